// k_cluster.cu -- instantiations of the single-cluster (DSMEM) kernel, see potts_cluster.cuh.
#include "potts_launch.cuh"

namespace potts {
namespace {

template <int CM>
const void *cluster_kernel_cm(int stream_spec, int nthreads)
{
    if (nthreads <= 256) return stream_spec == 2 ? (const void *)k_cluster_u8<CM, 2, 256> : (const void *)k_cluster_u8<CM, 1, 256>;
    return stream_spec == 2 ? (const void *)k_cluster_u8<CM, 2, 1024> : (const void *)k_cluster_u8<CM, 1, 1024>;
}

}  // namespace

const void *cluster_kernel(int cm, int stream_spec, int nthreads)
{
    switch (cm) {
    case CM_7BIT: return cluster_kernel_cm<CM_7BIT>(stream_spec, nthreads);
    case CM_8BIT: return cluster_kernel_cm<CM_8BIT>(stream_spec, nthreads);
    case CM_NIB4: return cluster_kernel_cm<CM_NIB4>(stream_spec, nthreads);
    default: return cluster_kernel_cm<CM_NIB3>(stream_spec, nthreads);
    }
}

}  // namespace potts
