// k_resident.cu -- instantiations of the persistent shared-memory kernel and of the replica-batch kernel,
// see potts_resident.cuh.
#include "potts_launch.cuh"

namespace potts {
namespace {

// register budget: 112 per thread for blocks up to 576 threads, 80 up to 768, else 64
template <int CM, int ST>
const void *resident_kernel_st(int W, int small)
{
    if (W == 3)          // W = 2 with the ColKeys table (potts_resident.cuh, COL)
        return small == 2 ? (const void *)k_resident_u8<CM, 2, ST, 576, true>
                          : (small == 1 ? (const void *)k_resident_u8<CM, 2, ST, 768, true> : (const void *)k_resident_u8<CM, 2, ST, 1024, true>);
    if (W == 1) return small == 2 ? (const void *)k_resident_u8<CM, 1, ST, 576> : (const void *)k_resident_u8<CM, 1, ST, 1024>;
    return small == 2 ? (const void *)k_resident_u8<CM, 2, ST, 576>
                      : (small == 1 ? (const void *)k_resident_u8<CM, 2, ST, 768> : (const void *)k_resident_u8<CM, 2, ST, 1024>);
}

template <int CM>
const void *resident_kernel_cm(int stream_spec, int W, int small)
{
    return stream_spec == 2 ? resident_kernel_st<CM, 2>(W, small) : resident_kernel_st<CM, 1>(W, small);
}

template <int CM, int ST, int MAXT>
cudaError_t launch_batch_fn(const BatchParams &B, const BatchTable &T, int n, int nthreads, size_t smem, cudaStream_t st)
{
    auto fn = k_resident_batch_u8<CM, ST, MAXT>;
    cudaError_t e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    fn<<<(unsigned)n, (unsigned)nthreads, smem, st>>>(B, T);
    return cudaGetLastError();
}

template <int CM, int ST>
cudaError_t launch_batch_st(const BatchParams &B, const BatchTable &T, int n, int nthreads, size_t smem, cudaStream_t st)
{
    // register budget by block size: up to 256 threads several blocks per SM, up to 512 threads 128 registers, else 64
    if (nthreads <= 256) return launch_batch_fn<CM, ST, 256>(B, T, n, nthreads, smem, st);
    return nthreads <= 512 ? launch_batch_fn<CM, ST, 512>(B, T, n, nthreads, smem, st) : launch_batch_fn<CM, ST, 1024>(B, T, n, nthreads, smem, st);
}

template <int CM>
cudaError_t launch_batch_cm(int stream_spec, const BatchParams &B, const BatchTable &T, int n, int nthreads, size_t smem, cudaStream_t st)
{
    return stream_spec == 2 ? launch_batch_st<CM, 2>(B, T, n, nthreads, smem, st) : launch_batch_st<CM, 1>(B, T, n, nthreads, smem, st);
}

}  // namespace

const void *resident_kernel(int cm, int stream_spec, int W, int small)
{
    switch (cm) {
    case CM_7BIT: return resident_kernel_cm<CM_7BIT>(stream_spec, W, small);
    case CM_8BIT: return resident_kernel_cm<CM_8BIT>(stream_spec, W, small);
    case CM_NIB4: return resident_kernel_cm<CM_NIB4>(stream_spec, W, small);
    default: return resident_kernel_cm<CM_NIB3>(stream_spec, W, small);
    }
}

cudaError_t launch_batch(int cm, int stream_spec, const BatchParams &B, const BatchTable &T, int n, int nthreads, size_t smem, cudaStream_t st)
{
    switch (cm) {
    case CM_7BIT: return launch_batch_cm<CM_7BIT>(stream_spec, B, T, n, nthreads, smem, st);
    case CM_8BIT: return launch_batch_cm<CM_8BIT>(stream_spec, B, T, n, nthreads, smem, st);
    case CM_NIB4: return launch_batch_cm<CM_NIB4>(stream_spec, B, T, n, nthreads, smem, st);
    default: return launch_batch_cm<CM_NIB3>(stream_spec, B, T, n, nthreads, smem, st);
    }
}

}  // namespace potts
