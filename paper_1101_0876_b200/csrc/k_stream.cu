// k_stream.cu -- instantiations of the streaming half-sweep kernel (U8 layout), see potts_kernels.cuh.
#include "potts_launch.cuh"

namespace potts {
namespace {

// grid = the blocks that are resident at once (the kernel draws its tiles from a counter), at most one per tile
template <int CM, int ST, bool MEASURE, bool HIST, bool DELTA>
void launch_hs(const SweepParams &P, int num_sms, size_t smem, cudaStream_t st)
{
    static size_t cached_smem = ~(size_t)0;
    static int per_sm = 1;
    if (cached_smem != smem) {
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_sweep_rows_u8<CM, ST, MEASURE, HIST, DELTA>, 32 * HS_WARPS, smem);
        if (per_sm < 1) per_sm = 1;
        cached_smem = smem;
    }
    const unsigned long long want = (unsigned long long)per_sm * (unsigned)num_sms;
    const unsigned grid = (unsigned)(want < P.total_tiles ? want : P.total_tiles);
    k_sweep_rows_u8<CM, ST, MEASURE, HIST, DELTA><<<grid, dim3(32, HS_WARPS), smem, st>>>(P);
}

template <int CM, int ST>
void launch_hs_st(const SweepParams &P, bool delta, int num_sms, size_t smem, cudaStream_t st)
{
    if (delta) { launch_hs<CM, ST, false, false, true>(P, num_sms, smem, st); return; }
    const int sel = (P.E_out ? 2 : 0) | (P.hist_out ? 1 : 0);
    switch (sel) {
    case 0: launch_hs<CM, ST, false, false, false>(P, num_sms, smem, st); break;
    case 1: launch_hs<CM, ST, false, true, false>(P, num_sms, smem, st); break;
    case 2: launch_hs<CM, ST, true, false, false>(P, num_sms, smem, st); break;
    default: launch_hs<CM, ST, true, true, false>(P, num_sms, smem, st); break;
    }
}

template <int CM>
void launch_hs_cm(int stream_spec, const SweepParams &P, bool delta, int num_sms, size_t smem, cudaStream_t st)
{
    if (stream_spec == 2) launch_hs_st<CM, 2>(P, delta, num_sms, smem, st);
    else launch_hs_st<CM, 1>(P, delta, num_sms, smem, st);
}

}  // namespace

void launch_sweep_rows_u8(int cm, int stream_spec, bool delta, const SweepParams &P, int num_sms, size_t smem, cudaStream_t st)
{
    switch (cm) {
    case CM_7BIT: launch_hs_cm<CM_7BIT>(stream_spec, P, delta, num_sms, smem, st); break;
    case CM_8BIT: launch_hs_cm<CM_8BIT>(stream_spec, P, delta, num_sms, smem, st); break;
    case CM_NIB4: launch_hs_cm<CM_NIB4>(stream_spec, P, delta, num_sms, smem, st); break;
    default: launch_hs_cm<CM_NIB3>(stream_spec, P, delta, num_sms, smem, st); break;
    }
}

}  // namespace potts
