// k_stream.inl -- instantiations of k_sweep_rows_u8 for one (stream definition, colour) pair; included by
// k_stream_s{1,2}c{0,1}.cu with POTTS_ST and POTTS_COLOUR defined, so that the four sets compile in parallel.
#include "potts_launch.cuh"

namespace potts {
namespace {

// grid = the blocks that are resident at once (the kernel draws its tiles from a counter), at most one per tile
template <int CM, bool MEASURE, bool HIST, bool DELTA, bool FAST>
void launch_hs(const SweepParams &P, int num_sms, size_t smem, cudaStream_t st)
{
    auto fn = k_sweep_rows_u8<CM, POTTS_ST, POTTS_COLOUR, MEASURE, HIST, DELTA, FAST>;
    static size_t cached_smem = ~(size_t)0;
    static int per_sm = 1;
    if (cached_smem != smem) {
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, fn, 32 * HS_WARPS, smem);
        if (per_sm < 1) per_sm = 1;
        cached_smem = smem;
    }
    const unsigned long long want = (unsigned long long)per_sm * (unsigned)num_sms;
    const unsigned grid = (unsigned)(want < P.total_tiles ? want : P.total_tiles);
    fn<<<grid, dim3(32, HS_WARPS), smem, st>>>(P);
}

// the staged form of the plain half-sweep (experiment, option stream_stage): dynamic shared memory = the warps' stages
template <int CM, bool FAST>
void launch_hs_bulk(const SweepParams &P, int num_sms, cudaStream_t st)
{
    auto fn = k_sweep_rows_u8<CM, POTTS_ST, POTTS_COLOUR, false, false, false, FAST, true>;
    const size_t smem = (size_t)HS_WARPS * (size_t)(P.rpw + 2) * BULK_ROW;
    static size_t cached_smem = ~(size_t)0;
    static int per_sm = 1;
    if (cached_smem != smem) {
        cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, 160 << 10);
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, fn, 32 * HS_WARPS, smem);
        if (per_sm < 1) per_sm = 1;
        cached_smem = smem;
    }
    const unsigned long long want = (unsigned long long)per_sm * (unsigned)num_sms;
    const unsigned grid = (unsigned)(want < P.total_tiles ? want : P.total_tiles);
    fn<<<grid, dim3(32, HS_WARPS), smem, st>>>(P);
}

template <int CM>
void launch_hs_cm(const SweepParams &P, bool delta, int num_sms, size_t smem, cudaStream_t st)
{
    if (P.bulk && !delta && !P.E_out && !P.hist_out) {
        if (accept_fast_ok(P.thr)) launch_hs_bulk<CM, true>(P, num_sms, st);
        else launch_hs_bulk<CM, false>(P, num_sms, st);
        return;
    }
    if (delta) { launch_hs<CM, false, false, true, false>(P, num_sms, smem, st); return; }
    const bool fast = accept_fast_ok(P.thr);          // no "never accept" entry: the one-compare form is exact
    if (P.E_out) {
#if POTTS_COLOUR == 1                                 // the energy is counted from the black sites only
        if (P.hist_out) launch_hs<CM, true, true, false, false>(P, num_sms, smem, st);
        else launch_hs<CM, true, false, false, false>(P, num_sms, smem, st);
#endif
        return;
    }
    if (P.hist_out) {
        if (fast) launch_hs<CM, false, true, false, true>(P, num_sms, smem, st);
        else launch_hs<CM, false, true, false, false>(P, num_sms, smem, st);
    } else {
        if (fast) launch_hs<CM, false, false, false, true>(P, num_sms, smem, st);
        else launch_hs<CM, false, false, false, false>(P, num_sms, smem, st);
    }
}

}  // namespace

#define POTTS_CAT2(a, b, c, d) a##b##c##d
#define POTTS_CAT(a, b, c, d) POTTS_CAT2(a, b, c, d)
void POTTS_CAT(launch_sweep_rows_u8_s, POTTS_ST, c, POTTS_COLOUR)(int cm, bool delta, const SweepParams &P, int num_sms, size_t smem, cudaStream_t st)
{
    switch (cm) {
    case CM_7BIT: launch_hs_cm<CM_7BIT>(P, delta, num_sms, smem, st); break;
    case CM_8BIT: launch_hs_cm<CM_8BIT>(P, delta, num_sms, smem, st); break;
    case CM_NIB4: launch_hs_cm<CM_NIB4>(P, delta, num_sms, smem, st); break;
    default: launch_hs_cm<CM_NIB3>(P, delta, num_sms, smem, st); break;
    }
}

}  // namespace potts
