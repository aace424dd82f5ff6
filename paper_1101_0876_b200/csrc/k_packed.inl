// k_packed.inl -- instantiations of k_sweep_rows_packed for one stream definition; included by k_packed_s{1,2}.cu
// with POTTS_ST defined.
#include "potts_launch.cuh"

namespace potts {
namespace {

constexpr size_t PK_COL_BYTES = 2 * PK_SITES * 32 * sizeof(uint4);      // ColKeys table; the histogram table follows it

template <bool FIVE, int COLOUR, bool MEASURE, bool HIST, bool DELTA, bool FAST>
void launch_pk_one(const PackedSweepParams &P, int num_sms, size_t smem, cudaStream_t st)
{
    auto fn = k_sweep_rows_packed<FIVE, POTTS_ST, COLOUR, MEASURE, HIST, DELTA, FAST>;
    smem += PK_COL_BYTES;
    static size_t cached_smem = ~(size_t)0;
    static int per_sm = 1;
    if (cached_smem != smem) {
        cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, 96 << 10);   // static + dynamic exceed the 48 KB default
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, fn, 32 * PK_WARPS, smem);
        if (per_sm < 1) per_sm = 1;
        cached_smem = smem;
    }
    const unsigned long long want = (unsigned long long)per_sm * (unsigned)num_sms;
    const unsigned grid = (unsigned)(want < P.total_tiles ? want : P.total_tiles);
    fn<<<grid, dim3(32, PK_WARPS), smem, st>>>(P);
}

template <bool FIVE, int COLOUR>
void launch_pk_c(bool delta, const PackedSweepParams &P, int num_sms, size_t smem, cudaStream_t st)
{
    if (delta) { launch_pk_one<FIVE, COLOUR, false, false, true, false>(P, num_sms, 0, st); return; }
    const bool fast = accept_fast_ok(P.thr);
    if (P.E_out) {
        if constexpr (COLOUR == 1) {                  // the energy is counted from the black sites only
            if (P.hist_out) launch_pk_one<FIVE, 1, true, true, false, false>(P, num_sms, smem, st);
            else launch_pk_one<FIVE, 1, true, false, false, false>(P, num_sms, smem, st);
        }
        return;
    }
    if (P.hist_out) {
        if (fast) launch_pk_one<FIVE, COLOUR, false, true, false, true>(P, num_sms, smem, st);
        else launch_pk_one<FIVE, COLOUR, false, true, false, false>(P, num_sms, smem, st);
    } else {
        if (fast) launch_pk_one<FIVE, COLOUR, false, false, false, true>(P, num_sms, smem, st);
        else launch_pk_one<FIVE, COLOUR, false, false, false, false>(P, num_sms, smem, st);
    }
}

}  // namespace

#define POTTS_CAT2(a, b) a##b
#define POTTS_CAT(a, b) POTTS_CAT2(a, b)
void POTTS_CAT(launch_sweep_rows_packed_s, POTTS_ST)(bool five, bool delta, const PackedSweepParams &P, int num_sms, size_t smem, cudaStream_t st)
{
    if (five) {
        if (P.colour) launch_pk_c<true, 1>(delta, P, num_sms, smem, st);
        else launch_pk_c<true, 0>(delta, P, num_sms, smem, st);
    } else {
        if (P.colour) launch_pk_c<false, 1>(delta, P, num_sms, smem, st);
        else launch_pk_c<false, 0>(delta, P, num_sms, smem, st);
    }
}

}  // namespace potts
