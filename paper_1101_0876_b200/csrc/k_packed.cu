// k_packed.cu -- instantiations of the streaming half-sweep kernel on the sub-byte packed layout, see potts_packed.cuh.
#include "potts_launch.cuh"

namespace potts {
namespace {

constexpr size_t PK_COL_BYTES = 2 * PK_SITES * 32 * sizeof(uint4);      // ColKeys table; the histogram table follows it

template <bool FIVE, int ST, bool MEASURE, bool HIST, bool DELTA>
void launch_pk_one(const PackedSweepParams &P, int num_sms, size_t smem, cudaStream_t st)
{
    auto fn = k_sweep_rows_packed<FIVE, ST, MEASURE, HIST, DELTA>;
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

template <bool FIVE, int ST>
void launch_pk_st(bool delta, const PackedSweepParams &P, int num_sms, size_t smem, cudaStream_t st)
{
    if (delta) { launch_pk_one<FIVE, ST, false, false, true>(P, num_sms, 0, st); return; }
    const int sel = (P.E_out ? 2 : 0) | (P.hist_out ? 1 : 0);
    switch (sel) {
    case 0: launch_pk_one<FIVE, ST, false, false, false>(P, num_sms, smem, st); break;
    case 1: launch_pk_one<FIVE, ST, false, true, false>(P, num_sms, smem, st); break;
    case 2: launch_pk_one<FIVE, ST, true, false, false>(P, num_sms, smem, st); break;
    default: launch_pk_one<FIVE, ST, true, true, false>(P, num_sms, smem, st); break;
    }
}

template <bool FIVE>
void launch_pk(int stream_spec, bool delta, const PackedSweepParams &P, int num_sms, size_t smem, cudaStream_t st)
{
    if (stream_spec == 2) launch_pk_st<FIVE, 2>(delta, P, num_sms, smem, st);
    else launch_pk_st<FIVE, 1>(delta, P, num_sms, smem, st);
}

}  // namespace

void launch_sweep_rows_packed(bool five, int stream_spec, bool delta, const PackedSweepParams &P, int num_sms, size_t smem, cudaStream_t st)
{
    if (five) launch_pk<true>(stream_spec, delta, P, num_sms, smem, st);
    else launch_pk<false>(stream_spec, delta, P, num_sms, smem, st);
}

}  // namespace potts
