// k_packed.cu -- instantiations of the streaming half-sweep kernel on the sub-byte packed layout, see potts_packed.cuh.
#include "potts_launch.cuh"

namespace potts {
namespace {

template <bool FIVE, int ST>
void launch_pk_st(bool delta, const PackedSweepParams &P, dim3 grid, size_t smem, cudaStream_t st)
{
    const dim3 block(32, PK_WARPS);
    if (delta) { k_half_sweep_packed<FIVE, ST, false, false, true><<<grid, block, 0, st>>>(P); return; }
    const int sel = (P.E_out ? 2 : 0) | (P.hist_out ? 1 : 0);
    switch (sel) {
    case 0: k_half_sweep_packed<FIVE, ST, false, false><<<grid, block, smem, st>>>(P); break;
    case 1: k_half_sweep_packed<FIVE, ST, false, true><<<grid, block, smem, st>>>(P); break;
    case 2: k_half_sweep_packed<FIVE, ST, true, false><<<grid, block, smem, st>>>(P); break;
    default: k_half_sweep_packed<FIVE, ST, true, true><<<grid, block, smem, st>>>(P); break;
    }
}

template <bool FIVE>
void launch_pk(int stream_spec, bool delta, const PackedSweepParams &P, dim3 grid, size_t smem, cudaStream_t st)
{
    if (stream_spec == 2) launch_pk_st<FIVE, 2>(delta, P, grid, smem, st);
    else launch_pk_st<FIVE, 1>(delta, P, grid, smem, st);
}

}  // namespace

void launch_sweep_rows_packed(bool five, int stream_spec, bool delta, const PackedSweepParams &P, dim3 grid, size_t smem, cudaStream_t st)
{
    if (five) launch_pk<true>(stream_spec, delta, P, grid, smem, st);
    else launch_pk<false>(stream_spec, delta, P, grid, smem, st);
}

}  // namespace potts
