// k_packed.cu -- dispatch of the streaming half-sweep kernel on the sub-byte packed layout; see k_packed.inl.
#include "potts_launch.cuh"

namespace potts {

void launch_sweep_rows_packed_s1(bool five, bool delta, const PackedSweepParams &P, int num_sms, size_t smem, cudaStream_t st);
void launch_sweep_rows_packed_s2(bool five, bool delta, const PackedSweepParams &P, int num_sms, size_t smem, cudaStream_t st);

void launch_sweep_rows_packed(bool five, int stream_spec, bool delta, const PackedSweepParams &P, int num_sms, size_t smem, cudaStream_t st)
{
    if (stream_spec == 2) launch_sweep_rows_packed_s2(five, delta, P, num_sms, smem, st);
    else launch_sweep_rows_packed_s1(five, delta, P, num_sms, smem, st);
}

}  // namespace potts
