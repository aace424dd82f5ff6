// k_stream.cu -- dispatch of the streaming half-sweep kernel (U8 layout) to the translation unit that holds its
// (stream definition, colour) instantiations; see k_stream.inl and potts_kernels.cuh.
#include "potts_launch.cuh"

namespace potts {

void launch_sweep_rows_u8_s1c0(int cm, bool delta, const SweepParams &P, int num_sms, size_t smem, cudaStream_t st);
void launch_sweep_rows_u8_s1c1(int cm, bool delta, const SweepParams &P, int num_sms, size_t smem, cudaStream_t st);
void launch_sweep_rows_u8_s2c0(int cm, bool delta, const SweepParams &P, int num_sms, size_t smem, cudaStream_t st);
void launch_sweep_rows_u8_s2c1(int cm, bool delta, const SweepParams &P, int num_sms, size_t smem, cudaStream_t st);

void launch_sweep_rows_u8(int cm, int stream_spec, bool delta, const SweepParams &P, int num_sms, size_t smem, cudaStream_t st)
{
    if (stream_spec == 2) {
        if (P.colour) launch_sweep_rows_u8_s2c1(cm, delta, P, num_sms, smem, st);
        else launch_sweep_rows_u8_s2c0(cm, delta, P, num_sms, smem, st);
    } else {
        if (P.colour) launch_sweep_rows_u8_s1c1(cm, delta, P, num_sms, smem, st);
        else launch_sweep_rows_u8_s1c0(cm, delta, P, num_sms, smem, st);
    }
}

}  // namespace potts
