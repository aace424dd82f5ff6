// potts_launch.cuh -- the template dispatch of the heavy kernels, one translation unit per kernel family so
// that the library builds in parallel (build.py).  potts_api.cu calls these; nothing else does.
#pragma once
#include "potts_kernels.cuh"
#include "potts_resident.cuh"
#include "potts_packed.cuh"
#include "potts_cluster.cuh"

namespace potts {

// k_stream.cu: k_sweep_rows_u8<CM, ST, MEASURE, HIST, DELTA>; MEASURE / HIST follow P.E_out / P.hist_out,
// delta = true selects the energy-change form (P.E_out receives the change, P.hist_out must be null)
void launch_sweep_rows_u8(int cm, int stream_spec, bool delta, const SweepParams &P, int num_sms, size_t smem, cudaStream_t st);

// k_packed.cu: k_sweep_rows_packed<FIVE, ST, MEASURE, HIST, DELTA>, same conventions
void launch_sweep_rows_packed(bool five, int stream_spec, bool delta, const PackedSweepParams &P, int num_sms, size_t smem, cudaStream_t st);

// k_resident.cu: the persistent kernel (small: 2 = blocks up to 576 threads, 1 = up to 768, 0 = up to 1024) and the batch launch
const void *resident_kernel(int cm, int stream_spec, int W, int small);
cudaError_t launch_batch(int cm, int stream_spec, const BatchParams &B, const BatchTable &T, int n, int nthreads, size_t smem, cudaStream_t st);

// k_cluster.cu
const void *cluster_kernel(int cm, int stream_spec, int nthreads);   // nthreads: block size (register budget)

}  // namespace potts
