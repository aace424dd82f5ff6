// potts_resident.cuh -- persistent multi-sweep kernel: the lattice lives in shared memory.
//
// For lattices that fit the shared memory of the GPU (2 planes x L x L/2 bytes spread over up to 148
// SMs: L <= ~4096) one cooperative launch runs ALL sweeps of a potts_sweep call.  CTA b owns the rows
// [r0, r1) of both colour planes in its shared memory.  A half-sweep of colour c reads only the other
// plane (sec. 3), so the only data that crosses CTAs are the two boundary rows of the
// plane just written; they go through the global planes (L2) and a per-CTA counter:
//
//   half-sweep hs (absolute index 2 t + c):
//     W  wait until both neighbour CTAs have published half-sweep hs-1      (skipped for the first)
//     H  copy their boundary rows of plane 1-c (global, L2) into the halo rows of shared memory
//     B  update the CTA's first and last row, store them to shared AND global memory
//     P  __syncthreads; one thread: fence, flags[b] = hs+1 (release)
//     I  update the interior rows (hides the latency of P -> neighbour's W)
//
// A neighbour overwrites a boundary row in global memory (its step B of hs+1) only after it has seen
// flags[b] = hs+1, which CTA b sets after its step H of hs has consumed the previous version, so one
// buffer per row is enough.  All rows are also written through to the global planes, so the global
// state is complete when the kernel ends and every other entry point keeps working unchanged.
// Energy and histogram of a sampled sweep are fused: per-thread sums, one block reduction, one
// atomicAdd per CTA into the series slot (sec. 3.4).
//
// The random stream is a pure function of (seed, t, colour, i, j), so the result does not depend on
// the number of CTAs or the row split; tests check that bit for bit.
#pragma once
#include "potts_core.cuh"

namespace potts {

struct ResidentParams {
    uint8_t *plane[2];
    int32_t L, pitch;                 // pitch = L/2 bytes per plane row
    uint32_t q;
    uint32_t key0, key1;
    uint32_t thr[4];
    uint32_t t0;                      // sweep counter of the first sweep
    uint32_t nsweeps;
    uint32_t every;                   // sample after every `every`-th sweep of this launch; 0 = never
    unsigned long long *E_series;     // device, nsweeps/every entries, may be null
    unsigned long long *hist_series;  // device, nsweeps/every rows of q, may be null
    unsigned long long *flags;        // [gridDim.x] published half-sweeps, absolute (2 t + c + 1)
    int *error;                       // set to 1 if a neighbour wait gave up
    int32_t rows_max;                 // rows of shared memory per plane = rows_max + 2
};

constexpr long long RESIDENT_SPIN_LIMIT = 1ll << 24;   // polls before a wait gives up (seconds)

__device__ __forceinline__ unsigned long long ld_acquire_u64(const unsigned long long *p)
{
    unsigned long long v;
    asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}

__device__ __forceinline__ void st_release_u64(unsigned long long *p, unsigned long long v)
{
    asm volatile("st.release.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}

__device__ __forceinline__ uint4 ld_cg_u4(const void *p)   // L2 only: never a stale L1 line
{
    return __ldcg(reinterpret_cast<const uint4 *>(p));
}

// Block = (wpr_threads = L/8 words per plane row, ty rows); thread (tx, ty) owns word tx of the row
// slots ty, ty + blockDim.y, ...  Slot 0 is the CTA's first row, slot 1 its last row, slots 2.. the
// interior rows, so the boundary rows are finished (and published) first.
template <bool WIDE>
__global__ void __launch_bounds__(1024, 1) k_resident_u8(const __grid_constant__ ResidentParams P)
{
    extern __shared__ __align__(16) uint8_t s_raw[];
    __shared__ uint32_t lut[12];
    __shared__ unsigned long long blockE;
    __shared__ HalfSweepKeys s_keys[2];                             // double-buffered by colour

    const uint32_t G = gridDim.x, b = blockIdx.x;
    const int L = P.L, pitch = P.pitch;
    const int r0 = (int)(((long long)b * L) / G), r1 = (int)(((long long)(b + 1) * L) / G);
    const int rows = r1 - r0;
    const uint32_t up_cta = (b + G - 1) % G, dn_cta = (b + 1) % G;
    const int srows = P.rows_max + 2;                               // local row 0 / rows+1 = halos
    const size_t plane_stride = (size_t)srows * pitch;
    uint32_t *s_hist = reinterpret_cast<uint32_t *>(s_raw + 2 * (size_t)srows * pitch);

    const uint32_t tx = threadIdx.x, ty = threadIdx.y;
    const uint32_t nthreads = blockDim.x * blockDim.y, tid = ty * blockDim.x + tx;
    const int wpr = pitch >> 2;
    const bool do_hist = P.hist_series != nullptr && P.every != 0;
    const bool do_E = P.E_series != nullptr && P.every != 0;

    if (tid < 9) lut[tid] = tid >= 5 ? P.thr[tid - 5] : 0u;
    if (tid == 0) blockE = 0ull;
    if (do_hist)
        for (uint32_t n = tid; n < hist_words(P.q); n += nthreads) s_hist[n] = 0u;
    // own rows of both planes: global -> shared (local row = global row - r0 + 1)
    {
        const int vpr = pitch >> 4;                                 // uint4 per row
        for (int c = 0; c < 2; ++c)
            for (int n = (int)tid; n < rows * vpr; n += (int)nthreads) {
                const int lr = n / vpr, v = n - lr * vpr;
                *reinterpret_cast<uint4 *>(s_raw + c * plane_stride + (size_t)(lr + 1) * pitch + 16 * v) =
                    ld_cg_u4(P.plane[c] + (size_t)(r0 + lr) * pitch + 16 * v);
            }
    }
    __syncthreads();

    const int nslots = rows;
    const int iters = (nslots + (int)blockDim.y - 1) / (int)blockDim.y;
    const int kb = ((rows < 2 ? rows : 2) - 1) / (int)blockDim.y;   // iteration that completes the boundary rows
    const int kl = (int)tx == 0 ? wpr - 1 : (int)tx - 1, kr = (int)tx + 1 == wpr ? 0 : (int)tx + 1;

    uint32_t until = P.every;                                       // sweeps until the next sample
    uint32_t sample_idx = 0;
    for (uint32_t n = 0; n < P.nsweeps; ++n) {
        const uint32_t t = P.t0 + n;
        const bool sample = P.every != 0 && --until == 0;
        if (sample) until = P.every;
        for (uint32_t c = 0; c < 2; ++c) {
            const unsigned long long hs = 2ull * t + c;
            uint8_t *own_p = s_raw + c * plane_stride;
            uint8_t *oth_p = s_raw + (1 - c) * plane_stride;
            if (tid == 0) s_keys[c] = half_sweep_keys(P.key0, P.key1, t, c);   // visible after the barrier below
            // ---- W: neighbours have published half-sweep hs-1
            if (n != 0 || c != 0) {
                if (tid < 2) {
                    const unsigned long long *f = P.flags + (tid == 0 ? up_cta : dn_cta);
                    long long spins = 0;
                    while (ld_acquire_u64(f) < hs)
                        if (++spins > RESIDENT_SPIN_LIMIT) { atomicExch(P.error, 1); break; }
                }
                __syncthreads();
            }
            // ---- H: halo rows of the other plane
            {
                const int vpr = pitch >> 4;
                const uint8_t *g = P.plane[1 - c];
                const int gu = wrap(r0 - 1, L), gd = wrap(r1, L);
                for (int v = (int)tid; v < 2 * vpr; v += (int)nthreads) {
                    const bool lower = v >= vpr;
                    const int vv = lower ? v - vpr : v;
                    *reinterpret_cast<uint4 *>(oth_p + (size_t)(lower ? rows + 1 : 0) * pitch + 16 * vv) =
                        ld_cg_u4(g + (size_t)(lower ? gd : gu) * pitch + 16 * vv);
                }
            }
            __syncthreads();

            const HalfSweepKeys K = s_keys[c];
            const uint32_t q = in_register(P.q);
            uint32_t nef_sum = 0, words_done = 0;
            for (int k = 0; k < iters; ++k) {
                const int slot = (int)ty + k * (int)blockDim.y;
                if (slot < nslots) {
                    const int lr = slot == 0 ? 1 : (slot == 1 ? rows : slot);        // local row 1..rows
                    const int i = r0 + lr - 1;
                    const uint32_t p = (uint32_t)(i + c) & 1u;
                    const uint32_t *own_row = reinterpret_cast<const uint32_t *>(own_p + (size_t)lr * pitch);
                    const uint32_t *mid_row = reinterpret_cast<const uint32_t *>(oth_p + (size_t)lr * pitch);
                    const uint32_t own = own_row[tx];
                    const uint32_t up = reinterpret_cast<const uint32_t *>(oth_p + (size_t)(lr - 1) * pitch)[tx];
                    const uint32_t dn = reinterpret_cast<const uint32_t *>(oth_p + (size_t)(lr + 1) * pitch)[tx];
                    const uint32_t mid = mid_row[tx];
                    const uint32_t adj = mid_row[p ? kr : kl];
                    uint32_t lf, rt, nef;
                    horizontal(p, mid, adj, lf, rt);
                    const RowKeys R = row_keys(K, (uint32_t)i);
                    const uint32_t out = update_word<WIDE>(own, up, dn, lf, rt, 8u * tx + p, q, K, R, lut, nef);
                    reinterpret_cast<uint32_t *>(own_p + (size_t)lr * pitch)[tx] = out;
                    reinterpret_cast<uint32_t *>(P.plane[c] + (size_t)i * pitch)[tx] = out;
                    if (sample) {
                        if (c == 1 && do_E) { nef_sum += nef; ++words_done; }
                        if (do_hist) hist_add_word(s_hist, P.q, out, tid & 31u);
                    }
                }
                if (k == kb) {
                    // ---- P: boundary rows are in global memory; publish half-sweep hs
                    __syncthreads();
                    if (tid == 0) {
                        __threadfence();
                        st_release_u64(P.flags + b, hs + 1ull);
                    }
                }
            }
            __syncthreads();                                        // own plane complete in shared memory

            if (sample && c == 1) {
                if (do_E) {
                    // satisfied bonds seen from this thread's black sites = 4 per site - unequal neighbours
                    // (nef_sum holds 4 byte counters, +<= 4 per word: the host keeps iters <= 60)
                    uint32_t satisfied = 16u * words_done - byte_sum(nef_sum);
#pragma unroll
                    for (int o = 16; o > 0; o >>= 1) satisfied += __shfl_xor_sync(0xffffffffu, satisfied, o);
                    if ((tid & 31u) == 0) atomicAdd(&blockE, (unsigned long long)satisfied);
                    __syncthreads();
                    if (tid == 0) {
                        atomicAdd(P.E_series + sample_idx, 0ull - blockE);
                        blockE = 0ull;
                    }
                }
                if (do_hist) hist_flush(s_hist, P.q, P.hist_series + (size_t)sample_idx * P.q, tid, nthreads);
                ++sample_idx;
                __syncthreads();
            }
        }
    }
}

}  // namespace potts
