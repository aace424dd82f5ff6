// potts_cluster.cuh -- tiny lattices: one thread-block cluster, boundary rows through distributed shared memory.
//
// A lattice of L <= 256 is a few thousand words: the resident kernel's L2 packets (~1 us per half-sweep of flight and
// polling) cost more than the update itself.  Here the whole lattice lives in the shared memory of ONE cluster of up to 16
// CTAs (CTA b owns rows [bL/G, (b+1)L/G) of both planes, plus one halo row above and below per plane); the thread that
// updates a word of a boundary row also stores it straight into the neighbour CTA's halo row (DSMEM,
// cluster.map_shared_rank), and one hardware cluster barrier per half-sweep is the only synchronisation: no polling, no
// inbox, no comm warps.  A half-sweep of colour c writes plane c (own rows, and the neighbours' plane-c halo rows) and
// reads plane 1-c only, so the barrier at the end of the half-sweep is all the ordering there is to do.
// Same arithmetic (potts_core.cuh), same chain: tests compare it bit for bit with the other kernels and the oracle.
#pragma once
#include <cooperative_groups.h>

#include "potts_core.cuh"
#include "potts_resident.cuh"

namespace potts {

constexpr int CLUSTER_MAX = 16;     // 8 is the portable cluster size; B200 takes 16 with the non-portable attribute

// Block = wpr x tyc threads (wpr = L/8 words per plane row); thread (tx, ty) updates word tx of local rows
// 1+ty, 1+ty+tyc, ...  P.inbox and P.error are unused.
template <int CM, int ST>
__global__ void __launch_bounds__(1024, 1) k_cluster_u8(const __grid_constant__ ResidentParams P)
{
    namespace cg = cooperative_groups;
    cg::cluster_group cluster = cg::this_cluster();
    extern __shared__ __align__(16) uint8_t s_raw[];
    __shared__ AcceptLutWide lut;

    const uint32_t G = cluster.num_blocks(), b = cluster.block_rank();
    const int L = P.L, pitch = P.pitch;
    const int r0 = (int)(((long long)b * L) / G), r1 = (int)(((long long)(b + 1) * L) / G);
    const int rows = r1 - r0;
    const uint32_t up_cta = (b + G - 1) % G, dn_cta = (b + 1) % G;
    const int rows_up = (int)(((long long)(up_cta + 1) * L) / G) - (int)(((long long)up_cta * L) / G);
    const int srows = P.rows_max + 2;
    const uint32_t plane_stride = (uint32_t)srows * (uint32_t)pitch;
    // two histogram tables used by alternate samples: one is flushed (and zeroed) while the next sample already counts
    uint32_t *const s_hist0 = reinterpret_cast<uint32_t *>(s_raw + 2 * plane_stride);
    // the same shared-memory layout in every CTA of the cluster: my pointers, seen in the neighbours' address space
    uint8_t *const up_raw = cluster.map_shared_rank(s_raw, up_cta);
    uint8_t *const dn_raw = cluster.map_shared_rank(s_raw, dn_cta);

    const uint32_t tid = threadIdx.x, nthreads = blockDim.x;
    const int wpr = pitch >> 2, tyc = P.tyc;
    const bool is_compute = (int)tid < wpr * tyc;
    const int ty = is_compute ? (int)tid / wpr : 0;
    const uint32_t col = is_compute ? 4u * (uint32_t)((int)tid - ty * wpr) : 0u;
    const uint32_t col_prev = col == 0u ? (uint32_t)pitch - 4u : col - 4u;
    const uint32_t col_next = col + 4u == (uint32_t)pitch ? 0u : col + 4u;
    const bool do_hist = P.hist_series != nullptr && P.every != 0;
    const bool do_E = P.E_series != nullptr && P.every != 0;
    const bool do_D = P.dE_series != nullptr;
    const uint32_t q = in_register(P.q);

    accept_lut_fill(&lut, P.thr, tid, nthreads);
    const uint32_t lane_off = accept_lane_offset<AcceptLutWide::slots>(tid);
    if (do_hist)
        for (uint32_t n = tid; n < 2u * hist_words(P.q); n += nthreads) s_hist0[n] = 0u;
    {
        const int vpr = pitch >> 4;
        for (int c = 0; c < 2; ++c)
            for (int n = (int)tid; n < (rows + 2) * vpr; n += (int)nthreads) {
                const int lr = n / vpr, v = n - lr * vpr;
                const int gr = wrap(r0 + lr - 1, L);
                *reinterpret_cast<uint4 *>(s_raw + c * plane_stride + (uint32_t)(lr * pitch + 16 * v)) =
                    __ldcg(reinterpret_cast<const uint4 *>(P.plane[c] + (size_t)gr * pitch + 16 * v));
            }
    }
    cluster.sync();      // nobody writes a neighbour's halo before every CTA has loaded its start state

    const HalfSweepKeys K0 = half_sweep_keys(P.key0, P.key1, 0u, 0u);
    uint32_t until = P.every, sample_idx = 0;
    for (uint32_t n = 0; n < P.nsweeps; ++n) {
        const uint32_t t = P.t0 + n;
        const bool sample = P.every != 0 && --until == 0;
        if (sample) until = P.every;
#pragma unroll
        for (uint32_t c = 0; c < 2; ++c) {
            uint8_t *const own_col = s_raw + c * plane_stride + col;
            const uint8_t *const oth_row = s_raw + (1u - c) * plane_stride;
            HalfSweepKeys K = K0;
            half_sweep_rekey(K, P.key0, P.key1, t, c);
            const bool count_E = sample && c == 1 && do_E, count_H = sample && do_hist;
            int d_sum = 0, ne_sum = 0;
            uint32_t words_done = 0;
            uint32_t *const s_hist = s_hist0 + (sample_idx & 1u) * hist_words(P.q);
            if (is_compute)
                for (int lr = 1 + ty; lr <= rows; lr += tyc) {
                    const uint32_t ro = (uint32_t)(lr * pitch);
                    const uint32_t i = (uint32_t)(r0 + lr - 1);
                    const uint32_t p = (i + c) & 1u;
                    const uint8_t *const orow = oth_row + ro;
                    const uint32_t own = *reinterpret_cast<const uint32_t *>(own_col + ro);
                    const uint32_t mid = *reinterpret_cast<const uint32_t *>(orow + col);
                    const uint32_t up = *reinterpret_cast<const uint32_t *>(orow + col - pitch);
                    const uint32_t dn = *reinterpret_cast<const uint32_t *>(orow + col + pitch);
                    const uint32_t adj = *reinterpret_cast<const uint32_t *>(orow + (p ? col_next : col_prev));
                    uint32_t lf, rt;
                    horizontal(p, mid, adj, lf, rt);
                    const RowKeys R = row_keys(K, i);
                    uint32_t code, mask;
                    const uint32_t out = update_word<CM, ST, AcceptLutWide::slots>(own, up, dn, lf, rt, 2u * col + p, q, K, R, &lut, lane_off, code, mask);
                    if (count_E) ne_sum += ne_final_sum(code, mask);
                    if (do_D) d_sum += delta_sum(code, mask);
                    *reinterpret_cast<uint32_t *>(own_col + ro) = out;
                    // my first row is the row below the last row of the CTA above, my last row the row above the first of the CTA below
                    if (lr == 1)
                        *reinterpret_cast<uint32_t *>(up_raw + c * plane_stride + (uint32_t)((rows_up + 1) * pitch) + col) = out;
                    if (lr == rows) *reinterpret_cast<uint32_t *>(dn_raw + c * plane_stride + col) = out;
                    ++words_done;
                    if (count_H) hist_add_word(s_hist, P.q, out, tid & 31u);
                }
            if (do_D) {
                int dd = d_sum;
                dd = __reduce_add_sync(0xffffffffu, dd);                     // one REDUX instead of a five-step shuffle tree
                if ((tid & 31u) == 0 && dd) atomicAdd(P.dE_series + n, (unsigned long long)(long long)dd);
            }
            if (count_E) {
                uint32_t satisfied = 16u * words_done - (uint32_t)ne_sum;
                satisfied = __reduce_add_sync(0xffffffffu, satisfied);                     // one REDUX instead of a five-step shuffle tree
                if ((tid & 31u) == 0 && satisfied) atomicAdd(P.E_series + sample_idx, 0ull - (unsigned long long)satisfied);
            }
            cluster.sync();                                         // plane c and its halos complete everywhere
            if (sample && c == 1) {
                // no barrier after the flush: the next sample counts into the other table
                if (do_hist) hist_flush(s_hist, P.q, P.hist_series + (size_t)sample_idx * P.q, tid, nthreads);
                ++sample_idx;
            }
        }
    }
    {
        const int vpr = pitch >> 4;
        for (int c = 0; c < 2; ++c)
            for (int n = (int)tid; n < rows * vpr; n += (int)nthreads) {
                const int lr = n / vpr, v = n - lr * vpr;
                *reinterpret_cast<uint4 *>(P.plane[c] + (size_t)(r0 + lr) * pitch + 16 * v) =
                    *reinterpret_cast<const uint4 *>(s_raw + c * plane_stride + (uint32_t)((lr + 1) * pitch + 16 * v));
            }
    }
    cluster.sync();      // no CTA exits while a neighbour may still write into its shared memory
}

}  // namespace potts
