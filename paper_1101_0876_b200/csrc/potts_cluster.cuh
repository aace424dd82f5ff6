// potts_cluster.cuh -- tiny lattices: one thread-block cluster, boundary rows through distributed shared memory.
//
// A lattice of L <= 256 is a few thousand words: the resident kernel's L2 packets (~1 us per half-sweep of flight and
// polling) cost more than the update itself.  Here the whole lattice lives in the shared memory of ONE cluster of up to 16
// CTAs (CTA b owns rows [bL/G, (b+1)L/G) of both planes, plus one halo row above and below per plane); the thread that
// updates a word of a boundary row also sends it straight into the neighbour CTA's halo row through distributed shared
// memory with `st.async ... mbarrier::complete_tx::bytes`: the store carries its own completion signal to an mbarrier in
// the RECEIVER's shared memory, which counts the bytes of the row.  So there is no cluster-wide barrier in the loop and no
// memory fence (a `barrier.cluster.arrive.release` is a MEMBAR.ALL.GPU plus ~380 cycles of barrier, and the fence waits
// for every global atomic of the measurement to be acknowledged by L2): a CTA synchronises only with its two neighbours,
// only its two boundary rows wait (the first row for the halo above, the last for the halo below), and the rest of the
// block is ordered by one __syncthreads per half-sweep.  A half-sweep of colour c writes plane c (own rows, and the
// neighbours' plane-c halo rows) and reads plane 1-c only.
//
// mbarrier protocol.  s_mbar[c][side] guards my halo row of plane c on that side (0: above my first row, written by the
// last row of the CTA above; 1: below my last row, written by the first row of the CTA below); one phase per sweep, armed
// by thread 0 with the row's byte count (arrive.expect_tx, pending count 1), completed by the neighbour's L/2 bytes.
//   * read after write: my boundary-row threads wait for the phase of the half-sweep before (acquire, cluster scope).
//   * write after read: the neighbour overwrites that halo two half-sweeps later, and only after it has received my
//     boundary row of the half-sweep in between, whose bytes are complete only when every thread of that row has read
//     the halo and sent its word.
//   * a phase is re-armed by thread 0 after the __syncthreads that ends the half-sweep which consumed it; bytes of the
//     next phase that arrive before the arming just drive the byte count negative for a while, which the mbarrier allows.
// Same arithmetic (potts_core.cuh), same chain: tests compare it bit for bit with the other kernels and the oracle.
#pragma once
#include <cooperative_groups.h>

#include "potts_core.cuh"
#include "potts_resident.cuh"

namespace potts {

// the shared::cluster address of my shared-memory address `a` in CTA `rank` of the cluster
__device__ __forceinline__ uint32_t map_to_cta(uint32_t a, uint32_t rank)
{
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(a), "r"(rank));
    return r;
}

__device__ __forceinline__ void mbar_init(uint32_t mbar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(mbar), "r"(count) : "memory");
}

__device__ __forceinline__ void mbar_arm(uint32_t mbar, uint32_t tx_bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(mbar), "r"(tx_bytes) : "memory");
}

// one 4-byte word into a neighbour's shared memory; its arrival takes 4 bytes off the neighbour's mbarrier
__device__ __forceinline__ void st_async_word(uint32_t remote_addr, uint32_t value, uint32_t remote_mbar)
{
    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.b32 [%0], %1, [%2];" ::"r"(remote_addr), "r"(value), "r"(remote_mbar) : "memory");
}

// true once the phase of parity `parity` is complete (the data of its st.async stores is visible after it)
__device__ __forceinline__ bool mbar_try_wait(uint32_t mbar, uint32_t parity)
{
    uint32_t done;
    asm volatile("{\n.reg .pred p;\nmbarrier.try_wait.parity.acquire.cluster.shared::cta.b64 p, [%1], %2;\nselp.u32 %0, 1, 0, p;\n}"
                 : "=r"(done) : "r"(mbar), "r"(parity) : "memory");
    return done != 0u;
}

constexpr long long CLUSTER_SPIN_LIMIT = 1ll << 22;   // try_wait calls (each suspends for a while) before a wait gives up

constexpr int CLUSTER_MAX = 16;     // 8 is the portable cluster size; B200 takes 16 with the non-portable attribute

// Block = wpr x tyc threads (wpr = L/8 words per plane row); thread (tx, ty) updates word tx of local rows
// 1+ty, 1+ty+tyc, ...  P.inbox is unused; P.error is set if a wait for a neighbour gives up.
// MAXT: the block size the registers are budgeted for (256: small blocks get what the compiler asks for, 1024: 64)
template <int CM, int ST, int MAXT>
__global__ void __launch_bounds__(MAXT, 1) k_cluster_u8(const __grid_constant__ ResidentParams P)
{
    namespace cg = cooperative_groups;
    cg::cluster_group cluster = cg::this_cluster();
    extern __shared__ __align__(16) uint8_t s_raw[];
    __shared__ AcceptLutWide lut;
    __shared__ __align__(8) unsigned long long s_mbar[2][2];         // [plane colour][side]

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
    // the same shared-memory layout in every CTA of the cluster: my addresses, seen in the neighbours' shared memory
    const uint32_t up_raw = map_to_cta(smem_u32(s_raw), up_cta), dn_raw = map_to_cta(smem_u32(s_raw), dn_cta);
    const uint32_t mbar = smem_u32(&s_mbar[0][0]);                   // + 16 c + 8 side
    const uint32_t up_mbar = map_to_cta(mbar, up_cta) + 8u;           // my first row lands below the last row of the CTA above
    const uint32_t dn_mbar = map_to_cta(mbar, dn_cta);                // my last row lands above the first row of the CTA below

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
    if (tid == 0) {
#pragma unroll
        for (uint32_t m = 0; m < 4; ++m) {
            mbar_init(mbar + 8u * m, 1u);
            mbar_arm(mbar + 8u * m, (uint32_t)pitch);                // first phase: the neighbour's row of the first sweep
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
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
    cluster.sync();      // nobody writes a neighbour's halo (or signals its mbarriers) before every CTA has loaded its start state

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
            // the halos of plane 1-c were sent during the half-sweep before (none before the first of the launch: loaded
            // from global memory); the phase of that half-sweep: sweep n for plane 0, sweep n-1 for plane 1
            const bool have_halo = c == 1u || n > 0u;
            const uint32_t halo_parity = (c == 1u ? n : n - 1u) & 1u;
            const uint32_t halo_mbar = mbar + 16u * (1u - c);
            if (is_compute)
                for (int lr = 1 + ty; lr <= rows; lr += tyc) {
                    const uint32_t ro = (uint32_t)(lr * pitch);
                    const uint32_t i = (uint32_t)(r0 + lr - 1);
                    const uint32_t p = (i + c) & 1u;
                    if (have_halo && (lr == 1 || lr == rows)) {
                        long long spins = 0;
                        if (lr == 1)
                            while (!mbar_try_wait(halo_mbar, halo_parity))
                                if (++spins > CLUSTER_SPIN_LIMIT) { atomicExch(P.error, 1); break; }
                        if (lr == rows)
                            while (!mbar_try_wait(halo_mbar + 8u, halo_parity))
                                if (++spins > CLUSTER_SPIN_LIMIT) { atomicExch(P.error, 1); break; }
                    }
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
                    // my first row is the row below the last row of the CTA above, my last row the row above the first of the CTA below
                    if (lr == 1) st_async_word(up_raw + c * plane_stride + (uint32_t)((rows_up + 1) * pitch) + col, out, up_mbar + 16u * c);
                    if (lr == rows) st_async_word(dn_raw + c * plane_stride + col, out, dn_mbar + 16u * c);
                    *reinterpret_cast<uint32_t *>(own_col + ro) = out;
                    if (count_E) ne_sum += ne_final_sum(code, mask);
                    if (do_D) d_sum += delta_sum(code, mask);
                    ++words_done;
                    if (count_H) hist_add_word(s_hist, P.q, out, tid & 31u);
                }
            __syncthreads();                                        // plane c complete in this CTA; its halos as the mbarriers say
            if (tid == 0 && have_halo) {                            // the phases this half-sweep consumed: armed for their next sweep
                mbar_arm(halo_mbar, (uint32_t)pitch);
                mbar_arm(halo_mbar + 8u, (uint32_t)pitch);
            }
            // global writes of the measurement: nothing in the loop waits for them
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
    // The last phases nobody waited for (the halos of the final half-sweeps): every CTA's stores have landed and every
    // mbarrier is quiet before a CTA exits and its shared memory is given away.
    {
        const uint32_t last = (P.nsweeps - 1u) & 1u;
        long long spins = 0;
        if (tid == 0 && P.nsweeps > 0) {
            // plane 1: sent in the last half-sweep, never consumed; plane 0: consumed by the last half-sweep and re-armed,
            // its new phase stays open (nothing is in flight for it)
            while (!mbar_try_wait(mbar + 16u, last) || !mbar_try_wait(mbar + 24u, last))
                if (++spins > CLUSTER_SPIN_LIMIT) { atomicExch(P.error, 1); break; }
        }
    }
    cluster.sync();      // no CTA exits while a neighbour may still write into its shared memory
}

}  // namespace potts
