// potts_cluster.cuh -- tiny lattices: one thread-block cluster, boundary rows through distributed shared memory.
//
// A lattice of L <= 256 is a few thousand words: the resident kernel's L2 packets (~1 us per half-sweep of flight and
// polling) cost more than the update itself.  Here the whole lattice lives in the shared memory of ONE cluster of up to 16
// CTAs (CTA b owns rows [bL/G, (b+1)L/G) of both planes, plus one halo row above and below per plane); the thread that
// updates a word of a boundary row also sends it straight to the neighbour CTA through distributed shared
// memory as ONE 8-byte packet {4 spins | half-sweep number << 32} into the neighbour's INBOX in its shared memory
// (`st.relaxed.cluster.shared::cluster.b64`: an aligned 64-bit scalar is single-copy atomic, so data and tag arrive
// together, exactly as the resident kernel's packets do through L2).  The thread that needs the word -- the one that
// updates the same column of the neighbour's first / last row -- polls its own slot until the number is that of the
// half-sweep before and uses the spins straight from the packet.  So there is no cluster-wide barrier in the loop, no
// memory fence and no mbarrier: a `barrier.cluster.arrive.release` is a MEMBAR.ALL.GPU plus ~380 cycles of barrier, and
// the fence waits for every global atomic of the measurement to be acknowledged by L2; an `st.async` with its
// completion counted by an mbarrier in the receiver's shared memory (the form this kernel had in between,
// profiles/r02h_cluster_exchange.md) has no fence but ~1000 cycles from store to wake-up.  A CTA synchronises only with
// its two neighbours, only its two boundary rows wait, and the rest of the block is ordered by one __syncthreads per
// half-sweep.  A half-sweep of colour c writes plane c and reads plane 1-c only.
//
// Hazards.  One inbox slot per (plane colour, side, word).
//   * read after write: the tag.  Packets carry the launch-local half-sweep number (from 1); the inbox starts zeroed.
//   * write after read: a sender overwrites the slot of colour c two half-sweeps later, and only after its thread of
//     that column has received the neighbour's packet of the half-sweep in between, which the neighbour's thread of the
//     same column sent after it had consumed the slot.
//   * the halo ROWS in shared memory are read in the first half-sweep of a launch only (loaded from global memory).
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

__device__ __forceinline__ void st_packet_cluster(uint32_t remote_addr, uint32_t spins, uint32_t seq)
{
    asm volatile("st.relaxed.cluster.shared::cluster.b64 [%0], %1;" ::"r"(remote_addr), "l"(make_packet(spins, seq)) : "memory");
}

__device__ __forceinline__ uint2 ld_packet_local(uint32_t addr)
{
    unsigned long long v;
    asm volatile("ld.relaxed.cluster.shared::cta.b64 %0, [%1];" : "=l"(v) : "r"(addr) : "memory");
    return make_uint2((uint32_t)v, (uint32_t)(v >> 32));
}

constexpr long long CLUSTER_SPIN_LIMIT = 1ll << 26;   // polls of a packet slot before a wait gives up (seconds)

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

    const uint32_t G = cluster.num_blocks(), b = cluster.block_rank();
    const int L = P.L, pitch = P.pitch;
    const int r0 = (int)(((long long)b * L) / G), r1 = (int)(((long long)(b + 1) * L) / G);
    const int rows = r1 - r0;
    const uint32_t up_cta = (b + G - 1) % G, dn_cta = (b + 1) % G;
    const int srows = P.rows_max + 2;
    const uint32_t plane_stride = (uint32_t)srows * (uint32_t)pitch;
    // two histogram tables used by alternate samples: one is flushed (and zeroed) while the next sample already counts
    uint32_t *const s_hist0 = reinterpret_cast<uint32_t *>(s_raw + 2 * plane_stride);
    // the same shared-memory layout in every CTA of the cluster.  Inbox: [plane colour][side][word of a row] packets
    // behind the two histogram tables; side 0 = the row above my first row, side 1 = the row below my last row
    const uint32_t wpr4 = (uint32_t)pitch >> 2;
    const uint32_t inbox = smem_u32(s_raw) + 2u * plane_stride + 8u * hist_words(P.q);
    const uint32_t up_inbox = map_to_cta(inbox, up_cta) + 8u * wpr4;  // my first row is the row below the last row of the CTA above
    const uint32_t dn_inbox = map_to_cta(inbox, dn_cta);              // my last row is the row above the first row of the CTA below

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
    for (uint32_t n = tid; n < 4u * wpr4; n += nthreads)             // no packet carries the number 0
        *reinterpret_cast<unsigned long long *>(s_raw + 2u * plane_stride + 8u * hist_words(P.q) + 8u * n) = 0ull;
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
    cluster.sync();      // nobody writes into a neighbour's inbox before every CTA has cleared it and loaded its start state

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
            // the rows above my first / below my last row were sent during the half-sweep before (none before the first of
            // the launch: those are the halo rows loaded from global memory)
            const uint32_t seq = 2u * n + c + 1u;                       // number of this half-sweep in the launch, from 1
            const bool have_halo = seq > 1u;
            const uint32_t halo_inbox = inbox + 16u * wpr4 * (1u - c);  // the packets of plane 1-c: side 0, then side 1
            if (is_compute)
                for (int lr = 1 + ty; lr <= rows; lr += tyc) {
                    const uint32_t ro = (uint32_t)(lr * pitch);
                    const uint32_t i = (uint32_t)(r0 + lr - 1);
                    const uint32_t p = (i + c) & 1u;
                    uint32_t halo_up = 0u, halo_dn = 0u;
                    const bool pk_up = have_halo && lr == 1, pk_dn = have_halo && lr == rows;
                    if (pk_up || pk_dn) {
                        const uint32_t slot = halo_inbox + 2u * col;            // 8 bytes per word of the row
                        long long spins = 0;
                        if (pk_up) {
                            uint2 v = ld_packet_local(slot);
                            while (v.y != seq - 1u) {
                                if (++spins > CLUSTER_SPIN_LIMIT) { atomicExch(P.error, 1); break; }
                                v = ld_packet_local(slot);
                            }
                            halo_up = v.x;
                        }
                        if (pk_dn) {
                            uint2 v = ld_packet_local(slot + 8u * wpr4);
                            while (v.y != seq - 1u) {
                                if (++spins > CLUSTER_SPIN_LIMIT) { atomicExch(P.error, 1); break; }
                                v = ld_packet_local(slot + 8u * wpr4);
                            }
                            halo_dn = v.x;
                        }
                    }
                    const uint8_t *const orow = oth_row + ro;
                    const uint32_t own = *reinterpret_cast<const uint32_t *>(own_col + ro);
                    const uint32_t mid = *reinterpret_cast<const uint32_t *>(orow + col);
                    const uint32_t up = pk_up ? halo_up : *reinterpret_cast<const uint32_t *>(orow + col - pitch);
                    const uint32_t dn = pk_dn ? halo_dn : *reinterpret_cast<const uint32_t *>(orow + col + pitch);
                    const uint32_t adj = *reinterpret_cast<const uint32_t *>(orow + (p ? col_next : col_prev));
                    uint32_t lf, rt;
                    horizontal(p, mid, adj, lf, rt);
                    const RowKeys R = row_keys(K, i);
                    uint32_t code, mask;
                    const uint32_t out = update_word<CM, ST, AcceptLutWide::slots>(own, up, dn, lf, rt, 2u * col + p, q, K, R, &lut, lane_off, code, mask);
                    // my first row is the row below the last row of the CTA above, my last row the row above the first of the CTA below
                    if (lr == 1) st_packet_cluster(up_inbox + 16u * wpr4 * c + 2u * col, out, seq);
                    if (lr == rows) st_packet_cluster(dn_inbox + 16u * wpr4 * c + 2u * col, out, seq);
                    *reinterpret_cast<uint32_t *>(own_col + ro) = out;
                    if (count_E) ne_sum += ne_final_sum(code, mask);
                    if (do_D) d_sum += delta_sum(code, mask);
                    ++words_done;
                    if (count_H) hist_add_word(s_hist, P.q, out, tid & 31u);
                }
            __syncthreads();                                        // plane c complete in this CTA
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
    cluster.sync();      // no CTA exits while a neighbour may still write into its shared memory
}

}  // namespace potts
