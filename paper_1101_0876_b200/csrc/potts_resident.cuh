// potts_resident.cuh -- persistent multi-sweep kernel: the lattice lives in shared memory.
//
// For lattices that fit the shared memory of the GPU (2 planes x L x L/2 bytes spread over up to 148
// SMs: L <= 4096) one cooperative launch runs ALL sweeps of a potts_sweep call.  CTA b owns the rows
// [r0, r1) of both colour planes in its shared memory.  A half-sweep of colour c reads only the other
// plane (sec. 3), so the only data that crosses CTAs are the two boundary rows of the
// plane just written.  They travel as 8-byte packets {4 spins, sequence number} written straight into
// the neighbour's inbox in global memory (L2) by the thread that computed them; a packet is one aligned
// 64-bit scalar, single-copy atomic in the PTX memory model, so the receiver just polls the packet until
// the sequence number is the one it expects: no fence, no separate flag, one L2 round trip.
//
//   Threads [0, ncw*32) compute: thread (cx, ty) owns the 8-site chunk cx (two words) of the rows dealt to
//   thread row ty (round-robin, interior rows first, the CTA's first and last row at the very end).
//   Threads [ncw*32, ncw*32 + L/16) only receive ("comm").  Eight sites per thread (not four) halves the
//   per-thread bookkeeping and leaves room for >64 registers.  Per half-sweep number s of colour c:
//     compute: interior rows (they read no halo row), then -- after named barrier 1 -- the two boundary
//              rows; each boundary chunk goes straight into the neighbour's inbox with tag s
//     comm:    poll the inbox for the packets tagged s-1 (plane 1-c, sent at the END of the previous
//              half-sweep), write them into the halo rows of plane 1-c, arrive at named barrier 1
//     __syncthreads
//   Boundary rows LAST means the packets have a whole interior phase to cross the chip, and every warp
//   has work from the first cycle of the half-sweep.
//
// Why one inbox slot per (CTA, colour, side) is enough: a sender overwrites the slot of colour c two
// half-sweeps later, after its boundary phase has consumed the receiver's packets of the half-sweep in
// between, and the receiver sent those after its own comm warps had consumed the slot.
// The global planes are written at the end of the launch only, so every other entry point
// (and the next launch) sees the complete state.  Energy and histogram of a sampled sweep are fused:
// per-thread sums, a warp shuffle and one int64 atomicAdd per warp into the series slot for the energy, the
// lane-privatised shared table and one atomicAdd per state and CTA for the histogram.
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
    unsigned long long *dE_series;    // device, nsweeps entries (zeroed), may be null: += energy change of every sweep
    uint2 *inbox;                     // [gridDim.x][2 colours][2 sides][wpr] packets, zeroed before the launch
    int *error;                       // set to 1 if a wait gave up
    int32_t rows_max;                 // rows of shared memory per plane = rows_max + 2
    int32_t tyc;                      // thread rows that compute
    uint32_t col_offset;              // COL kernels: byte offset of the ColKeys table (2 x pitch entries of 16 bytes) in the dynamic shared memory
};

constexpr long long RESIDENT_SPIN_LIMIT = 1ll << 24;   // polls before a wait gives up (seconds)

// A packet is ONE 64-bit scalar {4 spins | sequence number << 32}: the PTX memory model treats a vector access as
// independent accesses of its elements, so with 64-bit elements "spins and tag arrive together" is guaranteed by the
// model (single-copy atomicity of an aligned scalar), not by the hardware's habit.  Two packets (an 8-site chunk)
// travel as one .v2.b64 access: two such elements.
__device__ __forceinline__ uint4 ld_packet2(const uint2 *p)
{
    unsigned long long a, b;
    asm volatile("ld.relaxed.gpu.global.v2.b64 {%0, %1}, [%2];" : "=l"(a), "=l"(b) : "l"(p) : "memory");
    return make_uint4((uint32_t)a, (uint32_t)(a >> 32), (uint32_t)b, (uint32_t)(b >> 32));
}

__device__ __forceinline__ unsigned long long make_packet(uint32_t spins, uint32_t seq)
{
    unsigned long long v;
    asm("mov.b64 %0, {%1, %2};" : "=l"(v) : "r"(spins), "r"(seq));
    return v;
}

template <int W>
__device__ __forceinline__ void st_packets(uint2 *p, uint2 data, uint32_t seq)
{
    if (W == 2) asm volatile("st.relaxed.gpu.global.v2.b64 [%0], {%1, %2};" ::"l"(p), "l"(make_packet(data.x, seq)), "l"(make_packet(data.y, seq)) : "memory");
    else asm volatile("st.relaxed.gpu.global.b64 [%0], %1;" ::"l"(p), "l"(make_packet(data.x, seq)) : "memory");
}

__device__ __forceinline__ void named_barrier_sync(int id, int nthreads)
{
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}

__device__ __forceinline__ void named_barrier_arrive(int id, int nthreads)
{
    asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}

// What differs between one lattice split over the grid and a batch of independent lattices, one per CTA
struct ResidentLattice {
    uint32_t G, b;                    // CTAs sharing this lattice, my index among them
    uint8_t *plane[2];
    uint32_t key0, key1;
    uint32_t thr[4];
    unsigned long long *E_series, *hist_series, *dE_series;
};

// W = words (4 sites each) a compute thread updates per row visit: 2 (an 8-site chunk: less bookkeeping per site) or
// 1 (finer grain: the host picks it where chunks would leave the four sub-partitions of an SM unevenly loaded).
// COL (W = 2 only): the column part of Philox (ColKeys) of all L columns is rebuilt at the start of every half-sweep
// into shared memory and shared by the rows a thread visits: pays from ~3 visits per thread and half-sweep (L >= 2048).
template <int CM, int W, int ST, bool COL = false>
__device__ __forceinline__ void resident_run(const ResidentParams &P, const ResidentLattice &X)
{
    static_assert(!COL || W == 2, "ColKeys table: chunk-grained kernel only");
    extern __shared__ __align__(16) uint8_t s_raw[];
    __shared__ AcceptLutWide lut;

    const uint32_t G = X.G, b = X.b;
    const int L = P.L, pitch = P.pitch;
    const int r0 = (int)(((long long)b * L) / G), r1 = (int)(((long long)(b + 1) * L) / G);
    const int rows = r1 - r0;
    const uint32_t up_cta = (b + G - 1) % G, dn_cta = (b + 1) % G;
    const int srows = P.rows_max + 2;                               // local row 0 / rows+1 = halos
    const uint32_t plane_stride = (uint32_t)srows * (uint32_t)pitch;
    uint32_t *s_hist = reinterpret_cast<uint32_t *>(s_raw + 2 * plane_stride);

    const uint32_t tid = threadIdx.x, nthreads = blockDim.x;
    const int cpr = pitch / (4 * W);                                // compute threads per plane row
    const int ccomm = pitch >> 3;                                   // 8-site chunks (2 packets each) of a halo row; the comm threads share them
    const int tyc = P.tyc;
    const int ncompute = cpr * tyc;
    const int nbar = (ncompute + 31) & ~31;                         // compute warps, in threads
    const bool is_compute = (int)tid < ncompute;
    const int ctx = (int)tid - nbar;                                // comm thread index
    const int ncomm = (int)nthreads - nbar;                         // comm threads: chunk ctx, ctx + ncomm, ... each
    const bool is_comm = ctx >= 0 && ctx < ccomm;
    const int ty = is_compute ? (int)tid / cpr : 0;
    const int cx = is_compute ? (int)tid - ty * cpr : 0;
    const uint32_t col = is_comm ? 8u * (uint32_t)ctx : 4u * W * (uint32_t)cx;   // byte offset of my words in a plane row
    // Rows are dealt round-robin over the thread rows, interior rows (local 2..rows-1) first, the two
    // boundary rows (local 1 and `rows`) last: they are the only ones that read a halo row.
    const int ni = rows > 2 ? rows - 2 : 0;
    const int tb0 = ni % tyc, tb1 = (ni + 1) % tyc;                 // thread rows that own local row 1 / local row `rows`
    const bool two = rows >= 2;
    // warps that hold a thread of those thread rows wait for the halo (named barrier 1) before the boundary phase
    const int wid = (int)(tid >> 5);
    const int w0lo = (tb0 * cpr) >> 5, w0hi = ((tb0 + 1) * cpr - 1) >> 5;
    const int w1lo = (tb1 * cpr) >> 5, w1hi = ((tb1 + 1) * cpr - 1) >> 5;
    const bool warp_boundary = (wid >= w0lo && wid <= w0hi) || (two && wid >= w1lo && wid <= w1hi);
    int nbw = w0hi - w0lo + 1;
    if (two) {
        const int lo = w1lo > w0lo ? w1lo : w0lo, hi = w1hi < w0hi ? w1hi : w0hi;
        nbw += (w1hi - w1lo + 1) - (hi >= lo ? hi - lo + 1 : 0);
    }
    const bool do_hist = X.hist_series != nullptr && P.every != 0;
    const bool do_E = X.E_series != nullptr && P.every != 0;
    const bool do_D = X.dE_series != nullptr;

    accept_lut_fill(&lut, X.thr, tid, nthreads);
    const uint32_t lane_off = accept_lane_offset<AcceptLutWide::slots>(tid);
    if (do_hist)
        for (uint32_t n = tid; n < hist_words(P.q); n += nthreads) s_hist[n] = 0u;
    // own rows of both planes, and the halo rows of plane 1 (read by the first half-sweep, colour 0):
    // global -> shared (local row = global row - r0 + 1)
    {
        const int vpr = pitch >> 4;                                 // uint4 per row
        for (int c = 0; c < 2; ++c)
            for (int n = (int)tid; n < (rows + 2) * vpr; n += (int)nthreads) {
                const int lr = n / vpr, v = n - lr * vpr;
                if (c == 0 && (lr == 0 || lr == rows + 1)) continue;
                const int gr = wrap(r0 + lr - 1, L);
                *reinterpret_cast<uint4 *>(s_raw + c * plane_stride + (uint32_t)(lr * pitch + 16 * v)) =
                    __ldcg(reinterpret_cast<const uint4 *>(X.plane[c] + (size_t)gr * pitch + 16 * v));
            }
    }
    __syncthreads();

    // the other-colour word left of my chunk (p = 0) / right of it (p = 1), periodic
    const uint32_t col_prev = col == 0u ? (uint32_t)pitch - 4u : col - 4u;
    const uint32_t col_next = col + 4u * W == (uint32_t)pitch ? 0u : col + 4u * W;
    const uint32_t q = in_register(P.q);
    // inbox of CTA x, colour c, side s (0: the row above x's first row, 1: the row below x's last row);
    // one packet {4 spins, seq} per word, so a chunk is two packets = 16 bytes
    const uint32_t wpr = (uint32_t)pitch >> 2;
    auto inbox = [&](uint32_t x, uint32_t c, uint32_t s) { return P.inbox + ((size_t)(x * 2 + c) * 2 + s) * wpr + (col >> 2); };
    uint2 *const send_up0 = inbox(up_cta, 0, 1);     // my first row -> the row below the last row of the CTA above
    uint2 *const send_dn0 = inbox(dn_cta, 0, 0);     // my last row  -> the row above the first row of the CTA below
    const uint2 *const recv0 = inbox(b, 0, 0);       // colour c: + c * 2 * wpr, side s: + s * wpr, chunk ch beyond mine: + 2 (ch - ctx)
    const uint32_t cstride = 2u * wpr;
    const int halo_bar = 32 * nbw + ((int)nthreads - nbar);         // boundary warps + comm warps, in threads

    const HalfSweepKeys K0 = half_sweep_keys(X.key0, X.key1, 0u, 0u);
    uint32_t until = P.every;                                       // sweeps until the next sample
    uint32_t sample_idx = 0;
    uint32_t seq = 0;                                               // launch-local half-sweep number, from 1
    for (uint32_t n = 0; n < P.nsweeps; ++n) {
        const uint32_t t = P.t0 + n;
        const bool sample = P.every != 0 && --until == 0;
        if (sample) until = P.every;
#pragma unroll
        for (uint32_t c = 0; c < 2; ++c) {
            ++seq;
            uint8_t *const own_col = s_raw + c * plane_stride + col;                      // + lr*pitch: my chunk
            const uint8_t *const oth_row = s_raw + (1u - c) * plane_stride;               // + lr*pitch: row start
            int d_sum = 0, ne_sum = 0;                              // energy change / unequal neighbours of the final spins
            uint32_t words_done = 0;
            const bool count_E = sample && c == 1 && do_E, count_H = sample && do_hist;
            if (COL) {
                // every thread of the block (comm warps too) rebuilds the table for (t, c); nobody reads the old one any more
                // (the barrier that ended the previous half-sweep), nobody reads the new one before the barrier below
                HalfSweepKeys Kc = K0;
                half_sweep_rekey(Kc, X.key0, X.key1, t, c);
                uint4 *const tab = reinterpret_cast<uint4 *>(s_raw + P.col_offset);
                for (uint32_t n = tid; n < 2u * (uint32_t)pitch; n += nthreads) {
                    // entry (par, s, cx) = column 2 (8 cx + s) + par: the lanes of a warp (consecutive cx) read consecutive entries
                    const uint32_t par = n >= (uint32_t)pitch ? 1u : 0u, m = n - par * (uint32_t)pitch;
                    const uint32_t sx = m / (uint32_t)cpr, cxx = m - sx * (uint32_t)cpr;
                    const ColKeys C = col_keys(Kc, 2u * (8u * cxx + sx) + par);
                    tab[n] = make_uint4(C.l0, C.l1, C.ph, C.pl);
                }
                __syncthreads();
            }
            if ((int)tid < nbar) {
                HalfSweepKeys K = K0;                                                       // uniform registers; round keys built once
                half_sweep_rekey(K, X.key0, X.key1, t, c);
                const uint4 *const s_col = reinterpret_cast<const uint4 *>(s_raw + P.col_offset);
                // one visit: local row lr, my W words
                auto update = [&](int lr) -> uint2 {
                    const uint32_t ro = (uint32_t)(lr * pitch);
                    const uint32_t i = (uint32_t)(r0 + lr - 1);
                    const uint32_t p = (i + c) & 1u;
                    const uint8_t *const orow = oth_row + ro;
                    const uint32_t adj = *reinterpret_cast<const uint32_t *>(orow + (p ? col_next : col_prev));
                    const RowKeys R = row_keys(K, i);
                    uint2 out;
                    if (W == 2) {
                        const uint2 own = *reinterpret_cast<const uint2 *>(own_col + ro);
                        const uint2 mid = *reinterpret_cast<const uint2 *>(orow + col);
                        const uint2 up = *reinterpret_cast<const uint2 *>(orow + col - pitch);
                        const uint2 dn = *reinterpret_cast<const uint2 *>(orow + col + pitch);
                        uint32_t lf0, rt0, lf1, rt1;
                        horizontal(p, mid.x, p ? mid.y : adj, lf0, rt0);
                        horizontal(p, mid.y, p ? adj : mid.x, lf1, rt1);
                        uint32_t code0, mask0, code1, mask1;
                        if (COL) {
                            const RowKeysH RH = {R.xd, R.c3 ^ K.r1[2]};
                            const uint4 *const ck = s_col + p * (uint32_t)pitch + (uint32_t)cx;   // + s * cpr: site s of my chunk
                            out.x = update_word_h<CM, ST, AcceptLutWide::slots>(own.x, up.x, dn.x, lf0, rt0, ck, (uint32_t)cpr, q, K, RH, &lut, lane_off, code0, mask0);
                            out.y = update_word_h<CM, ST, AcceptLutWide::slots>(own.y, up.y, dn.y, lf1, rt1, ck + 4 * cpr, (uint32_t)cpr, q, K, RH, &lut, lane_off, code1, mask1);
                        } else {
                            out.x = update_word<CM, ST, AcceptLutWide::slots>(own.x, up.x, dn.x, lf0, rt0, 2u * col + p, q, K, R, &lut, lane_off, code0, mask0);
                            out.y = update_word<CM, ST, AcceptLutWide::slots>(own.y, up.y, dn.y, lf1, rt1, 2u * col + 8u + p, q, K, R, &lut, lane_off, code1, mask1);
                        }
                        if (count_E) ne_sum += ne_final_sum(code0, mask0) + ne_final_sum(code1, mask1);
                        if (do_D) d_sum += delta_sum(code0, mask0) + delta_sum(code1, mask1);
                        *reinterpret_cast<uint2 *>(own_col + ro) = out;
                        words_done += 2;
                        if (count_H) { hist_add_word(s_hist, P.q, out.x, tid & 31u); hist_add_word(s_hist, P.q, out.y, tid & 31u); }
                    } else {
                        const uint32_t own = *reinterpret_cast<const uint32_t *>(own_col + ro);
                        const uint32_t mid = *reinterpret_cast<const uint32_t *>(orow + col);
                        const uint32_t up = *reinterpret_cast<const uint32_t *>(orow + col - pitch);
                        const uint32_t dn = *reinterpret_cast<const uint32_t *>(orow + col + pitch);
                        uint32_t lf, rt;
                        horizontal(p, mid, adj, lf, rt);
                        uint32_t code, mask;
                        out.x = update_word<CM, ST, AcceptLutWide::slots>(own, up, dn, lf, rt, 2u * col + p, q, K, R, &lut, lane_off, code, mask);
                        if (count_E) ne_sum += ne_final_sum(code, mask);
                        if (do_D) d_sum += delta_sum(code, mask);
                        out.y = 0u;
                        *reinterpret_cast<uint32_t *>(own_col + ro) = out.x;
                        words_done += 1;
                        if (count_H) hist_add_word(s_hist, P.q, out.x, tid & 31u);
                    }
                    return out;
                };
                if (is_compute)
                    for (int lr = 2 + ty; lr < rows; lr += tyc) update(lr);
                // boundary rows last: by now the neighbours' rows of the previous half-sweep have had a whole
                // interior phase to arrive
                if (warp_boundary) {
                    if (G > 1) named_barrier_sync(1, halo_bar);      // comm warps have filled the halo rows of plane 1-c
#pragma unroll 1
                    for (int bb = 0; bb < (two ? 2 : 1); ++bb) {
                        if (is_compute && ty == (bb ? tb1 : tb0)) {
                            const int lr = bb ? rows : 1;
                            const uint2 out = update(lr);
                            if (G > 1) {
                                if (lr == 1) st_packets<W>(send_up0 + c * cstride, out, seq);
                                if (lr == rows) st_packets<W>(send_dn0 + c * cstride, out, seq);
                            }
                        }
                    }
                }
            } else if (G > 1) {
                // comm warps: receive the rows the neighbours sent at the end of the PREVIOUS half-sweep (plane 1-c,
                // tag seq-1) into the halo rows of plane 1-c, which only the boundary phase of this half-sweep reads
                if (is_comm && seq > 1) {
#pragma unroll 1
                    for (int ch = ctx; ch < ccomm; ch += ncomm) {
                        const uint32_t more = (uint32_t)(ch - ctx);                            // chunks beyond my first one
                        uint8_t *const halo = s_raw + (1u - c) * plane_stride + col + 8u * more;
#pragma unroll 1
                        for (int s = 0; s < 2; ++s) {
                            const uint2 *src = recv0 + (1u - c) * cstride + (uint32_t)s * wpr + 2u * more;
                            uint4 v = ld_packet2(src);
                            long long spins = 0;
                            while (v.y != seq - 1 || v.w != seq - 1) {
                                if (++spins > RESIDENT_SPIN_LIMIT) { atomicExch(P.error, 1); break; }
                                __nanosleep(40);
                                v = ld_packet2(src);
                            }
                            *reinterpret_cast<uint2 *>(halo + (s == 0 ? 0u : (uint32_t)((rows + 1) * pitch))) = make_uint2(v.x, v.z);
                        }
                    }
                }
                named_barrier_arrive(1, halo_bar);
            }
            __syncthreads();                                        // plane c complete in shared memory
            if (G == 1) {
                // a single CTA is its own neighbour: wrap the rows inside shared memory
                if (is_comm) {
                    for (int ch = ctx; ch < ccomm; ch += ncomm) {
                        uint8_t *const mine = s_raw + c * plane_stride + col + 8u * (uint32_t)(ch - ctx);
                        *reinterpret_cast<uint2 *>(mine) = *reinterpret_cast<const uint2 *>(mine + (uint32_t)(rows * pitch));
                        *reinterpret_cast<uint2 *>(mine + (uint32_t)((rows + 1) * pitch)) = *reinterpret_cast<const uint2 *>(mine + pitch);
                    }
                }
                __syncthreads();
            }

            if (do_D) {
                // energy change of this half-sweep = sum of d over its accepted moves (R5, R7): one int64 atomic per warp
                int dd = d_sum;
                dd = __reduce_add_sync(0xffffffffu, dd);                     // one REDUX instead of a five-step shuffle tree
                if ((tid & 31u) == 0 && dd) atomicAdd(X.dE_series + n, (unsigned long long)(long long)dd);
            }
            if (sample && c == 1) {
                if (do_E) {
                    // satisfied bonds seen from this thread's black sites = 4 per site - unequal neighbours of the final
                    // spins (ne_sum); one fire-and-forget int64 atomic per warp: no block-wide barrier for the energy
                    uint32_t satisfied = 16u * words_done - (uint32_t)ne_sum;
                    satisfied = __reduce_add_sync(0xffffffffu, satisfied);                     // one REDUX instead of a five-step shuffle tree
                    if ((tid & 31u) == 0 && satisfied) atomicAdd(X.E_series + sample_idx, 0ull - (unsigned long long)satisfied);
                }
                if (do_hist) {
                    hist_flush(s_hist, P.q, X.hist_series + (size_t)sample_idx * P.q, tid, nthreads);
                    __syncthreads();                                // the table is zero again before the next sample counts
                }
                ++sample_idx;
            }
        }
    }
    // final state: shared -> global
    {
        const int vpr = pitch >> 4;
        for (int c = 0; c < 2; ++c)
            for (int n = (int)tid; n < rows * vpr; n += (int)nthreads) {
                const int lr = n / vpr, v = n - lr * vpr;
                *reinterpret_cast<uint4 *>(X.plane[c] + (size_t)(r0 + lr) * pitch + 16 * v) =
                    *reinterpret_cast<const uint4 *>(s_raw + c * plane_stride + (uint32_t)((lr + 1) * pitch + 16 * v));
            }
    }
}

// One lattice over the whole grid (cooperative launch: the CTAs wait for each other's packets).
template <int CM, int W, int ST, int MAXT, bool COL = false>     // MAXT: block size the registers are budgeted for (576 -> 112 registers)
__global__ void __launch_bounds__(MAXT, 1) k_resident_u8(const __grid_constant__ ResidentParams P)
{
    ResidentLattice X;
    X.G = gridDim.x;
    X.b = blockIdx.x;
    X.plane[0] = P.plane[0];
    X.plane[1] = P.plane[1];
    X.key0 = P.key0;
    X.key1 = P.key1;
#pragma unroll
    for (int d = 0; d < 4; ++d) X.thr[d] = P.thr[d];
    X.E_series = P.E_series;
    X.hist_series = P.hist_series;
    X.dE_series = P.dE_series;
    resident_run<CM, W, ST, COL>(P, X);
}

// Replica batch: CTA r runs lattice r of a batch of independent lattices of the same (L, q), each with
// its own seed and temperature, entirely in its shared memory: no packets, no co-residency requirement, any grid
// size.  Small lattices (the paper's L <= 256 studies with hundreds of samples) fill the GPU this
// way.  Seeds and thresholds travel in the launch parameters, so they stay in uniform registers.
constexpr int BATCH_MAX = 1024;       // lattices per launch (24 KB of launch parameters)

struct BatchTable {
    uint32_t key[BATCH_MAX][2];
    uint32_t thr[BATCH_MAX][4];
};

struct BatchParams {
    ResidentParams P;                 // plane[], E_series, hist_series: those of lattice 0; inbox unused
    unsigned long long lattice_stride;   // bytes from one lattice's planes to the next one's
    unsigned long long series_stride;    // samples per lattice in E_series (hist_series: x q)
    unsigned long long delta_stride;     // entries per lattice in dE_series
};

// One CTA = one whole lattice, so the body is much simpler than resident_run: no packets, no comm warps, no halo rows
// to fill (the row above local row 1 IS local row L, read in place), one block barrier per half-sweep.  Block =
// L/8 x tyc threads with tyc EVEN: thread row ty visits the rows 1+ty, 1+ty+tyc, ..., all of one parity, so the column
// part of Philox (ColKeys) of its four columns is computed once per half-sweep into registers and serves every visit.
// Register budget: blocks of up to 256 threads (L <= 64: two visits per thread) are compiled for three blocks per SM = 78
// registers (measured at 888 cfg1 lattices: 3.44 ps per update; four blocks = 64 registers: 3.52; the 60 registers of the
// shared resident body before: 4.37), up to 512 threads for one block = up to 128 registers, larger ones 64.
constexpr int BATCH_MIN_BLOCKS = 3;
template <int CM, int ST, int MAXT>
__global__ void __launch_bounds__(MAXT, MAXT <= 256 ? BATCH_MIN_BLOCKS : 1) k_resident_batch_u8(const __grid_constant__ BatchParams B, const __grid_constant__ BatchTable T)
{
    extern __shared__ __align__(16) uint8_t s_raw[];
    __shared__ AcceptLutWide lut;
    const ResidentParams &P = B.P;
    const uint32_t r = blockIdx.x;
    uint8_t *const plane0 = P.plane[0] + r * B.lattice_stride, *const plane1 = P.plane[1] + r * B.lattice_stride;
    const uint32_t key0 = T.key[r][0], key1 = T.key[r][1];
    unsigned long long *const E_series = P.E_series ? P.E_series + r * B.series_stride : nullptr;
    unsigned long long *const hist_series = P.hist_series ? P.hist_series + r * B.series_stride * P.q : nullptr;
    unsigned long long *const dE_series = P.dE_series ? P.dE_series + r * B.delta_stride : nullptr;

    const int L = P.L, pitch = P.pitch, rows = L;
    const uint32_t plane_stride = (uint32_t)(rows + 2) * (uint32_t)pitch;   // local row lr at lr * pitch; rows 0 and L+1 unused
    uint32_t *s_hist = reinterpret_cast<uint32_t *>(s_raw + 2 * plane_stride);
    const uint32_t tid = threadIdx.x, nthreads = blockDim.x;
    const int wpr = pitch >> 2, tyc = P.tyc;
    const bool is_compute = (int)tid < wpr * tyc;
    const int ty = is_compute ? (int)tid / wpr : 0;
    const uint32_t col = is_compute ? 4u * (uint32_t)((int)tid - ty * wpr) : 0u;
    const uint32_t col_prev = col == 0u ? (uint32_t)pitch - 4u : col - 4u;
    const uint32_t col_next = col + 4u == (uint32_t)pitch ? 0u : col + 4u;
    const bool do_hist = hist_series != nullptr && P.every != 0;
    const bool do_E = E_series != nullptr && P.every != 0;
    const bool do_D = dE_series != nullptr;
    const uint32_t q = in_register(P.q);

    accept_lut_fill(&lut, T.thr[r], tid, nthreads);
    const uint32_t lane_off = accept_lane_offset<AcceptLutWide::slots>(tid);
    if (do_hist)
        for (uint32_t n = tid; n < hist_words(P.q); n += nthreads) s_hist[n] = 0u;
    {
        const int vpr = pitch >> 4;
        for (int c = 0; c < 2; ++c)
            for (int n = (int)tid; n < rows * vpr; n += (int)nthreads) {
                const int gr = n / vpr, v = n - gr * vpr;
                *reinterpret_cast<uint4 *>(s_raw + c * plane_stride + (uint32_t)((gr + 1) * pitch + 16 * v)) =
                    __ldcg(reinterpret_cast<const uint4 *>((c ? plane1 : plane0) + (size_t)gr * pitch + 16 * v));
            }
    }
    __syncthreads();

    const HalfSweepKeys K0 = half_sweep_keys(key0, key1, 0u, 0u);
    uint32_t until = P.every, sample_idx = 0;
    for (uint32_t n = 0; n < P.nsweeps; ++n) {
        const uint32_t t = P.t0 + n;
        const bool sample = P.every != 0 && --until == 0;
        if (sample) until = P.every;
#pragma unroll
        for (uint32_t c = 0; c < 2; ++c) {
            uint8_t *const own_col = s_raw + c * plane_stride + col;
            const uint8_t *const oth = s_raw + (1u - c) * plane_stride;
            HalfSweepKeys K = K0;
            half_sweep_rekey(K, key0, key1, t, c);
            const bool count_E = sample && c == 1 && do_E, count_H = sample && do_hist;
            int d_sum = 0, ne_sum = 0;
            uint32_t words_done = 0;
            if (is_compute) {
                // global row i = lr - 1; every row of this thread has the parity of ty, so p and the columns are fixed
                const uint32_t p = ((uint32_t)ty + c) & 1u;
                ColKeys ck[4];
#pragma unroll
                for (int s = 0; s < 4; ++s) ck[s] = col_keys(K, 2u * col + p + 2u * (uint32_t)s);
                for (int lr = 1 + ty; lr <= rows; lr += tyc) {
                    const uint32_t ro = (uint32_t)(lr * pitch);
                    const uint32_t ro_up = lr == 1 ? (uint32_t)(rows * pitch) : ro - (uint32_t)pitch;      // periodic, in place
                    const uint32_t ro_dn = lr == rows ? (uint32_t)pitch : ro + (uint32_t)pitch;
                    const uint32_t own = *reinterpret_cast<const uint32_t *>(own_col + ro);
                    const uint32_t mid = *reinterpret_cast<const uint32_t *>(oth + ro + col);
                    const uint32_t up = *reinterpret_cast<const uint32_t *>(oth + ro_up + col);
                    const uint32_t dn = *reinterpret_cast<const uint32_t *>(oth + ro_dn + col);
                    const uint32_t adj = *reinterpret_cast<const uint32_t *>(oth + ro + (p ? col_next : col_prev));
                    uint32_t lf, rt;
                    horizontal(p, mid, adj, lf, rt);
                    const RowKeysH R = row_keys_h(K, (uint32_t)(lr - 1));
                    uint32_t code, mask;
                    const uint32_t out = update_word_r<CM, ST, AcceptLutWide::slots>(own, up, dn, lf, rt, ck, q, K, R, &lut, lane_off, code, mask);
                    *reinterpret_cast<uint32_t *>(own_col + ro) = out;
                    if (count_E) ne_sum += ne_final_sum(code, mask);
                    if (do_D) d_sum += delta_sum(code, mask);
                    ++words_done;
                    if (count_H) hist_add_word(s_hist, P.q, out, tid & 31u);
                }
            }
            __syncthreads();                                        // plane c complete
            if (do_D) {
                int dd = d_sum;
                dd = __reduce_add_sync(0xffffffffu, dd);                     // one REDUX instead of a five-step shuffle tree
                if ((tid & 31u) == 0 && dd) atomicAdd(dE_series + n, (unsigned long long)(long long)dd);
            }
            if (sample && c == 1) {
                if (do_E) {
                    uint32_t satisfied = 16u * words_done - (uint32_t)ne_sum;
                    satisfied = __reduce_add_sync(0xffffffffu, satisfied);                     // one REDUX instead of a five-step shuffle tree
                    if ((tid & 31u) == 0 && satisfied) atomicAdd(E_series + sample_idx, 0ull - (unsigned long long)satisfied);
                }
                if (do_hist) {
                    hist_flush(s_hist, P.q, hist_series + (size_t)sample_idx * P.q, tid, nthreads);
                    __syncthreads();                                // the table is zero again before the next sample counts
                }
                ++sample_idx;
            }
        }
    }
    {
        const int vpr = pitch >> 4;
        for (int c = 0; c < 2; ++c)
            for (int n = (int)tid; n < rows * vpr; n += (int)nthreads) {
                const int gr = n / vpr, v = n - gr * vpr;
                *reinterpret_cast<uint4 *>((c ? plane1 : plane0) + (size_t)gr * pitch + 16 * v) =
                    *reinterpret_cast<const uint4 *>(s_raw + c * plane_stride + (uint32_t)((gr + 1) * pitch + 16 * v));
            }
    }
}

}  // namespace potts
