// potts_kernels.cuh -- streaming kernels of the checkerboard Potts sweep for sm_100a (U8 layout):
// one half-sweep per launch reading the planes through L2/HBM, the standalone measurement, the
// random start and the layout converters.  The per-site arithmetic is in potts_core.cuh.
//
// Spin layout "U8 split planes" (PAPER.md:159 packs whites then blacks; the exact map is ours):
//   plane[c][i][k], c = (i+j)&1, k = j>>1, one byte per spin, row pitch L/2 bytes.
// A colour-c site (i,k) with p = (i+c)&1 sits at column j = 2k+p; its neighbours are all in
// plane 1-c:  up [i-1][k], down [i+1][k], and horizontally [i][k],[i][k+1] if p = 1 or
// [i][k-1],[i][k] if p = 0 (indices periodic).
#pragma once
#include <type_traits>

#include "potts_core.cuh"

namespace potts {

struct SweepParams {
    uint8_t *plane_own;         // plane of the colour being updated
    const uint8_t *plane_oth;   // plane of the other colour
    int32_t L;                  // lattice size
    int32_t pitch;              // L/2, bytes per plane row
    uint32_t q;
    uint32_t colour;            // 0 = white ((i+j) even), 1 = black
    HalfSweepKeys K;            // Philox key material of (seed, t, colour), built on the host
    uint32_t thr[4];            // floor(2^32 exp(-d/T)), d = 1..4
    unsigned long long *E_out;  // MEASURE: -= satisfied bonds seen from this colour's sites; DELTA: += energy change
    unsigned long long *hist_out;  // HIST: += occupancies of this colour's sites after the update
    int32_t rpw;                // rows per warp (even, divides L / HS_WARPS)
    int32_t row_groups;         // tiles per column block = L / (HS_WARPS * rpw)
    uint32_t total_tiles;       // column blocks x row_groups
    uint32_t *tile_counter;     // device word, 0 at launch and again after it: the blocks draw their tiles from it
    int32_t bulk;               // 1: plain half-sweeps take the BULK (cp.async.bulk staging) form of the kernel
    // Row strip of a lattice split over several GPUs: the planes hold `rows` rows, local row r = global row
    // row0 + r (row0 even), with one halo row above local row 0 and one below local row rows-1 that the host fills
    // from the neighbouring strips; plane_own / plane_oth point at local row 0.  rows = L, row0 = 0, strip = 0: the whole
    // (periodic) lattice.
    int32_t rows, row0, strip;
};

// ---------------------------------------------------------------------------------------------
// Half-sweep, U8 layout, one launch per colour.  A block is HS_WARPS warps; it owns a tile of 32 x 16 = 512
// same-colour sites (1024 lattice columns) x HS_WARPS * rpw rows.  Warp w walks DOWN its rpw consecutive rows; a
// lane updates one 16-byte chunk (16 consecutive same-colour sites) per row.  Walking down means
//   * the other-colour rows i-1, i, i+1 roll through registers: one 16-byte load of row i+1 per row visit
//     instead of three (the word left / right of the chunk is a fourth, 4-byte load from L1);
//   * the nibble-doubling of a neighbour word (prep_nbr) is done once per loaded word, not once per use;
//   * the column part of Philox (ColKeys: 3 of the 17 multiplies, 2 of the 18 XORs per site) is computed once
//     per block for the tile's 2 x 512 columns (both row parities), kept in 16 KB of shared memory and read
//     back with one conflict-free 16-byte load per site.
// grid = as many blocks as are resident at once (or fewer tiles); tiles drawn dynamically.  Requires L % 32 == 0.
// MEASURE: E -= satisfied bonds seen from this colour's sites (colour 1 of a sampled sweep).  HIST: occupancy of
// the words just written.  DELTA (potts_sweep_delta: "a parallel accumulation of local energy
// changes on-the-fly"): E_out += sum over accepted moves of d = n_old - n_new (R5, R7), no energy recount.
constexpr int HS_WARPS = 4;
constexpr int HS_SITES = 16;          // same-colour sites per lane and row

// COLOUR = P.colour as a template argument: with it the row parity of every visit is a literal, the row loop
// handles two rows per trip and the next row's loads alternate between two register sets instead of being copied.
// FAST: the one-compare form of the acceptance (accept_lut_fill); the host selects it for launches without the
// energy / energy-change sums when no threshold is zero.
// BULK (experiment of round 2, option stream_stage = 1, profiles/r02e_bulk_staging.md): the other-colour rows of a
// warp's strip (rpw + 2 rows of 512 bytes + a 16-byte halo on either side) are staged in shared memory with
// cp.async.bulk copies that complete on the warp's mbarrier, and the visits read them from there instead of from
// global memory.  Needs pitch % 512 == 0 (every lane active) and no histogram (the dynamic shared memory is the stage).
constexpr int BULK_ROW = 544;                                 // 16 + 512 + 16 bytes

template <int CM, int ST, int COLOUR, bool MEASURE, bool HIST, bool DELTA, bool FAST, bool BULK = false>
__global__ void __launch_bounds__(32 * HS_WARPS) k_sweep_rows_u8(const __grid_constant__ SweepParams P)
{
    constexpr bool EX = MEASURE || DELTA;
    static_assert(!(FAST && EX), "the sums need the exact form of the acceptance");
    static_assert(!(BULK && HIST), "the staging buffer takes the dynamic shared memory");
    extern __shared__ __align__(16) uint32_t s_dyn[];         // HIST: the block's histogram table; BULK: the staged rows
    __shared__ __align__(8) unsigned long long s_mbar[HS_WARPS];
    __shared__ uint4 s_col[2][HS_SITES][32];                  // ColKeys of [row parity p][site of the chunk][lane]
    __shared__ AcceptLut lut;
    __shared__ int blockAcc;
    const uint32_t lane = threadIdx.x, wy = threadIdx.y, tid = wy * 32u + lane;
    accept_lut_fill(&lut, P.thr, tid, 32 * HS_WARPS, FAST);
    if (EX && tid == 0) blockAcc = 0;
    if (HIST)
        for (uint32_t n = tid; n < hist_words(P.q); n += 32 * HS_WARPS) s_dyn[n] = 0u;
    uint32_t bulk_phase = 0;
    const uint32_t mbar = smem_u32(&s_mbar[threadIdx.y]);
    const uint32_t stage = smem_u32(s_dyn) + threadIdx.y * (uint32_t)((P.rpw + 2) * BULK_ROW);   // this warp's rows
    if (BULK && threadIdx.x == 0) {
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(mbar));
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }

    const int chunks = P.pitch >> 4;                                  // 16-byte chunks per row
    const HalfSweepKeys &K = P.K;
    const uint32_t lane_off = accept_lane_offset(lane);
    const uint32_t q = in_register(P.q);
    const int L = P.rows, pitch = P.pitch;                            // L: rows of this plane (the lattice's, or the strip's)
    int acc = 0, rows_done = 0;                                       // acc: MEASURE unequal neighbours of the final spins; DELTA energy change
    // Tiles (column block cb, row group rg) are drawn from a global counter: tile = cb * row_groups + rg, so a block
    // mostly stays in its column block and keeps its ColKeys.  atomicInc wraps to 0 after the last of the
    // total_tiles + gridDim.x draws of a launch (every block draws exactly one tile number >= total_tiles and stops).
    __shared__ uint32_t s_tile[2];
    int cb_cur = -1;
    for (uint32_t it = 0;; ++it) {
    if (tid == 0) s_tile[it & 1u] = atomicInc(P.tile_counter, P.total_tiles + gridDim.x - 1u);
    __syncthreads();                                                  // also: every thread is done with the previous tile
    const uint32_t tile = s_tile[it & 1u];
    if (tile >= P.total_tiles) break;
    const int cb = (int)(tile / (uint32_t)P.row_groups), rg = (int)(tile - (uint32_t)cb * (uint32_t)P.row_groups);
    const int x = cb * 32 + (int)lane;
    const bool active = x < chunks;
    const int k0 = x << 4;
    if (cb != cb_cur) {
    cb_cur = cb;
    if (active) {
        // site n of my chunk in a row of parity p sits at column j = 2 (k0 + n) + p
#pragma unroll
        for (int nn = 0; nn < HS_SITES / HS_WARPS; ++nn) {
            const int n = (int)wy * (HS_SITES / HS_WARPS) + nn;
#pragma unroll
            for (int p = 0; p < 2; ++p) {
                const ColKeys C = col_keys(K, 2u * (uint32_t)(k0 + n) + (uint32_t)p);
                s_col[p][n][lane] = make_uint4(C.l0, C.l1, C.ph, C.pl);
            }
        }
    }
    __syncthreads();
    }

    if (active) {
        rows_done += P.rpw;
        const int i0 = (rg * HS_WARPS + (int)wy) * P.rpw;
        const int kn = wrap(k0 + 16, pitch), kp = wrap(k0 - 4, pitch);
        const uint8_t *const oth = P.plane_oth + k0;
        uint8_t *const ownp = P.plane_own + k0;
        if (BULK) {
            // the previous tile's reads of the stage are done (generic proxy) before the copies overwrite it (async proxy)
            __syncwarp();
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            const uint32_t bytes = (uint32_t)((P.rpw + 2) * BULK_ROW);
            if (lane == 0) asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(mbar), "r"(bytes) : "memory");
            __syncwarp();
            if ((int)lane < P.rpw + 2) {
                const int kb = cb * 512;                                   // first byte of the block's columns in a plane row
                const uint8_t *src = P.plane_oth + (long long)(P.strip ? i0 - 1 + (int)lane : wrap(i0 - 1 + (int)lane, L)) * pitch;
                const uint32_t dst = stage + lane * BULK_ROW;
                asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], 512, [%2];" ::"r"(dst + 16), "l"(src + kb), "r"(mbar) : "memory");
                asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], 16, [%2];" ::"r"(dst), "l"(src + wrap(kb - 16, pitch)), "r"(mbar) : "memory");
                asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], 16, [%2];" ::"r"(dst + 528), "l"(src + wrap(kb + 512, pitch)), "r"(mbar) : "memory");
            }
            uint32_t done = 0;
            while (!done)
                asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2; selp.u32 %0, 1, 0, p; }" : "=r"(done) : "r"(mbar), "r"(bulk_phase) : "memory");
            bulk_phase ^= 1u;
        }
        // other-colour row i (rr = i - (i0 - 1) in the stage): my chunk, and the word beside it a visit of parity par needs
        auto oth16 = [&](int i) {
            if (BULK) {
                uint4 v;
                asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(stage + (uint32_t)((i - i0 + 1) * BULK_ROW) + 16u + lane * 16u));
                return v;
            }
            return *reinterpret_cast<const uint4 *>(oth + (long long)(P.strip ? i : wrap(i, L)) * pitch);   // a strip has halo rows at -1 and L
        };
        auto oth_adj = [&](int i, int par, int kcol) {
            if (BULK) {
                uint32_t v;
                asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(stage + (uint32_t)((i - i0 + 1) * BULK_ROW) + 16u + lane * 16u + (par ? 16u : 0xfffffffcu)));
                return v;
            }
            return *reinterpret_cast<const uint32_t *>(P.plane_oth + (size_t)i * pitch + kcol);
        };

        // one row visit; PAR = (i + colour) & 1 is uniform over the block row
        auto visit = [&](auto par, int i, const uint4 &own4, const uint32_t (&up)[4], const uint32_t (&mid)[4], uint32_t adjp,
                         const uint32_t (&dn)[4]) {
            constexpr int PAR = decltype(par)::value;
            const RowKeysH R = row_keys_h(K, (uint32_t)(i + P.row0));
            const uint32_t own[4] = {own4.x, own4.y, own4.z, own4.w};
            uint32_t out[4];
#pragma unroll
            for (int n = 0; n < 4; ++n) {
                uint32_t nb[4];
                nb[0] = up[n];
                nb[1] = dn[n];
                if (PAR) {      // horizontal neighbours at k and k+1
                    nb[2] = mid[n];
                    nb[3] = __funnelshift_r(mid[n], n < 3 ? mid[n < 3 ? n + 1 : 3] : adjp, 8);
                } else {        // at k-1 and k
                    nb[2] = __funnelshift_l(n > 0 ? mid[n > 0 ? n - 1 : 0] : adjp, mid[n], 8);
                    nb[3] = mid[n];
                }
                uint32_t w0[4], w1[4];
                if (ST == 1) {
#pragma unroll
                    for (int b = 0; b < 4; ++b) {
                        const uint4 c = s_col[PAR][4 * n + b][lane];
                        philox_site_h(K, R, ColKeys{c.x, c.y, c.z, c.w}, w0[b], w1[b]);
                    }
                } else {
#pragma unroll
                    for (int m = 0; m < 2; ++m) {
                        const uint4 c = s_col[PAR][4 * n + 2 * m][lane];
                        uint32_t w[4];
                        philox_pair_h(K, R, ColKeys{c.x, c.y, c.z, c.w}, w);
                        w0[2 * m] = w[0]; w1[2 * m] = w[1]; w0[2 * m + 1] = w[2]; w1[2 * m + 1] = w[3];
                    }
                }
                uint32_t code, mask;
                out[n] = metropolis_word<CM, FAST>(own[n], nb, q, w0, w1, &lut, lane_off, code, mask);
                if (MEASURE) acc += ne_final_sum(code, mask);
                if (DELTA) acc += delta_sum(code, mask);
                if (HIST) hist_add_word(s_dyn, P.q, out[n], lane);
            }
            *reinterpret_cast<uint4 *>(ownp + (size_t)i * pitch) = make_uint4(out[0], out[1], out[2], out[3]);
        };
        auto ld16 = [](const uint8_t *p) { return *reinterpret_cast<const uint4 *>(p); };
        auto prep4 = [](const uint4 &v, uint32_t (&w)[4]) {
            w[0] = prep_nbr<CM>(v.x); w[1] = prep_nbr<CM>(v.y); w[2] = prep_nbr<CM>(v.z); w[3] = prep_nbr<CM>(v.w);
        };

        // rows i0 (parity COLOUR: i0 is even), i0 + 1 (the other parity), ...: two visits per trip.  Register sets a / b
        // hold the loads of the even / odd visit; each visit first issues the loads of the NEXT row into the other
        // set, so they have a whole visit to arrive (the tile's last visit reloads its own row, unused).
        uint32_t up[4], mid[4], dn[4], dn2[4];
        prep4(oth16(i0 - 1), up);
        prep4(oth16(i0), mid);
        constexpr int PA = COLOUR, PB = 1 - COLOUR;
        const int k_a = PA ? kn : kp, k_b = PB ? kn : kp;             // column of the word outside the chunk
        uint4 own_a = ld16(ownp + (size_t)i0 * pitch);
        uint4 dn_a = oth16(i0 + 1);
        uint32_t adj_a = oth_adj(i0, PA, k_a);
#pragma unroll 1
        for (int r = 0; r < P.rpw; r += 2) {
            const int i = i0 + r;
            const uint4 own_b = ld16(ownp + (size_t)(i + 1) * pitch);
            const uint4 dn_b = oth16(i + 2);
            const uint32_t adj_b = oth_adj(i + 1, PB, k_b);
            prep4(dn_a, dn);
            visit(std::integral_constant<int, PA>{}, i, own_a, up, mid, prep_nbr<CM>(adj_a), dn);
            const int inx = r + 2 < P.rpw ? i + 2 : i + 1;
            own_a = ld16(ownp + (size_t)inx * pitch);
            dn_a = oth16(inx + 1);
            adj_a = oth_adj(inx, PA, k_a);
            prep4(dn_b, dn2);
            visit(std::integral_constant<int, PB>{}, i + 1, own_b, mid, dn, prep_nbr<CM>(adj_b), dn2);
#pragma unroll
            for (int n = 0; n < 4; ++n) { up[n] = dn[n]; mid[n] = dn2[n]; }
        }
    }
    }   // tiles
    if (EX) {
        // MEASURE: satisfied bonds = 4 per site - unequal neighbours of the final spins = 64 per row visit - acc
        int v = DELTA ? acc : 64 * rows_done - acc;
        v = __reduce_add_sync(0xffffffffu, v);                     // one REDUX instead of a five-step shuffle tree
        if (lane == 0) atomicAdd(&blockAcc, v);
        __syncthreads();
        // E = -(satisfied bonds): accumulate the two's-complement negative into the int64 slot; DELTA: += the change
        if (tid == 0) atomicAdd(P.E_out, DELTA ? (unsigned long long)(long long)blockAcc : 0ull - (unsigned long long)(long long)blockAcc);
    }
    if (HIST) {
        __syncthreads();
        hist_flush(s_dyn, P.q, P.hist_out, tid, 32 * HS_WARPS);
    }
}

// ---------------------------------------------------------------------------------------------
// Standalone measurement: energy from the black plane's sites (every bond joins a black and a
// white site, so summing equal neighbours over black sites counts each bond once) and the
// histogram of both planes.  One thread per 16-byte chunk of the black plane; the white chunk
// at the same (row, k-range) is the thread's "mid" word, so every white site is counted once.
struct MeasureParams {
    const uint8_t *plane0, *plane1;
    int32_t L, pitch;               // L: rows of the planes (the lattice's, or the strip's); pitch = lattice L / 2
    int32_t row0, strip;            // row strip (see SweepParams): halo rows instead of the periodic wrap
    uint32_t q;
    unsigned long long *E_out;      // may be null
    unsigned long long *hist_out;   // q entries, may be null
};

template <bool WIDE>
__global__ void __launch_bounds__(256) k_measure_u8(const MeasureParams P)
{
    extern __shared__ uint32_t s_hist[];            // hist_words(q) counters, see potts_core.cuh
    __shared__ unsigned long long blockE;
    const bool do_hist = P.hist_out != nullptr;
    if (do_hist)
        for (uint32_t n = threadIdx.x; n < hist_words(P.q); n += blockDim.x) s_hist[n] = 0;
    if (threadIdx.x == 0) blockE = 0ull;
    __syncthreads();

    const int chunks = P.pitch >> 4;
    const long long total = (long long)P.L * chunks;
    uint32_t satisfied = 0;
    for (long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x; gid < total;
         gid += (long long)gridDim.x * blockDim.x) {
        const int i = (int)(gid / chunks);
        const int x = (int)(gid - (long long)i * chunks);
        const int k0 = x << 4;
        const uint32_t p = (uint32_t)(i + P.row0 + 1) & 1u;          // colour 1 sites
        const long long iu = P.strip ? i - 1 : wrap(i - 1, P.L), id = P.strip ? i + 1 : wrap(i + 1, P.L);
        const size_t row = (size_t)i * P.pitch;
        const uint4 own4 = *reinterpret_cast<const uint4 *>(P.plane1 + row + k0);
        const uint4 mid4 = *reinterpret_cast<const uint4 *>(P.plane0 + row + k0);
        const uint32_t own[4] = {own4.x, own4.y, own4.z, own4.w};
        if (P.E_out) {
            const uint4 up4 = *reinterpret_cast<const uint4 *>(P.plane0 + iu * P.pitch + k0);
            const uint4 dn4 = *reinterpret_cast<const uint4 *>(P.plane0 + id * P.pitch + k0);
            const int ka = p ? wrap(k0 + 16, P.pitch) : wrap(k0 - 4, P.pitch);
            const uint32_t adj = *reinterpret_cast<const uint32_t *>(P.plane0 + row + ka);
            const uint32_t mid[6] = {adj, mid4.x, mid4.y, mid4.z, mid4.w, adj};
            const uint32_t up[4] = {up4.x, up4.y, up4.z, up4.w};
            const uint32_t dn[4] = {dn4.x, dn4.y, dn4.z, dn4.w};
            uint32_t nef = 0;
#pragma unroll
            for (int n = 0; n < 4; ++n) {
                uint32_t lf, rt;
                horizontal(p, mid[n + 1], p ? mid[n + 2] : mid[n], lf, rt);
                nef += ne_count4<WIDE>(own[n], up[n], dn[n], lf, rt);
            }
            satisfied += 64u - byte_sum(nef);
        }
        if (do_hist) {
            const uint32_t oth[4] = {mid4.x, mid4.y, mid4.z, mid4.w};
#pragma unroll
            for (int n = 0; n < 4; ++n) {
                hist_add_word(s_hist, P.q, own[n], threadIdx.x & 31u);
                hist_add_word(s_hist, P.q, oth[n], threadIdx.x & 31u);
            }
        }
    }
    if (P.E_out) {
        satisfied = __reduce_add_sync(0xffffffffu, satisfied);                     // one REDUX instead of a five-step shuffle tree
        if ((threadIdx.x & 31) == 0) atomicAdd(&blockE, (unsigned long long)satisfied);
    }
    __syncthreads();
    if (P.E_out && threadIdx.x == 0) atomicAdd(P.E_out, 0ull - blockE);
    if (do_hist) hist_flush(s_hist, P.q, P.hist_out, threadIdx.x, blockDim.x);
}

// ---------------------------------------------------------------------------------------------
// Random start (R9): s(i,j) = floor(w0 q / 2^32), (w0,..) = Philox((j, i, 0, 2), seed).
// One thread per 4 consecutive k of one plane row.
// L = rows of the planes; row0 = global index of their first row (0 unless the planes are a row strip; even).
static __global__ void k_init_random_u8(uint8_t *plane0, uint8_t *plane1, int L, int pitch, uint32_t q,
                                 uint32_t key0, uint32_t key1, int row0 = 0)
{
    const long long words_per_plane = (long long)L * (pitch >> 2);
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (gid >= 2 * words_per_plane) return;
    const int c = gid >= words_per_plane;
    const long long r = gid - (long long)c * words_per_plane;
    const int i = (int)(r / (pitch >> 2));
    const int kw = (int)(r - (long long)i * (pitch >> 2));
    const uint32_t p = (uint32_t)(i + c) & 1u;
    uint32_t word = 0;
#pragma unroll
    for (int b = 0; b < 4; ++b) {
        uint32_t ctr[4] = {2u * (uint32_t)(4 * kw + b) + p, (uint32_t)(i + row0), 0u, 2u};
        philox4x32_10(ctr, key0, key1);
        word |= __umulhi(ctr[0], q) << (8 * b);
    }
    uint8_t *plane = c ? plane1 : plane0;
    *reinterpret_cast<uint32_t *>(plane + (size_t)i * pitch + 4 * kw) = word;
}

// ---------------------------------------------------------------------------------------------
// Layout conversion: split planes <-> canonical row-major s[i*L + j], for `rows` rows starting
// at row i0.  One thread per 4 sites of a plane row (= 8 columns of the lattice row).
static __global__ void k_planes_to_rowmajor(const uint8_t *plane0, const uint8_t *plane1, uint8_t *out,
                                     int L, int pitch, int i0, int rows)
{
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const int wpr = pitch >> 2;
    if (gid >= (long long)rows * wpr) return;
    const int r = (int)(gid / wpr), kw = (int)(gid - (long long)r * wpr);
    const int i = i0 + r;
    const uint32_t a = *reinterpret_cast<const uint32_t *>(plane0 + (size_t)i * pitch + 4 * kw);
    const uint32_t b = *reinterpret_cast<const uint32_t *>(plane1 + (size_t)i * pitch + 4 * kw);
    // row parity decides which plane holds the even columns
    const uint32_t ev = (i & 1) ? b : a, od = (i & 1) ? a : b;
    uint2 o;
    o.x = __byte_perm(ev, od, 0x5140);   // ev0 od0 ev1 od1
    o.y = __byte_perm(ev, od, 0x7362);   // ev2 od2 ev3 od3
    *reinterpret_cast<uint2 *>(out + (size_t)r * L + 8 * kw) = o;
}

static __global__ void k_rowmajor_to_planes(const uint8_t *in, uint8_t *plane0, uint8_t *plane1, int L,
                                     int pitch, int i0, int rows, uint32_t q, int *bad)
{
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const int wpr = pitch >> 2;
    if (gid >= (long long)rows * wpr) return;
    const int r = (int)(gid / wpr), kw = (int)(gid - (long long)r * wpr);
    const int i = i0 + r;
    const uint2 v = *reinterpret_cast<const uint2 *>(in + (size_t)r * L + 8 * kw);
    const uint32_t ev = __byte_perm(v.x, v.y, 0x6420);
    const uint32_t od = __byte_perm(v.x, v.y, 0x7531);
    if (q < 256) {
        bool b = false;
#pragma unroll
        for (int n = 0; n < 4; ++n)
            b |= ((ev >> (8 * n)) & 0xffu) >= q || ((od >> (8 * n)) & 0xffu) >= q;
        if (b) atomicExch(bad, 1);
    }
    *reinterpret_cast<uint32_t *>(((i & 1) ? plane1 : plane0) + (size_t)i * pitch + 4 * kw) = ev;
    *reinterpret_cast<uint32_t *>(((i & 1) ? plane0 : plane1) + (size_t)i * pitch + 4 * kw) = od;
}

}  // namespace potts
