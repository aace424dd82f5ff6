// potts_packed.cuh -- sub-byte packed spin layout (BASELINE config 4) for sm_100a.
//
// b = 4 bits per spin for q <= 16, 5 bits for 16 < q <= 32 (PAPER.md:161 uses a byte for every q; the
// paper's own limit, 1.5 GB for L = 32768, is what a narrower spin relaxes).  Each colour plane is
// split again into
//   nibble plane  row pitch L/4 bytes: a 32-bit word holds 8 consecutive same-colour sites of a row,
//                 sites 0..3 in the low nibbles of bytes 0..3, sites 4..7 in the high nibbles, so
//                 `w & 0x0f0f0f0f` and `(w >> 4) & 0x0f0f0f0f` are the two byte-per-site words;
//   high-bit plane (5-bit only) row pitch L/16 bytes: a 32-bit word holds bit 4 of 32 consecutive
//                 sites = 4 nibble words m = 0..3; site j of the low half of nibble word m sits at
//                 bit 8j+m, of the high half at bit 8j+4+m, so one shift and one mask per half put
//                 the bit where the byte-per-site word wants it.
// Algorithmic HBM traffic per update: read own + read other (once) + write own = 3 b/8 bytes
// (1.5 B at 4 bits, 1.875 B at 5 bits, against 3 B for the U8 layout).
// The arithmetic is the one of potts_core.cuh on unpacked words: results are bit-identical to U8.
// A thread handles 32 consecutive same-colour sites (16 bytes of nibbles + 4 bytes of high bits), so
// the packed layout needs L % 64 == 0.
#pragma once
#include <type_traits>

#include "potts_core.cuh"

namespace potts {

// 32 sites -> 8 words of one byte per site; w[n] = sites 4n..4n+3
template <bool FIVE>
__device__ __forceinline__ void unpack_pair(uint32_t nib, uint32_t hb, int m, uint32_t &lo, uint32_t &hi)
{
    lo = nib & 0x0f0f0f0fu;
    hi = (nib >> 4) & 0x0f0f0f0fu;
    if (FIVE) {
        lo |= (hb << (4 - m)) & 0x10101010u;
        hi |= (hb >> m) & 0x10101010u;
    }
}

template <bool FIVE>
__device__ __forceinline__ void unpack32(uint4 nib, uint32_t hb, uint32_t w[8])
{
    const uint32_t nw[4] = {nib.x, nib.y, nib.z, nib.w};
#pragma unroll
    for (int m = 0; m < 4; ++m) unpack_pair<FIVE>(nw[m], hb, m, w[2 * m], w[2 * m + 1]);
}

template <bool FIVE>
__device__ __forceinline__ uint32_t pack_pair(uint32_t lo, uint32_t hi, int m, uint32_t &hb)
{
    if (FIVE) hb |= (((lo >> 4) & 0x01010101u) | (hi & 0x10101010u)) << m;
    return (lo & 0x0f0f0f0fu) | ((hi << 4) & 0xf0f0f0f0u);
}

struct PackedPlanes {
    uint8_t *nib[2];      // nibble planes of colour 0 / 1
    uint8_t *hb[2];       // high-bit planes (5-bit layout only)
    int32_t L;
    int32_t pn, ph;       // row pitches: L/4 and L/16 bytes
};

template <bool FIVE>
__device__ __forceinline__ void load32(const PackedPlanes &S, int c, int i, int x, uint32_t w[8])
{
    const uint4 nib = *reinterpret_cast<const uint4 *>(S.nib[c] + (size_t)i * S.pn + 16 * x);
    const uint32_t hb = FIVE ? *reinterpret_cast<const uint32_t *>(S.hb[c] + (size_t)i * S.ph + 4 * x) : 0u;
    unpack32<FIVE>(nib, hb, w);
}

struct PackedSweepParams {
    PackedPlanes S;
    uint32_t q;
    uint32_t colour;
    HalfSweepKeys K;
    uint32_t thr[4];
    unsigned long long *E_out;
    unsigned long long *hist_out;
    int32_t rpw;                 // rows per warp (even, divides L / PK_WARPS)
    int32_t row_groups;          // tiles per column block = L / (PK_WARPS * rpw)
    uint32_t total_tiles;        // column blocks x row_groups
    uint32_t *tile_counter;      // device word, 0 at launch and again after it (see k_sweep_rows_u8)
};

// 8 warps share a block's 48 KB of tables (ColKeys + accept table), three blocks per SM (80 registers): 24 warps per SM.
// With 4 warps per block the shared memory held an SM to 4 blocks = 16 warps: cfg4 3.02 -> 2.75 ps per update.
constexpr int PK_WARPS = 8;
constexpr int PK_MIN_BLOCKS = 3;
constexpr int PK_SITES = 32;     // same-colour sites per lane and row: 16 bytes of nibbles (+ 4 bytes of high bits)

// Half-sweep, packed layout, one launch per colour: k_sweep_rows_u8 (potts_kernels.cuh) on packed planes.  A block owns
// 32 x 32 = 1024 same-colour sites (2048 lattice columns) x PK_WARPS * rpw rows; warp w walks DOWN its rpw rows, a lane
// updates one 32-site chunk per row.  The other-colour rows i-1, i, i+1 roll through registers UNPACKED (and doubled
// for the nibble compare), so a loaded word is unpacked once instead of once per use (three rows use it); the column
// part of Philox (ColKeys) of the tile's 2 x 1024 columns is computed once per block into 32 KB of shared memory.
// grid = as many blocks as are resident at once (or fewer tiles), block = (32, PK_WARPS = 8); tiles drawn dynamically.
// DELTA (potts_sweep_delta): instead of the energy, add the sum of the accepted moves'
// d = n_old - n_new of this half-sweep to *P.E_out (two's-complement int64).
template <bool FIVE, int ST, int COLOUR, bool MEASURE, bool HIST, bool DELTA, bool FAST>
__global__ void __launch_bounds__(32 * PK_WARPS, PK_MIN_BLOCKS) k_sweep_rows_packed(const __grid_constant__ PackedSweepParams P)
{
    constexpr bool EX = MEASURE || DELTA;
    static_assert(!(FAST && EX), "the sums need the exact form of the acceptance");
    constexpr int CM = FIVE ? CM_7BIT : CM_NIB4;
    extern __shared__ __align__(16) uint8_t s_dyn_raw[];
    uint4 (*s_col)[PK_SITES][32] = reinterpret_cast<uint4 (*)[PK_SITES][32]>(s_dyn_raw);          // [2][32][32]: 32 KB
    uint32_t *s_hist = reinterpret_cast<uint32_t *>(s_dyn_raw + 2 * PK_SITES * 32 * sizeof(uint4));  // HIST table
    __shared__ AcceptLut lut;
    __shared__ int blockAcc;
    const uint32_t lane = threadIdx.x, wy = threadIdx.y, tid = wy * 32u + lane;
    accept_lut_fill(&lut, P.thr, tid, 32 * PK_WARPS, FAST);
    if (EX && tid == 0) blockAcc = 0;
    if (HIST)
        for (uint32_t n = tid; n < hist_words(P.q); n += 32 * PK_WARPS) s_hist[n] = 0u;

    const PackedPlanes &S = P.S;
    const int chunks = S.L >> 6;                                       // 32-site chunks per plane row
    const HalfSweepKeys &K = P.K;
    constexpr int c = COLOUR, o = 1 - COLOUR;
    const uint32_t lane_off = accept_lane_offset(lane);
    const uint32_t q = in_register(P.q);
    const int L = S.L;
    int acc = 0, rows_done = 0;                                       // acc: MEASURE unequal neighbours of the final spins; DELTA energy change
    __shared__ uint32_t s_tile[2];                                    // dynamic tiles, as k_sweep_rows_u8
    int cb_cur = -1;
    for (uint32_t it = 0;; ++it) {
    if (tid == 0) s_tile[it & 1u] = atomicInc(P.tile_counter, P.total_tiles + gridDim.x - 1u);
    __syncthreads();
    const uint32_t tile = s_tile[it & 1u];
    if (tile >= P.total_tiles) break;
    const int cb = (int)(tile / (uint32_t)P.row_groups), rg = (int)(tile - (uint32_t)cb * (uint32_t)P.row_groups);
    const int x = cb * 32 + (int)lane;
    const bool active = x < chunks;
    if (cb != cb_cur) {
    cb_cur = cb;
    if (active) {
        // site n of my chunk in a row of parity p sits at column j = 2 (32 x + n) + p
#pragma unroll
        for (int nn = 0; nn < PK_SITES / PK_WARPS; ++nn) {
            const int n = (int)wy * (PK_SITES / PK_WARPS) + nn;
#pragma unroll
            for (int p = 0; p < 2; ++p) {
                const ColKeys C = col_keys(K, 2u * (uint32_t)(32 * x + n) + (uint32_t)p);
                s_col[p][n][lane] = make_uint4(C.l0, C.l1, C.ph, C.pl);
            }
        }
    }
    __syncthreads();
    }

    if (active) {
        rows_done += P.rpw;
        const int i0 = (rg * PK_WARPS + (int)wy) * P.rpw;
        const int xn = x + 1 == chunks ? 0 : x + 1, xp = x == 0 ? chunks - 1 : x - 1;
        struct Raw { uint4 nib; uint32_t hb; };
        auto ld_row = [&](int pl, int i) {
            Raw r;
            r.nib = *reinterpret_cast<const uint4 *>(S.nib[pl] + (size_t)i * S.pn + 16 * x);
            r.hb = FIVE ? *reinterpret_cast<const uint32_t *>(S.hb[pl] + (size_t)i * S.ph + 4 * x) : 0u;
            return r;
        };
        // the word outside my chunk a row of parity p needs: sites 32..35 (p = 1) or -4..-1 (p = 0) of plane o
        auto ld_adj = [&](int i, uint32_t p) {
            Raw r;
            const int xa = p ? xn : xp;
            r.nib.x = *reinterpret_cast<const uint32_t *>(S.nib[o] + (size_t)i * S.pn + 16 * xa + (p ? 0 : 12));
            r.hb = FIVE ? *reinterpret_cast<const uint32_t *>(S.hb[o] + (size_t)i * S.ph + 4 * xa) : 0u;
            return r;
        };
        auto prep8 = [](const Raw &r, uint32_t (&w)[8]) {
            unpack32<FIVE>(r.nib, r.hb, w);
#pragma unroll
            for (int n = 0; n < 8; ++n) w[n] = prep_nbr<CM>(w[n]);
        };
        auto prep_adj = [](const Raw &r, uint32_t p) {
            uint32_t lo, hi;
            unpack_pair<FIVE>(r.nib.x, r.hb, p ? 0 : 3, lo, hi);
            return prep_nbr<CM>(p ? lo : hi);
        };

        auto visit = [&](auto par, int i, const Raw &own_raw, const uint32_t (&up)[8], const uint32_t (&mid)[8], uint32_t adjp,
                         const uint32_t (&dn)[8]) {
            constexpr int PAR = decltype(par)::value;
            const RowKeysH R = row_keys_h(K, (uint32_t)i);
            uint32_t own[8], out[8];
            unpack32<FIVE>(own_raw.nib, own_raw.hb, own);
#pragma unroll
            for (int n = 0; n < 8; ++n) {
                uint32_t nb[4];
                nb[0] = up[n];
                nb[1] = dn[n];
                if (PAR) {      // horizontal neighbours at k and k+1
                    nb[2] = mid[n];
                    nb[3] = __funnelshift_r(mid[n], n < 7 ? mid[n < 7 ? n + 1 : 7] : adjp, 8);
                } else {        // at k-1 and k
                    nb[2] = __funnelshift_l(n > 0 ? mid[n > 0 ? n - 1 : 0] : adjp, mid[n], 8);
                    nb[3] = mid[n];
                }
                uint32_t w0[4], w1[4];
                if (ST == 1) {
#pragma unroll
                    for (int b = 0; b < 4; ++b) {
                        const uint4 ck = s_col[PAR][4 * n + b][lane];
                        philox_site_h(K, R, ColKeys{ck.x, ck.y, ck.z, ck.w}, w0[b], w1[b]);
                    }
                } else {
#pragma unroll
                    for (int m = 0; m < 2; ++m) {
                        const uint4 ck = s_col[PAR][4 * n + 2 * m][lane];
                        uint32_t w[4];
                        philox_pair_h(K, R, ColKeys{ck.x, ck.y, ck.z, ck.w}, w);
                        w0[2 * m] = w[0]; w1[2 * m] = w[1]; w0[2 * m + 1] = w[2]; w1[2 * m + 1] = w[3];
                    }
                }
                uint32_t code, mask;
                out[n] = metropolis_word<CM, FAST>(own[n], nb, q, w0, w1, &lut, lane_off, code, mask);
                if (MEASURE) acc += ne_final_sum(code, mask);
                if (DELTA) acc += delta_sum(code, mask);
                if (HIST) hist_add_word(s_hist, P.q, out[n], lane);
            }
            uint32_t out_h = 0, out_w[4];
#pragma unroll
            for (int m = 0; m < 4; ++m) out_w[m] = pack_pair<FIVE>(out[2 * m], out[2 * m + 1], m, out_h);
            *reinterpret_cast<uint4 *>(S.nib[c] + (size_t)i * S.pn + 16 * x) = make_uint4(out_w[0], out_w[1], out_w[2], out_w[3]);
            if (FIVE) *reinterpret_cast<uint32_t *>(S.hb[c] + (size_t)i * S.ph + 4 * x) = out_h;
        };

        // two visits per trip, loads alternating between register sets a / b (see k_sweep_rows_u8)
        uint32_t up[8], mid[8], dn[8], dn2[8];
        prep8(ld_row(o, wrap(i0 - 1, L)), up);
        prep8(ld_row(o, i0), mid);
        constexpr uint32_t PA = COLOUR, PB = 1 - COLOUR;             // i0 is even
        Raw own_a = ld_row(c, i0), dn_a = ld_row(o, wrap(i0 + 1, L)), adj_a = ld_adj(i0, PA);
#pragma unroll 1
        for (int r = 0; r < P.rpw; r += 2) {
            const int i = i0 + r;
            const Raw own_b = ld_row(c, i + 1), dn_b = ld_row(o, wrap(i + 2, L)), adj_b = ld_adj(i + 1, PB);
            prep8(dn_a, dn);
            visit(std::integral_constant<int, (int)PA>{}, i, own_a, up, mid, prep_adj(adj_a, PA), dn);
            const int inx = r + 2 < P.rpw ? i + 2 : i + 1;
            own_a = ld_row(c, inx); dn_a = ld_row(o, wrap(inx + 1, L)); adj_a = ld_adj(inx, PA);
            prep8(dn_b, dn2);
            visit(std::integral_constant<int, (int)PB>{}, i + 1, own_b, mid, dn, prep_adj(adj_b, PB), dn2);
#pragma unroll
            for (int n = 0; n < 8; ++n) { up[n] = dn[n]; mid[n] = dn2[n]; }
        }
    }
    }   // tiles
    if (EX) {
        // MEASURE: satisfied bonds = 4 per site - unequal neighbours of the final spins = 128 per row visit - acc; DELTA: the change
        int v = DELTA ? acc : 128 * rows_done - acc;
        v = __reduce_add_sync(0xffffffffu, v);                     // one REDUX instead of a five-step shuffle tree
        if (lane == 0) atomicAdd(&blockAcc, v);
        __syncthreads();
        if (tid == 0) atomicAdd(P.E_out, DELTA ? (unsigned long long)(long long)blockAcc : 0ull - (unsigned long long)(long long)blockAcc);
    }
    if (HIST) {
        __syncthreads();
        hist_flush(s_hist, P.q, P.hist_out, tid, 32 * PK_WARPS);
    }
}

// ---------------------------------------------------------------------------------------------
// Standalone measurement, packed layout (see k_measure_u8): one thread per 32-site chunk of the black
// plane; the white chunk at the same place is its "mid" row, so every white site is counted once.
struct PackedMeasureParams {
    PackedPlanes S;
    uint32_t q;
    unsigned long long *E_out;
    unsigned long long *hist_out;
};

template <bool FIVE>
__global__ void __launch_bounds__(256) k_measure_packed(const PackedMeasureParams P)
{
    extern __shared__ uint32_t s_hist[];
    __shared__ unsigned long long blockE;
    const bool do_hist = P.hist_out != nullptr;
    if (do_hist)
        for (uint32_t n = threadIdx.x; n < hist_words(P.q); n += blockDim.x) s_hist[n] = 0;
    if (threadIdx.x == 0) blockE = 0ull;
    __syncthreads();
    const PackedPlanes &S = P.S;
    const int chunks = S.L >> 6;
    const long long total = (long long)S.L * chunks;
    uint32_t satisfied = 0;
    for (long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x; gid < total;
         gid += (long long)gridDim.x * blockDim.x) {
        const int i = (int)(gid / chunks);
        const int x = (int)(gid - (long long)i * chunks);
        const uint32_t p = (uint32_t)(i + 1) & 1u;                    // colour 1 sites
        uint32_t own[8], mid[10];
        load32<FIVE>(S, 1, i, x, own);
        load32<FIVE>(S, 0, i, x, mid + 1);
        if (P.E_out) {
            uint32_t up[8], dn[8];
            load32<FIVE>(S, 0, wrap(i - 1, S.L), x, up);
            load32<FIVE>(S, 0, wrap(i + 1, S.L), x, dn);
            const int xa = p ? (x + 1 == chunks ? 0 : x + 1) : (x == 0 ? chunks - 1 : x - 1);
            const uint32_t an = *reinterpret_cast<const uint32_t *>(S.nib[0] + (size_t)i * S.pn + 16 * xa + (p ? 0 : 12));
            const uint32_t ah = FIVE ? *reinterpret_cast<const uint32_t *>(S.hb[0] + (size_t)i * S.ph + 4 * xa) : 0u;
            unpack_pair<FIVE>(an, ah, p ? 0 : 3, mid[9], mid[0]);
            uint32_t nef = 0;
#pragma unroll
            for (int n = 0; n < 8; ++n) {
                uint32_t lf, rt;
                horizontal(p, mid[n + 1], p ? mid[n + 2] : mid[n], lf, rt);
                nef += ne_count4<false>(own[n], up[n], dn[n], lf, rt);
            }
            satisfied += 128u - byte_sum(nef);
        }
        if (do_hist) {
#pragma unroll
            for (int n = 0; n < 8; ++n) {
                hist_add_word(s_hist, P.q, own[n], threadIdx.x & 31u);
                hist_add_word(s_hist, P.q, mid[n + 1], threadIdx.x & 31u);
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
// Random start (R9), packed layout: one thread per 32-site chunk of one plane row.
template <bool FIVE>
__global__ void k_init_random_packed(PackedPlanes S, uint32_t q, uint32_t key0, uint32_t key1)
{
    const int chunks = S.L >> 6;
    const long long per_plane = (long long)S.L * chunks;
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (gid >= 2 * per_plane) return;
    const int c = gid >= per_plane;
    const long long r = gid - (long long)c * per_plane;
    const int i = (int)(r / chunks), x = (int)(r - (long long)i * chunks);
    const uint32_t p = (uint32_t)(i + c) & 1u;
    uint32_t nw[4], hb = 0;
#pragma unroll
    for (int m = 0; m < 4; ++m) {
        uint32_t w[2] = {0u, 0u};
#pragma unroll
        for (int s = 0; s < 8; ++s) {
            uint32_t ctr[4] = {2u * (uint32_t)(32 * x + 8 * m + s) + p, (uint32_t)i, 0u, 2u};
            philox4x32_10(ctr, key0, key1);
            w[s >> 2] |= __umulhi(ctr[0], q) << (8 * (s & 3));
        }
        nw[m] = pack_pair<FIVE>(w[0], w[1], m, hb);
    }
    *reinterpret_cast<uint4 *>(S.nib[c] + (size_t)i * S.pn + 16 * x) = make_uint4(nw[0], nw[1], nw[2], nw[3]);
    if (FIVE) *reinterpret_cast<uint32_t *>(S.hb[c] + (size_t)i * S.ph + 4 * x) = hb;
}

// ---------------------------------------------------------------------------------------------
// Layout conversion, packed planes <-> canonical row-major s[i*L + j], for `rows` rows starting at
// row i0.  One thread per 32-site chunk of a plane row, both colours (= 64 columns of the lattice row).
template <bool FIVE>
__global__ void k_packed_to_rowmajor(PackedPlanes S, uint8_t *out, int i0, int rows)
{
    const int chunks = S.L >> 6;
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (gid >= (long long)rows * chunks) return;
    const int r = (int)(gid / chunks), x = (int)(gid - (long long)r * chunks);
    const int i = i0 + r;
    uint32_t a[8], b[8];
    load32<FIVE>(S, 0, i, x, a);
    load32<FIVE>(S, 1, i, x, b);
    uint4 *dst = reinterpret_cast<uint4 *>(out + (size_t)r * S.L + 64 * x);
#pragma unroll
    for (int n = 0; n < 8; n += 2) {
        // row parity decides which plane holds the even columns
        const uint32_t ev0 = (i & 1) ? b[n] : a[n], od0 = (i & 1) ? a[n] : b[n];
        const uint32_t ev1 = (i & 1) ? b[n + 1] : a[n + 1], od1 = (i & 1) ? a[n + 1] : b[n + 1];
        dst[n >> 1] = make_uint4(__byte_perm(ev0, od0, 0x5140), __byte_perm(ev0, od0, 0x7362),
                                 __byte_perm(ev1, od1, 0x5140), __byte_perm(ev1, od1, 0x7362));
    }
}

template <bool FIVE>
__global__ void k_rowmajor_to_packed(const uint8_t *in, PackedPlanes S, int i0, int rows, uint32_t q, int *bad)
{
    const int chunks = S.L >> 6;
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (gid >= (long long)rows * chunks) return;
    const int r = (int)(gid / chunks), x = (int)(gid - (long long)r * chunks);
    const int i = i0 + r;
    const uint4 *src = reinterpret_cast<const uint4 *>(in + (size_t)r * S.L + 64 * x);
    uint32_t ev[8], od[8];
    bool oob = false;
#pragma unroll
    for (int n = 0; n < 8; n += 2) {
        const uint4 v = src[n >> 1];
        ev[n] = __byte_perm(v.x, v.y, 0x6420);
        od[n] = __byte_perm(v.x, v.y, 0x7531);
        ev[n + 1] = __byte_perm(v.z, v.w, 0x6420);
        od[n + 1] = __byte_perm(v.z, v.w, 0x7531);
    }
#pragma unroll
    for (int n = 0; n < 8; ++n)
#pragma unroll
        for (int s = 0; s < 4; ++s) oob |= ((ev[n] >> (8 * s)) & 0xffu) >= q || ((od[n] >> (8 * s)) & 0xffu) >= q;
    if (oob) { atomicExch(bad, 1); return; }
    uint32_t n0[4], n1[4], h0 = 0, h1 = 0;
#pragma unroll
    for (int m = 0; m < 4; ++m) {
        n0[m] = pack_pair<FIVE>((i & 1) ? od[2 * m] : ev[2 * m], (i & 1) ? od[2 * m + 1] : ev[2 * m + 1], m, h0);
        n1[m] = pack_pair<FIVE>((i & 1) ? ev[2 * m] : od[2 * m], (i & 1) ? ev[2 * m + 1] : od[2 * m + 1], m, h1);
    }
    *reinterpret_cast<uint4 *>(S.nib[0] + (size_t)i * S.pn + 16 * x) = make_uint4(n0[0], n0[1], n0[2], n0[3]);
    *reinterpret_cast<uint4 *>(S.nib[1] + (size_t)i * S.pn + 16 * x) = make_uint4(n1[0], n1[1], n1[2], n1[3]);
    if (FIVE) {
        *reinterpret_cast<uint32_t *>(S.hb[0] + (size_t)i * S.ph + 4 * x) = h0;
        *reinterpret_cast<uint32_t *>(S.hb[1] + (size_t)i * S.ph + 4 * x) = h1;
    }
}

}  // namespace potts
