// potts3d.cuh -- the 3D generalisation of the checkerboard sweep ("the checkerboard scheme defining two
// independent sub-networks persists, however the cell-packing scheme should be updated"): simple-cubic L x L x L
// periodic lattice, 6 nearest neighbours, same Metropolis rule (reading S16).  First CUDA path of this
// row of SURVEY 8(f)4: one launch per half-sweep, one 16-site chunk per thread, no row walking yet.
//
// Cell packing: plane[c][z][y][k], c = (x+y+z)&1, k = x>>1, one byte per spin, row pitch L/2 bytes.  A colour-c site
// (z, y, k) with p = (z+y+c)&1 sits at x = 2k+p.  Its neighbours are all in plane 1-c: (z, y+-1, k) and (z+-1, y, k)
// at the SAME k (those rows have the same p), and in its own row (z, y) the words at k and k+1 (p = 1) or k-1 and k
// (p = 0), periodic.
// Random stream: Philox4x32-10(counter = (x, y, t, colour + 4 z), key = seed), words 0 and 1: the 2D HalfSweepKeys /
// RowKeys / philox_site of potts_core.cuh apply with "colour" := colour + 4 z (a per-thread value here).
#pragma once
#include "potts_core.cuh"

#include <type_traits>

namespace potts {

struct Sweep3Params {
    uint8_t *plane_own;
    const uint8_t *plane_oth;
    int32_t L, pitch;            // pitch = L/2
    uint32_t q, colour;
    uint32_t key0, key1, t;
    unsigned long long neg_thr[13];   // 2^64 - threshold(d), d = -6..6 (threshold = 2^32 for d <= 0): index d + 6
};

// per-byte "differs" counts of a word against six neighbour words, for the current spins and the proposals at once
template <int CM>
__device__ __forceinline__ void ne_counts6(uint32_t own, uint32_t prop, const uint32_t nb[6], uint32_t &c_old, uint32_t &c_new)
{
    if (is_nibble_mode(CM)) {
        const uint32_t both = prop * 16u + own;
        uint32_t s = 0;
#pragma unroll
        for (int k = 0; k < 6; ++k) {
            const uint32_t n2 = nb[k] * 0x11u;
            uint32_t u;
            if (CM == CM_NIB3) u = (both ^ n2) + 0x77777777u;
            else u = lop3<LOP_OR_XOR>(lop3<LOP_XOR_AND>(both, n2, 0x77777777u) + 0x77777777u, both, n2);
            s += (u >> 3) & 0x11111111u;                              // nibble counters: at most 6
        }
        c_old = s & 0x0f0f0f0fu;
        c_new = (s >> 4) & 0x0f0f0f0fu;
    } else {
        c_old = c_new = 0;
#pragma unroll
        for (int k = 0; k < 6; ++k) {
            c_old += ne_flags<CM == CM_8BIT>(own, nb[k]) >> 7;
            c_new += ne_flags<CM == CM_8BIT>(prop, nb[k]) >> 7;
        }
    }
}

// Half-sweep of colour P.colour.  One thread per 16-byte chunk of the own plane; grid-stride over all chunks.
template <int CM>
__global__ void __launch_bounds__(128) k_sweep3_u8(const __grid_constant__ Sweep3Params P)
{
    __shared__ unsigned long long lut[16];
    if (threadIdx.x < 13) lut[threadIdx.x] = P.neg_thr[threadIdx.x];
    __syncthreads();
    const int L = P.L, pitch = P.pitch, cpr = pitch >> 4;              // 16-byte chunks per row
    const long long total = (long long)L * L * cpr;
    const uint32_t q = in_register(P.q);
    for (long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x; gid < total; gid += (long long)gridDim.x * blockDim.x) {
        const int cx = (int)(gid % cpr);
        const long long row = gid / cpr;
        const int y = (int)(row % L), z = (int)(row / L);
        const uint32_t p = (uint32_t)(z + y + (int)P.colour) & 1u;
        const int k0 = cx << 4;
        const size_t r_mid = ((size_t)z * L + y) * pitch;
        const size_t r_up = ((size_t)z * L + wrap(y - 1, L)) * pitch, r_dn = ((size_t)z * L + wrap(y + 1, L)) * pitch;
        const size_t r_lo = ((size_t)wrap(z - 1, L) * L + y) * pitch, r_hi = ((size_t)wrap(z + 1, L) * L + y) * pitch;
        const uint4 own4 = *reinterpret_cast<const uint4 *>(P.plane_own + r_mid + k0);
        const uint4 mid4 = *reinterpret_cast<const uint4 *>(P.plane_oth + r_mid + k0);
        const uint4 up4 = *reinterpret_cast<const uint4 *>(P.plane_oth + r_up + k0);
        const uint4 dn4 = *reinterpret_cast<const uint4 *>(P.plane_oth + r_dn + k0);
        const uint4 lo4 = *reinterpret_cast<const uint4 *>(P.plane_oth + r_lo + k0);
        const uint4 hi4 = *reinterpret_cast<const uint4 *>(P.plane_oth + r_hi + k0);
        const uint32_t adj = *reinterpret_cast<const uint32_t *>(P.plane_oth + r_mid + (p ? wrap(k0 + 16, pitch) : wrap(k0 - 4, pitch)));
        const HalfSweepKeys K = half_sweep_keys(P.key0, P.key1, P.t, P.colour + 4u * (uint32_t)z);
        const RowKeys R = row_keys(K, (uint32_t)y);
        const uint32_t own[4] = {own4.x, own4.y, own4.z, own4.w};
        const uint32_t mid[6] = {adj, mid4.x, mid4.y, mid4.z, mid4.w, adj};
        const uint32_t up[4] = {up4.x, up4.y, up4.z, up4.w}, dn[4] = {dn4.x, dn4.y, dn4.z, dn4.w};
        const uint32_t lo[4] = {lo4.x, lo4.y, lo4.z, lo4.w}, hi[4] = {hi4.x, hi4.y, hi4.z, hi4.w};
        uint32_t out[4];
#pragma unroll
        for (int n = 0; n < 4; ++n) {
            uint32_t nb[6];
            horizontal(p, mid[n + 1], p ? mid[n + 2] : mid[n], nb[0], nb[1]);
            nb[2] = up[n]; nb[3] = dn[n]; nb[4] = lo[n]; nb[5] = hi[n];
            uint32_t w0[4], w1[4];
#pragma unroll
            for (int b = 0; b < 4; ++b) philox_site(K, R, 2u * (uint32_t)(k0 + 4 * n + b) + p, w0[b], w1[b]);
            const uint32_t s01 = __byte_perm(__umulhi(w0[0], q), __umulhi(w0[1], q), 0x0040);
            const uint32_t s23 = __byte_perm(__umulhi(w0[2], q), __umulhi(w0[3], q), 0x0040);
            const uint32_t prop = __byte_perm(s01, s23, 0x5410);                       // R4
            uint32_t c_old, c_new;
            ne_counts6<CM>(own[n], prop, nb, c_old, c_new);                            // R5'
            const uint32_t dw8 = (c_new + 0x06060606u - c_old) << 3;                   // byte b = 8 (d + 6): table offsets
            uint32_t a[4];
#pragma unroll
            for (int b = 0; b < 4; ++b) {                                              // R6': high word of w1 + (2^64 - threshold)
                const unsigned long long e = *reinterpret_cast<const unsigned long long *>(
                    reinterpret_cast<const char *>(lut) + ((dw8 >> (8 * b)) & 0xffu));
                a[b] = (uint32_t)((e + (unsigned long long)w1[b]) >> 32);
            }
            const uint32_t m01 = lop3<LOP_SEL>(a[0], a[1], 0x000000ffu), m23 = lop3<LOP_SEL>(a[2], a[3], 0x00ffffffu);
            out[n] = lop3<LOP_SEL>(prop, own[n], lop3<LOP_SEL>(m01, m23, 0x0000ffffu));   // R7
        }
        *reinterpret_cast<uint4 *>(P.plane_own + r_mid + k0) = make_uint4(out[0], out[1], out[2], out[3]);
    }
}

// ---------------------------------------------------------------------------------------------
// Row-walking form (the 2D streaming kernel k_sweep_rows_u8 carried to three dimensions).  A block of H3_WARPS
// warps owns a tile of one z.  A lane updates 4 W same-colour sites per row visit and walks down a window of rpw rows
// at fixed z: the other-colour rows y-1, y, y+1 of plane z roll through registers (one load per visit), the rows
// (z-1, y) and (z+1, y) are two more loads.  A row narrower than a warp of such lanes (L < 256 W) takes 2^lpr_log2
// lanes, and the 32 >> lpr_log2 lane groups of the warp walk different windows of the same columns, so that no lane
// idles down to L = 32 W.  Every window starts at a row of parity (z & 1): the first visit of every tile has row
// parity COLOUR and the parities are literals as in 2D.  ColKeys depend on z through
// xb = (colour + 4 z) ^ key1: the table of the tile's columns is rebuilt whenever (column block, z) changes; tiles
// are numbered (cb, z, row group) so that a block draws the row groups of one z in a row.
//
// Compare: the six "differs" flag words of a 4-site word are added bit-sliced by a carry-save tree of three-input
// logic ops (8 for six neighbours) into the bit planes ones / twos / fours; code byte = c_old in bits 0-2 and c_new
// in bits 4-6 (bits 3, 7 are garbage and masked out of the table offset).  Accept table: AcceptLut indexed by that
// code, entry = 2^64 - threshold(c_new - c_old) (FAST: threshold - 1), as in 2D.
constexpr int H3_WARPS = 4;
constexpr uint32_t CODE3_BITS = 0x77u;

struct Sweep3RowsParams {
    uint8_t *plane_own;
    const uint8_t *plane_oth;
    int32_t L, pitch;
    uint32_t q, key1;             // xb(z) = (colour + 4 z) ^ key1
    HalfSweepKeys K;              // of (seed, t): xb is redone per z
    uint32_t thr[6];              // threshold(d) for d = 1..6 (R6')
    int32_t rpw, row_groups;      // rows per window; tiles per (column block, z)
    int32_t lpr_log2;             // log2 of the lanes that cover a row (5 if the row is a warp wide or wider)
    uint32_t total_tiles;
    uint32_t *tile_counter;
};

__host__ __device__ inline bool accept_fast_ok3(const uint32_t thr[6]) { return thr[0] && thr[1] && thr[2] && thr[3] && thr[4] && thr[5]; }

template <int SLOTS>
__device__ __forceinline__ void accept_lut_fill3(AcceptLutT<SLOTS> *lut, const uint32_t thr[6], uint32_t tid, uint32_t nthreads, bool fast)
{
    for (uint32_t n = tid; n < (uint32_t)(128 * SLOTS); n += nthreads) {
        const uint32_t code = n / SLOTS;
        const int c_old = (int)(code & 7u), c_new = (int)((code >> 4) & 7u);
        const int d = c_new - c_old > 6 ? 6 : c_new - c_old;          // counts of 7 never occur
        const unsigned long long th = d <= 0 ? (1ull << 32) : (unsigned long long)thr[d - 1];
        const unsigned long long e = fast ? th - 1ull : 0ull - th;
        (&lut->e[0][0])[n] = make_uint2((uint32_t)e, (uint32_t)(e >> 32));
    }
}

// carry-save count of six flag words: bit planes of the per-position sum (0..6)
__device__ __forceinline__ void csa6(const uint32_t u[6], uint32_t &ones, uint32_t &twos, uint32_t &fours)
{
    constexpr int XOR3 = 0x96, MAJ = 0xE8;
    const uint32_t s1 = lop3<XOR3>(u[0], u[1], u[2]), c1 = lop3<MAJ>(u[0], u[1], u[2]);
    const uint32_t s2 = lop3<XOR3>(u[3], u[4], u[5]), c2 = lop3<MAJ>(u[3], u[4], u[5]);
    ones = s1 ^ s2;
    const uint32_t c3 = s1 & s2;
    twos = lop3<XOR3>(c1, c2, c3);
    fours = lop3<MAJ>(c1, c2, c3);
}

// code byte per site: bits 0-2 = neighbours that differ from the current spin, bits 4-6 = from the proposal
template <int CM>
__device__ __forceinline__ uint32_t ne_code6(uint32_t own, uint32_t prop, const uint32_t nb[6])
{
    if (is_nibble_mode(CM)) {
        const uint32_t both = prop * 16u + own;
        uint32_t u[6];
#pragma unroll
        for (int k = 0; k < 6; ++k) {
            if (CM == CM_NIB3) u[k] = (both ^ nb[k]) + 0x77777777u;
            else u[k] = lop3<LOP_OR_XOR>(lop3<LOP_XOR_AND>(both, nb[k], 0x77777777u) + 0x77777777u, both, nb[k]);
        }
        uint32_t ones, twos, fours;                                    // flags in bits 3 and 7 of every byte
        csa6(u, ones, twos, fours);
        const uint32_t c = lop3<LOP_SEL>(ones >> 3, twos >> 2, 0x11111111u);
        return lop3<LOP_SEL>(c, fours >> 1, 0x33333333u);
    } else {
        uint32_t o[6], n[6];
#pragma unroll
        for (int k = 0; k < 6; ++k) {
            if (CM == CM_7BIT) {
                o[k] = (own ^ nb[k]) + 0x7f7f7f7fu;
                n[k] = (prop ^ nb[k]) + 0x7f7f7f7fu;
            } else {
                o[k] = lop3<LOP_OR_XOR>(lop3<LOP_XOR_AND>(own, nb[k], 0x7f7f7f7fu) + 0x7f7f7f7fu, own, nb[k]);
                n[k] = lop3<LOP_OR_XOR>(lop3<LOP_XOR_AND>(prop, nb[k], 0x7f7f7f7fu) + 0x7f7f7f7fu, prop, nb[k]);
            }
        }
        uint32_t o1, o2, o4, n1, n2, n4;                               // flags in bit 7 of every byte
        csa6(o, o1, o2, o4);
        csa6(n, n1, n2, n4);
        uint32_t a = lop3<LOP_SEL>(o1 >> 7, o2 >> 6, 0x01010101u);
        a = lop3<LOP_SEL>(a, o4 >> 5, 0x03030303u);
        uint32_t b = lop3<LOP_SEL>(n1 >> 3, n2 >> 2, 0x10101010u);
        b = lop3<LOP_SEL>(b, n4 >> 1, 0x30303030u);
        return lop3<LOP_SEL>(a, b, 0x0f0f0f0fu);
    }
}

template <int W> struct Words3 { uint32_t w[W]; };

template <int W>
__device__ __forceinline__ Words3<W> ld_words3(const uint8_t *p)
{
    Words3<W> r;
    if constexpr (W == 4) { const uint4 v = *reinterpret_cast<const uint4 *>(p); r.w[0] = v.x; r.w[1] = v.y; r.w[2] = v.z; r.w[3] = v.w; }
    else if constexpr (W == 2) { const uint2 v = *reinterpret_cast<const uint2 *>(p); r.w[0] = v.x; r.w[1] = v.y; }
    else r.w[0] = *reinterpret_cast<const uint32_t *>(p);
    return r;
}

template <int W>
__device__ __forceinline__ void st_words3(uint8_t *p, const uint32_t (&o)[W])
{
    if constexpr (W == 4) *reinterpret_cast<uint4 *>(p) = make_uint4(o[0], o[1], o[2], o[3]);
    else if constexpr (W == 2) *reinterpret_cast<uint2 *>(p) = make_uint2(o[0], o[1]);
    else *reinterpret_cast<uint32_t *>(p) = o[0];
}

template <int CM, int COLOUR, int W, bool FAST>
__global__ void __launch_bounds__(32 * H3_WARPS) k_sweep3_rows_u8(const __grid_constant__ Sweep3RowsParams P)
{
    constexpr int SITES = 4 * W;                                      // same-colour sites per lane and row
    __shared__ uint4 s_col[2][SITES][32];                             // ColKeys of [row parity][site of the chunk][lane]
    __shared__ AcceptLut lut;
    __shared__ uint32_t s_tile[2];
    const uint32_t lane = threadIdx.x, wy = threadIdx.y, tid = wy * 32u + lane;
    accept_lut_fill3(&lut, P.thr, tid, 32 * H3_WARPS, FAST);
    const HalfSweepKeys &K = P.K;
    const uint32_t lane_off = accept_lane_offset(lane);
    const uint32_t q = in_register(P.q);
    const int L = P.L, pitch = P.pitch, chunks = pitch / SITES;
    const size_t plane_z = (size_t)L * pitch;                         // bytes of one z of a colour plane
    int key_cur = -1;
    for (uint32_t it = 0;; ++it) {
    if (tid == 0) s_tile[it & 1u] = atomicInc(P.tile_counter, P.total_tiles + gridDim.x - 1u);
    __syncthreads();                                                  // also: every thread is done with the previous tile
    const uint32_t tile = s_tile[it & 1u];
    if (tile >= P.total_tiles) break;
    const int cz = (int)(tile / (uint32_t)P.row_groups), rg = (int)(tile - (uint32_t)cz * (uint32_t)P.row_groups);
    const int cb = cz / L, z = cz - cb * L;
    const int xl = (int)lane & ((1 << P.lpr_log2) - 1), sub = (int)lane >> P.lpr_log2;   // lane of the row, window of the warp
    const int x = cb * 32 + xl;
    const int win = ((rg * H3_WARPS + (int)wy) << (5 - P.lpr_log2)) + sub;                 // window of the plane
    const bool active = x < chunks && win * P.rpw < L;
    const int k0 = x * SITES;
    if (cz != key_cur) {
        key_cur = cz;
        if (x < chunks && sub == 0) {
            const uint32_t xb = ((uint32_t)COLOUR + 4u * (uint32_t)z) ^ P.key1;
            for (int n = (int)wy; n < SITES; n += H3_WARPS) {
#pragma unroll
                for (int p = 0; p < 2; ++p) {
                    const ColKeys C = col_keys(xb, K.xc, 2u * (uint32_t)(k0 + n) + (uint32_t)p);
                    s_col[p][n][xl] = make_uint4(C.l0, C.l1, C.ph, C.pl);
                }
            }
        }
        __syncthreads();
    }

    if (active) {
        const int ys = win * P.rpw + (z & 1);                         // first row of the window: parity of visit r is (r + COLOUR) & 1
        const uint8_t *const oth_z = P.plane_oth + (size_t)z * plane_z + k0;
        const uint8_t *const oth_lo = P.plane_oth + (size_t)wrap(z - 1, L) * plane_z + k0;
        const uint8_t *const oth_hi = P.plane_oth + (size_t)wrap(z + 1, L) * plane_z + k0;
        uint8_t *const own_z = P.plane_own + (size_t)z * plane_z + k0;
        const int kn = wrap(k0 + SITES, pitch) - k0, kp = wrap(k0 - 4, pitch) - k0;
        struct Loads { Words3<W> own, dn, lo, hi; uint32_t adj; };
        auto load_row = [&](int y, int kadj) {
            const size_t r = (size_t)wrap(y, L) * pitch;
            Loads l;
            l.own = ld_words3<W>(own_z + r);
            l.dn = ld_words3<W>(oth_z + (size_t)wrap(wrap(y, L) + 1, L) * pitch);
            l.lo = ld_words3<W>(oth_lo + r);
            l.hi = ld_words3<W>(oth_hi + r);
            l.adj = *reinterpret_cast<const uint32_t *>(oth_z + (ptrdiff_t)r + kadj);
            return l;
        };
        auto prep = [](const Words3<W> &v, uint32_t (&w)[W]) {
#pragma unroll
            for (int n = 0; n < W; ++n) w[n] = prep_nbr<CM>(v.w[n]);
        };
        auto visit = [&](auto par, int y, const Loads &ld, const uint32_t (&up)[W], const uint32_t (&mid)[W], const uint32_t (&dn)[W]) {
            constexpr int PAR = decltype(par)::value;
            const int yw = wrap(y, L);
            const RowKeysH R = row_keys_h(K, (uint32_t)yw);
            const uint32_t adjp = prep_nbr<CM>(ld.adj);
            uint32_t lo[W], hi[W], out[W];
            prep(ld.lo, lo);
            prep(ld.hi, hi);
#pragma unroll
            for (int n = 0; n < W; ++n) {
                uint32_t nb[6];
                nb[0] = up[n];
                nb[1] = dn[n];
                if (PAR) {
                    nb[2] = mid[n];
                    nb[3] = __funnelshift_r(mid[n], n < W - 1 ? mid[n < W - 1 ? n + 1 : W - 1] : adjp, 8);
                } else {
                    nb[2] = __funnelshift_l(n > 0 ? mid[n > 0 ? n - 1 : 0] : adjp, mid[n], 8);
                    nb[3] = mid[n];
                }
                nb[4] = lo[n];
                nb[5] = hi[n];
                uint32_t w0[4], w1[4];
#pragma unroll
                for (int b = 0; b < 4; ++b) {
                    const uint4 c = s_col[PAR][4 * n + b][xl];
                    philox_site_h(K, R, ColKeys{c.x, c.y, c.z, c.w}, w0[b], w1[b]);
                }
                const uint32_t s01 = __byte_perm(__umulhi(w0[0], q), __umulhi(w0[1], q), 0x0040);
                const uint32_t s23 = __byte_perm(__umulhi(w0[2], q), __umulhi(w0[3], q), 0x0040);
                const uint32_t prop = __byte_perm(s01, s23, 0x5410);                       // R4
                const uint32_t code = ne_code6<CM>(ld.own.w[n], prop, nb);                 // R5'
                if (FAST) out[n] = accept_insert<8, CODE3_BITS>(ld.own.w[n], prop, code, w1, &lut, lane_off);   // R6', R7
                else out[n] = lop3<LOP_SEL>(prop, ld.own.w[n], accept_mask<8, CODE3_BITS>(code, w1, &lut, lane_off));
            }
            st_words3<W>(own_z + (size_t)yw * pitch, out);
        };

        uint32_t up[W], mid[W], dn[W], dn2[W];
        prep(ld_words3<W>(oth_z + (size_t)wrap(ys - 1, L) * pitch), up);
        prep(ld_words3<W>(oth_z + (size_t)wrap(ys, L) * pitch), mid);
        constexpr int PA = COLOUR, PB = 1 - COLOUR;
        const int k_a = PA ? kn : kp, k_b = PB ? kn : kp;
        Loads a = load_row(ys, k_a);
#pragma unroll 1
        for (int r = 0; r < P.rpw; r += 2) {
            const int y = ys + r;
            const Loads b = load_row(y + 1, k_b);
            prep(a.dn, dn);
            visit(std::integral_constant<int, PA>{}, y, a, up, mid, dn);
            a = load_row(r + 2 < P.rpw ? y + 2 : y + 1, k_a);
            prep(b.dn, dn2);
            visit(std::integral_constant<int, PB>{}, y + 1, b, mid, dn, dn2);
#pragma unroll
            for (int n = 0; n < W; ++n) { up[n] = dn[n]; mid[n] = dn2[n]; }
        }
    }
    }   // tiles
}

// Energy (from the colour-1 sites: every bond joins the two colours) and histogram of both planes.
struct Measure3Params {
    const uint8_t *plane0, *plane1;
    int32_t L, pitch;
    uint32_t q;
    unsigned long long *E_out, *hist_out;      // either may be null
};

template <bool WIDE>
__global__ void __launch_bounds__(256) k_measure3_u8(const Measure3Params P)
{
    extern __shared__ uint32_t s_hist[];
    __shared__ unsigned long long blockE;
    const bool do_hist = P.hist_out != nullptr;
    if (do_hist)
        for (uint32_t n = threadIdx.x; n < hist_words(P.q); n += blockDim.x) s_hist[n] = 0;
    if (threadIdx.x == 0) blockE = 0ull;
    __syncthreads();
    const int L = P.L, pitch = P.pitch, cpr = pitch >> 4;
    const long long total = (long long)L * L * cpr;
    uint32_t satisfied = 0;
    for (long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x; gid < total; gid += (long long)gridDim.x * blockDim.x) {
        const int cx = (int)(gid % cpr);
        const long long row = gid / cpr;
        const int y = (int)(row % L), z = (int)(row / L), k0 = cx << 4;
        const uint32_t p = (uint32_t)(z + y + 1) & 1u;
        const size_t r_mid = ((size_t)z * L + y) * pitch;
        const uint4 own4 = *reinterpret_cast<const uint4 *>(P.plane1 + r_mid + k0);
        const uint4 mid4 = *reinterpret_cast<const uint4 *>(P.plane0 + r_mid + k0);
        const uint32_t own[4] = {own4.x, own4.y, own4.z, own4.w};
        if (P.E_out) {
            const uint4 up4 = *reinterpret_cast<const uint4 *>(P.plane0 + ((size_t)z * L + wrap(y - 1, L)) * pitch + k0);
            const uint4 dn4 = *reinterpret_cast<const uint4 *>(P.plane0 + ((size_t)z * L + wrap(y + 1, L)) * pitch + k0);
            const uint4 lo4 = *reinterpret_cast<const uint4 *>(P.plane0 + ((size_t)wrap(z - 1, L) * L + y) * pitch + k0);
            const uint4 hi4 = *reinterpret_cast<const uint4 *>(P.plane0 + ((size_t)wrap(z + 1, L) * L + y) * pitch + k0);
            const uint32_t adj = *reinterpret_cast<const uint32_t *>(P.plane0 + r_mid + (p ? wrap(k0 + 16, pitch) : wrap(k0 - 4, pitch)));
            const uint32_t mid[6] = {adj, mid4.x, mid4.y, mid4.z, mid4.w, adj};
            const uint32_t up[4] = {up4.x, up4.y, up4.z, up4.w}, dn[4] = {dn4.x, dn4.y, dn4.z, dn4.w};
            const uint32_t lo[4] = {lo4.x, lo4.y, lo4.z, lo4.w}, hi[4] = {hi4.x, hi4.y, hi4.z, hi4.w};
            uint32_t nef = 0;
#pragma unroll
            for (int n = 0; n < 4; ++n) {
                uint32_t lf, rt;
                horizontal(p, mid[n + 1], p ? mid[n + 2] : mid[n], lf, rt);
                nef += ne_count4<WIDE>(own[n], up[n], dn[n], lf, rt) + (ne_flags<WIDE>(own[n], lo[n]) >> 7) + (ne_flags<WIDE>(own[n], hi[n]) >> 7);
            }
            satisfied += 96u - byte_sum(nef);                             // 16 sites x 6 neighbours - unequal ones
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

// Random start (R9'): s(x,y,z) = floor(w0 q / 2^32), (w0,..) = Philox((x, y, 0, 2 + 4 z), seed).  One thread per word.
static __global__ void k_init_random3_u8(uint8_t *plane0, uint8_t *plane1, int L, int pitch, uint32_t q, uint32_t key0, uint32_t key1)
{
    const long long words_per_plane = (long long)L * L * (pitch >> 2);
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (gid >= 2 * words_per_plane) return;
    const int c = gid >= words_per_plane;
    const long long r = gid - (long long)c * words_per_plane;
    const int kw = (int)(r % (pitch >> 2));
    const long long row = r / (pitch >> 2);
    const int y = (int)(row % L), z = (int)(row / L);
    const uint32_t p = (uint32_t)(z + y + c) & 1u;
    uint32_t word = 0;
#pragma unroll
    for (int b = 0; b < 4; ++b) {
        uint32_t ctr[4] = {2u * (uint32_t)(4 * kw + b) + p, (uint32_t)y, 0u, 2u + 4u * (uint32_t)z};
        philox4x32_10(ctr, key0, key1);
        word |= __umulhi(ctr[0], q) << (8 * b);
    }
    *reinterpret_cast<uint32_t *>((c ? plane1 : plane0) + (size_t)row * pitch + 4 * kw) = word;
}

// planes <-> canonical s[(z L + y) L + x] for `rows` rows (row = z L + y) starting at row0; one thread per 4 sites of a plane row
static __global__ void k_planes_to_rowmajor3(const uint8_t *plane0, const uint8_t *plane1, uint8_t *out, int L, int pitch, long long row0, int rows)
{
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const int wpr = pitch >> 2;
    if (gid >= (long long)rows * wpr) return;
    const int r = (int)(gid / wpr), kw = (int)(gid - (long long)r * wpr);
    const long long row = row0 + r;
    const int y = (int)(row % L), z = (int)(row / L);
    const uint32_t a = *reinterpret_cast<const uint32_t *>(plane0 + (size_t)row * pitch + 4 * kw);
    const uint32_t b = *reinterpret_cast<const uint32_t *>(plane1 + (size_t)row * pitch + 4 * kw);
    const bool odd = ((z + y) & 1) != 0;                              // colour 0 holds the even columns iff z + y is even
    const uint32_t ev = odd ? b : a, od = odd ? a : b;
    uint2 o;
    o.x = __byte_perm(ev, od, 0x5140);
    o.y = __byte_perm(ev, od, 0x7362);
    *reinterpret_cast<uint2 *>(out + (size_t)r * L + 8 * kw) = o;
}

static __global__ void k_rowmajor_to_planes3(const uint8_t *in, uint8_t *plane0, uint8_t *plane1, int L, int pitch, long long row0, int rows,
                                             uint32_t q, int *bad)
{
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const int wpr = pitch >> 2;
    if (gid >= (long long)rows * wpr) return;
    const int r = (int)(gid / wpr), kw = (int)(gid - (long long)r * wpr);
    const long long row = row0 + r;
    const int y = (int)(row % L), z = (int)(row / L);
    const uint2 v = *reinterpret_cast<const uint2 *>(in + (size_t)r * L + 8 * kw);
    const uint32_t ev = __byte_perm(v.x, v.y, 0x6420), od = __byte_perm(v.x, v.y, 0x7531);
    if (q < 256) {
        bool b = false;
#pragma unroll
        for (int n = 0; n < 4; ++n) b |= ((ev >> (8 * n)) & 0xffu) >= q || ((od >> (8 * n)) & 0xffu) >= q;
        if (b) atomicExch(bad, 1);
    }
    const bool odd = ((z + y) & 1) != 0;
    *reinterpret_cast<uint32_t *>((odd ? plane1 : plane0) + (size_t)row * pitch + 4 * kw) = ev;
    *reinterpret_cast<uint32_t *>((odd ? plane0 : plane1) + (size_t)row * pitch + 4 * kw) = od;
}

}  // namespace potts
