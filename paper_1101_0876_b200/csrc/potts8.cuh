// potts8.cuh -- the 2D generalisation with first AND second neighbour interactions ("there are nine
// independent sub-networks to update instead of two"; reading S17).  First CUDA path of this row of
// one launch per sub-network, one 4-site word per thread.
//
// Cell packing: nine planes plane[c][I][J], c = 3 (i mod 3) + (j mod 3), I = i / 3, J = j / 3, one byte per spin,
// row pitch L/3 bytes.  The neighbour (i + di, j + dj) of a site of sub-network (a, b) lies in plane
// ((a + di) mod 3, (b + dj) mod 3), at row I + (-1, 0 or +1) and at column J + (-1, 0 or +1): which of the three is
// the same for every site of the sub-network, so the host passes one descriptor per direction and a word's four
// neighbours in a direction are one word of that plane, shifted by at most one byte (funnel shift with the word beside).
// Random stream: Philox4x32-10(counter = (j, i, t, 16 + c), key = seed): the 2D keys with "colour" := 16 + c.
#pragma once
#include "potts_core.cuh"

namespace potts {

struct Nbr8 {
    int32_t plane;      // sub-network of the neighbour
    int32_t dI;         // its row is I + dI (periodic in L/3)
    int32_t shift;      // its column is J + shift
};

struct Sweep8Params {
    uint8_t *planes;              // nine planes, plane_bytes apart
    unsigned long long plane_bytes;
    int32_t L, pitch, rows;       // pitch = rows = L/3
    uint32_t q, c;                // sub-network being updated
    uint32_t key0, key1, t;
    Nbr8 nbr[8];
    unsigned long long neg_thr[17];   // 2^64 - threshold(d), d = -8..8: index d + 8
};

// word at columns 4 w + shift .. + 3 of a plane row (wpr words, periodic)
__device__ __forceinline__ uint32_t load_shifted(const uint8_t *row, int w, int shift, int wpr)
{
    const uint32_t *r = reinterpret_cast<const uint32_t *>(row);
    const uint32_t w0 = r[w];
    if (shift == 0) return w0;
    if (shift > 0) return __funnelshift_r(w0, r[w + 1 == wpr ? 0 : w + 1], 8);
    return __funnelshift_l(r[w == 0 ? wpr - 1 : w - 1], w0, 8);
}

template <int CM>
__device__ __forceinline__ void ne_counts8(uint32_t own, uint32_t prop, const uint32_t nb[8], uint32_t &c_old, uint32_t &c_new)
{
    if (is_nibble_mode(CM)) {
        const uint32_t both = prop * 16u + own;
        uint32_t s = 0;
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            const uint32_t n2 = nb[k] * 0x11u;
            uint32_t u;
            if (CM == CM_NIB3) u = (both ^ n2) + 0x77777777u;
            else u = lop3<LOP_OR_XOR>(lop3<LOP_XOR_AND>(both, n2, 0x77777777u) + 0x77777777u, both, n2);
            s += (u >> 3) & 0x11111111u;                              // nibble counters: at most 8
        }
        c_old = s & 0x0f0f0f0fu;
        c_new = (s >> 4) & 0x0f0f0f0fu;
    } else {
        c_old = c_new = 0;
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            c_old += ne_flags<CM == CM_8BIT>(own, nb[k]) >> 7;
            c_new += ne_flags<CM == CM_8BIT>(prop, nb[k]) >> 7;
        }
    }
}

// Update of sub-network P.c.  One thread per 4-site word of its plane; grid-stride.
template <int CM>
__global__ void __launch_bounds__(128) k_sweep8_u8(const __grid_constant__ Sweep8Params P)
{
    __shared__ unsigned long long lut[20];
    if (threadIdx.x < 17) lut[threadIdx.x] = P.neg_thr[threadIdx.x];
    __syncthreads();
    const int wpr = P.pitch >> 2, rows = P.rows;
    const long long total = (long long)rows * wpr;
    const uint32_t q = in_register(P.q);
    const uint32_t a = P.c / 3u, b = P.c % 3u;
    const HalfSweepKeys K = half_sweep_keys(P.key0, P.key1, P.t, 16u + P.c);
    uint8_t *const own_plane = P.planes + P.c * P.plane_bytes;
    for (long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x; gid < total; gid += (long long)gridDim.x * blockDim.x) {
        const int I = (int)(gid / wpr), w = (int)(gid - (long long)I * wpr);
        const uint32_t own = *reinterpret_cast<const uint32_t *>(own_plane + (size_t)I * P.pitch + 4 * w);
        uint32_t nb[8];
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            const int In = wrap(I + P.nbr[k].dI, rows);
            nb[k] = load_shifted(P.planes + P.nbr[k].plane * P.plane_bytes + (size_t)In * P.pitch, w, P.nbr[k].shift, wpr);
        }
        const RowKeys R = row_keys(K, 3u * (uint32_t)I + a);
        uint32_t w0[4], w1[4];
#pragma unroll
        for (int s = 0; s < 4; ++s) philox_site(K, R, 3u * (uint32_t)(4 * w + s) + b, w0[s], w1[s]);
        const uint32_t s01 = __byte_perm(__umulhi(w0[0], q), __umulhi(w0[1], q), 0x0040);
        const uint32_t s23 = __byte_perm(__umulhi(w0[2], q), __umulhi(w0[3], q), 0x0040);
        const uint32_t prop = __byte_perm(s01, s23, 0x5410);                           // R4
        uint32_t c_old, c_new;
        ne_counts8<CM>(own, prop, nb, c_old, c_new);                                   // R5"
        const uint32_t dw8 = (c_new + 0x08080808u - c_old) << 3;                       // byte = 8 (d + 8): table offsets
        uint32_t acc[4];
#pragma unroll
        for (int s = 0; s < 4; ++s) {                                                  // R6"
            const unsigned long long e = *reinterpret_cast<const unsigned long long *>(reinterpret_cast<const char *>(lut) + ((dw8 >> (8 * s)) & 0xffu));
            acc[s] = (uint32_t)((e + (unsigned long long)w1[s]) >> 32);
        }
        const uint32_t m01 = lop3<LOP_SEL>(acc[0], acc[1], 0x000000ffu), m23 = lop3<LOP_SEL>(acc[2], acc[3], 0x00ffffffu);
        *reinterpret_cast<uint32_t *>(own_plane + (size_t)I * P.pitch + 4 * w) = lop3<LOP_SEL>(prop, own, lop3<LOP_SEL>(m01, m23, 0x0000ffffu));   // R7
    }
}

// ---------------------------------------------------------------------------------------------
// Row-walking form.  A lane updates 16 sites (one 16-byte chunk of a plane row, columns J = k0..k0+15) per row visit
// and walks a window of rpw rows; a block of H8_WARPS warps owns a tile of 32 chunks x its windows (rows narrower than
// a warp: 2^lpr_log2 lanes per row and several windows per warp, as in k_sweep3_rows_u8); tiles are drawn from a
// counter.  What walking buys here is not load reuse (the eight neighbours of consecutive rows lie in eight different
// (plane, row) pairs) but everything per column and per visit: the ColKeys of the tile's columns j = 3 J + b (the
// column part of Philox, shared by all rows) sit in shared memory, the row keys, addresses and neighbour preparation
// are paid once per 16 sites.  B = c mod 3 is a template argument: the column shift of every direction is a literal.
// Compare: the eight flag words are added bit-sliced by a carry-save tree (14 three-input logic ops) into the planes
// ones / twos / fours / eights; code byte = c_old in bits 0-3, c_new in bits 4-7, index of the 2D accept table filled
// with threshold(c_new - c_old).  Needs pitch % 16 == 0 (L % 48 == 0).
constexpr int H8_WARPS = 4;

struct Sweep8RowsParams {
    uint8_t *planes;
    unsigned long long plane_bytes;
    int32_t pitch, rows;          // both L/3
    uint32_t q, c;
    HalfSweepKeys K;              // of (seed, t, 16 + c)
    Nbr8 nbr[8];                  // directions in the order (di, dj) = (0,1) (1,0) (1,1) (1,-1) (0,-1) (-1,0) (-1,-1) (-1,1)
    uint32_t thr[8];              // threshold(d), d = 1..8 (R6")
    int32_t rpw, row_groups, lpr_log2;
    uint32_t total_tiles;
    uint32_t *tile_counter;
};

__host__ __device__ constexpr int dir8_dj(int k) { return (k == 0 || k == 2 || k == 7) ? 1 : ((k == 1 || k == 5) ? 0 : -1); }
// column shift of direction k for the sites of column residue b (Nbr8::shift, as a literal)
__host__ __device__ constexpr int dir8_shift(int b, int k) { return (b == 0 && dir8_dj(k) < 0) ? -1 : ((b == 2 && dir8_dj(k) > 0) ? 1 : 0); }

__host__ __device__ inline bool accept_fast_ok8(const uint32_t thr[8])
{
    bool ok = true;
    for (int d = 0; d < 8; ++d) ok = ok && thr[d] != 0u;
    return ok;
}

template <int SLOTS>
__device__ __forceinline__ void accept_lut_fill8(AcceptLutT<SLOTS> *lut, const uint32_t thr[8], uint32_t tid, uint32_t nthreads, bool fast)
{
    for (uint32_t n = tid; n < (uint32_t)(ACCEPT_ENTRIES * SLOTS); n += nthreads) {
        const uint32_t code = n / SLOTS;
        int d = (int)(code >> 4) - (int)(code & 15u);
        d = d > 8 ? 8 : d;                                             // counts above 8 never occur
        const unsigned long long th = d <= 0 ? (1ull << 32) : (unsigned long long)thr[d - 1];
        const unsigned long long e = fast ? th - 1ull : 0ull - th;
        (&lut->e[0][0])[n] = make_uint2((uint32_t)e, (uint32_t)(e >> 32));
    }
}

// carry-save count of eight flag words: bit planes of the per-position sum (0..8)
__device__ __forceinline__ void csa8(const uint32_t u[8], uint32_t &ones, uint32_t &twos, uint32_t &fours, uint32_t &eights)
{
    constexpr int XOR3 = 0x96, MAJ = 0xE8;
    const uint32_t s1 = lop3<XOR3>(u[0], u[1], u[2]), c1 = lop3<MAJ>(u[0], u[1], u[2]);
    const uint32_t s2 = lop3<XOR3>(u[3], u[4], u[5]), c2 = lop3<MAJ>(u[3], u[4], u[5]);
    const uint32_t s3 = lop3<XOR3>(s1, s2, u[6]), c3 = lop3<MAJ>(s1, s2, u[6]);
    ones = s3 ^ u[7];
    const uint32_t c4 = s3 & u[7];
    const uint32_t t1 = lop3<XOR3>(c1, c2, c3), d1 = lop3<MAJ>(c1, c2, c3);
    twos = t1 ^ c4;
    const uint32_t d2 = t1 & c4;
    fours = d1 ^ d2;
    eights = d1 & d2;
}

template <int CM>
__device__ __forceinline__ uint32_t ne_code8(uint32_t own, uint32_t prop, const uint32_t nb[8])
{
    if (is_nibble_mode(CM)) {
        const uint32_t both = prop * 16u + own;
        uint32_t u[8];
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            if (CM == CM_NIB3) u[k] = (both ^ nb[k]) + 0x77777777u;
            else u[k] = lop3<LOP_OR_XOR>(lop3<LOP_XOR_AND>(both, nb[k], 0x77777777u) + 0x77777777u, both, nb[k]);
        }
        uint32_t c1, c2, c4, c8;                                       // flags in bits 3 and 7 of every byte
        csa8(u, c1, c2, c4, c8);
        uint32_t c = lop3<LOP_SEL>(c1 >> 3, c2 >> 2, 0x11111111u);
        c = lop3<LOP_SEL>(c, c4 >> 1, 0x33333333u);
        return lop3<LOP_SEL>(c, c8, 0x77777777u);
    } else {
        uint32_t o[8], n[8];
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            if (CM == CM_7BIT) {
                o[k] = (own ^ nb[k]) + 0x7f7f7f7fu;
                n[k] = (prop ^ nb[k]) + 0x7f7f7f7fu;
            } else {
                o[k] = lop3<LOP_OR_XOR>(lop3<LOP_XOR_AND>(own, nb[k], 0x7f7f7f7fu) + 0x7f7f7f7fu, own, nb[k]);
                n[k] = lop3<LOP_OR_XOR>(lop3<LOP_XOR_AND>(prop, nb[k], 0x7f7f7f7fu) + 0x7f7f7f7fu, prop, nb[k]);
            }
        }
        uint32_t o1, o2, o4, o8, n1, n2, n4, n8;                       // flags in bit 7 of every byte
        csa8(o, o1, o2, o4, o8);
        csa8(n, n1, n2, n4, n8);
        uint32_t a = lop3<LOP_SEL>(o1 >> 7, o2 >> 6, 0x01010101u);
        a = lop3<LOP_SEL>(a, o4 >> 5, 0x03030303u);
        a = lop3<LOP_SEL>(a, o8 >> 4, 0x07070707u);
        uint32_t b = lop3<LOP_SEL>(n1 >> 3, n2 >> 2, 0x10101010u);
        b = lop3<LOP_SEL>(b, n4 >> 1, 0x30303030u);
        b = lop3<LOP_SEL>(b, n8, 0x70707070u);
        return lop3<LOP_SEL>(a, b, 0x0f0f0f0fu);
    }
}

template <int CM, int B, bool FAST>
__global__ void __launch_bounds__(32 * H8_WARPS, 5) k_sweep8_rows_u8(const __grid_constant__ Sweep8RowsParams P)
{
    __shared__ uint4 s_col[16][32];                                   // ColKeys of [site of the chunk][lane of the row]
    __shared__ AcceptLut lut;
    __shared__ uint32_t s_tile[2];
    const uint32_t lane = threadIdx.x, wy = threadIdx.y, tid = wy * 32u + lane;
    accept_lut_fill8(&lut, P.thr, tid, 32 * H8_WARPS, FAST);
    const HalfSweepKeys &K = P.K;
    const uint32_t lane_off = accept_lane_offset(lane);
    const uint32_t q = in_register(P.q);
    const int pitch = P.pitch, rows = P.rows, chunks = pitch >> 4;
    const uint32_t a = P.c / 3u;
    uint8_t *const own_plane = P.planes + P.c * P.plane_bytes;
    int cb_cur = -1;
    for (uint32_t it = 0;; ++it) {
    if (tid == 0) s_tile[it & 1u] = atomicInc(P.tile_counter, P.total_tiles + gridDim.x - 1u);
    __syncthreads();                                                  // also: every thread is done with the previous tile
    const uint32_t tile = s_tile[it & 1u];
    if (tile >= P.total_tiles) break;
    const int cb = (int)(tile / (uint32_t)P.row_groups), rg = (int)(tile - (uint32_t)cb * (uint32_t)P.row_groups);
    const int xl = (int)lane & ((1 << P.lpr_log2) - 1), sub = (int)lane >> P.lpr_log2;
    const int x = cb * 32 + xl;
    const int win = ((rg * H8_WARPS + (int)wy) << (5 - P.lpr_log2)) + sub;
    const bool active = x < chunks && win * P.rpw < rows;
    const int k0 = x << 4;
    if (cb != cb_cur) {
        cb_cur = cb;
        if (x < chunks && sub == 0)
            for (int n = (int)wy; n < 16; n += H8_WARPS) {
                const ColKeys C = col_keys(K, 3u * (uint32_t)(k0 + n) + (uint32_t)B);
                s_col[n][xl] = make_uint4(C.l0, C.l1, C.ph, C.pl);
            }
        __syncthreads();
    }
    if (active) {
        const int kn = wrap(k0 + 16, pitch) - k0, kp = wrap(k0 - 4, pitch) - k0;
        const int I0 = win * P.rpw;
#pragma unroll 1
        for (int r = 0; r < P.rpw; ++r) {
            const int I = I0 + r;
            // the ColKeys of the lane's columns do not depend on the row: without this the compiler hoists the 16
            // loads out of the row loop and spills the 64 registers they need
            int xc = xl;
            asm volatile("" : "+r"(xc));
            // byte offsets of rows I-1, I, I+1 inside a plane (32 bit: nine planes stay below 4 GB)
            const uint32_t r_0 = (uint32_t)(I * pitch + k0), r_m = (uint32_t)(wrap(I - 1, rows) * pitch + k0), r_p = (uint32_t)(wrap(I + 1, rows) * pitch + k0);
            const uint4 own4 = *reinterpret_cast<const uint4 *>(own_plane + r_0);
            uint32_t nbw[8][4];
#pragma unroll
            for (int k = 0; k < 8; ++k) {
                const int dI = P.nbr[k].dI;
                const uint32_t ro = dI == 0 ? r_0 : (dI < 0 ? r_m : r_p);
                const uint8_t *rowp = P.planes + ((uint32_t)P.nbr[k].plane * (uint32_t)P.plane_bytes + ro);
                const uint4 v = *reinterpret_cast<const uint4 *>(rowp);
                const int sh = dir8_shift(B, k);
                if (sh > 0) {
                    const uint32_t adj = *reinterpret_cast<const uint32_t *>(rowp + kn);
                    nbw[k][0] = __funnelshift_r(v.x, v.y, 8); nbw[k][1] = __funnelshift_r(v.y, v.z, 8);
                    nbw[k][2] = __funnelshift_r(v.z, v.w, 8); nbw[k][3] = __funnelshift_r(v.w, adj, 8);
                } else if (sh < 0) {
                    const uint32_t adj = *reinterpret_cast<const uint32_t *>(rowp + kp);
                    nbw[k][0] = __funnelshift_l(adj, v.x, 8); nbw[k][1] = __funnelshift_l(v.x, v.y, 8);
                    nbw[k][2] = __funnelshift_l(v.y, v.z, 8); nbw[k][3] = __funnelshift_l(v.z, v.w, 8);
                } else {
                    nbw[k][0] = v.x; nbw[k][1] = v.y; nbw[k][2] = v.z; nbw[k][3] = v.w;
                }
#pragma unroll
                for (int n = 0; n < 4; ++n) nbw[k][n] = prep_nbr<CM>(nbw[k][n]);
            }
            const RowKeysH R = row_keys_h(K, 3u * (uint32_t)I + a);
            const uint32_t own[4] = {own4.x, own4.y, own4.z, own4.w};
            uint32_t out[4];
#pragma unroll
            for (int n = 0; n < 4; ++n) {
                uint32_t nb[8];
#pragma unroll
                for (int k = 0; k < 8; ++k) nb[k] = nbw[k][n];
                uint32_t w0[4], w1[4];
#pragma unroll
                for (int b = 0; b < 4; ++b) {
                    const uint4 c = s_col[4 * n + b][xc];
                    philox_site_h(K, R, ColKeys{c.x, c.y, c.z, c.w}, w0[b], w1[b]);
                }
                const uint32_t s01 = __byte_perm(__umulhi(w0[0], q), __umulhi(w0[1], q), 0x0040);
                const uint32_t s23 = __byte_perm(__umulhi(w0[2], q), __umulhi(w0[3], q), 0x0040);
                const uint32_t prop = __byte_perm(s01, s23, 0x5410);                       // R4
                const uint32_t code = ne_code8<CM>(own[n], prop, nb);                      // R5"
                if (FAST) out[n] = accept_insert(own[n], prop, code, w1, &lut, lane_off);  // R6", R7
                else out[n] = lop3<LOP_SEL>(prop, own[n], accept_mask(code, w1, &lut, lane_off));
            }
            *reinterpret_cast<uint4 *>(own_plane + r_0) = make_uint4(out[0], out[1], out[2], out[3]);
        }
    }
    }   // tiles
}

// Energy: for every word of sub-network P.c the equal neighbours in the four FORWARD directions (0,1), (1,0), (1,1),
// (1,-1) (descriptors nbr[0..3]), so that every bond is counted once over the nine launches; histogram of the plane.
template <bool WIDE>
__global__ void __launch_bounds__(256) k_measure8_u8(const Sweep8Params P, unsigned long long *E_out, unsigned long long *hist_out)
{
    extern __shared__ uint32_t s_hist[];
    __shared__ unsigned long long blockE;
    const bool do_hist = hist_out != nullptr;
    if (do_hist)
        for (uint32_t n = threadIdx.x; n < hist_words(P.q); n += blockDim.x) s_hist[n] = 0;
    if (threadIdx.x == 0) blockE = 0ull;
    __syncthreads();
    const int wpr = P.pitch >> 2, rows = P.rows;
    const long long total = (long long)rows * wpr;
    const uint8_t *const own_plane = P.planes + P.c * P.plane_bytes;
    uint32_t satisfied = 0;
    for (long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x; gid < total; gid += (long long)gridDim.x * blockDim.x) {
        const int I = (int)(gid / wpr), w = (int)(gid - (long long)I * wpr);
        const uint32_t own = *reinterpret_cast<const uint32_t *>(own_plane + (size_t)I * P.pitch + 4 * w);
        if (E_out) {
            uint32_t nef = 0;
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const int In = wrap(I + P.nbr[k].dI, rows);
                const uint32_t nb = load_shifted(P.planes + P.nbr[k].plane * P.plane_bytes + (size_t)In * P.pitch, w, P.nbr[k].shift, wpr);
                nef += ne_flags<WIDE>(own, nb) >> 7;
            }
            satisfied += 16u - byte_sum(nef);
        }
        if (do_hist) hist_add_word(s_hist, P.q, own, threadIdx.x & 31u);
    }
    if (E_out) {
        satisfied = __reduce_add_sync(0xffffffffu, satisfied);                     // one REDUX instead of a five-step shuffle tree
        if ((threadIdx.x & 31) == 0) atomicAdd(&blockE, (unsigned long long)satisfied);
    }
    __syncthreads();
    if (E_out && threadIdx.x == 0) atomicAdd(E_out, 0ull - blockE);
    if (do_hist) hist_flush(s_hist, P.q, hist_out, threadIdx.x, blockDim.x);
}

// Random start (R9, the 2D rule): s(i,j) = floor(w0 q / 2^32), Philox((j, i, 0, 2), seed).  One thread per site.
static __global__ void k_init_random8_u8(uint8_t *planes, unsigned long long plane_bytes, int L, int pitch, uint32_t q, uint32_t key0, uint32_t key1)
{
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (gid >= (long long)L * L) return;
    const int i = (int)(gid / L), j = (int)(gid - (long long)i * L);
    uint32_t ctr[4] = {(uint32_t)j, (uint32_t)i, 0u, 2u};
    philox4x32_10(ctr, key0, key1);
    planes[(size_t)(3 * (i % 3) + (j % 3)) * plane_bytes + (size_t)(i / 3) * pitch + (j / 3)] = (uint8_t)__umulhi(ctr[0], q);
}

// planes <-> canonical row-major s[i L + j]; one thread per site (not on the timed path)
static __global__ void k_planes_to_rowmajor8(const uint8_t *planes, unsigned long long plane_bytes, uint8_t *out, int L, int pitch)
{
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (gid >= (long long)L * L) return;
    const int i = (int)(gid / L), j = (int)(gid - (long long)i * L);
    out[gid] = planes[(size_t)(3 * (i % 3) + (j % 3)) * plane_bytes + (size_t)(i / 3) * pitch + (j / 3)];
}

static __global__ void k_rowmajor_to_planes8(const uint8_t *in, uint8_t *planes, unsigned long long plane_bytes, int L, int pitch, uint32_t q, int *bad)
{
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (gid >= (long long)L * L) return;
    const int i = (int)(gid / L), j = (int)(gid - (long long)i * L);
    const uint8_t v = in[gid];
    if (v >= q) atomicExch(bad, 1);
    planes[(size_t)(3 * (i % 3) + (j % 3)) * plane_bytes + (size_t)(i / 3) * pitch + (j / 3)] = v;
}

}  // namespace potts
