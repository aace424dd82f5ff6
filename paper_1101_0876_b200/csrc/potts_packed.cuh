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
    int32_t rpt;                 // rows per thread
};

constexpr int PK_WARPS = 4;

// Half-sweep, packed layout: a thread updates 32 consecutive same-colour sites of P.rpt consecutive rows.
// grid = (ceil(L/64 / 32), L / (PK_WARPS * rpt)), block = (32, PK_WARPS).
// DELTA (potts_sweep_delta; see k_half_sweep_delta_u8): instead of the energy, add the sum of the
// accepted moves' d = n_old - n_new of this half-sweep to *P.E_out (two's-complement int64).
template <bool FIVE, int ST, bool MEASURE, bool HIST, bool DELTA = false>
__global__ void __launch_bounds__(32 * PK_WARPS) k_half_sweep_packed(const __grid_constant__ PackedSweepParams P)
{
    constexpr bool EX = MEASURE || DELTA;
    constexpr int CM = FIVE ? CM_7BIT : CM_NIB4;
    extern __shared__ uint32_t s_dyn[];
    __shared__ AcceptLut lut;
    __shared__ int blockAcc;
    const uint32_t tid = threadIdx.y * 32u + threadIdx.x;
    accept_lut_fill(&lut, P.thr, tid, 32 * PK_WARPS);
    if (EX && tid == 0) blockAcc = 0;
    if (HIST)
        for (uint32_t n = tid; n < hist_words(P.q); n += 32 * PK_WARPS) s_dyn[n] = 0u;
    __syncthreads();

    const PackedPlanes &S = P.S;
    const int chunks = S.L >> 6;                                       // 32-site chunks per plane row
    const int x = (int)(blockIdx.x * 32u + threadIdx.x);
    const int i0 = (int)(blockIdx.y * PK_WARPS + threadIdx.y) * P.rpt;
    const int c = (int)P.colour, o = 1 - c;
    int acc = 0, rows_done = 0;
    if (x < chunks) {
        const uint32_t lane_off = accept_lane_offset(threadIdx.x);
        const HalfSweepKeys &K = P.K;
        const uint32_t q = in_register(P.q);
        const int xn = x + 1 == chunks ? 0 : x + 1, xp = x == 0 ? chunks - 1 : x - 1;
#pragma unroll 1
        for (int r = 0; r < P.rpt; ++r) {
            const int i = i0 + r;
            const uint32_t p = (uint32_t)(i + c) & 1u;
            const int iu = wrap(i - 1, S.L), id = wrap(i + 1, S.L);
            const uint4 own_n = *reinterpret_cast<const uint4 *>(S.nib[c] + (size_t)i * S.pn + 16 * x);
            const uint4 up_n = *reinterpret_cast<const uint4 *>(S.nib[o] + (size_t)iu * S.pn + 16 * x);
            const uint4 dn_n = *reinterpret_cast<const uint4 *>(S.nib[o] + (size_t)id * S.pn + 16 * x);
            uint32_t own_h = 0, up_h = 0, dn_h = 0;
            if (FIVE) {
                own_h = *reinterpret_cast<const uint32_t *>(S.hb[c] + (size_t)i * S.ph + 4 * x);
                up_h = *reinterpret_cast<const uint32_t *>(S.hb[o] + (size_t)iu * S.ph + 4 * x);
                dn_h = *reinterpret_cast<const uint32_t *>(S.hb[o] + (size_t)id * S.ph + 4 * x);
            }
            // other-colour sites of my row: mid[1..8] = my 32 columns, mid[0] / mid[9] = the word before / after
            uint32_t mid[10];
            load32<FIVE>(S, o, i, x, mid + 1);
            {
                // p = 1 needs site 32 (first site of the next chunk), p = 0 site -1 (last site of the previous one)
                const int xa = p ? xn : xp;
                const uint32_t an = *reinterpret_cast<const uint32_t *>(S.nib[o] + (size_t)i * S.pn + 16 * xa + (p ? 0 : 12));
                const uint32_t ah = FIVE ? *reinterpret_cast<const uint32_t *>(S.hb[o] + (size_t)i * S.ph + 4 * xa) : 0u;
                uint32_t lo, hi;
                unpack_pair<FIVE>(an, ah, p ? 0 : 3, lo, hi);
                mid[0] = hi;     // used when p = 0: sites -4..-1
                mid[9] = lo;     // used when p = 1: sites 32..35
            }
            const RowKeys R = row_keys(K, (uint32_t)i);
            const uint32_t own_w[4] = {own_n.x, own_n.y, own_n.z, own_n.w};
            const uint32_t up_w[4] = {up_n.x, up_n.y, up_n.z, up_n.w};
            const uint32_t dn_w[4] = {dn_n.x, dn_n.y, dn_n.z, dn_n.w};
            uint32_t out_w[4], out_h = 0;
#pragma unroll
            for (int m = 0; m < 4; ++m) {
                uint32_t own[2], up[2], dn[2], out[2];
                unpack_pair<FIVE>(own_w[m], own_h, m, own[0], own[1]);
                unpack_pair<FIVE>(up_w[m], up_h, m, up[0], up[1]);
                unpack_pair<FIVE>(dn_w[m], dn_h, m, dn[0], dn[1]);
#pragma unroll
                for (int hlf = 0; hlf < 2; ++hlf) {
                    const int n = 2 * m + hlf;                        // byte-per-site word n: sites 4n..4n+3
                    uint32_t lf, rt, w0[4], w1[4];
                    horizontal(p, mid[n + 1], p ? mid[n + 2] : mid[n], lf, rt);
                    draw_words<ST>(K, R, 2u * (uint32_t)(32 * x + 4 * n) + p, w0, w1);
                    const uint32_t nb[4] = {prep_nbr<CM>(up[hlf]), prep_nbr<CM>(dn[hlf]), prep_nbr<CM>(lf), prep_nbr<CM>(rt)};
                    uint32_t code, mask;
                    out[hlf] = metropolis_word<CM>(own[hlf], nb, q, w0, w1, &lut, lane_off, code, mask);
                    if (MEASURE) acc += ne_final_sum(code, mask);
                    if (DELTA) acc += delta_sum(code, mask);
                    if (HIST) hist_add_word(s_dyn, P.q, out[hlf], threadIdx.x);
                }
                out_w[m] = pack_pair<FIVE>(out[0], out[1], m, out_h);
            }
            *reinterpret_cast<uint4 *>(S.nib[c] + (size_t)i * S.pn + 16 * x) = make_uint4(out_w[0], out_w[1], out_w[2], out_w[3]);
            if (FIVE) *reinterpret_cast<uint32_t *>(S.hb[c] + (size_t)i * S.ph + 4 * x) = out_h;
            ++rows_done;
        }
    }
    if (EX) {
        // MEASURE: satisfied bonds = 4 per site - unequal neighbours of the final spins; DELTA: the change
        int v = DELTA ? acc : 128 * rows_done - acc;
#pragma unroll
        for (int s = 16; s > 0; s >>= 1) v += __shfl_xor_sync(0xffffffffu, v, s);
        if (threadIdx.x == 0) atomicAdd(&blockAcc, v);
        __syncthreads();
        if (tid == 0) atomicAdd(P.E_out, DELTA ? (unsigned long long)(long long)blockAcc : 0ull - (unsigned long long)(long long)blockAcc);
    }
    if (HIST) {
        __syncthreads();
        hist_flush(s_dyn, P.q, P.hist_out, tid, 32 * PK_WARPS);
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
#pragma unroll
        for (int s = 16; s > 0; s >>= 1) satisfied += __shfl_xor_sync(0xffffffffu, satisfied, s);
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
