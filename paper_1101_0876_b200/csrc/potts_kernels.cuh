// potts_kernels.cuh -- device code of the checkerboard Potts sweep for sm_100a.
//
// Everything on the device is integer arithmetic: Philox4x32-10 keyed by
// (seed; j, i, t, colour), multiply-high proposal, byte-parallel neighbour comparison, integer
// threshold acceptance (PAPER.md:94 sec. 3, :145 sec. 3.2), and integer energy / histogram
// reductions (sec. 3.4).  Not shared with oracle/ in any way.
//
// Spin layout "U8 split planes" (PAPER.md:159 packs whites then blacks; the exact map is ours):
//   plane[c][i][k], c = (i+j)&1, k = j>>1, one byte per spin, row pitch L/2 bytes.
// A colour-c site (i,k) with p = (i+c)&1 sits at column j = 2k+p; its neighbours are all in
// plane 1-c:  up [i-1][k], down [i+1][k], and horizontally [i][k],[i][k+1] if p = 1 or
// [i][k-1],[i][k] if p = 0 (indices periodic).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace potts {

constexpr uint32_t PHILOX_M0 = 0xD2511F53u;
constexpr uint32_t PHILOX_M1 = 0xCD9E8D57u;
constexpr uint32_t PHILOX_W0 = 0x9E3779B9u;
constexpr uint32_t PHILOX_W1 = 0xBB67AE85u;

struct SweepParams {
    uint8_t *plane_own;         // plane of the colour being updated
    const uint8_t *plane_oth;   // plane of the other colour
    int32_t L;                  // lattice size
    int32_t pitch;              // L/2, bytes per plane row
    uint32_t q;
    uint32_t colour;            // 0 = white ((i+j) even), 1 = black
    uint32_t t;                 // sweep counter (Philox counter word 2)
    uint32_t key0, key1;        // seed low / high
    uint32_t thr[4];            // floor(2^32 exp(-d/T)), d = 1..4
    unsigned long long *E_out;  // MEASURE: -= satisfied bonds seen from this colour's sites
};

// ---------------------------------------------------------------------------------------------
// Philox4x32-10, words 0 and 1 only (the update rule uses w0 for the proposal and w1 for the
// acceptance).  The last round therefore needs only the M1*c2 product.
__device__ __forceinline__ void philox4x32_10_w01(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                                  uint32_t k0, uint32_t k1, uint32_t &w0, uint32_t &w1)
{
#pragma unroll
    for (int r = 0; r < 9; ++r) {
        const uint32_t hi0 = __umulhi(PHILOX_M0, c0), lo0 = PHILOX_M0 * c0;
        const uint32_t hi1 = __umulhi(PHILOX_M1, c2), lo1 = PHILOX_M1 * c2;
        c0 = hi1 ^ c1 ^ k0;
        c1 = lo1;
        c2 = hi0 ^ c3 ^ k1;
        c3 = lo0;
        k0 += PHILOX_W0;
        k1 += PHILOX_W1;
    }
    w0 = __umulhi(PHILOX_M1, c2) ^ c1 ^ k0;
    w1 = PHILOX_M1 * c2;
}

// full 4-word version (init kernel, tests)
__device__ __forceinline__ void philox4x32_10(uint32_t c[4], uint32_t k0, uint32_t k1)
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t hi0 = __umulhi(PHILOX_M0, c[0]), lo0 = PHILOX_M0 * c[0];
        const uint32_t hi1 = __umulhi(PHILOX_M1, c[2]), lo1 = PHILOX_M1 * c[2];
        c[0] = hi1 ^ c[1] ^ k0;
        c[1] = lo1;
        c[2] = hi0 ^ c[3] ^ k1;
        c[3] = lo0;
        k0 += PHILOX_W0;
        k1 += PHILOX_W1;
    }
}

// ---------------------------------------------------------------------------------------------
// Byte-parallel "not equal" flags: bit 7 of every byte of the result is set iff the bytes of a
// and b differ.  WIDE = false assumes all spin values < 128 (q <= 128), so a^b has bit 7 clear
// in every byte and adding 0x7f cannot carry across bytes.
template <bool WIDE>
__device__ __forceinline__ uint32_t ne_flags(uint32_t a, uint32_t b)
{
    const uint32_t x = a ^ b;
    if (!WIDE) return (x + 0x7f7f7f7fu) & 0x80808080u;
    return (((x & 0x7f7f7f7fu) + 0x7f7f7f7fu) | x) & 0x80808080u;
}

// per-byte count (0..4) of neighbours that differ from the bytes of s
template <bool WIDE>
__device__ __forceinline__ uint32_t ne_count4(uint32_t s, uint32_t up, uint32_t dn, uint32_t lf, uint32_t rt)
{
    return (ne_flags<WIDE>(s, up) >> 7) + (ne_flags<WIDE>(s, dn) >> 7) +
           (ne_flags<WIDE>(s, lf) >> 7) + (ne_flags<WIDE>(s, rt) >> 7);
}

__device__ __forceinline__ uint32_t byte_sum(uint32_t v)   // sum of the 4 bytes (each <= 63)
{
    return (v * 0x01010101u) >> 24;
}

__device__ __forceinline__ int wrap(int x, int n) { return x < 0 ? x + n : (x >= n ? x - n : x); }

// ---------------------------------------------------------------------------------------------
// One word (4 same-colour sites, consecutive k) of the Metropolis update.
//   own      current spins of the 4 sites
//   up,dn,lf,rt  the 4 neighbour words, byte b = that neighbour of site b
//   j0       column of byte 0 (columns advance by 2 per byte), i = row
// Returns the new word; *ne_final receives the per-byte count of unequal neighbours of the
// final spins (for the fused energy).
template <bool WIDE>
__device__ __forceinline__ uint32_t update_word(uint32_t own, uint32_t up, uint32_t dn, uint32_t lf,
                                                uint32_t rt, uint32_t j0, uint32_t i,
                                                const SweepParams &P, const uint32_t *lut,
                                                uint32_t *ne_final)
{
    uint32_t w0[4], w1[4];
#pragma unroll
    for (int b = 0; b < 4; ++b)
        philox4x32_10_w01(j0 + 2u * b, i, P.t, P.colour, P.key0, P.key1, w0[b], w1[b]);
    uint32_t prop = 0;
#pragma unroll
    for (int b = 0; b < 4; ++b) prop |= __umulhi(w0[b], P.q) << (8 * b);

    const uint32_t c_old = ne_count4<WIDE>(own, up, dn, lf, rt);
    const uint32_t c_new = ne_count4<WIDE>(prop, up, dn, lf, rt);
    // d = n_old - n_new = ne_new - ne_old; biased by 4 per byte so that bytes stay in 0..8
    const uint32_t dw = c_new + 0x04040404u - c_old;
    uint32_t mask = 0;
#pragma unroll
    for (int b = 0; b < 4; ++b) {
        const uint32_t dd = (dw >> (8 * b)) & 0xffu;       // d + 4
        const bool acc = (dd <= 4u) || (w1[b] < lut[dd]);
        mask |= acc ? (0xffu << (8 * b)) : 0u;
    }
    *ne_final = (c_new & mask) | (c_old & ~mask);
    return (prop & mask) | (own & ~mask);
}

// ---------------------------------------------------------------------------------------------
// Half-sweep, U8 layout, one thread per 16 consecutive same-colour sites of one row.
// Requires L % 32 == 0.  grid = ceil(L * (L/32) / blockDim).
template <bool WIDE, bool MEASURE>
__global__ void __launch_bounds__(128) k_half_sweep_u8(const SweepParams P)
{
    __shared__ uint32_t lut[16];
    __shared__ unsigned long long blockE;
    if (threadIdx.x < 16) {
        const int dd = threadIdx.x;
        lut[dd] = (dd >= 5 && dd <= 8) ? P.thr[dd - 5] : 0xFFFFFFFFu;
    }
    if (MEASURE && threadIdx.x == 0) blockE = 0ull;
    __syncthreads();

    const int chunks = P.pitch >> 4;                                  // 16-byte chunks per row
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long total = (long long)P.L * chunks;
    uint32_t satisfied = 0;
    if (gid < total) {
        const int i = (int)(gid / chunks);
        const int x = (int)(gid - (long long)i * chunks);
        const int k0 = x << 4;
        const uint32_t p = (uint32_t)(i + P.colour) & 1u;
        const int iu = wrap(i - 1, P.L), id = wrap(i + 1, P.L);
        const size_t row = (size_t)i * P.pitch;

        const uint4 own4 = *reinterpret_cast<const uint4 *>(P.plane_own + row + k0);
        const uint4 mid4 = *reinterpret_cast<const uint4 *>(P.plane_oth + row + k0);
        const uint4 up4 = *reinterpret_cast<const uint4 *>(P.plane_oth + (size_t)iu * P.pitch + k0);
        const uint4 dn4 = *reinterpret_cast<const uint4 *>(P.plane_oth + (size_t)id * P.pitch + k0);
        // the one byte outside the chunk: [i][k0+16] if p = 1, [i][k0-1] if p = 0 (periodic)
        const int ka = p ? wrap(k0 + 16, P.pitch) : wrap(k0 - 1, P.pitch);
        const uint32_t adj = P.plane_oth[row + ka];

        const uint32_t own[4] = {own4.x, own4.y, own4.z, own4.w};
        const uint32_t mid[4] = {mid4.x, mid4.y, mid4.z, mid4.w};
        const uint32_t up[4] = {up4.x, up4.y, up4.z, up4.w};
        const uint32_t dn[4] = {dn4.x, dn4.y, dn4.z, dn4.w};
        uint32_t out[4];
#pragma unroll
        for (int n = 0; n < 4; ++n) {
            uint32_t lf, rt;
            if (p) {   // neighbours at k and k+1
                lf = mid[n];
                const uint32_t nxt = (n < 3) ? mid[n < 3 ? n + 1 : 3] : adj;
                rt = __funnelshift_r(mid[n], nxt, 8);
            } else {   // neighbours at k-1 and k
                const uint32_t prv = (n > 0) ? mid[n > 0 ? n - 1 : 0] : (adj << 24);
                lf = __funnelshift_l(prv, mid[n], 8);
                rt = mid[n];
            }
            uint32_t nef;
            out[n] = update_word<WIDE>(own[n], up[n], dn[n], lf, rt, 2u * (uint32_t)(k0 + 4 * n) + p,
                                       (uint32_t)i, P, lut, &nef);
            if (MEASURE) satisfied += 16u - byte_sum(nef);
        }
        *reinterpret_cast<uint4 *>(P.plane_own + row + k0) = make_uint4(out[0], out[1], out[2], out[3]);
    }
    if (MEASURE) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) satisfied += __shfl_xor_sync(0xffffffffu, satisfied, o);
        if ((threadIdx.x & 31) == 0) atomicAdd(&blockE, (unsigned long long)satisfied);
        __syncthreads();
        // E = -(satisfied bonds): accumulate the two's-complement negative into the int64 slot
        if (threadIdx.x == 0) atomicAdd(P.E_out, 0ull - blockE);
    }
}

// ---------------------------------------------------------------------------------------------
// Standalone measurement: energy from the black plane's sites (every bond joins a black and a
// white site, so summing equal neighbours over black sites counts each bond once) and the
// histogram of both planes.  One thread per 16-byte chunk of the black plane; the white chunk
// at the same (row, k-range) is the thread's "mid" word, so every white site is counted once.
struct MeasureParams {
    const uint8_t *plane0, *plane1;
    int32_t L, pitch;
    uint32_t q;
    unsigned long long *E_out;      // may be null
    unsigned long long *hist_out;   // q entries, may be null
};

template <bool WIDE>
__global__ void __launch_bounds__(256) k_measure_u8(const MeasureParams P)
{
    extern __shared__ uint32_t s_hist[];            // [warps][q]
    __shared__ unsigned long long blockE;
    const int warps = blockDim.x >> 5, warp = threadIdx.x >> 5;
    const bool do_hist = P.hist_out != nullptr;
    if (do_hist)
        for (int n = threadIdx.x; n < warps * (int)P.q; n += blockDim.x) s_hist[n] = 0;
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
        const uint32_t p = (uint32_t)(i + 1) & 1u;                   // colour 1 sites
        const int iu = wrap(i - 1, P.L), id = wrap(i + 1, P.L);
        const size_t row = (size_t)i * P.pitch;
        const uint4 own4 = *reinterpret_cast<const uint4 *>(P.plane1 + row + k0);
        const uint4 mid4 = *reinterpret_cast<const uint4 *>(P.plane0 + row + k0);
        const uint32_t own[4] = {own4.x, own4.y, own4.z, own4.w};
        const uint32_t mid[4] = {mid4.x, mid4.y, mid4.z, mid4.w};
        if (P.E_out) {
            const uint4 up4 = *reinterpret_cast<const uint4 *>(P.plane0 + (size_t)iu * P.pitch + k0);
            const uint4 dn4 = *reinterpret_cast<const uint4 *>(P.plane0 + (size_t)id * P.pitch + k0);
            const int ka = p ? wrap(k0 + 16, P.pitch) : wrap(k0 - 1, P.pitch);
            const uint32_t adj = P.plane0[row + ka];
            const uint32_t up[4] = {up4.x, up4.y, up4.z, up4.w};
            const uint32_t dn[4] = {dn4.x, dn4.y, dn4.z, dn4.w};
#pragma unroll
            for (int n = 0; n < 4; ++n) {
                uint32_t lf, rt;
                if (p) {
                    lf = mid[n];
                    const uint32_t nxt = (n < 3) ? mid[n < 3 ? n + 1 : 3] : adj;
                    rt = __funnelshift_r(mid[n], nxt, 8);
                } else {
                    const uint32_t prv = (n > 0) ? mid[n > 0 ? n - 1 : 0] : (adj << 24);
                    lf = __funnelshift_l(prv, mid[n], 8);
                    rt = mid[n];
                }
                satisfied += 16u - byte_sum(ne_count4<WIDE>(own[n], up[n], dn[n], lf, rt));
            }
        }
        if (do_hist) {
            uint32_t *h = s_hist + warp * P.q;
#pragma unroll
            for (int n = 0; n < 4; ++n)
#pragma unroll
                for (int b = 0; b < 4; ++b) {
                    atomicAdd(&h[(own[n] >> (8 * b)) & 0xffu], 1u);
                    atomicAdd(&h[(mid[n] >> (8 * b)) & 0xffu], 1u);
                }
        }
    }
    if (P.E_out) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) satisfied += __shfl_xor_sync(0xffffffffu, satisfied, o);
        if ((threadIdx.x & 31) == 0) atomicAdd(&blockE, (unsigned long long)satisfied);
    }
    __syncthreads();
    if (P.E_out && threadIdx.x == 0) atomicAdd(P.E_out, 0ull - blockE);
    if (do_hist)
        for (int b = threadIdx.x; b < (int)P.q; b += blockDim.x) {
            unsigned long long tot = 0;
            for (int w = 0; w < warps; ++w) tot += s_hist[w * P.q + b];
            if (tot) atomicAdd(&P.hist_out[b], tot);
        }
}

// ---------------------------------------------------------------------------------------------
// Random start (R9): s(i,j) = floor(w0 q / 2^32), (w0,..) = Philox((j, i, 0, 2), seed).
// One thread per 4 consecutive k of one plane row.
__global__ void k_init_random_u8(uint8_t *plane0, uint8_t *plane1, int L, int pitch, uint32_t q,
                                 uint32_t key0, uint32_t key1)
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
        uint32_t ctr[4] = {2u * (uint32_t)(4 * kw + b) + p, (uint32_t)i, 0u, 2u};
        philox4x32_10(ctr, key0, key1);
        word |= __umulhi(ctr[0], q) << (8 * b);
    }
    uint8_t *plane = c ? plane1 : plane0;
    *reinterpret_cast<uint32_t *>(plane + (size_t)i * pitch + 4 * kw) = word;
}

// ---------------------------------------------------------------------------------------------
// Layout conversion: split planes <-> canonical row-major s[i*L + j], for `rows` rows starting
// at row i0.  One thread per 4 sites of a plane row (= 8 columns of the lattice row).
__global__ void k_planes_to_rowmajor(const uint8_t *plane0, const uint8_t *plane1, uint8_t *out,
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

__global__ void k_rowmajor_to_planes(const uint8_t *in, uint8_t *plane0, uint8_t *plane1, int L,
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
