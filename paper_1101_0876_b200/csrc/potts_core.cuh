// potts_core.cuh -- per-site arithmetic of the checkerboard Potts sweep for sm_100a.
//
// Everything on the device is integer arithmetic: Philox4x32-10 keyed by
// (seed; j, i, t, colour), multiply-high proposal, byte-parallel neighbour comparison and integer
// threshold acceptance (PAPER.md:94 sec. 3, :145 sec. 3.2).  Not shared with oracle/ in any way.
//
// Cost model this file is written against (profiles/r01b_pipe_model.md, measured on B200): for this
// integer mix an SM sub-partition retires one warp instruction every 2 clocks whichever pipe it goes to
// (IMAD.WIDE, IMAD, LOP3, IADD3, SHF, PRMT alike; IMAD.HI and POPC take 4), so the time of an update is
// its instruction count.  One update needs 17 IMAD.WIDE + 18 LOP3 of Philox (fixed by the stream
// definition) + 1 multiply for the proposal; everything else (neighbour compare, acceptance, packing,
// loads and stores: ~22 instructions per update at 16 sites per thread) is overhead to keep small.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace potts {

constexpr uint32_t PHILOX_M0 = 0xD2511F53u;
constexpr uint32_t PHILOX_M1 = 0xCD9E8D57u;
constexpr uint32_t PHILOX_W0 = 0x9E3779B9u;
constexpr uint32_t PHILOX_W1 = 0xBB67AE85u;

__device__ __forceinline__ void mul_wide(uint32_t a, uint32_t b, uint32_t &hi, uint32_t &lo)
{
    // one IMAD.WIDE; written in PTX so that the compiler does not split it into IMAD.HI + IMAD
    // (twice the issue cost) where only part of the product looks live
    unsigned long long p;
    asm("mul.wide.u32 %0, %1, %2;" : "=l"(p) : "r"(a), "r"(b));
    asm("mov.b64 {%0, %1}, %2;" : "=r"(lo), "=r"(hi) : "l"(p));
}

// Copy of a kernel-uniform value held in an ordinary register.  Multiplies cannot take a uniform-
// register operand, and the compiler otherwise re-materialises the copy (one more instruction)
// before every use.
__device__ __forceinline__ uint32_t in_register(uint32_t v)
{
    uint32_t r;
    asm volatile("mov.u32 %0, %1;" : "=r"(r) : "r"(v));
    return r;
}

// full 4-word Philox4x32-10 (random start, R9)
__device__ __forceinline__ void philox4x32_10(uint32_t c[4], uint32_t k0, uint32_t k1)
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        uint32_t hi0, lo0, hi1, lo1;
        mul_wide(PHILOX_M0, c[0], hi0, lo0);
        mul_wide(PHILOX_M1, c[2], hi1, lo1);
        c[0] = hi1 ^ c[1] ^ k0;
        c[1] = lo1;
        c[2] = hi0 ^ c[3] ^ k1;
        c[3] = lo0;
        k0 += PHILOX_W0;
        k1 += PHILOX_W1;
    }
}

// ---------------------------------------------------------------------------------------------
// Philox4x32-10 of counter (j, i, t, colour), words w0 and w1 only, split by what each part
// depends on so that nothing is computed twice:
//   HalfSweepKeys  depends on (seed, t, colour)   -- uniform over a half-sweep
//   RowKeys        adds the row i                 -- one wide multiply per thread and row
//   philox_site    adds the column j              -- 17 wide multiplies + 18 three-input XORs
// Round 1 multiplies the counter words c0 = j and c2 = t; round 2 multiplies c0' = hi(M1 t)^i^k0,
// which does not depend on j.
struct HalfSweepKeys {
    uint32_t xa;      // hi(M1*t) ^ k0[0]          c0 after round 1 is xa ^ i
    uint32_t xb;      // colour ^ k1[0]            c2 after round 1 is hi(M0*j) ^ xb
    uint32_t xc;      // lo(M1*t) ^ k0[1]          c0 after round 2 is hi(M1*c2') ^ xc
    uint32_t k0, k1;  // the key itself (round r uses k + r*W)
};

// Host and device: the streaming kernels get the keys as launch parameters (if every thread derived
// xb from two uniform operands the compiler would fold the XOR into each use and re-copy a uniform
// register for every site); the resident kernel unrolls the colour loop, so there the colour is a
// literal and the keys stay in uniform registers.
__host__ __device__ inline HalfSweepKeys half_sweep_keys(uint32_t key0, uint32_t key1, uint32_t t, uint32_t colour)
{
    HalfSweepKeys K;
    const unsigned long long p = (unsigned long long)PHILOX_M1 * (unsigned long long)t;
    const uint32_t hi = (uint32_t)(p >> 32), lo = (uint32_t)p;
    K.xa = hi ^ key0;
    K.xb = colour ^ key1;
    K.xc = lo ^ (key0 + PHILOX_W0);
    K.k0 = key0;
    K.k1 = key1;
    return K;
}

struct RowKeys {
    uint32_t xd;      // hi(M0*(xa^i)) ^ k1[1]     c2 after round 2 is lo(M0*j) ^ xd
    uint32_t c3;      // lo(M0*(xa^i))             c3 after round 2
};

__device__ __forceinline__ RowKeys row_keys(const HalfSweepKeys &K, uint32_t i)
{
    RowKeys R;
    uint32_t hi;
    mul_wide(PHILOX_M0, K.xa ^ i, hi, R.c3);
    R.xd = hi ^ (K.k1 + PHILOX_W1);
    return R;
}

__device__ __forceinline__ void philox_site(const HalfSweepKeys &K, const RowKeys &R, uint32_t j,
                                            uint32_t &w0, uint32_t &w1)
{
    uint32_t h0, l0, h1, l1;
    mul_wide(PHILOX_M0, j, h0, l0);                  // round 1, the M0*c0 product
    mul_wide(PHILOX_M1, h0 ^ K.xb, h1, l1);          // round 2, the M1*c2 product
    uint32_t c0 = h1 ^ K.xc, c1 = l1, c2 = l0 ^ R.xd, c3 = R.c3;
    uint32_t k0 = K.k0 + 2u * PHILOX_W0, k1 = K.k1 + 2u * PHILOX_W1;
#pragma unroll
    for (int r = 2; r < 9; ++r) {
        mul_wide(PHILOX_M0, c0, h0, l0);
        mul_wide(PHILOX_M1, c2, h1, l1);
        c0 = h1 ^ c1 ^ k0;
        c1 = l1;
        c2 = h0 ^ c3 ^ k1;
        c3 = l0;
        k0 += PHILOX_W0;
        k1 += PHILOX_W1;
    }
    mul_wide(PHILOX_M1, c2, h1, l1);                 // round 10: only words 0 and 1 are used
    w0 = h1 ^ c1 ^ k0;
    w1 = l1;
}

// Stream-spec v2 (reading S15): all four words of the block of counter (j, i, t, colour); the pair of
// same-colour sites (j, j+2) shares it.  18 wide multiplies + 18 XORs per pair: half of v1's work per site.
__device__ __forceinline__ void philox_pair(const HalfSweepKeys &K, const RowKeys &R, uint32_t j, uint32_t w[4])
{
    uint32_t h0, l0, h1, l1;
    mul_wide(PHILOX_M0, j, h0, l0);
    mul_wide(PHILOX_M1, h0 ^ K.xb, h1, l1);
    uint32_t c0 = h1 ^ K.xc, c1 = l1, c2 = l0 ^ R.xd, c3 = R.c3;
    uint32_t k0 = K.k0 + 2u * PHILOX_W0, k1 = K.k1 + 2u * PHILOX_W1;
#pragma unroll
    for (int r = 2; r < 10; ++r) {
        mul_wide(PHILOX_M0, c0, h0, l0);
        mul_wide(PHILOX_M1, c2, h1, l1);
        c0 = h1 ^ c1 ^ k0;
        c1 = l1;
        c2 = h0 ^ c3 ^ k1;
        c3 = l0;
        k0 += PHILOX_W0;
        k1 += PHILOX_W1;
    }
    w[0] = c0; w[1] = c1; w[2] = c2; w[3] = c3;
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
    return ((ne_flags<WIDE>(s, up) >> 7) + (ne_flags<WIDE>(s, dn) >> 7)) +
           ((ne_flags<WIDE>(s, lf) >> 7) + (ne_flags<WIDE>(s, rt) >> 7));
}

// Compare modes of update_word: how the per-byte counts of unequal neighbours are formed.
//   CM_7BIT  q <= 128: one flag word per (spin word, neighbour word) pair, 8 pairs per 4 sites
//   CM_8BIT  q <= 256: the same with the carry-safe test
//   CM_NIB4  q <= 16:  the current spin sits in the low nibble and the proposal in the high nibble of one byte,
//                      the neighbour is doubled into both nibbles (x 0x11): ONE xor and one zero-nibble test give
//                      the flags of both comparisons, and the shifted sum leaves n_old and n_new in the two nibbles
//   CM_NIB3  q <= 8:   as CM_NIB4, but a 3-bit difference cannot carry out of its nibble: a shorter zero test
constexpr int CM_7BIT = 0, CM_8BIT = 1, CM_NIB4 = 2, CM_NIB3 = 3;

__host__ __device__ constexpr int compare_mode_of(int q) { return q > 128 ? CM_8BIT : (q > 16 ? CM_7BIT : (q > 8 ? CM_NIB4 : CM_NIB3)); }

template <int CM>
__device__ __forceinline__ void ne_counts(uint32_t own, uint32_t prop, uint32_t up, uint32_t dn, uint32_t lf, uint32_t rt,
                                          uint32_t &c_old, uint32_t &c_new)
{
    if (CM == CM_7BIT || CM == CM_8BIT) {
        c_old = ne_count4<CM == CM_8BIT>(own, up, dn, lf, rt);
        c_new = ne_count4<CM == CM_8BIT>(prop, up, dn, lf, rt);
    } else {
        const uint32_t both = own | (prop << 4);
        const uint32_t nb[4] = {up, dn, lf, rt};
        uint32_t s = 0;
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const uint32_t x = both ^ (nb[k] * 0x11u);
            const uint32_t f = CM == CM_NIB3 ? (x + 0x77777777u) & 0x88888888u
                                             : (((x & 0x77777777u) + 0x77777777u) | x) & 0x88888888u;
            s += f >> 3;
        }
        c_old = s & 0x0f0f0f0fu;
        c_new = (s >> 4) & 0x0f0f0f0fu;
    }
}

__device__ __forceinline__ uint32_t byte_sum(uint32_t v)   // sum of the 4 bytes (sum < 256)
{
    return __dp4a(v, 0x01010101u, 0u);
}

// every byte of the result = 0xff if bit 7 of that byte of v is set, else 0x00 (PRMT with the
// "replicate sign" bit of each selector nibble; __byte_perm masks that bit off)
__device__ __forceinline__ uint32_t msb_to_bytemask(uint32_t v)
{
    uint32_t r;
    asm("prmt.b32 %0, %1, %1, 0xba98;" : "=r"(r) : "r"(v));
    return r;
}

__device__ __forceinline__ int wrap(int x, int n) { return x < 0 ? x + n : (x >= n ? x - n : x); }

// The two horizontal neighbour words of a 4-site word.  mid = other-colour word at the same
// (row, k); adj = the other-colour word at k+1 (p = 1) or k-1 (p = 0), periodic.
__device__ __forceinline__ void horizontal(uint32_t p, uint32_t mid, uint32_t adj, uint32_t &lf, uint32_t &rt)
{
    if (p) {   // neighbours at k and k+1
        lf = mid;
        rt = __funnelshift_r(mid, adj, 8);
    } else {   // neighbours at k-1 and k
        lf = __funnelshift_l(adj, mid, 8);
        rt = mid;
    }
}

// ---------------------------------------------------------------------------------------------
// One word (4 same-colour sites, consecutive k) of the Metropolis update (R4-R7).
//   own          current spins of the 4 sites
//   up,dn,lf,rt  the 4 neighbour words, byte b = that neighbour of site b
//   j0           column of byte 0 (columns advance by 2 per byte)
//   lut          shared memory, 9 words: lut[d+4] = floor(2^32 exp(-d/T)) for d = 1..4 (entries 0..4 unused)
// Returns the new word; ne_final = per-byte count of unequal neighbours of the final spins, ne_old = the same of
// the spins before the update (so that, per byte, ne_final - ne_old = d of an accepted move and 0 otherwise).
template <int CM, int ST>     // ST: random-stream definition, 1 = one Philox block per site (R3), 2 = per pair (R3')
__device__ __forceinline__ uint32_t update_word_ex(uint32_t own, uint32_t up, uint32_t dn, uint32_t lf, uint32_t rt,
                                                   uint32_t j0, uint32_t q, const HalfSweepKeys &K, const RowKeys &R,
                                                   const uint32_t *lut, uint32_t &ne_final, uint32_t &ne_old)
{
    uint32_t w0[4], w1[4];
    if (ST == 1) {
#pragma unroll
        for (int b = 0; b < 4; ++b) philox_site(K, R, j0 + 2u * b, w0[b], w1[b]);
    } else {
        // byte 0 of a word is an even same-colour site, so the word holds two whole pairs
#pragma unroll
        for (int m = 0; m < 2; ++m) {
            uint32_t w[4];
            philox_pair(K, R, j0 + 4u * m, w);
            w0[2 * m] = w[0]; w1[2 * m] = w[1]; w0[2 * m + 1] = w[2]; w1[2 * m + 1] = w[3];
        }
    }
    // R4: proposal floor(w0 q / 2^32), packed one byte per site
    const uint32_t s01 = __byte_perm(__umulhi(w0[0], q), __umulhi(w0[1], q), 0x0040);
    const uint32_t s23 = __byte_perm(__umulhi(w0[2], q), __umulhi(w0[3], q), 0x0040);
    const uint32_t prop = __byte_perm(s01, s23, 0x5410);

    // R5: d = n_old - n_new = ne_new - ne_old, biased by 4 so that every byte stays in 0..8
    uint32_t c_old, c_new;
    ne_counts<CM>(own, prop, up, dn, lf, rt, c_old, c_new);
    const uint32_t dw = c_new + 0x04040404u - c_old;
    // R6: d <= 0 always accepts: byte <= 4  <=>  bit 7 of (0x84 - byte); replicate it over the byte
    uint32_t mask = msb_to_bytemask(0x84848484u - dw);
    const uint32_t dw4 = dw << 2;                                   // byte offsets into lut
#pragma unroll
    for (int b = 0; b < 4; ++b) {
        const uint32_t off = (dw4 >> (8 * b)) & 0xffu;
        const uint32_t thr = *reinterpret_cast<const uint32_t *>(reinterpret_cast<const char *>(lut) + off);
        if (w1[b] < thr) mask |= 0xffu << (8 * b);
    }
    ne_final = (c_new & mask) | (c_old & ~mask);
    ne_old = c_old;
    return (prop & mask) | (own & ~mask);                           // R7
}

template <int CM, int ST>
__device__ __forceinline__ uint32_t update_word(uint32_t own, uint32_t up, uint32_t dn, uint32_t lf, uint32_t rt,
                                                uint32_t j0, uint32_t q, const HalfSweepKeys &K, const RowKeys &R,
                                                const uint32_t *lut, uint32_t &ne_final)
{
    uint32_t ne_old;
    return update_word_ex<CM, ST>(own, up, dn, lf, rt, j0, q, K, R, lut, ne_final, ne_old);
}

// ---------------------------------------------------------------------------------------------
// Histogram helpers.  Counters live in shared memory, privatised per lane (s_hist[k*32 + lane]) so
// that the 32 lanes of a warp never collide, even in the ordered phase where ~90 % of the sites
// hold one state; different warps meet through the shared-memory atomic.  For q > HIST_LANE_QMAX
// the table would be too large: one counter per state and a warp-aggregated add instead.
constexpr uint32_t HIST_LANE_QMAX = 64;

__device__ __forceinline__ uint32_t hist_words(uint32_t q) { return q <= HIST_LANE_QMAX ? q * 32u : q; }

__device__ __forceinline__ void hist_add_word(uint32_t *s_hist, uint32_t q, uint32_t word, uint32_t lane)
{
    if (q <= HIST_LANE_QMAX) {
        uint32_t *mine = s_hist + lane;
#pragma unroll
        for (int b = 0; b < 4; ++b) atomicAdd(mine + (((word >> (8 * b)) & 0xffu) << 5), 1u);
    } else {
        const uint32_t active = __activemask();
#pragma unroll
        for (int b = 0; b < 4; ++b) {
            const uint32_t s = (word >> (8 * b)) & 0xffu;
            const uint32_t peers = __match_any_sync(active, s);
            if (lane == (uint32_t)(__ffs(peers) - 1)) atomicAdd(s_hist + s, (uint32_t)__popc(peers));
        }
    }
}

// add this block's shared histogram to hist_out (int64 per state) and leave the table zeroed;
// call with all threads of the block (a multiple of 32), after a __syncthreads()
__device__ __forceinline__ void hist_flush(uint32_t *s_hist, uint32_t q, unsigned long long *hist_out, uint32_t tid,
                                           uint32_t nthreads)
{
    if (q <= HIST_LANE_QMAX) {
        // one warp per state: lanes read the 32 private counters, shuffle-reduce
        const uint32_t warp = tid >> 5, lane = tid & 31u, nwarps = nthreads >> 5;
        for (uint32_t k = warp; k < q; k += nwarps) {
            uint32_t v = s_hist[k * 32u + lane];
            s_hist[k * 32u + lane] = 0u;
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
            if (lane == 0 && v) atomicAdd(hist_out + k, (unsigned long long)v);
        }
    } else {
        for (uint32_t k = tid; k < q; k += nthreads) {
            const uint32_t v = s_hist[k];
            s_hist[k] = 0u;
            if (v) atomicAdd(hist_out + k, (unsigned long long)v);
        }
    }
}

}  // namespace potts
