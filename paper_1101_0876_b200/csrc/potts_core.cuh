// potts_core.cuh -- per-site arithmetic of the checkerboard Potts sweep for sm_100a.
//
// Everything on the device is integer arithmetic: Philox4x32-10 keyed by
// (seed; j, i, t, colour), multiply-high proposal, byte-parallel neighbour comparison and integer
// threshold acceptance (PAPER.md:94 sec. 3, :145 sec. 3.2).  Not shared with oracle/ in any way.
//
// Cost model this file is written against (profiles/r01b_pipe_model.md, measured on B200): for this
// integer mix an SM sub-partition retires one warp instruction every 2 clocks whichever pipe it goes to
// (IMAD.WIDE, IMAD, LOP3, IADD3, SHF, PRMT alike; IMAD.HI and POPC take 4), so the time of an update is
// its instruction count.  Round 2 (profiles/r02a_update_word.md) therefore cut instructions:
//   * Philox: the three multiplies and two XORs of rounds 1-3 that depend on the column j only (not on the
//     row) are computed once per column and half-sweep (ColKeys) and reused by every row of the tile:
//     14 IMAD.WIDE + 16 LOP3 per site instead of 17 + 18;
//   * neighbour compare: the four "differs" flags of the current spin and the four of the proposal are
//     gathered into ONE code byte per site (no counting, no subtraction);
//   * acceptance: the code byte indexes a 256-entry shared table of 64-bit values 2^64 - threshold(d),
//     and the 64-bit sum  w1 + entry  (add, add-with-carry) leaves the accept mask (0 / 0xffffffff) in its
//     high word: d <= 0 ("always") and threshold 0 ("never") need no special case and no mask start-up;
//   * the energy / energy-change sums of sampled sweeps are two population counts of the masked code word.
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

// 32-bit shared-window address of a shared-memory pointer (operand of mbarrier / bulk-copy / st.async instructions)
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

// three-input logic in one LOP3; LUT = f(0xF0, 0xCC, 0xAA)
template <int LUT>
__device__ __forceinline__ uint32_t lop3(uint32_t a, uint32_t b, uint32_t c)
{
    uint32_t r;
    asm("lop3.b32 %0, %1, %2, %3, %4;" : "=r"(r) : "r"(a), "r"(b), "r"(c), "n"(LUT));
    return r;
}
constexpr int LOP_XOR_AND = (0xF0 ^ 0xCC) & 0xAA;              // (a ^ b) & c
constexpr int LOP_OR_XOR = 0xF0 | (0xCC ^ 0xAA);               // a | (b ^ c)
constexpr int LOP_SEL = (0xF0 & 0xAA) | (0xCC & ~0xAA & 0xFF); // (a & c) | (b & ~c): bits of a where c is set, else b

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
//   ColKeys        adds the column j, NOT the row -- three wide multiplies per column and half-sweep
//   philox_site    adds the column j to a row     -- 17 wide multiplies + 18 three-input XORs (no ColKeys)
//   philox_site_h  the same from ColKeys          -- 14 wide multiplies + 16 XORs
// Round 1 multiplies the counter words c0 = j and c2 = t; round 2 multiplies c0' = hi(M1 t)^i^k0 (no j) and
// c2' = hi(M0 j)^colour^k1 (no i); round 3 multiplies c0'' = hi(M1 c2')^lo(M1 t)^k0' (no i).
struct HalfSweepKeys {
    uint32_t xa;      // hi(M1*t) ^ k0[0]          c0 after round 1 is xa ^ i
    uint32_t xb;      // colour ^ k1[0]            c2 after round 1 is hi(M0*j) ^ xb
    uint32_t xc;      // lo(M1*t) ^ k0[1]          c0 after round 2 is hi(M1*c2') ^ xc
    uint32_t r0[10], r1[10];  // the round keys: round r (0-based) uses r0[r] = key0 + r W0, r1[r] = key1 + r W1
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
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        K.r0[r] = key0 + (uint32_t)r * PHILOX_W0;
        K.r1[r] = key1 + (uint32_t)r * PHILOX_W1;
    }
    return K;
}

// the (t, colour) part only: the round keys depend on the seed alone (persistent kernels build them once per launch)
__host__ __device__ inline void half_sweep_rekey(HalfSweepKeys &K, uint32_t key0, uint32_t key1, uint32_t t, uint32_t colour)
{
    const unsigned long long p = (unsigned long long)PHILOX_M1 * (unsigned long long)t;
    K.xa = (uint32_t)(p >> 32) ^ key0;
    K.xb = colour ^ key1;
    K.xc = (uint32_t)p ^ (key0 + PHILOX_W0);
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
    R.xd = hi ^ K.r1[1];
    return R;
}

__device__ __forceinline__ void philox_site(const HalfSweepKeys &K, const RowKeys &R, uint32_t j,
                                            uint32_t &w0, uint32_t &w1)
{
    uint32_t h0, l0, h1, l1;
    mul_wide(PHILOX_M0, j, h0, l0);                  // round 1, the M0*c0 product
    mul_wide(PHILOX_M1, h0 ^ K.xb, h1, l1);          // round 2, the M1*c2 product
    uint32_t c0 = h1 ^ K.xc, c1 = l1, c2 = l0 ^ R.xd, c3 = R.c3;
#pragma unroll
    for (int r = 2; r < 9; ++r) {
        mul_wide(PHILOX_M0, c0, h0, l0);
        mul_wide(PHILOX_M1, c2, h1, l1);
        c0 = h1 ^ c1 ^ K.r0[r];
        c1 = l1;
        c2 = h0 ^ c3 ^ K.r1[r];
        c3 = l0;
    }
    mul_wide(PHILOX_M1, c2, h1, l1);                 // round 10: only words 0 and 1 are used
    w0 = h1 ^ c1 ^ K.r0[9];
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
#pragma unroll
    for (int r = 2; r < 10; ++r) {
        mul_wide(PHILOX_M0, c0, h0, l0);
        mul_wide(PHILOX_M1, c2, h1, l1);
        c0 = h1 ^ c1 ^ K.r0[r];
        c1 = l1;
        c2 = h0 ^ c3 ^ K.r1[r];
        c3 = l0;
    }
    w[0] = c0; w[1] = c1; w[2] = c2; w[3] = c3;
}

// The column part: everything of rounds 1-3 that depends on j but not on the row i.  One uint4 per column.
struct ColKeys {
    uint32_t l0;      // lo(M0*j)                      c2 after round 2 is l0 ^ R.xd
    uint32_t l1;      // lo(M1*(hi(M0*j)^xb))          c1 after round 2
    uint32_t ph, pl;  // M0 * (hi(M1*(hi(M0*j)^xb)) ^ xc): round 3's M0*c0 product
};

__device__ __forceinline__ ColKeys col_keys(uint32_t xb, uint32_t xc, uint32_t j)
{
    ColKeys C;
    uint32_t h0, h1;
    mul_wide(PHILOX_M0, j, h0, C.l0);
    mul_wide(PHILOX_M1, h0 ^ xb, h1, C.l1);
    mul_wide(PHILOX_M0, h1 ^ xc, C.ph, C.pl);
    return C;
}

__device__ __forceinline__ ColKeys col_keys(const HalfSweepKeys &K, uint32_t j) { return col_keys(K.xb, K.xc, j); }

// row part for the hoisted form: RowKeys plus c3 ^ (k1 of round 3)
struct RowKeysH {
    uint32_t xd;      // as RowKeys
    uint32_t rc;      // R.c3 ^ (k1 + 2 W1): c2 after round 3 is C.ph ^ rc
};

__device__ __forceinline__ RowKeysH row_keys_h(const HalfSweepKeys &K, uint32_t i)
{
    const RowKeys R = row_keys(K, i);
    RowKeysH H;
    H.xd = R.xd;
    H.rc = R.c3 ^ K.r1[2];
    return H;
}

// rounds 3-9 from (ColKeys, RowKeysH); leaves the state before round 10 and the keys of round 10
__device__ __forceinline__ void philox_rounds_h(const HalfSweepKeys &K, const RowKeysH &R, const ColKeys &C,
                                                uint32_t &c0, uint32_t &c1, uint32_t &c2, uint32_t &c3)
{
    uint32_t h0, l0, h1, l1;
    mul_wide(PHILOX_M1, C.l0 ^ R.xd, h1, l1);        // round 3: the M1*c2 product (M0*c0 is in C)
    c0 = h1 ^ C.l1 ^ K.r0[2];
    c1 = l1;
    c2 = C.ph ^ R.rc;
    c3 = C.pl;
#pragma unroll
    for (int r = 3; r < 9; ++r) {
        mul_wide(PHILOX_M0, c0, h0, l0);
        mul_wide(PHILOX_M1, c2, h1, l1);
        c0 = h1 ^ c1 ^ K.r0[r];
        c1 = l1;
        c2 = h0 ^ c3 ^ K.r1[r];
        c3 = l0;
    }
}

__device__ __forceinline__ void philox_site_h(const HalfSweepKeys &K, const RowKeysH &R, const ColKeys &C,
                                              uint32_t &w0, uint32_t &w1)
{
    uint32_t c0, c1, c2, c3, h1, l1;
    philox_rounds_h(K, R, C, c0, c1, c2, c3);
    mul_wide(PHILOX_M1, c2, h1, l1);                 // round 10: only words 0 and 1 are used
    w0 = h1 ^ c1 ^ K.r0[9];
    w1 = l1;
}

__device__ __forceinline__ void philox_pair_h(const HalfSweepKeys &K, const RowKeysH &R, const ColKeys &C, uint32_t w[4])
{
    uint32_t c0, c1, c2, c3, h0, l0, h1, l1;
    philox_rounds_h(K, R, C, c0, c1, c2, c3);
    mul_wide(PHILOX_M0, c0, h0, l0);
    mul_wide(PHILOX_M1, c2, h1, l1);
    w[0] = h1 ^ c1 ^ K.r0[9]; w[1] = l1; w[2] = h0 ^ c3 ^ K.r1[9]; w[3] = l0;
}

// ---------------------------------------------------------------------------------------------
// Compare modes: how the "differs" flags of a word's four sites against one neighbour word are formed.
//   CM_7BIT  q <= 128: own and proposal are compared separately, flag in bit 7 of ((a^b) + 0x7f)
//   CM_8BIT  q <= 256: the same with the carry-safe test
//   CM_NIB4  q <= 16:  the current spin sits in the low nibble and the proposal in the high nibble of one byte,
//                      the neighbour is doubled into both nibbles (x 0x11, once per loaded word): ONE three-input
//                      logic op, one add and one more logic op give the flags of both comparisons (bits 3 and 7)
//   CM_NIB3  q <= 8:   as CM_NIB4, but a 3-bit difference cannot carry out of its nibble: one XOR and one add
constexpr int CM_7BIT = 0, CM_8BIT = 1, CM_NIB4 = 2, CM_NIB3 = 3;

__host__ __device__ constexpr int compare_mode_of(int q) { return q > 128 ? CM_8BIT : (q > 16 ? CM_7BIT : (q > 8 ? CM_NIB4 : CM_NIB3)); }
__host__ __device__ constexpr bool is_nibble_mode(int cm) { return cm == CM_NIB4 || cm == CM_NIB3; }

// a neighbour word as the compare wants it: doubled into both nibbles for the nibble modes
template <int CM>
__device__ __forceinline__ uint32_t prep_nbr(uint32_t w) { return is_nibble_mode(CM) ? w * 0x11u : w; }

// One code byte per site: bit k (k = 0..3) = neighbour k differs from the CURRENT spin, bit 4+k = neighbour k
// differs from the PROPOSAL.  nb[] = the four neighbour words, prepared by prep_nbr.  The flags of neighbour k
// are moved to their bit by one shift and merged by one bit-select; bits the select leaves behind are garbage
// of an earlier stage that a later select overwrites.
template <int CM>
__device__ __forceinline__ uint32_t ne_code(uint32_t own, uint32_t prop, const uint32_t nb[4])
{
    if (is_nibble_mode(CM)) {
        const uint32_t both = prop * 16u + own;                       // one IMAD: the nibbles do not overlap
        uint32_t u[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            if (CM == CM_NIB3) {
                u[k] = (both ^ nb[k]) + 0x77777777u;                  // bit 3 of a nibble = its 3-bit difference is non-zero
            } else {
                const uint32_t m = lop3<LOP_XOR_AND>(both, nb[k], 0x77777777u);
                u[k] = lop3<LOP_OR_XOR>(m + 0x77777777u, both, nb[k]);
            }
        }
        uint32_t c = lop3<LOP_SEL>(u[0] >> 3, u[1] >> 2, 0x11111111u);
        c = lop3<LOP_SEL>(c, u[2] >> 1, 0x33333333u);
        return lop3<LOP_SEL>(c, u[3], 0x77777777u);
    } else {
        uint32_t o[4], n[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            if (CM == CM_7BIT) {
                o[k] = (own ^ nb[k]) + 0x7f7f7f7fu;                   // bit 7 of a byte = its 7-bit difference is non-zero
                n[k] = (prop ^ nb[k]) + 0x7f7f7f7fu;
            } else {
                o[k] = lop3<LOP_OR_XOR>(lop3<LOP_XOR_AND>(own, nb[k], 0x7f7f7f7fu) + 0x7f7f7f7fu, own, nb[k]);
                n[k] = lop3<LOP_OR_XOR>(lop3<LOP_XOR_AND>(prop, nb[k], 0x7f7f7f7fu) + 0x7f7f7f7fu, prop, nb[k]);
            }
        }
        uint32_t a = lop3<LOP_SEL>(o[0] >> 7, o[1] >> 6, 0x01010101u);
        a = lop3<LOP_SEL>(a, o[2] >> 5, 0x03030303u);
        a = lop3<LOP_SEL>(a, o[3] >> 4, 0x07070707u);                 // bits 0..3 of every byte
        uint32_t b = lop3<LOP_SEL>(n[0] >> 3, n[1] >> 2, 0x10101010u);
        b = lop3<LOP_SEL>(b, n[2] >> 1, 0x30303030u);
        b = lop3<LOP_SEL>(b, n[3], 0x70707070u);                      // bits 4..7 of every byte
        return lop3<LOP_SEL>(a, b, 0x0f0f0f0fu);
    }
}

__device__ __forceinline__ int wrap(int x, int n) { return x < 0 ? x + n : (x >= n ? x - n : x); }

// The two horizontal neighbour words of a 4-site word.  mid = other-colour word at the same
// (row, k); adj = the other-colour word at k+1 (p = 1) or k-1 (p = 0), periodic.  Works on prepared
// (doubled) words as well: the shift is a whole byte.
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
// Acceptance table (shared memory), indexed by the code byte.  With c_old = popc(code & 15) neighbours that
// differ from the current spin and c_new = popc(code >> 4) that differ from the proposal,
//   d = n_old - n_new = c_new - c_old                                   (R5)
//   threshold(d) = 2^32 for d <= 0 (always accept), thr[d-1] = floor(2^32 exp(-d/T)) for d = 1..4   (R6)
//   entry = 2^64 - threshold(d)  (mod 2^64)
// so that the high word of  w1 + entry  is 0xffffffff iff w1 < threshold(d) and 0 otherwise: exact for every
// threshold in [0, 2^32].  The 32 lanes of a warp look up 32 different codes, so a single copy of the table
// would serialise on its banks (measured: the 9-word table of round 1 never did); the table is therefore stored
// in SLOTS copies, entry (code, slot) at byte code * 8 * SLOTS + slot * 8, and lane l reads slot
// l % SLOTS: the 16 lanes of a half-warp meet on a bank pair only if they share a slot AND differ in code.
constexpr int ACCEPT_ENTRIES = 256;
template <int SLOTS>
struct AcceptLutT {
    static_assert(SLOTS == 4 || SLOTS == 8 || SLOTS == 16, "slot copies: 4, 8 or 16");
    static constexpr int slots = SLOTS;
    static constexpr int shift = SLOTS == 4 ? 5 : (SLOTS == 8 ? 6 : 7);     // log2(8 bytes * SLOTS)
    uint2 e[ACCEPT_ENTRIES][SLOTS];
};
using AcceptLut = AcceptLutT<8>;           // streaming kernels: 16 KB beside the 16 KB of ColKeys
using AcceptLutWide = AcceptLutT<16>;      // persistent kernels: 32 KB, no two lanes of a half-warp share a slot

// fast = true (allowed only if every thr[d] >= 1, i.e. no "never accept" entry): the entry's first word is
// threshold(d) - 1 instead, and a site accepts iff w1 <= that word (0xffffffff for d <= 0): one 32-bit compare.
template <int SLOTS>
__device__ __forceinline__ void accept_lut_fill(AcceptLutT<SLOTS> *lut, const uint32_t thr[4], uint32_t tid, uint32_t nthreads, bool fast = false)
{
    for (uint32_t n = tid; n < (uint32_t)(ACCEPT_ENTRIES * SLOTS); n += nthreads) {
        const uint32_t code = n / SLOTS;
        const int d = __popc(code >> 4) - __popc(code & 15u);
        const unsigned long long th = d <= 0 ? (1ull << 32) : (unsigned long long)(d == 1 ? thr[0] : (d == 2 ? thr[1] : (d == 3 ? thr[2] : thr[3])));
        const unsigned long long e = fast ? th - 1ull : 0ull - th;
        (&lut->e[0][0])[n] = make_uint2((uint32_t)e, (uint32_t)(e >> 32));
    }
}

__host__ __device__ inline bool accept_fast_ok(const uint32_t thr[4]) { return thr[0] && thr[1] && thr[2] && thr[3]; }

// byte offset of this lane's slot inside a table row
template <int SLOTS = 8>
__device__ __forceinline__ uint32_t accept_lane_offset(uint32_t lane) { return (lane % SLOTS) * 8u; }

// accept masks of the four sites of a word: byte b = 0xff iff site b accepts its proposal
// CODE_BITS: the bits of a code byte that index the table (the 3D code leaves garbage in bits 3 and 7: 0x77)
template <int SLOTS, uint32_t CODE_BITS = 0xffu>
__device__ __forceinline__ uint32_t accept_mask(uint32_t code, const uint32_t w1[4], const AcceptLutT<SLOTS> *lut, uint32_t lane_off)
{
    constexpr int ACCEPT_SHIFT = AcceptLutT<SLOTS>::shift;
    constexpr uint32_t M = CODE_BITS << ACCEPT_SHIFT;
    uint32_t a[4];
#pragma unroll
    for (int b = 0; b < 4; ++b) {
        const uint32_t sh = b == 0 ? code << ACCEPT_SHIFT : code >> (8 * b - ACCEPT_SHIFT);
        const uint32_t off = lop3<0xEA>(sh, M, lane_off);              // (sh & M) | lane_off
        const uint2 v = *reinterpret_cast<const uint2 *>(reinterpret_cast<const char *>(lut) + off);
        unsigned long long e;
        asm("mov.b64 %0, {%1, %2};" : "=l"(e) : "r"(v.x), "r"(v.y));
        a[b] = (uint32_t)((e + (unsigned long long)w1[b]) >> 32);
    }
    const uint32_t m01 = lop3<LOP_SEL>(a[0], a[1], 0x000000ffu);
    const uint32_t m23 = lop3<LOP_SEL>(a[2], a[3], 0x00ffffffu);
    return lop3<LOP_SEL>(m01, m23, 0x0000ffffu);
}

// Fast form (table filled with fast = true): the new word directly, one compare and one predicated byte insert per site.
template <int SLOTS, uint32_t CODE_BITS = 0xffu>
__device__ __forceinline__ uint32_t accept_insert(uint32_t own, uint32_t prop, uint32_t code, const uint32_t w1[4], const AcceptLutT<SLOTS> *lut,
                                                  uint32_t lane_off)
{
    constexpr int ACCEPT_SHIFT = AcceptLutT<SLOTS>::shift;
    constexpr uint32_t M = CODE_BITS << ACCEPT_SHIFT;
    uint32_t out = own;
#pragma unroll
    for (int b = 0; b < 4; ++b) {
        const uint32_t sh = b == 0 ? code << ACCEPT_SHIFT : code >> (8 * b - ACCEPT_SHIFT);
        const uint32_t off = lop3<0xEA>(sh, M, lane_off);
        const uint32_t t = *reinterpret_cast<const uint32_t *>(reinterpret_cast<const char *>(lut) + off);
        const uint32_t ins = __byte_perm(out, prop, b == 0 ? 0x3214 : (b == 1 ? 0x3250 : (b == 2 ? 0x3610 : 0x7210)));
        out = w1[b] <= t ? ins : out;
    }
    return out;
}

// Sums over the four sites of a word from its code word and accept mask (sampled sweeps and the energy-change
// series only).  ne_final_sum: unequal neighbours of the FINAL spins (accepted: the proposal's flags, else the
// current spin's).  delta_sum: sum of d = n_old - n_new = c_new - c_old over the accepted sites.
__device__ __forceinline__ int ne_final_sum(uint32_t code, uint32_t mask)
{
    return __popc(lop3<LOP_SEL>(code >> 4, code, mask) & 0x0f0f0f0fu);
}

__device__ __forceinline__ int delta_sum(uint32_t code, uint32_t mask)
{
    const uint32_t cm = code & mask;
    return __popc(cm & 0xf0f0f0f0u) - __popc(cm & 0x0f0f0f0fu);
}

// ---------------------------------------------------------------------------------------------
// One word (4 same-colour sites, consecutive k) of the Metropolis update (R4-R7), random words given.
//   own      current spins of the 4 sites
//   nb[4]    the 4 neighbour words (up, down, left, right: any order), prepared by prep_nbr<CM>
//   w0, w1   Philox words of the 4 sites: proposal and acceptance
// Returns the new word; code / mask = the word's code bytes and accept mask for ne_final_sum / delta_sum.
template <int CM, bool FAST = false, int SLOTS = 8>
__device__ __forceinline__ uint32_t metropolis_word(uint32_t own, const uint32_t nb[4], uint32_t q, const uint32_t w0[4],
                                                    const uint32_t w1[4], const AcceptLutT<SLOTS> *lut, uint32_t lane_off,
                                                    uint32_t &code, uint32_t &mask)
{
    // R4: proposal floor(w0 q / 2^32), packed one byte per site
    const uint32_t s01 = __byte_perm(__umulhi(w0[0], q), __umulhi(w0[1], q), 0x0040);
    const uint32_t s23 = __byte_perm(__umulhi(w0[2], q), __umulhi(w0[3], q), 0x0040);
    const uint32_t prop = __byte_perm(s01, s23, 0x5410);
    code = ne_code<CM>(own, prop, nb);                                // R5
    if (FAST) {
        mask = 0u;                                                    // not formed: the sums need the exact form
        return accept_insert(own, prop, code, w1, lut, lane_off);     // R6, R7
    }
    mask = accept_mask(code, w1, lut, lane_off);                      // R6
    return lop3<LOP_SEL>(prop, own, mask);                            // R7
}

// The random words of a word's four sites drawn without ColKeys (kernels that keep the lattice in shared memory):
//   j0  column of byte 0 (columns advance by 2 per byte)
template <int ST>     // ST: random-stream definition, 1 = one Philox block per site (R3), 2 = per pair (R3')
__device__ __forceinline__ void draw_words(const HalfSweepKeys &K, const RowKeys &R, uint32_t j0, uint32_t w0[4], uint32_t w1[4])
{
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
}

// One word of the update from the neighbour words as loaded (byte b = that neighbour of site b).
template <int CM, int ST, int SLOTS>
__device__ __forceinline__ uint32_t update_word(uint32_t own, uint32_t up, uint32_t dn, uint32_t lf, uint32_t rt,
                                                uint32_t j0, uint32_t q, const HalfSweepKeys &K, const RowKeys &R,
                                                const AcceptLutT<SLOTS> *lut, uint32_t lane_off, uint32_t &code, uint32_t &mask)
{
    uint32_t w0[4], w1[4];
    draw_words<ST>(K, R, j0, w0, w1);
    const uint32_t nb[4] = {prep_nbr<CM>(up), prep_nbr<CM>(dn), prep_nbr<CM>(lf), prep_nbr<CM>(rt)};
    return metropolis_word<CM, false, SLOTS>(own, nb, q, w0, w1, lut, lane_off, code, mask);
}

// The same with the column part of Philox read from a table: ck[b * ck_stride] = ColKeys of the word's column b, in the
// row parity of this visit (persistent kernels that visit a column often enough to share it: L >= 2048).
template <int CM, int ST, int SLOTS>
__device__ __forceinline__ uint32_t update_word_h(uint32_t own, uint32_t up, uint32_t dn, uint32_t lf, uint32_t rt,
                                                  const uint4 *ck, uint32_t ck_stride, uint32_t q, const HalfSweepKeys &K, const RowKeysH &R,
                                                  const AcceptLutT<SLOTS> *lut, uint32_t lane_off, uint32_t &code, uint32_t &mask)
{
    uint32_t w0[4], w1[4];
    if (ST == 1) {
#pragma unroll
        for (int b = 0; b < 4; ++b) {
            const uint4 c = ck[b * ck_stride];
            philox_site_h(K, R, ColKeys{c.x, c.y, c.z, c.w}, w0[b], w1[b]);
        }
    } else {
#pragma unroll
        for (int m = 0; m < 2; ++m) {
            const uint4 c = ck[2 * m * ck_stride];
            uint32_t w[4];
            philox_pair_h(K, R, ColKeys{c.x, c.y, c.z, c.w}, w);
            w0[2 * m] = w[0]; w1[2 * m] = w[1]; w0[2 * m + 1] = w[2]; w1[2 * m + 1] = w[3];
        }
    }
    const uint32_t nb[4] = {prep_nbr<CM>(up), prep_nbr<CM>(dn), prep_nbr<CM>(lf), prep_nbr<CM>(rt)};
    return metropolis_word<CM, false, SLOTS>(own, nb, q, w0, w1, lut, lane_off, code, mask);
}

// The same with the ColKeys of the word's four columns in the caller's registers (the replica-batch kernel, whose
// threads visit rows of one parity only).
template <int CM, int ST, int SLOTS>
__device__ __forceinline__ uint32_t update_word_r(uint32_t own, uint32_t up, uint32_t dn, uint32_t lf, uint32_t rt,
                                                  const ColKeys *ck, uint32_t q, const HalfSweepKeys &K, const RowKeysH &R,
                                                  const AcceptLutT<SLOTS> *lut, uint32_t lane_off, uint32_t &code, uint32_t &mask)
{
    uint32_t w0[4], w1[4];
    if (ST == 1) {
#pragma unroll
        for (int b = 0; b < 4; ++b) philox_site_h(K, R, ck[b], w0[b], w1[b]);
    } else {
#pragma unroll
        for (int m = 0; m < 2; ++m) {
            uint32_t w[4];
            philox_pair_h(K, R, ck[2 * m], w);
            w0[2 * m] = w[0]; w1[2 * m] = w[1]; w0[2 * m + 1] = w[2]; w1[2 * m + 1] = w[3];
        }
    }
    const uint32_t nb[4] = {prep_nbr<CM>(up), prep_nbr<CM>(dn), prep_nbr<CM>(lf), prep_nbr<CM>(rt)};
    return metropolis_word<CM, false, SLOTS>(own, nb, q, w0, w1, lut, lane_off, code, mask);
}

// ---------------------------------------------------------------------------------------------
// Standalone measurement helpers: byte-parallel "not equal" flags (bit 7 of every byte of the result is
// set iff the bytes of a and b differ).  WIDE = false assumes all spin values < 128.
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

__device__ __forceinline__ uint32_t byte_sum(uint32_t v)   // sum of the 4 bytes (sum < 256)
{
    return __dp4a(v, 0x01010101u, 0u);
}

// ---------------------------------------------------------------------------------------------
// Histogram helpers.  Counters live in shared memory, privatised per lane (s_hist[k*32 + lane]) so
// that the 32 lanes of a warp never collide, even in the ordered phase where ~90 % of the sites
// hold one state; different warps meet through the shared-memory atomic.  For q > HIST_LANE_QMAX
// the table would be too large: one counter per state and a warp-aggregated add instead.
constexpr uint32_t HIST_LANE_QMAX = 64;

__host__ __device__ inline uint32_t hist_words(uint32_t q) { return q <= HIST_LANE_QMAX ? q * 32u : q; }

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
        // one warp per state: lanes read the 32 private counters, one REDUX per state.  Four states per trip, so that the
        // loads, the reductions and the atomics of a warp's states overlap instead of forming one dependent chain per state
        // (the flush sits between two half-sweeps of the persistent kernels: its latency is on their critical path)
        const uint32_t warp = tid >> 5, lane = tid & 31u, nwarps = nthreads >> 5;
        for (uint32_t k0 = warp; k0 < q; k0 += 4u * nwarps) {
            uint32_t v[4];
#pragma unroll
            for (uint32_t u = 0; u < 4; ++u) {
                const uint32_t k = k0 + u * nwarps;
                v[u] = 0u;
                if (k < q) {
                    v[u] = s_hist[k * 32u + lane];
                    s_hist[k * 32u + lane] = 0u;
                }
            }
#pragma unroll
            for (uint32_t u = 0; u < 4; ++u) v[u] = __reduce_add_sync(0xffffffffu, v[u]);
#pragma unroll
            for (uint32_t u = 0; u < 4; ++u)
                if (lane == 0 && v[u]) atomicAdd(hist_out + k0 + u * nwarps, (unsigned long long)v[u]);
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
