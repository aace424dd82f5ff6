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
