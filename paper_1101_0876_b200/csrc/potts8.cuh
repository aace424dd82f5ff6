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
