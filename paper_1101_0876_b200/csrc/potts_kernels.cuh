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
    unsigned long long *E_out;  // MEASURE: -= satisfied bonds seen from this colour's sites
    unsigned long long *hist_out;  // HIST: += occupancies of this colour's sites after the update
    int32_t rpt;                // rows per thread (divides L / HS_WARPS)
};

// ---------------------------------------------------------------------------------------------
// Half-sweep, U8 layout.  A thread updates 16 consecutive same-colour sites (one 16-byte chunk) of
// P.rpt consecutive rows; a warp covers 32 chunks, a block HS_WARPS groups of rows.
// grid = (ceil(L/32 / 32), L / (HS_WARPS * rpt)).  Requires L % 32 == 0.  rpt up to 8 amortises the
// prologue and the block turnover on large lattices; small ones keep rpt low to fill the GPU.
constexpr int HS_WARPS = 4;

template <int CM, int ST, bool MEASURE, bool HIST>
__global__ void __launch_bounds__(32 * HS_WARPS) k_half_sweep_u8(const __grid_constant__ SweepParams P)
{
    extern __shared__ uint32_t s_dyn[];             // HIST: the block's histogram table
    __shared__ uint32_t lut[12];
    __shared__ uint32_t blockE;
    const uint32_t tid = threadIdx.y * 32u + threadIdx.x;
    if (tid < 9) lut[tid] = tid >= 5 ? P.thr[tid - 5] : 0u;
    if (MEASURE && tid == 0) blockE = 0u;
    if (HIST)
        for (uint32_t n = tid; n < hist_words(P.q); n += 32 * HS_WARPS) s_dyn[n] = 0u;
    __syncthreads();

    const int chunks = P.pitch >> 4;                                  // 16-byte chunks per row
    const int x = (int)(blockIdx.x * 32u + threadIdx.x);
    const int i0 = (int)(blockIdx.y * HS_WARPS + threadIdx.y) * P.rpt;
    uint32_t satisfied = 0;
    if (x < chunks) {
        const int k0 = x << 4;
        const HalfSweepKeys &K = P.K;
        const uint32_t q = in_register(P.q);
        const int kn = wrap(k0 + 16, P.pitch), kp = wrap(k0 - 4, P.pitch);
#pragma unroll 1
        for (int r = 0; r < P.rpt; ++r) {
            const int i = i0 + r;
            const uint32_t p = (uint32_t)(i + P.colour) & 1u;
            const int iu = wrap(i - 1, P.L), id = wrap(i + 1, P.L);
            const size_t row = (size_t)i * P.pitch;
            const uint4 own4 = *reinterpret_cast<const uint4 *>(P.plane_own + row + k0);
            const uint4 mid4 = *reinterpret_cast<const uint4 *>(P.plane_oth + row + k0);
            const uint4 up4 = *reinterpret_cast<const uint4 *>(P.plane_oth + (size_t)iu * P.pitch + k0);
            const uint4 dn4 = *reinterpret_cast<const uint4 *>(P.plane_oth + (size_t)id * P.pitch + k0);
            // the one word outside the chunk: [i][k0+16..] if p = 1, [i][..k0-1] if p = 0 (periodic)
            const uint32_t adj = *reinterpret_cast<const uint32_t *>(P.plane_oth + row + (p ? kn : kp));

            const RowKeys R = row_keys(K, (uint32_t)i);
            const uint32_t own[4] = {own4.x, own4.y, own4.z, own4.w};
            const uint32_t mid[6] = {adj, mid4.x, mid4.y, mid4.z, mid4.w, adj};
            const uint32_t up[4] = {up4.x, up4.y, up4.z, up4.w};
            const uint32_t dn[4] = {dn4.x, dn4.y, dn4.z, dn4.w};
            uint32_t out[4], nef_sum = 0;
#pragma unroll
            for (int n = 0; n < 4; ++n) {
                uint32_t lf, rt, nef;
                horizontal(p, mid[n + 1], p ? mid[n + 2] : mid[n], lf, rt);
                out[n] = update_word<CM, ST>(own[n], up[n], dn[n], lf, rt, 2u * (uint32_t)(k0 + 4 * n) + p, q, K, R, lut, nef);
                if (MEASURE) nef_sum += nef;                          // bytes stay <= 16
                if (HIST) hist_add_word(s_dyn, P.q, out[n], threadIdx.x);
            }
            *reinterpret_cast<uint4 *>(P.plane_own + row + k0) = make_uint4(out[0], out[1], out[2], out[3]);
            if (MEASURE) satisfied += 64u - byte_sum(nef_sum);
        }
    }
    if (MEASURE) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) satisfied += __shfl_xor_sync(0xffffffffu, satisfied, o);
        if (threadIdx.x == 0) atomicAdd(&blockE, satisfied);
        __syncthreads();
        // E = -(satisfied bonds): accumulate the two's-complement negative into the int64 slot
        if (tid == 0) atomicAdd(P.E_out, 0ull - (unsigned long long)blockE);
    }
    if (HIST) {
        __syncthreads();
        hist_flush(s_dyn, P.q, P.hist_out, tid, 32 * HS_WARPS);
    }
}

// ---------------------------------------------------------------------------------------------
// Half-sweep with the on-the-fly energy change ("keeping track of the energy changes at
// each spin flip ... a parallel accumulation of local energy changes on-the-fly" for reweighting runs):
// adds  sum over accepted moves of d = n_old - n_new  (R5, R7) of this half-sweep to *dE_out, as a
// two's-complement int64.  No energy recount: per site d_accepted = ne(final spin) - ne(old spin), where ne is
// the count of unequal neighbours, so the half-sweep's sum is byte_sum(ne_final) - byte_sum(ne_old).
// Same thread map as k_half_sweep_u8 (P.rpt rows per thread); a separate kernel so that the plain path's code
// generation is untouched.
template <int CM, int ST>
__global__ void __launch_bounds__(32 * HS_WARPS) k_half_sweep_delta_u8(const __grid_constant__ SweepParams P,
                                                                       unsigned long long *dE_out)
{
    __shared__ uint32_t lut[12];
    __shared__ int blockD;
    const uint32_t tid = threadIdx.y * 32u + threadIdx.x;
    if (tid < 9) lut[tid] = tid >= 5 ? P.thr[tid - 5] : 0u;
    if (tid == 0) blockD = 0;
    __syncthreads();

    const int chunks = P.pitch >> 4;
    const int x = (int)(blockIdx.x * 32u + threadIdx.x);
    const int i0 = (int)(blockIdx.y * HS_WARPS + threadIdx.y) * P.rpt;
    int delta = 0;                                                     // |delta| <= 4 * 16 * rpt per thread
    if (x < chunks) {
        const int k0 = x << 4;
        const HalfSweepKeys &K = P.K;
        const uint32_t q = in_register(P.q);
        const int kn = wrap(k0 + 16, P.pitch), kp = wrap(k0 - 4, P.pitch);
#pragma unroll 1
        for (int r = 0; r < P.rpt; ++r) {
            const int i = i0 + r;
            const uint32_t p = (uint32_t)(i + P.colour) & 1u;
            const int iu = wrap(i - 1, P.L), id = wrap(i + 1, P.L);
            const size_t row = (size_t)i * P.pitch;
            const uint4 own4 = *reinterpret_cast<const uint4 *>(P.plane_own + row + k0);
            const uint4 mid4 = *reinterpret_cast<const uint4 *>(P.plane_oth + row + k0);
            const uint4 up4 = *reinterpret_cast<const uint4 *>(P.plane_oth + (size_t)iu * P.pitch + k0);
            const uint4 dn4 = *reinterpret_cast<const uint4 *>(P.plane_oth + (size_t)id * P.pitch + k0);
            const uint32_t adj = *reinterpret_cast<const uint32_t *>(P.plane_oth + row + (p ? kn : kp));
            const RowKeys R = row_keys(K, (uint32_t)i);
            const uint32_t own[4] = {own4.x, own4.y, own4.z, own4.w};
            const uint32_t mid[6] = {adj, mid4.x, mid4.y, mid4.z, mid4.w, adj};
            const uint32_t up[4] = {up4.x, up4.y, up4.z, up4.w};
            const uint32_t dn[4] = {dn4.x, dn4.y, dn4.z, dn4.w};
            uint32_t out[4], d_sum = 0;
#pragma unroll
            for (int n = 0; n < 4; ++n) {
                uint32_t lf, rt, nef, neo;
                horizontal(p, mid[n + 1], p ? mid[n + 2] : mid[n], lf, rt);
                out[n] = update_word_ex<CM, ST>(own[n], up[n], dn[n], lf, rt, 2u * (uint32_t)(k0 + 4 * n) + p, q, K, R, lut, nef, neo);
                d_sum += nef + 0x04040404u - neo;                       // d + 4 per byte; bytes stay <= 32
            }
            *reinterpret_cast<uint4 *>(P.plane_own + row + k0) = make_uint4(out[0], out[1], out[2], out[3]);
            delta += (int)byte_sum(d_sum) - 64;
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) delta += __shfl_xor_sync(0xffffffffu, delta, o);
    if (threadIdx.x == 0) atomicAdd(&blockD, delta);
    __syncthreads();
    if (tid == 0) atomicAdd(dE_out, (unsigned long long)(long long)blockD);
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
        const uint32_t p = (uint32_t)(i + 1) & 1u;                   // colour 1 sites
        const int iu = wrap(i - 1, P.L), id = wrap(i + 1, P.L);
        const size_t row = (size_t)i * P.pitch;
        const uint4 own4 = *reinterpret_cast<const uint4 *>(P.plane1 + row + k0);
        const uint4 mid4 = *reinterpret_cast<const uint4 *>(P.plane0 + row + k0);
        const uint32_t own[4] = {own4.x, own4.y, own4.z, own4.w};
        if (P.E_out) {
            const uint4 up4 = *reinterpret_cast<const uint4 *>(P.plane0 + (size_t)iu * P.pitch + k0);
            const uint4 dn4 = *reinterpret_cast<const uint4 *>(P.plane0 + (size_t)id * P.pitch + k0);
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
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) satisfied += __shfl_xor_sync(0xffffffffu, satisfied, o);
        if ((threadIdx.x & 31) == 0) atomicAdd(&blockE, (unsigned long long)satisfied);
    }
    __syncthreads();
    if (P.E_out && threadIdx.x == 0) atomicAdd(P.E_out, 0ull - blockE);
    if (do_hist) hist_flush(s_hist, P.q, P.hist_out, threadIdx.x, blockDim.x);
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
