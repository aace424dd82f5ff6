// microbench_issue.cu -- measurement tool, not part of the library: the integer issue model of a B200 SM
// sub-partition for the instruction mix of the Potts update, and the cost of each stage of update_word.
//
//   python -m paper_1101_0876_b200.build --microbench   ->  paper_1101_0876_b200/microbench_issue
//   ./paper_1101_0876_b200/microbench_issue             (one B200; prints cycles at 1965 MHz)
//
// Part 1: a Philox-like round (2 IMAD.WIDE + 2 LOP3 per chain, 4 independent chains per thread) plus K extra
// instructions of one kind per round on independent accumulators.  If the extra instructions ran on another
// pipe in parallel, the time per round would not move until that pipe filled up.
// Part 2: update_word of potts_core.cuh on register-resident data, stage by stage, at several occupancies.
// Results of round 1: profiles/r01b_pipe_model.md.
#include "potts_core.cuh"
#include <cstdio>
using namespace potts;

// ---- part 1 ---------------------------------------------------------------------------------------
template <int KA, int OP>
__global__ void __launch_bounds__(256) k_mix(uint32_t *out, int iters, uint32_t seed, uint32_t k0, uint32_t k1)
{
    constexpr int CH = 4;
    uint32_t c0[CH], c1[CH], c2[CH], c3[CH], a[8], m[8];
#pragma unroll
    for (int i = 0; i < CH; ++i) { c0[i] = seed + threadIdx.x * 8 + i; c1[i] = c0[i] * 3; c2[i] = c0[i] * 5; c3[i] = c0[i] * 7; }
#pragma unroll
    for (int i = 0; i < 8; ++i) { a[i] = seed * 11 + threadIdx.x + i; m[i] = a[i] * 3 + 1; }
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < 8; ++r) {
#pragma unroll
            for (int i = 0; i < CH; ++i) {
                uint32_t h0, l0, h1, l1;
                mul_wide(PHILOX_M0, c0[i], h0, l0);
                mul_wide(PHILOX_M1, c2[i], h1, l1);
                c0[i] = h1 ^ c1[i] ^ k0; c1[i] = l1; c2[i] = h0 ^ c3[i] ^ k1; c3[i] = l0;
            }
            k0 += PHILOX_W0; k1 += PHILOX_W1;
#pragma unroll
            for (int n = 0; n < KA * CH; ++n) {
                const int c = n & 7;
                if (OP == 0) asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(a[c]) : "r"(m[c]), "r"(m[(c + 1) & 7]));
                if (OP == 1) asm volatile("shf.r.wrap.b32 %0, %0, %1, 7;" : "+r"(a[c]) : "r"(m[c]));
                if (OP == 2) asm volatile("prmt.b32 %0, %0, %1, 0x5410;" : "+r"(a[c]) : "r"(m[c]));
                if (OP == 3) asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(a[c]) : "r"(m[c]), "r"(m[(c + 1) & 7]));
                if (OP == 4) asm volatile("{.reg .f32 t; mov.b32 t, %0; fma.rn.f32 t, t, %1, %2; mov.b32 %0, t;}" : "+r"(a[c]) : "f"(__uint_as_float(m[c])), "f"(__uint_as_float(m[(c + 1) & 7])));
                if (OP == 5) asm volatile("vabsdiff4.u32.u32.u32.add %0, %0, %1, %2;" : "+r"(a[c]) : "r"(m[c]), "r"(m[(c + 1) & 7]));
                if (OP == 6) asm volatile("mul.hi.u32 %0, %0, %1;" : "+r"(a[c]) : "r"(m[c]));
                if (OP == 7) asm volatile("popc.b32 %0, %0;" : "+r"(a[c]));
                if (OP == 8) asm volatile("dp4a.u32.u32 %0, %0, %1, %2;" : "+r"(a[c]) : "r"(m[c]), "r"(m[(c + 1) & 7]));
            }
        }
    }
    uint32_t r = 0;
#pragma unroll
    for (int i = 0; i < CH; ++i) r ^= c0[i] ^ c1[i] ^ c2[i] ^ c3[i];
#pragma unroll
    for (int i = 0; i < 8; ++i) r ^= a[i];
    out[blockIdx.x * blockDim.x + threadIdx.x] = r;
}

static float timed(void (*launch)(void))
{
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    launch(); cudaDeviceSynchronize();
    cudaEventRecord(e0); launch(); cudaEventRecord(e1); cudaEventSynchronize(e1);
    float ms; cudaEventElapsedTime(&ms, e0, e1);
    return ms;
}

static uint32_t *g_out, *g_thr;
constexpr int BPS = 8, MIX_ITERS = 500;

template <int KA, int OP>
void run_mix(const char *op)
{
    const float ms = timed([] { k_mix<KA, OP><<<148 * BPS, 256>>>(g_out, MIX_ITERS, 1, 5, 7); });
    const double rounds = (double)BPS * 8 / 4 * MIX_ITERS * 8 * 4;      // warp-rounds per sub-partition
    printf("round = 2 IMAD.WIDE + 2 LOP3, + %d x %-14s: %6.2f cycles per round\n", KA, op, ms * 1e-3 * 1.965e9 / rounds);
}

// ---- part 2 ---------------------------------------------------------------------------------------
template <int MODE>
__global__ void __launch_bounds__(256) kb(uint32_t *out, HalfSweepKeys K, uint32_t q, int iters, const uint32_t *thr)
{
    __shared__ uint32_t lut[12];
    if (threadIdx.x < 9) lut[threadIdx.x] = threadIdx.x >= 5 ? thr[threadIdx.x - 5] : 0u;
    __syncthreads();
    uint32_t own = threadIdx.x * 0x01020304u & 0x07070707u, up = own ^ 0x01000100u, dn = own ^ 0x00010000u, lf = own, rt = up;
    uint32_t acc = 0;
    const uint32_t qq = in_register(q);
    uint32_t j0 = blockIdx.x * 1024u + threadIdx.x * 8u;
    for (int it = 0; it < iters; ++it) {
        const RowKeys R = row_keys(K, (uint32_t)it);
        if (MODE == 0) {            // philox only
            uint32_t w0, w1;
#pragma unroll
            for (int b = 0; b < 4; ++b) { philox_site(K, R, j0 + 2u * b, w0, w1); acc ^= w0 + w1; }
        } else if (MODE == 1) {     // full update
            uint32_t nef;
            own = update_word<CM_7BIT, 1>(own, up, dn, lf, rt, j0, qq, K, R, lut, nef);
            acc += nef; up ^= own; 
        } else if (MODE == 2) {     // philox + proposal only
            uint32_t w0[4], w1[4];
#pragma unroll
            for (int b = 0; b < 4; ++b) philox_site(K, R, j0 + 2u * b, w0[b], w1[b]);
            const uint32_t s01 = __byte_perm(__umulhi(w0[0], qq), __umulhi(w0[1], qq), 0x0040);
            const uint32_t s23 = __byte_perm(__umulhi(w0[2], qq), __umulhi(w0[3], qq), 0x0040);
            acc ^= __byte_perm(s01, s23, 0x5410) ^ w1[0] ^ w1[1] ^ w1[2] ^ w1[3];
        } else if (MODE == 3) {     // philox + proposal + compares (no acceptance)
            uint32_t w0[4], w1[4];
#pragma unroll
            for (int b = 0; b < 4; ++b) philox_site(K, R, j0 + 2u * b, w0[b], w1[b]);
            const uint32_t s01 = __byte_perm(__umulhi(w0[0], qq), __umulhi(w0[1], qq), 0x0040);
            const uint32_t s23 = __byte_perm(__umulhi(w0[2], qq), __umulhi(w0[3], qq), 0x0040);
            const uint32_t prop = __byte_perm(s01, s23, 0x5410);
            const uint32_t c_old = ne_count4<false>(own, up, dn, lf, rt);
            const uint32_t c_new = ne_count4<false>(prop, up, dn, lf, rt);
            const uint32_t dw = c_new + 0x04040404u - c_old;
            acc ^= dw ^ w1[0] ^ w1[1] ^ w1[2] ^ w1[3]; up ^= dw; own ^= prop & 0x07070707u;
        }
        j0 += 8u;
    }
    out[blockIdx.x * blockDim.x + threadIdx.x] = acc ^ own;
}

template <int MODE>
void run_stage(const char *name, int blocks_per_sm, int iters, uint32_t *d_out, uint32_t *d_thr)
{
    HalfSweepKeys K = half_sweep_keys(12345u, 678u, 42u, 1u);
    cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
    const int grid = 148 * blocks_per_sm;
    kb<MODE><<<grid, 256>>>(d_out, K, 9u, iters, d_thr);
    cudaDeviceSynchronize();
    cudaEventRecord(e0);
    kb<MODE><<<grid, 256>>>(d_out, K, 9u, iters, d_thr);
    cudaEventRecord(e1); cudaEventSynchronize(e1);
    float ms; cudaEventElapsedTime(&ms, e0, e1);
    // warp-updates per SMSP: blocks_per_sm * 8 warps / 4 SMSPs * iters * 4 sites
    const double wu = (double)blocks_per_sm * 8 / 4 * iters * 4;
    const double cyc = ms * 1e-3 * 1.965e9 / wu;
    printf("%-28s occ=%2d warps/SMSP  %.2f cycles/warp-update  %.3f ps/update\n", name, blocks_per_sm * 2, cyc,
           ms * 1e9 / ((double)grid * 256 * iters * 4));
}


int main()
{
    cudaMalloc(&g_out, 148 * 8 * 256 * 4);
    cudaMalloc(&g_thr, 16);
    const uint32_t thr[4] = {1066287806u, 264721383u, 65720915u, 16316168u};     // config 5's thresholds
    cudaMemcpy(g_thr, thr, 16, cudaMemcpyHostToDevice);
    printf("part 1: 16 warps per sub-partition, 4 chains per thread\n");
    run_mix<0, 0>("(nothing)");
    run_mix<1, 0>("LOP3"); run_mix<2, 0>("LOP3"); run_mix<4, 0>("LOP3"); run_mix<6, 0>("LOP3");
    run_mix<2, 1>("SHF"); run_mix<2, 2>("PRMT"); run_mix<2, 3>("IMAD"); run_mix<2, 4>("FFMA"); run_mix<2, 5>("VABSDIFF4.ACC");
    run_mix<2, 6>("IMAD.HI"); run_mix<2, 7>("POPC"); run_mix<2, 8>("IDP.4A");
    printf("part 2: update_word, register-resident, stage by stage\n");
    for (int bps : {1, 2, 4, 8}) {
        run_stage<0>("philox only", bps, 2000, g_out, g_thr);
        run_stage<2>("philox+proposal", bps, 2000, g_out, g_thr);
        run_stage<3>("philox+proposal+compare", bps, 2000, g_out, g_thr);
        run_stage<1>("full update_word", bps, 2000, g_out, g_thr);
    }
    printf("%s\n", cudaGetErrorString(cudaGetLastError()));
    return 0;
}
