// potts_api.cu -- the C-ABI of include/potts.h: argument checking, device memory, launches.
// Every step of the hot path runs in the kernels of potts_kernels.cuh; this file only marshals.
#include "../../include/potts.h"
#include "potts_launch.cuh"

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>
#include <thread>
#include <vector>

namespace {

thread_local std::string g_err;

int fail(int code, const char *fmt, ...)
{
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    g_err = buf;
    return code;
}

#define CUDA_TRY(expr)                                                                          \
    do {                                                                                        \
        cudaError_t e_ = (expr);                                                                \
        if (e_ != cudaSuccess)                                                                  \
            return fail(e_ == cudaErrorMemoryAllocation ? POTTS_ERR_NOMEM : POTTS_ERR_CUDA,     \
                        "%s failed: %s", #expr, cudaGetErrorString(e_));                        \
    } while (0)

// Entry points run on the handle's device whatever the caller's current device is (and restore it afterwards).
struct DeviceGuard {
    int prev = -1;
    explicit DeviceGuard(int dev)
    {
        if (cudaGetDevice(&prev) != cudaSuccess) { prev = -1; return; }
        if (prev != dev) cudaSetDevice(dev); else prev = -1;
    }
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};
#define ON_DEVICE_OF(x) DeviceGuard guard_((x) ? (x)->device : current_device())
inline int current_device() { int d = 0; cudaGetDevice(&d); return d; }

constexpr size_t ALIGN = 256;
constexpr size_t align_up(size_t x) { return (x + ALIGN - 1) / ALIGN * ALIGN; }
constexpr int MAX_CTAS = 160;             // upper bound on the resident kernel's grid (>= SM count of B200)
constexpr int RESIDENT_L_MAX = 4096;       // largest lattice the resident kernel can hold (512 words per row)
constexpr int CLUSTER_AUTO_L_MAX = 288;    // lattices up to this size go to the cluster (DSMEM) kernel by default (measured, profiles/r02h_cluster_exchange.md: 2.3x the resident kernel at L = 128, 1.2x at L = 288, 0.96x at L = 320)
constexpr int ACC_WORDS = 1 + 256 + 2;    // E, hist[256], flag/error word, tile counter of the streaming kernels
constexpr size_t STATIC_SMEM = sizeof(potts::AcceptLutWide) + 1024;   // static shared memory of the persistent kernels

}  // namespace

namespace potts {
// the thread-local error message of potts_last_error(), for the other host translation units (potts3d_api.cu)
int set_error(int code, const char *msg) { g_err = msg; return code; }
}  // namespace potts

struct potts_s {
    int32_t L = 0, q = 0, layout = 0;
    int32_t rows = 0, row0 = 0;          // rows held by this handle: the whole lattice (rows = L, row0 = 0) or a row strip of it
    bool strip = false;                  // row strip of a lattice split over several GPUs: halo rows instead of the periodic wrap
    int device = 0;                      // the CUDA device the handle lives on; every entry point runs on it
    uint64_t seed = 0, t = 0;
    uint8_t *ws = nullptr;
    bool owns_ws = false;
    size_t plane_bytes = 0;
    uint8_t *plane[2] = {nullptr, nullptr};
    potts::PackedPlanes pk = {};          // PACKED layout: nibble / high-bit planes inside plane[c]
    unsigned long long *acc = nullptr;   // device scratch: [0] = E, [1..q] = histogram
    int *flag = nullptr;                 // device scratch flag (upload validation)
    int *error = nullptr;                // device: set by the resident kernel if a neighbour wait gave up
    uint32_t *tile_counter = nullptr;    // device: tile counter of the streaming kernels (0 between launches)
    uint8_t *inbox = nullptr;            // device: resident kernel's boundary-row packets (null if L too large)
    cudaStream_t stream = nullptr;
    uint64_t launches = 0;
    int num_sms = 0;
    size_t smem_optin = 0;
    int coop = 0;                        // device supports cooperative launches (the resident kernel needs one)
    uint8_t *scratch = nullptr;          // device scratch kept between calls (staging for up/download, host-series buffers)
    size_t scratch_bytes = 0;
    cudaStream_t copy_stream = nullptr;  // up/download: PCIe copies run here, conversions on `stream`
    cudaEvent_t ev_copied[2] = {nullptr, nullptr}, ev_converted[2] = {nullptr, nullptr}, ev_start = nullptr;
    // options (how to launch, never what is computed)
    int32_t stream_spec = 1;             // random-stream definition (1 = R3, 2 = R3'): changes the chain, not an option
    int64_t opt_variant = 0;             // 0 auto, 1 streaming (one launch per half-sweep), 2 resident
    int64_t opt_resident_ctas = 0;       // 0 auto, else the resident kernel's grid size
    int64_t opt_resident_words = 0;      // 0 auto, 1 / 2: 4-site words per thread and row visit
    int64_t opt_resident_rows = 0;       // 0 auto, else at most this many thread rows in a resident block
    int64_t opt_cluster_ctas = 0;        // 0 auto, else the cluster kernel's cluster size (1..16)
    int cluster_checked = 0;             // cluster size whose co-residency was confirmed (cudaOccupancyMaxActiveClusters)
    int64_t opt_resident_col = 1;        // 1: ColKeys table in the resident kernel where it pays; 0: never
    int64_t opt_stream_stage = 0;        // 0: other-colour rows through registers; 1: staged in shared memory by cp.async.bulk (experiment)
    int64_t opt_stream_rows = 0;         // 0 auto, else rows per warp of the streaming kernel (even, divides L/4)
};

namespace {

int check_shape(int32_t L, int32_t q, int32_t layout)
{
    if (L < 2 || (L & 1)) return fail(POTTS_ERR_ARG, "L = %d must be even and >= 2", L);
    if (q < 2 || q > 256) return fail(POTTS_ERR_ARG, "q = %d outside [2, 256]", q);
    if (layout != POTTS_LAYOUT_U8 && layout != POTTS_LAYOUT_PACKED)
        return fail(POTTS_ERR_ARG, "unknown layout %d", layout);
    if (L % 32 != 0)
        return fail(POTTS_ERR_UNSUPPORTED, "L = %d is not a multiple of 32 (kernel vector width)", L);
    if (layout == POTTS_LAYOUT_PACKED) {
        if (q > 32) return fail(POTTS_ERR_UNSUPPORTED, "packed layout holds at most 5 bits per spin: q = %d > 32", q);
        if (L % 64 != 0) return fail(POTTS_ERR_UNSUPPORTED, "packed layout needs L %% 64 == 0, L = %d", L);
    }
    return POTTS_OK;
}

// bytes of ONE colour plane: U8 L*L/2; packed L*L/4 of nibbles (+ L*L/16 of high bits when q > 16)
size_t nib_bytes_of(int32_t L) { return align_up((size_t)L * (size_t)(L / 4)); }
size_t hb_bytes_of(int32_t L, int32_t q) { return q > 16 ? align_up((size_t)L * (size_t)(L / 16)) : 0; }
size_t plane_bytes_of(int32_t L, int32_t q, int32_t layout)
{
    return layout == POTTS_LAYOUT_PACKED ? nib_bytes_of(L) + hb_bytes_of(L, q) : align_up((size_t)L * (size_t)(L / 2));
}

// resident kernel: per CTA 2 colours x 2 sides x L/8 packets of 8 bytes
size_t inbox_bytes_of(int32_t L) { return L <= RESIDENT_L_MAX ? align_up((size_t)MAX_CTAS * 4 * (size_t)L) : 0; }

size_t workspace_bytes_of(int32_t L, int32_t q, int32_t layout)
{
    return 2 * plane_bytes_of(L, q, layout) + align_up(ACC_WORDS * sizeof(unsigned long long)) + inbox_bytes_of(L) + ALIGN;
}

void thresholds(double T, uint32_t thr[4])
{
    // reading R6: exactly floor(ldexp(exp(-d/T), 32)) in double
    for (int d = 1; d <= 4; ++d) thr[d - 1] = (uint32_t)std::floor(std::ldexp(std::exp(-(double)d / T), 32));
}

// device scratch of at least `bytes`, kept in the handle so that repeated calls do not pay cudaMalloc / cudaFree
int get_scratch(potts_t *h, size_t bytes, uint8_t **out)
{
    if (h->scratch_bytes < bytes) {
        if (h->scratch) { cudaStreamSynchronize(h->stream); cudaFree(h->scratch); h->scratch = nullptr; h->scratch_bytes = 0; }
        CUDA_TRY(cudaMalloc(&h->scratch, bytes));
        h->scratch_bytes = bytes;
    }
    *out = h->scratch;
    return POTTS_OK;
}

int check_launch(potts_t *h, const char *what)
{
    h->launches += 1;
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(POTTS_ERR_CUDA, "launch of %s failed: %s", what, cudaGetErrorString(e));
    return POTTS_OK;
}

potts::SweepParams sweep_params(const potts_t *h, uint32_t colour, const uint32_t thr[4], unsigned long long *E_out)
{
    potts::SweepParams P;
    P.plane_own = h->plane[colour];
    P.plane_oth = h->plane[1 - colour];
    P.L = h->L;
    P.pitch = h->L / 2;
    P.q = (uint32_t)h->q;
    P.colour = colour;
    P.K = potts::half_sweep_keys((uint32_t)(h->seed & 0xFFFFFFFFull), (uint32_t)(h->seed >> 32), (uint32_t)h->t, colour);
    for (int d = 0; d < 4; ++d) P.thr[d] = thr[d];
    P.E_out = E_out;
    P.rows = h->rows;
    P.row0 = h->row0;
    P.strip = h->strip ? 1 : 0;
    return P;
}

// Rows per warp of a tile of the streaming kernels (L % 32 == 0, so 8 divides L / HS_WARPS).  Tiles are drawn from a
// counter by as many blocks as are resident at once, so small tiles cost nothing but the two neighbour rows a warp
// loads before its first visit; measured on B200 (profiles/r02b_kernels.md).
constexpr int STREAM_ROWS_PER_WARP = 8;

// delta = true: E_out receives the sum of the accepted moves' d instead of the energy (hist_out must be null)
int launch_half_sweep(potts_t *h, uint32_t colour, const uint32_t thr[4], unsigned long long *E_out,
                      unsigned long long *hist_out, bool delta = false)
{
    potts::SweepParams P = sweep_params(h, colour, thr, E_out);
    P.hist_out = hist_out;
    const int chunks = h->L / 32;
    const unsigned gx = (unsigned)((chunks + 31) / 32);
    P.rpw = h->opt_stream_rows > 0 ? (int)h->opt_stream_rows : STREAM_ROWS_PER_WARP;
    P.row_groups = h->rows / (potts::HS_WARPS * P.rpw);
    P.total_tiles = gx * (uint32_t)P.row_groups;
    P.tile_counter = h->tile_counter;
    P.bulk = (h->opt_stream_stage == 1 && (h->L / 2) % 512 == 0 && P.rpw + 2 <= 32) ? 1 : 0;
    const size_t smem = hist_out ? (size_t)potts::hist_words((uint32_t)h->q) * 4 : 0;
    potts::launch_sweep_rows_u8(potts::compare_mode_of(h->q), h->stream_spec, delta, P, h->num_sms, smem, h->stream);
    return check_launch(h, "k_sweep_rows_u8");
}

// delta = true: E_out receives the sum of the accepted moves' d instead of the energy (hist_out must be null)
int launch_half_sweep_packed(potts_t *h, uint32_t colour, const uint32_t thr[4], unsigned long long *E_out,
                             unsigned long long *hist_out, bool delta = false)
{
    potts::PackedSweepParams P;
    P.S = h->pk;
    P.q = (uint32_t)h->q;
    P.colour = colour;
    P.K = potts::half_sweep_keys((uint32_t)(h->seed & 0xFFFFFFFFull), (uint32_t)(h->seed >> 32), (uint32_t)h->t, colour);
    for (int d = 0; d < 4; ++d) P.thr[d] = thr[d];
    P.E_out = E_out;
    P.hist_out = hist_out;
    const int chunks = h->L / 64;
    const unsigned gx = (unsigned)((chunks + 31) / 32);
    // rows per warp: 8, or 4 while that leaves fewer than four tiles per resident block (3 per SM): L = 8192 is 1024 tiles
    // of 32 rows instead of 512 of 64 (measured 2.75 against 3.11 ps per update; L = 16384: 2.29 with 8, 2.32 with 4)
    P.rpw = STREAM_ROWS_PER_WARP;
    if ((long long)gx * (h->L / (potts::PK_WARPS * P.rpw)) < 4ll * potts::PK_MIN_BLOCKS * h->num_sms) P.rpw = 4;
    if (h->opt_stream_rows > 0) P.rpw = (int)h->opt_stream_rows;
    while ((h->L / potts::PK_WARPS) % P.rpw) P.rpw >>= 1;               // L % 64 == 0: 2, 4 and 8 always divide
    P.row_groups = h->L / (potts::PK_WARPS * P.rpw);
    P.total_tiles = gx * (uint32_t)P.row_groups;
    P.tile_counter = h->tile_counter;
    const size_t smem = hist_out ? (size_t)potts::hist_words((uint32_t)h->q) * 4 : 0;
    potts::launch_sweep_rows_packed(h->q > 16, h->stream_spec, delta, P, h->num_sms, smem, h->stream);
    return check_launch(h, "k_sweep_rows_packed");
}

int launch_measure(potts_t *h, unsigned long long *E_out, unsigned long long *hist_out)
{
    if (h->layout == POTTS_LAYOUT_PACKED) {
        potts::PackedMeasureParams M;
        M.S = h->pk;
        M.q = (uint32_t)h->q;
        M.E_out = E_out;
        M.hist_out = hist_out;
        long long blocks = ((long long)h->L * (h->L / 64) + 255) / 256;
        if (blocks > 148 * 8) blocks = 148 * 8;
        const size_t smem = hist_out ? (size_t)h->q * 32 * 4 : 0;
        if (h->q > 16) potts::k_measure_packed<true><<<(unsigned)blocks, 256, smem, h->stream>>>(M);
        else potts::k_measure_packed<false><<<(unsigned)blocks, 256, smem, h->stream>>>(M);
        return check_launch(h, "k_measure_packed");
    }
    potts::MeasureParams M;
    M.plane0 = h->plane[0];
    M.plane1 = h->plane[1];
    M.L = h->rows;
    M.pitch = h->L / 2;
    M.row0 = h->row0;
    M.strip = h->strip ? 1 : 0;
    M.q = (uint32_t)h->q;
    M.E_out = E_out;
    M.hist_out = hist_out;
    const long long threads = (long long)h->rows * (h->L / 32);
    const int block = 256;
    long long blocks = (threads + block - 1) / block;
    if (blocks > 148 * 8) blocks = 148 * 8;
    const size_t smem = hist_out ? (size_t)(h->q <= (int)potts::HIST_LANE_QMAX ? h->q * 32 : h->q) * 4 : 0;
    if (h->q > 128) potts::k_measure_u8<true><<<(unsigned)blocks, block, smem, h->stream>>>(M);
    else potts::k_measure_u8<false><<<(unsigned)blocks, block, smem, h->stream>>>(M);
    return check_launch(h, "k_measure_u8");
}

int check_sweep_args(potts_t *h, double T, int64_t nsweeps)
{
    if (!h) return fail(POTTS_ERR_ARG, "null handle");
    if (h->strip) return fail(POTTS_ERR_UNSUPPORTED, "a row strip is advanced half-sweep by half-sweep (potts_strip_half_sweep): its halo rows must be exchanged in between");
    if (!(T > 0.0) || !std::isfinite(T)) return fail(POTTS_ERR_ARG, "T = %g must be finite and > 0", T);
    if (nsweeps < 0) return fail(POTTS_ERR_ARG, "nsweeps = %lld < 0", (long long)nsweeps);
    if (h->t + (uint64_t)nsweeps > 0xFFFFFFFFull)
        return fail(POTTS_ERR_ARG, "sweep counter would pass 2^32 - 1 (Philox counter word)");
    return POTTS_OK;
}

// ---- resident (persistent, shared-memory) path ------------------------------------------------
struct ResidentPlan {
    bool ok = false;
    int G = 0, tyc = 0, wpr = 0, rows_max = 0, nthreads = 0, W = 2;
    size_t smem = 0;
    bool col = false;                    // ColKeys table in shared memory (W = 2, >= 3 visits per thread)
    uint32_t col_offset = 0;
    const char *why = "";
};

ResidentPlan plan_resident(const potts_t *h)
{
    ResidentPlan R;
    const int L = h->L;
    R.wpr = L / 8;
    if (h->layout != POTTS_LAYOUT_U8) { R.why = "the resident kernel holds the U8 layout only"; return R; }
    if (!h->coop) { R.why = "the device does not support cooperative launches"; return R; }
    if (L > RESIDENT_L_MAX || !h->inbox) { R.why = "L exceeds the resident kernel's 512 words per row"; return R; }
    const long long words = (long long)L * R.wpr;                   // 4-site words per half-sweep
    long long G = h->opt_resident_ctas > 0 ? h->opt_resident_ctas : words / 256;   // measured (profiles/r01c_kernels.md): one CTA per 256 words of a half-sweep
    if (G < 1) G = 1;
    if (G > h->num_sms) G = h->num_sms;
    if (G > L) G = L;
    if (G > MAX_CTAS) G = MAX_CTAS;
    R.G = (int)G;
    R.rows_max = (L + R.G - 1) / R.G;
    // block = compute warps (L/16 chunks x tyc rows at a time) + comm warps (L/16 threads)
    const int cpr = L / 16;
    // comm threads: one 8-site chunk of a halo row each up to L = 2048; beyond that 64 threads share the chunks: they need
    // few registers but are allocated the compute threads' budget, and 576 instead of 768 threads per block at L = 4096
    // lets the compute threads have 112 registers instead of 80 (measured: cfg3 2.79 -> 2.67 ps; at L = 2048, where the
    // block stays under 576 threads either way, sharing costs 2 %)
    const int comm = cpr <= 128 ? (cpr + 31) / 32 * 32 : 64;
    int tyc = (1024 - comm) / cpr;
    if (tyc > R.rows_max) tyc = R.rows_max;
    if (tyc < 1) { R.why = "no room for a compute row in a 1024-thread block"; return R; }
    int threads_per_row = cpr;
    // One 4-site word per thread and row visit (W = 1) instead of an 8-site chunk (W = 2) wherever every thread still
    // visits at most two rows inside a 576-thread block (112 registers): twice the warps for the latency-bound small
    // lattices, and at L = 1024 on 148 SMs an even load on the four sub-partitions of an SM (7 rows as chunks are
    // 14 warps -> 4,4,3,3; as words over 4 thread rows of 4 warps each: three thread rows with 2 rows, one with 1).
    // Measured (profiles/r01c_kernels.md): 4 % faster at L = 1024, 20 - 40 % at L <= 512.  Larger lattices keep W = 2.
    {
        int t1 = (576 - comm) / (2 * cpr);
        if (t1 > R.rows_max) t1 = R.rows_max;
        const bool fits = t1 >= 1 && t1 >= (R.rows_max + 1) / 2;
        if (h->opt_resident_words == 1 ? (t1 >= 1) : (h->opt_resident_words == 0 && fits)) {
            R.W = 1;
            threads_per_row = 2 * cpr;
            tyc = t1;
        }
    }
    if (R.W == 2 && h->opt_resident_rows == 0) {
        // thread rows for the chunk-grained kernel: fewer rows than fit can be better, because the last visit of an
        // uneven deal idles part of the block and blocks above 768 threads are held to 64 registers.  Cost model fitted
        // to the measurements in profiles/r01c_kernels.md (L = 2048: 3 rows, L = 4096: 2 rows).
        double best = 1e30;
        int best_t = tyc;
        for (int t = tyc; t >= 1; --t) {
            const int visits = (R.rows_max + t - 1) / t;
            const int threads = (cpr * t + 31) / 32 * 32 + comm, warps = cpr * t / 32;
            double cost = (double)visits * t / R.rows_max;
            if (threads > 768) cost *= 1.08;
            if (warps < 12) cost *= 1.0 + 0.025 * (12 - warps);
            if (visits > 30) continue;
            if (cost < best - 1e-9) { best = cost; best_t = t; }
        }
        tyc = best_t;
    }
    if (h->opt_resident_rows > 0 && h->opt_resident_rows < tyc) tyc = (int)h->opt_resident_rows;
    R.tyc = tyc;
    R.nthreads = (threads_per_row * tyc + 31) / 32 * 32 + comm;
    if ((R.rows_max + tyc - 1) / tyc > 30) { R.why = "too many rows per thread"; return R; }
    const size_t hist = (size_t)(h->q <= (int)potts::HIST_LANE_QMAX ? h->q * 32 : h->q) * 4;
    R.smem = 2 * (size_t)(R.rows_max + 2) * (L / 2) + hist;
    if (R.smem + STATIC_SMEM > h->smem_optin) { R.why = "lattice does not fit the shared memory of the grid"; return R; }
    // the column part of Philox shared by a thread's visits of a half-sweep: 16 L bytes more, if they fit
    const int visits = (R.rows_max + tyc - 1) / tyc;
    const size_t col_at = (R.smem + 15) / 16 * 16;
    if (R.W == 2 && visits >= 3 && h->opt_resident_col != 0 && col_at + 16 * (size_t)L + STATIC_SMEM <= h->smem_optin) {
        R.col = true;
        R.col_offset = (uint32_t)col_at;
        R.smem = col_at + 16 * (size_t)L;
    }
    R.ok = true;
    return R;
}

int launch_resident(potts_t *h, const ResidentPlan &R, const uint32_t thr[4], int64_t nsweeps, int64_t every,
                    unsigned long long *E_series_dev, unsigned long long *hist_series_dev, unsigned long long *dE_series_dev)
{
    potts::ResidentParams P;
    P.plane[0] = h->plane[0];
    P.plane[1] = h->plane[1];
    P.L = h->L;
    P.pitch = h->L / 2;
    P.q = (uint32_t)h->q;
    P.key0 = (uint32_t)(h->seed & 0xFFFFFFFFull);
    P.key1 = (uint32_t)(h->seed >> 32);
    for (int d = 0; d < 4; ++d) P.thr[d] = thr[d];
    P.t0 = (uint32_t)h->t;
    P.nsweeps = (uint32_t)nsweeps;
    P.every = (uint32_t)every;
    P.E_series = E_series_dev;
    P.hist_series = hist_series_dev;
    P.dE_series = dE_series_dev;
    P.inbox = (uint2 *)h->inbox;
    P.error = h->error;
    P.rows_max = R.rows_max;
    P.tyc = R.tyc;
    P.col_offset = R.col_offset;
    const void *fn = potts::resident_kernel(potts::compare_mode_of(h->q), h->stream_spec, R.col ? 3 : R.W, R.nthreads <= 576 ? 2 : (R.nthreads <= 768 ? 1 : 0));
    CUDA_TRY(cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)R.smem));
    int per_sm = 0;
    CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, fn, R.nthreads, R.smem));
    if (per_sm < 1 || (long long)per_sm * h->num_sms < R.G)
        return fail(POTTS_ERR_UNSUPPORTED, "resident kernel: %d CTAs cannot be co-resident", R.G);
    // packet sequence numbers restart at 1 in every launch: clear what the previous launch left
    if (R.G > 1) CUDA_TRY(cudaMemsetAsync(h->inbox, 0, (size_t)R.G * 4 * (size_t)h->L, h->stream));
    void *args[] = {(void *)&P};
    CUDA_TRY(cudaLaunchCooperativeKernel(fn, dim3((unsigned)R.G), dim3((unsigned)R.nthreads), args, R.smem, h->stream));
    h->launches += 1;
    return POTTS_OK;
}

// ---- cluster (DSMEM) path for tiny lattices -------------------------------------------------------
struct ClusterPlan { bool ok = false; int G = 0, tyc = 0, rows_max = 0, nthreads = 0; size_t smem = 0; const char *why = ""; };

ClusterPlan plan_cluster(const potts_t *h)
{
    ClusterPlan R;
    const int L = h->L, wpr = L / 8;
    if (h->layout != POTTS_LAYOUT_U8) { R.why = "the cluster kernel holds the U8 layout only"; return R; }
    if (wpr > 1024) { R.why = "L/8 words per row exceed 1024 threads"; return R; }
    long long G = h->opt_cluster_ctas > 0 ? h->opt_cluster_ctas : ((long long)L * wpr) / 128;   // measured: one CTA per 128 words of a half-sweep: L = 64 -> 4, L = 128 -> 16 (beyond 8 is the non-portable cluster size)
    if (G < 1) G = 1;
    if (G > potts::CLUSTER_MAX) G = potts::CLUSTER_MAX;
    if (G > L) G = L;
    R.G = (int)G;
    R.rows_max = (L + R.G - 1) / R.G;
    int tyc = 1024 / wpr;
    if (tyc > R.rows_max) tyc = R.rows_max;
    R.tyc = tyc;
    R.nthreads = (wpr * tyc + 31) / 32 * 32;
    if ((R.rows_max + tyc - 1) / tyc > 60) { R.why = "too many rows per thread"; return R; }
    const size_t hist = 2 * (size_t)(h->q <= (int)potts::HIST_LANE_QMAX ? h->q * 32 : h->q) * 4;   // two tables
    R.smem = 2 * (size_t)(R.rows_max + 2) * (L / 2) + hist + 8 * (size_t)(L / 2);   // planes, histogram tables, packet inbox
    if (R.smem + STATIC_SMEM > h->smem_optin) { R.why = "lattice does not fit the shared memory of one cluster"; return R; }
    R.ok = true;
    return R;
}

int launch_cluster(potts_t *h, const ClusterPlan &R, const uint32_t thr[4], int64_t nsweeps, int64_t every,
                   unsigned long long *E_series_dev, unsigned long long *hist_series_dev, unsigned long long *dE_series_dev)
{
    potts::ResidentParams P = {};
    P.plane[0] = h->plane[0];
    P.plane[1] = h->plane[1];
    P.L = h->L;
    P.pitch = h->L / 2;
    P.q = (uint32_t)h->q;
    P.key0 = (uint32_t)(h->seed & 0xFFFFFFFFull);
    P.key1 = (uint32_t)(h->seed >> 32);
    for (int d = 0; d < 4; ++d) P.thr[d] = thr[d];
    P.t0 = (uint32_t)h->t;
    P.nsweeps = (uint32_t)nsweeps;
    P.every = (uint32_t)every;
    P.E_series = E_series_dev;
    P.hist_series = hist_series_dev;
    P.dE_series = dE_series_dev;
    P.error = h->error;
    P.rows_max = R.rows_max;
    P.tyc = R.tyc;
    const void *fn = potts::cluster_kernel(potts::compare_mode_of(h->q), h->stream_spec, R.nthreads);
    CUDA_TRY(cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)R.smem));
    if (R.G > 8) CUDA_TRY(cudaFuncSetAttribute(fn, cudaFuncAttributeNonPortableClusterSizeAllowed, 1));
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)R.G);
    cfg.blockDim = dim3((unsigned)R.nthreads);
    cfg.dynamicSmemBytes = R.smem;
    cfg.stream = h->stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = (unsigned)R.G;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    if (h->cluster_checked != R.G) {
        // a cluster of this size may not be schedulable here (MIG slice, partial GPC): say so, the caller falls back
        int nclusters = 0;
        const cudaError_t eo = cudaOccupancyMaxActiveClusters(&nclusters, fn, &cfg);
        if (eo != cudaSuccess || nclusters < 1) {
            cudaGetLastError();
            return fail(POTTS_ERR_UNSUPPORTED, "a cluster of %d CTAs x %d threads with %zu bytes of shared memory cannot be scheduled on this device", R.G, R.nthreads, R.smem);
        }
        h->cluster_checked = R.G;
    }
    void *args[] = {(void *)&P};
    CUDA_TRY(cudaLaunchKernelExC(&cfg, fn, args));
    h->launches += 1;
    return POTTS_OK;
}

// The sweep loop shared by every entry point that sweeps.  every = 0: no samples.  dE_series_dev (nsweeps zeroed
// int64 slots, or null): slot n += the energy change of sweep n, summed over its accepted moves.
int run_sweeps(potts_t *h, double T, int64_t nsweeps, int64_t every, unsigned long long *E_series_dev,
               unsigned long long *hist_series_dev, unsigned long long *dE_series_dev = nullptr)
{
    uint32_t thr[4];
    thresholds(T, thr);
    if (nsweeps == 0) return POTTS_OK;
    // the persistent kernels' sweep and sample counters are 32-bit: long calls are split into pieces of whole samples
    const int64_t piece = every > 0 ? ((1ll << 30) / every) * every : (1ll << 30);
    if (h->opt_variant == 3 || (h->opt_variant == 0 && h->layout == POTTS_LAYOUT_U8 && h->L <= CLUSTER_AUTO_L_MAX)) {
        const ClusterPlan C = plan_cluster(h);
        bool cluster_ok = true;
        if (C.ok) {
            for (int64_t done = 0; done < nsweeps;) {
                const int64_t n = nsweeps - done < piece ? nsweeps - done : piece;
                const int64_t s0 = every > 0 ? done / every : 0;
                int rc = launch_cluster(h, C, thr, n, every > 0 ? every : 0, E_series_dev ? E_series_dev + s0 : nullptr,
                                        hist_series_dev ? hist_series_dev + s0 * h->q : nullptr,
                                        dE_series_dev ? dE_series_dev + done : nullptr);
                if (rc == POTTS_ERR_UNSUPPORTED && done == 0 && h->opt_variant == 0) { cluster_ok = false; break; }
                if (rc) return rc;
                h->t += (uint64_t)n;
                done += n;
            }
            if (cluster_ok) return POTTS_OK;                         // else: automatic mode falls through to the resident kernel
        }
        if (h->opt_variant == 3) return fail(POTTS_ERR_UNSUPPORTED, "cluster variant unavailable: %s", C.why);
    }
    if (h->opt_variant != 1) {
        const ResidentPlan R = plan_resident(h);
        if (R.ok) {
            for (int64_t done = 0; done < nsweeps;) {
                const int64_t n = nsweeps - done < piece ? nsweeps - done : piece;
                const int64_t s0 = every > 0 ? done / every : 0;
                int rc = launch_resident(h, R, thr, n, every > 0 ? every : 0,
                                         E_series_dev ? E_series_dev + s0 : nullptr,
                                         hist_series_dev ? hist_series_dev + s0 * h->q : nullptr,
                                         dE_series_dev ? dE_series_dev + done : nullptr);
                if (rc) return rc;
                h->t += (uint64_t)n;
                done += n;
            }
            return POTTS_OK;
        }
        if (h->opt_variant == 2) return fail(POTTS_ERR_UNSUPPORTED, "resident variant unavailable: %s", R.why);
    }
    const bool pk = h->layout == POTTS_LAYOUT_PACKED;
    for (int64_t n = 0; n < nsweeps; ++n) {
        int rc;
        if (dE_series_dev) {
            // streaming kernels: the energy-change form of the half-sweep (no samples in the same call)
            for (uint32_t c = 0; c < 2; ++c) {
                rc = pk ? launch_half_sweep_packed(h, c, thr, dE_series_dev + n, nullptr, true)
                        : launch_half_sweep(h, c, thr, dE_series_dev + n, nullptr, true);
                if (rc) return rc;
            }
            h->t += 1;
            continue;
        }
        const bool sample = every > 0 && ((n + 1) % every == 0);
        const int64_t idx = sample ? (n + 1) / every - 1 : 0;
        unsigned long long *Hs = (sample && hist_series_dev) ? hist_series_dev + idx * h->q : nullptr;
        unsigned long long *Es = (sample && E_series_dev) ? E_series_dev + idx : nullptr;
        rc = pk ? launch_half_sweep_packed(h, 0u, thr, nullptr, Hs) : launch_half_sweep(h, 0u, thr, nullptr, Hs);
        if (rc) return rc;
        rc = pk ? launch_half_sweep_packed(h, 1u, thr, Es, Hs) : launch_half_sweep(h, 1u, thr, Es, Hs);
        if (rc) return rc;
        h->t += 1;
    }
    return POTTS_OK;
}

// after a stream sync: did a resident launch give up waiting for a neighbour?
int check_device_error(potts_t *h)
{
    int e = 0;
    CUDA_TRY(cudaMemcpyAsync(&e, h->error, sizeof(int), cudaMemcpyDeviceToHost, h->stream));
    CUDA_TRY(cudaStreamSynchronize(h->stream));
    if (e) return fail(POTTS_ERR_CUDA, "resident kernel: a neighbour wait timed out (results are invalid)");
    return POTTS_OK;
}

}  // namespace

extern "C" {

const char *potts_last_error(void) { return g_err.c_str(); }
const char *potts_version(void) { return "potts-b200 0.1 (sm_100a)"; }

int potts_workspace_bytes(int32_t L, int32_t q, int32_t layout, size_t *bytes)
{
    if (!bytes) return fail(POTTS_ERR_ARG, "null bytes pointer");
    int rc = check_shape(L, q, layout);
    if (rc) return rc;
    *bytes = workspace_bytes_of(L, q, layout);
    return POTTS_OK;
}

int potts_create_ex(potts_t **out, int32_t L, int32_t q, uint64_t seed, int32_t init, int32_t layout,
                    void *dev_workspace, size_t workspace_bytes, void *cuda_stream)
{
    if (!out) return fail(POTTS_ERR_ARG, "null out pointer");
    if (init != POTTS_INIT_ORDERED && init != POTTS_INIT_RANDOM) return fail(POTTS_ERR_ARG, "bad init %d", init);
    int rc = check_shape(L, q, layout);
    if (rc) return rc;
    const size_t need = workspace_bytes_of(L, q, layout);
    if (dev_workspace) {
        if (workspace_bytes < need)
            return fail(POTTS_ERR_NOMEM, "workspace of %zu bytes < %zu needed", workspace_bytes, need);
        if ((uintptr_t)dev_workspace % ALIGN) return fail(POTTS_ERR_ARG, "workspace not %zu-byte aligned", ALIGN);
    }
    int ndev = 0;
    CUDA_TRY(cudaGetDeviceCount(&ndev));
    if (ndev < 1) return fail(POTTS_ERR_CUDA, "no CUDA device");
    potts_t *h = new (std::nothrow) potts_s;
    if (!h) return fail(POTTS_ERR_NOMEM, "host allocation failed");
    h->L = L; h->q = q; h->layout = layout; h->seed = seed; h->t = 0;
    h->rows = L;
    cudaGetDevice(&h->device);
    h->stream = (cudaStream_t)cuda_stream;
    if (dev_workspace) {
        h->ws = (uint8_t *)dev_workspace;
    } else {
        cudaError_t e = cudaMalloc(&h->ws, need);
        if (e != cudaSuccess) {
            delete h;
            return fail(e == cudaErrorMemoryAllocation ? POTTS_ERR_NOMEM : POTTS_ERR_CUDA,
                        "cudaMalloc(%zu) failed: %s", need, cudaGetErrorString(e));
        }
        h->owns_ws = true;
    }
    h->plane_bytes = plane_bytes_of(L, q, layout);
    h->plane[0] = h->ws;
    h->plane[1] = h->ws + h->plane_bytes;
    if (layout == POTTS_LAYOUT_PACKED) {
        for (int c = 0; c < 2; ++c) {
            h->pk.nib[c] = h->plane[c];
            h->pk.hb[c] = q > 16 ? h->plane[c] + nib_bytes_of(L) : nullptr;
        }
        h->pk.L = L;
        h->pk.pn = L / 4;
        h->pk.ph = L / 16;
    }
    h->acc = (unsigned long long *)(h->ws + 2 * h->plane_bytes);
    h->flag = (int *)(h->acc + 257);
    h->error = h->flag + 1;
    h->tile_counter = (uint32_t *)(h->acc + 258);
    h->inbox = inbox_bytes_of(L) ? h->ws + 2 * h->plane_bytes + align_up(ACC_WORDS * sizeof(unsigned long long)) : nullptr;
    {
        int dev = 0, v = 0;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev);
        h->num_sms = v;
        cudaDeviceGetAttribute(&v, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
        h->smem_optin = (size_t)v;
        cudaDeviceGetAttribute(&v, cudaDevAttrCooperativeLaunch, dev);
        h->coop = v;
        cudaMemsetAsync(h->acc, 0, ACC_WORDS * sizeof(unsigned long long), h->stream);
    }

    cudaError_t e = cudaSuccess;
    if (init == POTTS_INIT_ORDERED) {
        e = cudaMemsetAsync(h->ws, 0, 2 * h->plane_bytes, h->stream);
    } else if (layout == POTTS_LAYOUT_PACKED) {
        const long long threads = 2ll * L * (L / 64);
        const unsigned grid = (unsigned)((threads + 127) / 128);
        const uint32_t k0 = (uint32_t)(seed & 0xFFFFFFFFull), k1 = (uint32_t)(seed >> 32);
        if (q > 16) potts::k_init_random_packed<true><<<grid, 128, 0, h->stream>>>(h->pk, (uint32_t)q, k0, k1);
        else potts::k_init_random_packed<false><<<grid, 128, 0, h->stream>>>(h->pk, (uint32_t)q, k0, k1);
        h->launches += 1;
        e = cudaGetLastError();
    } else {
        const long long words = 2ll * L * (L / 8);
        const int block = 256;
        potts::k_init_random_u8<<<(unsigned)((words + block - 1) / block), block, 0, h->stream>>>(
            h->plane[0], h->plane[1], L, L / 2, (uint32_t)q, (uint32_t)(seed & 0xFFFFFFFFull), (uint32_t)(seed >> 32));
        h->launches += 1;
        e = cudaGetLastError();
    }
    if (e != cudaSuccess) {
        potts_destroy(h);
        return fail(POTTS_ERR_CUDA, "initialisation failed: %s", cudaGetErrorString(e));
    }
    *out = h;
    return POTTS_OK;
}

int potts_create(potts_t **out, int32_t L, int32_t q, uint64_t seed, int32_t init)
{
    return potts_create_ex(out, L, q, seed, init, POTTS_LAYOUT_U8, nullptr, 0, nullptr);
}

void potts_destroy(potts_t *h)
{
    ON_DEVICE_OF(h);
    if (!h) return;
    if (h->scratch || (h->owns_ws && h->ws)) cudaStreamSynchronize(h->stream);
    if (h->scratch) cudaFree(h->scratch);
    if (h->copy_stream) {
        cudaStreamDestroy(h->copy_stream);
        for (int k = 0; k < 2; ++k) { cudaEventDestroy(h->ev_copied[k]); cudaEventDestroy(h->ev_converted[k]); }
        cudaEventDestroy(h->ev_start);
    }
    if (h->owns_ws && h->ws) cudaFree(h->ws);
    delete h;
}

int potts_set_stream(potts_t *h, void *cuda_stream)
{
    ON_DEVICE_OF(h);
    if (!h) return fail(POTTS_ERR_ARG, "null handle");
    h->stream = (cudaStream_t)cuda_stream;
    return POTTS_OK;
}

int potts_sweep(potts_t *h, double T, int64_t nsweeps)
{
    ON_DEVICE_OF(h);
    int rc = check_sweep_args(h, T, nsweeps);
    if (rc) return rc;
    return run_sweeps(h, T, nsweeps, 0, nullptr, nullptr);
}

int potts_sweep_measured_dev(potts_t *h, double T, int64_t nsweeps, int64_t every, int64_t *E_series_dev,
                             int64_t *hist_series_dev)
{
    ON_DEVICE_OF(h);
    int rc = check_sweep_args(h, T, nsweeps);
    if (rc) return rc;
    if (every < 1 || every > (1ll << 30) || nsweeps % every != 0)
        return fail(POTTS_ERR_ARG, "every = %lld must be in [1, 2^30] and divide nsweeps = %lld", (long long)every,
                    (long long)nsweeps);
    const int64_t ns = nsweeps / every;
    if (ns == 0) return POTTS_OK;
    if (E_series_dev) CUDA_TRY(cudaMemsetAsync(E_series_dev, 0, (size_t)ns * 8, h->stream));
    if (hist_series_dev) CUDA_TRY(cudaMemsetAsync(hist_series_dev, 0, (size_t)ns * h->q * 8, h->stream));
    return run_sweeps(h, T, nsweeps, every, (unsigned long long *)E_series_dev,
                      (unsigned long long *)hist_series_dev);
}

int potts_sweep_measured(potts_t *h, double T, int64_t nsweeps, int64_t every, int64_t *E_series,
                         int64_t *hist_series)
{
    ON_DEVICE_OF(h);
    int rc = check_sweep_args(h, T, nsweeps);
    if (rc) return rc;
    if (every < 1 || every > (1ll << 30) || nsweeps % every != 0)
        return fail(POTTS_ERR_ARG, "every = %lld must be in [1, 2^30] and divide nsweeps = %lld", (long long)every,
                    (long long)nsweeps);
    const int64_t ns = nsweeps / every;
    if (ns == 0) return POTTS_OK;
    const size_t eb = E_series ? (size_t)ns * 8 : 0, hb = hist_series ? (size_t)ns * h->q * 8 : 0;
    uint8_t *dev = nullptr;
    if (eb + hb) {
        rc = get_scratch(h, eb + hb, &dev);
        if (rc) return rc;
    }
    int64_t *dE = E_series ? (int64_t *)dev : nullptr;
    int64_t *dH = hist_series ? (int64_t *)(dev + eb) : nullptr;
    rc = potts_sweep_measured_dev(h, T, nsweeps, every, dE, dH);
    cudaError_t e = cudaSuccess;
    if (rc == POTTS_OK && eb) e = cudaMemcpyAsync(E_series, dE, eb, cudaMemcpyDeviceToHost, h->stream);
    if (rc == POTTS_OK && e == cudaSuccess && hb)
        e = cudaMemcpyAsync(hist_series, dH, hb, cudaMemcpyDeviceToHost, h->stream);
    cudaError_t e2 = cudaStreamSynchronize(h->stream);
    if (rc) return rc;
    if (e != cudaSuccess || e2 != cudaSuccess)
        return fail(POTTS_ERR_CUDA, "series copy/sync failed: %s", cudaGetErrorString(e != cudaSuccess ? e : e2));
    return check_device_error(h);
}

int potts_sweep_delta(potts_t *h, double T, int64_t nsweeps, int64_t *dE_series)
{
    ON_DEVICE_OF(h);
    int rc = check_sweep_args(h, T, nsweeps);
    if (rc) return rc;
    if (!dE_series) return fail(POTTS_ERR_ARG, "null dE_series");
    if (nsweeps == 0) return POTTS_OK;
    uint32_t thr[4];
    thresholds(T, thr);
    uint8_t *dev = nullptr;
    rc = get_scratch(h, (size_t)nsweeps * 8, &dev);
    if (rc) return rc;
    unsigned long long *d = (unsigned long long *)dev;
    CUDA_TRY(cudaMemsetAsync(d, 0, (size_t)nsweeps * 8, h->stream));
    rc = run_sweeps(h, T, nsweeps, 0, nullptr, nullptr, d);
    cudaError_t e = cudaSuccess;
    if (rc == POTTS_OK) e = cudaMemcpyAsync(dE_series, d, (size_t)nsweeps * 8, cudaMemcpyDeviceToHost, h->stream);
    cudaError_t e2 = cudaStreamSynchronize(h->stream);
    if (rc) return rc;
    if (e != cudaSuccess || e2 != cudaSuccess)
        return fail(POTTS_ERR_CUDA, "series copy/sync failed: %s", cudaGetErrorString(e != cudaSuccess ? e : e2));
    return check_device_error(h);
}

int potts_ladder(potts_t *h, const double *T, int32_t nT, int64_t t_tran, int64_t t_max, int64_t dt, int64_t *E_series,
                 int64_t *hist_series)
{
    ON_DEVICE_OF(h);
    if (!h || !T) return fail(POTTS_ERR_ARG, "null argument");
    if (nT < 0 || t_tran < 0 || t_max < 0) return fail(POTTS_ERR_ARG, "negative count");
    if (dt < 1 || t_max % dt != 0)
        return fail(POTTS_ERR_ARG, "dt = %lld must be >= 1 and divide t_max = %lld", (long long)dt, (long long)t_max);
    for (int32_t k = 0; k < nT; ++k)
        if (!(T[k] > 0.0) || !std::isfinite(T[k])) return fail(POTTS_ERR_ARG, "T[%d] = %g must be finite and > 0", k, T[k]);
    if (h->t + (uint64_t)nT * (uint64_t)(t_tran + t_max) > 0xFFFFFFFFull)
        return fail(POTTS_ERR_ARG, "sweep counter would pass 2^32 - 1 (Philox counter word)");
    const int64_t per_T = t_max / dt, ns = per_T * nT;
    const size_t eb = E_series ? (size_t)ns * 8 : 0, hb = hist_series ? (size_t)ns * h->q * 8 : 0;
    uint8_t *dev = nullptr;
    if (eb + hb) {
        int rc0 = get_scratch(h, eb + hb, &dev);
        if (rc0) return rc0;
        cudaMemsetAsync(dev, 0, eb + hb, h->stream);
    }
    unsigned long long *dE = eb ? (unsigned long long *)dev : nullptr;
    unsigned long long *dH = hb ? (unsigned long long *)(dev + eb) : nullptr;
    int rc = POTTS_OK;
    for (int32_t k = 0; k < nT && rc == POTTS_OK; ++k) {
        rc = run_sweeps(h, T[k], t_tran, 0, nullptr, nullptr);
        if (rc == POTTS_OK && per_T > 0)
            rc = run_sweeps(h, T[k], t_max, dt, dE ? dE + k * per_T : nullptr, dH ? dH + k * per_T * h->q : nullptr);
    }
    cudaError_t e = cudaSuccess;
    if (rc == POTTS_OK && eb) e = cudaMemcpyAsync(E_series, dE, eb, cudaMemcpyDeviceToHost, h->stream);
    if (rc == POTTS_OK && e == cudaSuccess && hb) e = cudaMemcpyAsync(hist_series, dH, hb, cudaMemcpyDeviceToHost, h->stream);
    const cudaError_t e2 = cudaStreamSynchronize(h->stream);
    if (rc) return rc;
    if (e != cudaSuccess || e2 != cudaSuccess)
        return fail(POTTS_ERR_CUDA, "ladder copy/sync failed: %s", cudaGetErrorString(e != cudaSuccess ? e : e2));
    return check_device_error(h);
}

int potts_energy(potts_t *h, int64_t *E)
{
    ON_DEVICE_OF(h);
    if (!h || !E) return fail(POTTS_ERR_ARG, "null argument");
    CUDA_TRY(cudaMemsetAsync(h->acc, 0, 8, h->stream));
    int rc = launch_measure(h, h->acc, nullptr);
    if (rc) return rc;
    int64_t v = 0;
    CUDA_TRY(cudaMemcpyAsync(&v, h->acc, 8, cudaMemcpyDeviceToHost, h->stream));
    rc = check_device_error(h);
    if (rc) return rc;
    *E = v;
    return POTTS_OK;
}

int potts_histogram(potts_t *h, int64_t *counts)
{
    ON_DEVICE_OF(h);
    if (!h || !counts) return fail(POTTS_ERR_ARG, "null argument");
    CUDA_TRY(cudaMemsetAsync(h->acc + 1, 0, 8 * (size_t)h->q, h->stream));
    int rc = launch_measure(h, nullptr, h->acc + 1);
    if (rc) return rc;
    int64_t tmp[256];
    CUDA_TRY(cudaMemcpyAsync(tmp, h->acc + 1, 8 * (size_t)h->q, cudaMemcpyDeviceToHost, h->stream));
    rc = check_device_error(h);
    if (rc) return rc;
    std::memcpy(counts, tmp, 8 * (size_t)h->q);
    return POTTS_OK;
}

// ---- host <-> device transfer of the configuration ---------------------------------------------------
// Rows per staging buffer: two buffers of <= 32 MiB each, so that the PCIe copy of one chunk overlaps the layout
// conversion of the other (copies on the handle's own copy stream, conversions on the caller's stream, one
// event per buffer and direction; no synchronisation inside the loop).
static int chunk_rows(int L) { long long r = (32ll << 20) / L; return (int)(r < 1 ? 1 : (r > L ? L : r)); }

static int ensure_copy_objects(potts_t *h)
{
    if (h->copy_stream) return POTTS_OK;
    CUDA_TRY(cudaStreamCreateWithFlags(&h->copy_stream, cudaStreamNonBlocking));
    for (int k = 0; k < 2; ++k) {
        CUDA_TRY(cudaEventCreateWithFlags(&h->ev_copied[k], cudaEventDisableTiming));
        CUDA_TRY(cudaEventCreateWithFlags(&h->ev_converted[k], cudaEventDisableTiming));
    }
    CUDA_TRY(cudaEventCreateWithFlags(&h->ev_start, cudaEventDisableTiming));
    return POTTS_OK;
}

int potts_download(potts_t *h, uint8_t *spins)
{
    ON_DEVICE_OF(h);
    if (!h || !spins) return fail(POTTS_ERR_ARG, "null argument");
    const int L = h->L, rows = chunk_rows(L);
    const size_t buf_bytes = (size_t)rows * L;
    uint8_t *stage = nullptr;
    int rc = get_scratch(h, 2 * buf_bytes, &stage);
    if (rc) return rc;
    rc = ensure_copy_objects(h);
    if (rc) return rc;
    int k = 0;
    for (int i0 = 0; i0 < h->rows && rc == POTTS_OK; i0 += rows, ++k) {          // h->rows = L, or the rows of a strip
        const int r = (h->rows - i0 < rows) ? h->rows - i0 : rows, b = k & 1;
        uint8_t *buf = stage + (size_t)b * buf_bytes;
        if (k >= 2) CUDA_TRY(cudaStreamWaitEvent(h->stream, h->ev_copied[b], 0));      // the copy out of this buffer is done
        const long long threads = (long long)r * (L / 8);
        if (h->layout == POTTS_LAYOUT_PACKED) {
            const unsigned grid = (unsigned)(((long long)r * (L / 64) + 127) / 128);
            if (h->q > 16) potts::k_packed_to_rowmajor<true><<<grid, 128, 0, h->stream>>>(h->pk, buf, i0, r);
            else potts::k_packed_to_rowmajor<false><<<grid, 128, 0, h->stream>>>(h->pk, buf, i0, r);
        } else {
            potts::k_planes_to_rowmajor<<<(unsigned)((threads + 255) / 256), 256, 0, h->stream>>>(
                h->plane[0], h->plane[1], buf, L, L / 2, i0, r);
        }
        rc = check_launch(h, "k_planes_to_rowmajor");
        if (rc) break;
        CUDA_TRY(cudaEventRecord(h->ev_converted[b], h->stream));
        CUDA_TRY(cudaStreamWaitEvent(h->copy_stream, h->ev_converted[b], 0));
        CUDA_TRY(cudaMemcpyAsync(spins + (size_t)i0 * L, buf, (size_t)r * L, cudaMemcpyDeviceToHost, h->copy_stream));
        CUDA_TRY(cudaEventRecord(h->ev_copied[b], h->copy_stream));
    }
    const cudaError_t e1 = cudaStreamSynchronize(h->copy_stream), e2 = cudaStreamSynchronize(h->stream);
    if (rc) return rc;
    if (e1 != cudaSuccess || e2 != cudaSuccess)
        return fail(POTTS_ERR_CUDA, "download copy failed: %s", cudaGetErrorString(e1 != cudaSuccess ? e1 : e2));
    return check_device_error(h);
}

// is any byte of spins[0, n) >= q?  Word-parallel, a few host threads: ~20 ms per GiB, against ~40 ms of PCIe copy.
static bool host_has_value_ge(const uint8_t *spins, size_t n, int q)
{
    if (q >= 256) return false;
    unsigned nt = std::thread::hardware_concurrency();
    if (nt > 8) nt = 8;
    if (nt < 1 || n < (1u << 22)) nt = 1;
    std::vector<unsigned char> bad(nt, 0);
    auto scan = [&](unsigned t) {
        const size_t a = n * t / nt, b = n * (t + 1) / nt;
        unsigned char m = 0;
        for (size_t k = a; k < b; ++k) m |= (unsigned char)(spins[k] >= q);     // vectorised by the host compiler
        bad[t] = m;
    };
    if (nt == 1) scan(0);
    else {
        std::vector<std::thread> th;
        for (unsigned t = 0; t < nt; ++t) th.emplace_back(scan, t);
        for (auto &x : th) x.join();
    }
    for (unsigned t = 0; t < nt; ++t)
        if (bad[t]) return true;
    return false;
}

int potts_upload(potts_t *h, const uint8_t *spins)
{
    ON_DEVICE_OF(h);
    if (!h || !spins) return fail(POTTS_ERR_ARG, "null argument");
    const int L = h->L, rows = chunk_rows(L);
    // validate on the host first so that a rejected upload leaves the lattice untouched; the converter checks again
    // on the device and its flag is read back below
    if (host_has_value_ge(spins, (size_t)h->rows * L, h->q)) return fail(POTTS_ERR_ARG, "a spin value is >= q = %d", h->q);
    const size_t buf_bytes = (size_t)rows * L;
    uint8_t *stage = nullptr;
    int rc = get_scratch(h, 2 * buf_bytes, &stage);
    if (rc) return rc;
    rc = ensure_copy_objects(h);
    if (rc) return rc;
    CUDA_TRY(cudaMemsetAsync(h->flag, 0, sizeof(int), h->stream));
    // the staging buffers may still be read by earlier work on the caller's stream
    CUDA_TRY(cudaEventRecord(h->ev_start, h->stream));
    CUDA_TRY(cudaStreamWaitEvent(h->copy_stream, h->ev_start, 0));
    int k = 0;
    for (int i0 = 0; i0 < h->rows && rc == POTTS_OK; i0 += rows, ++k) {          // h->rows = L, or the rows of a strip
        const int r = (h->rows - i0 < rows) ? h->rows - i0 : rows, b = k & 1;
        uint8_t *buf = stage + (size_t)b * buf_bytes;
        if (k >= 2) CUDA_TRY(cudaStreamWaitEvent(h->copy_stream, h->ev_converted[b], 0));   // the converter has read this buffer
        CUDA_TRY(cudaMemcpyAsync(buf, spins + (size_t)i0 * L, (size_t)r * L, cudaMemcpyHostToDevice, h->copy_stream));
        CUDA_TRY(cudaEventRecord(h->ev_copied[b], h->copy_stream));
        CUDA_TRY(cudaStreamWaitEvent(h->stream, h->ev_copied[b], 0));
        const long long threads = (long long)r * (L / 8);
        if (h->layout == POTTS_LAYOUT_PACKED) {
            const unsigned grid = (unsigned)(((long long)r * (L / 64) + 127) / 128);
            if (h->q > 16) potts::k_rowmajor_to_packed<true><<<grid, 128, 0, h->stream>>>(buf, h->pk, i0, r, (uint32_t)h->q, h->flag);
            else potts::k_rowmajor_to_packed<false><<<grid, 128, 0, h->stream>>>(buf, h->pk, i0, r, (uint32_t)h->q, h->flag);
        } else
            potts::k_rowmajor_to_planes<<<(unsigned)((threads + 255) / 256), 256, 0, h->stream>>>(
                buf, h->plane[0], h->plane[1], L, L / 2, i0, r, (uint32_t)h->q, h->flag);
        rc = check_launch(h, "k_rowmajor_to_planes");
        if (rc) break;
        CUDA_TRY(cudaEventRecord(h->ev_converted[b], h->stream));
    }
    int bad = 0;
    cudaError_t e = cudaSuccess;
    if (rc == POTTS_OK) e = cudaMemcpyAsync(&bad, h->flag, sizeof(int), cudaMemcpyDeviceToHost, h->stream);
    const cudaError_t e1 = cudaStreamSynchronize(h->copy_stream), e2 = cudaStreamSynchronize(h->stream);
    if (rc) return rc;
    if (e != cudaSuccess || e1 != cudaSuccess || e2 != cudaSuccess) return fail(POTTS_ERR_CUDA, "upload copy failed");
    if (bad) return fail(POTTS_ERR_ARG, "a spin value is >= q = %d (device check; the lattice is now undefined)", h->q);
    return POTTS_OK;
}

// ---- one lattice split into row strips over several GPUs ------------------------------------------
int potts_create_strip(potts_t **out, int32_t L, int32_t q, uint64_t seed, int32_t init, int32_t row0, int32_t rows,
                       void *cuda_stream)
{
    if (!out) return fail(POTTS_ERR_ARG, "null out pointer");
    if (init != POTTS_INIT_ORDERED && init != POTTS_INIT_RANDOM) return fail(POTTS_ERR_ARG, "bad init %d", init);
    int rc = check_shape(L, q, POTTS_LAYOUT_U8);
    if (rc) return rc;
    if (row0 < 0 || rows < 32 || row0 + rows > L || row0 % 32 || rows % 32)
        return fail(POTTS_ERR_ARG, "strip rows [%d, %d) must lie in [0, %d) with both ends multiples of 32", row0, row0 + rows, L);
    int ndev = 0;
    CUDA_TRY(cudaGetDeviceCount(&ndev));
    if (ndev < 1) return fail(POTTS_ERR_CUDA, "no CUDA device");
    potts_t *h = new (std::nothrow) potts_s;
    if (!h) return fail(POTTS_ERR_NOMEM, "host allocation failed");
    h->L = L; h->q = q; h->layout = POTTS_LAYOUT_U8; h->seed = seed; h->t = 0;
    h->rows = rows; h->row0 = row0; h->strip = true;
    h->opt_variant = 1;                                                  // streaming kernels only
    h->stream = (cudaStream_t)cuda_stream;
    cudaGetDevice(&h->device);
    const size_t pitch = (size_t)L / 2;
    h->plane_bytes = align_up((size_t)(rows + 2) * pitch);              // one halo row above and one below
    const size_t need = 2 * h->plane_bytes + align_up(ACC_WORDS * sizeof(unsigned long long)) + ALIGN;
    cudaError_t e = cudaMalloc(&h->ws, need);
    if (e != cudaSuccess) {
        delete h;
        return fail(e == cudaErrorMemoryAllocation ? POTTS_ERR_NOMEM : POTTS_ERR_CUDA, "cudaMalloc(%zu) failed: %s", need, cudaGetErrorString(e));
    }
    h->owns_ws = true;
    h->plane[0] = h->ws + pitch;                                         // local row 0; the halo row above it is at -pitch
    h->plane[1] = h->ws + h->plane_bytes + pitch;
    h->acc = (unsigned long long *)(h->ws + 2 * h->plane_bytes);
    h->flag = (int *)(h->acc + 257);
    h->error = h->flag + 1;
    h->tile_counter = (uint32_t *)(h->acc + 258);
    {
        int v = 0;
        cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, h->device);
        h->num_sms = v;
        cudaDeviceGetAttribute(&v, cudaDevAttrMaxSharedMemoryPerBlockOptin, h->device);
        h->smem_optin = (size_t)v;
    }
    e = cudaMemsetAsync(h->ws, 0, need, h->stream);
    if (e == cudaSuccess && init == POTTS_INIT_RANDOM) {
        const long long words = 2ll * rows * (L / 8);
        potts::k_init_random_u8<<<(unsigned)((words + 255) / 256), 256, 0, h->stream>>>(
            h->plane[0], h->plane[1], rows, L / 2, (uint32_t)q, (uint32_t)(seed & 0xFFFFFFFFull), (uint32_t)(seed >> 32), row0);
        h->launches += 1;
        e = cudaGetLastError();
    }
    if (e != cudaSuccess) {
        potts_destroy(h);
        return fail(POTTS_ERR_CUDA, "strip initialisation failed: %s", cudaGetErrorString(e));
    }
    *out = h;
    return POTTS_OK;
}

int potts_strip_half_sweep(potts_t *h, double T, int32_t colour, int64_t *E_dev, int64_t *hist_dev)
{
    ON_DEVICE_OF(h);
    if (!h || !h->strip) return fail(POTTS_ERR_ARG, "not a strip handle");
    if (!(T > 0.0) || !std::isfinite(T)) return fail(POTTS_ERR_ARG, "T = %g must be finite and > 0", T);
    if (colour != 0 && colour != 1) return fail(POTTS_ERR_ARG, "colour must be 0 or 1");
    if (E_dev && colour != 1) return fail(POTTS_ERR_ARG, "the energy is counted from the colour-1 sites");
    if (h->t >= 0xFFFFFFFFull) return fail(POTTS_ERR_ARG, "sweep counter would pass 2^32 - 1");
    uint32_t thr[4];
    thresholds(T, thr);
    return launch_half_sweep(h, (uint32_t)colour, thr, (unsigned long long *)E_dev, (unsigned long long *)hist_dev);
}

int potts_strip_advance(potts_t *h)
{
    if (!h || !h->strip) return fail(POTTS_ERR_ARG, "not a strip handle");
    h->t += 1;
    return POTTS_OK;
}

int potts_strip_rows(potts_t *h, int32_t colour, void **first_row, void **last_row, void **halo_above, void **halo_below,
                     size_t *row_bytes)
{
    if (!h || !h->strip || !first_row || !last_row || !halo_above || !halo_below || !row_bytes) return fail(POTTS_ERR_ARG, "bad argument");
    if (colour != 0 && colour != 1) return fail(POTTS_ERR_ARG, "colour must be 0 or 1");
    const size_t pitch = (size_t)h->L / 2;
    uint8_t *p = h->plane[colour];
    *first_row = p;
    *last_row = p + (size_t)(h->rows - 1) * pitch;
    *halo_above = p - pitch;
    *halo_below = p + (size_t)h->rows * pitch;
    *row_bytes = pitch;
    return POTTS_OK;
}

int potts_sweep_count(potts_t *h, uint64_t *t)
{
    ON_DEVICE_OF(h);
    if (!h || !t) return fail(POTTS_ERR_ARG, "null argument");
    *t = h->t;
    return POTTS_OK;
}

int potts_set_sweep_count(potts_t *h, uint64_t t)
{
    ON_DEVICE_OF(h);
    if (!h) return fail(POTTS_ERR_ARG, "null handle");
    if (t > 0xFFFFFFFFull) return fail(POTTS_ERR_ARG, "t must be < 2^32");
    h->t = t;
    return POTTS_OK;
}

int potts_set_stream_spec(potts_t *h, int32_t spec)
{
    ON_DEVICE_OF(h);
    if (!h) return fail(POTTS_ERR_ARG, "null handle");
    if (spec != 1 && spec != 2) return fail(POTTS_ERR_ARG, "stream spec must be 1 or 2");
    h->stream_spec = spec;
    return POTTS_OK;
}

int potts_get_stream_spec(potts_t *h, int32_t *spec)
{
    ON_DEVICE_OF(h);
    if (!h || !spec) return fail(POTTS_ERR_ARG, "null argument");
    *spec = h->stream_spec;
    return POTTS_OK;
}

int potts_launch_count(potts_t *h, uint64_t *n)
{
    ON_DEVICE_OF(h);
    if (!h || !n) return fail(POTTS_ERR_ARG, "null argument");
    *n = h->launches;
    return POTTS_OK;
}

int potts_set_option(potts_t *h, const char *key, int64_t value)
{
    ON_DEVICE_OF(h);
    if (!h || !key) return fail(POTTS_ERR_ARG, "null argument");
    if (!std::strcmp(key, "variant")) {
        if (value < 0 || value > 3) return fail(POTTS_ERR_ARG, "variant must be 0 (auto), 1 (streaming), 2 (resident) or 3 (cluster)");
        h->opt_variant = value; return POTTS_OK;
    }
    if (!std::strcmp(key, "resident_ctas")) {
        if (value < 0 || value > MAX_CTAS) return fail(POTTS_ERR_ARG, "resident_ctas must be in [0, %d]", MAX_CTAS);
        h->opt_resident_ctas = value; return POTTS_OK;
    }
    if (!std::strcmp(key, "cluster_ctas")) {
        if (value < 0 || value > potts::CLUSTER_MAX) return fail(POTTS_ERR_ARG, "cluster_ctas must be in [0, %d]", potts::CLUSTER_MAX);
        h->opt_cluster_ctas = value; return POTTS_OK;
    }
    if (!std::strcmp(key, "resident_rows")) {
        if (value < 0 || value > 1024) return fail(POTTS_ERR_ARG, "resident_rows must be in [0, 1024]");
        h->opt_resident_rows = value; return POTTS_OK;
    }
    if (!std::strcmp(key, "resident_words")) {
        if (value < 0 || value > 2) return fail(POTTS_ERR_ARG, "resident_words must be 0 (auto), 1 or 2");
        h->opt_resident_words = value; return POTTS_OK;
    }
    if (!std::strcmp(key, "resident_col")) {
        if (value < 0 || value > 1) return fail(POTTS_ERR_ARG, "resident_col must be 0 or 1");
        h->opt_resident_col = value; return POTTS_OK;
    }
    if (!std::strcmp(key, "stream_stage")) {
        if (value < 0 || value > 1) return fail(POTTS_ERR_ARG, "stream_stage must be 0 (registers) or 1 (cp.async.bulk staging)");
        h->opt_stream_stage = value; return POTTS_OK;
    }
    if (!std::strcmp(key, "stream_rows")) {
        if (value < 0 || (value > 0 && ((value & 1) || (h->L / potts::HS_WARPS) % value)))
            return fail(POTTS_ERR_ARG, "stream_rows must be 0 (auto) or an even divisor of L / %d", potts::HS_WARPS);
        h->opt_stream_rows = value; return POTTS_OK;
    }
    return fail(POTTS_ERR_ARG, "unknown option '%s'", key);
}

int potts_get_option(potts_t *h, const char *key, int64_t *value)
{
    ON_DEVICE_OF(h);
    if (!h || !key || !value) return fail(POTTS_ERR_ARG, "null argument");
    if (!std::strcmp(key, "variant")) { *value = h->opt_variant; return POTTS_OK; }
    if (!std::strcmp(key, "resident_ctas")) { *value = h->opt_resident_ctas; return POTTS_OK; }
    if (!std::strcmp(key, "resident_words")) { *value = h->opt_resident_words; return POTTS_OK; }
    if (!std::strcmp(key, "resident_rows")) { *value = h->opt_resident_rows; return POTTS_OK; }
    if (!std::strcmp(key, "cluster_ctas")) { *value = h->opt_cluster_ctas; return POTTS_OK; }
    if (!std::strcmp(key, "stream_rows")) { *value = h->opt_stream_rows; return POTTS_OK; }
    if (!std::strcmp(key, "stream_stage")) { *value = h->opt_stream_stage; return POTTS_OK; }
    if (!std::strcmp(key, "resident_col")) { *value = h->opt_resident_col; return POTTS_OK; }
    if (!std::strcmp(key, "cluster_active")) {             // read-only: cluster size the next sweep call would use (0 = not the cluster kernel)
        const bool want = h->opt_variant == 3 || (h->opt_variant == 0 && h->layout == POTTS_LAYOUT_U8 && h->L <= CLUSTER_AUTO_L_MAX);
        *value = (want && plan_cluster(h).ok) ? plan_cluster(h).G : 0; return POTTS_OK;
    }
    if (!std::strcmp(key, "resident_active")) {            // read-only: would the next sweep call run resident?
        const bool cluster = h->opt_variant == 3 || (h->opt_variant == 0 && h->layout == POTTS_LAYOUT_U8 && h->L <= CLUSTER_AUTO_L_MAX && plan_cluster(h).ok);
        *value = (!cluster && h->opt_variant != 1 && plan_resident(h).ok) ? plan_resident(h).G : 0; return POTTS_OK;
    }
    return fail(POTTS_ERR_ARG, "unknown option '%s'", key);
}

// ---- host-side derived observables (R10) -------------------------------------------------------
int potts_observables(const int64_t *E_series, int64_t n, int64_t N, double T, double *mean_e, double *cv,
                      double *binder)
{
    if (!E_series || n < 1 || N < 1 || !(T > 0.0) || !std::isfinite(T))
        return fail(POTTS_ERR_ARG, "bad arguments to potts_observables");
    typedef __int128 i128;
    i128 s1 = 0, s2 = 0;
    long double s4 = 0.0L, comp = 0.0L;            // Kahan-compensated sum of E^4
    for (int64_t k = 0; k < n; ++k) {
        const i128 e = (i128)E_series[k];
        const i128 e2 = e * e;                      // < 2^63 for |E| <= 2^31.5: exact
        s1 += e;
        s2 += e2;
        const long double e4 = (long double)e2 * (long double)e2;
        const long double y = e4 - comp;
        const long double tsum = s4 + y;
        comp = (tsum - s4) - y;
        s4 = tsum;
    }
    // <E^2> - <E>^2 = (n s2 - s1^2) / n^2, formed exactly in 128-bit integers
    const i128 num = (i128)n * s2 - s1 * s1;
    if (mean_e) *mean_e = (double)((long double)s1 / ((long double)n * (long double)N));
    if (cv) *cv = (double)((long double)num / ((long double)n * (long double)n) / ((long double)N * (long double)T * (long double)T));
    if (binder) {
        if (s2 == 0) return fail(POTTS_ERR_ARG, "Binder cumulant undefined: all energies are zero");
        *binder = (double)(1.0L - ((long double)n * s4) / (3.0L * (long double)s2 * (long double)s2));
    }
    return POTTS_OK;
}

int potts_magnetisation(const int64_t *counts, int32_t q, double *m)
{
    if (!counts || !m || q < 2 || q > 256) return fail(POTTS_ERR_ARG, "bad arguments to potts_magnetisation");
    int64_t N = 0, mx = 0;
    for (int k = 0; k < q; ++k) {
        if (counts[k] < 0) return fail(POTTS_ERR_ARG, "negative count");
        N += counts[k];
        if (counts[k] > mx) mx = counts[k];
    }
    if (N == 0) return fail(POTTS_ERR_ARG, "empty histogram");
    *m = (double)((((long double)q * (long double)mx) / (long double)N - 1.0L) / (long double)(q - 1));
    return POTTS_OK;
}

int potts_susceptibility(const int64_t *hist_series, int64_t n, int32_t q, double T, double *mean_m, double *mean_m2,
                         double *chi)
{
    if (!hist_series || n < 1 || q < 2 || q > 256 || !(T > 0.0) || !std::isfinite(T))
        return fail(POTTS_ERR_ARG, "bad arguments to potts_susceptibility");
    typedef __int128 i128;
    i128 s1 = 0, s2 = 0;
    int64_t N = 0;
    for (int64_t k = 0; k < n; ++k) {
        const int64_t *row = hist_series + k * q;
        int64_t sum = 0, mx = 0;
        for (int s = 0; s < q; ++s) {
            if (row[s] < 0) return fail(POTTS_ERR_ARG, "negative count in histogram %lld", (long long)k);
            sum += row[s];
            if (row[s] > mx) mx = row[s];
        }
        if (k == 0) N = sum;
        if (sum != N || N <= 0) return fail(POTTS_ERR_ARG, "histogram %lld sums to %lld, expected N = %lld > 0", (long long)k, (long long)sum, (long long)N);
        const i128 a = (i128)q * mx - N;                 // m_k = a / ((q-1) N), 0 <= a <= (q-1) N
        s1 += a;
        s2 += a * a;
    }
    const long double den = (long double)(q - 1) * (long double)N;          // m = a / den
    if (mean_m) *mean_m = (double)((long double)s1 / ((long double)n * den));
    if (mean_m2) *mean_m2 = (double)((long double)s2 / ((long double)n * den * den));
    if (chi) {
        // <m^2> - <m>^2 = (n s2 - s1^2) / (n den)^2, the numerator exact while it fits 126 bits
        long double num;
        const long double est = (long double)n * (long double)s2;
        if (est < 0x1p125L) num = (long double)((i128)n * s2 - s1 * s1);
        else num = est - (long double)s1 * (long double)s1;
        *chi = (double)((long double)N / (long double)T * num / ((long double)n * den * (long double)n * den));
    }
    return POTTS_OK;
}

}  // extern "C"

// ---- replica batch -------------------------------------------------------------------------------
struct potts_batch_s {
    int32_t n = 0, L = 0, q = 0;
    int device = 0;
    uint64_t t = 0, launches = 0;
    int32_t stream_spec = 1;
    uint64_t *seeds = nullptr;            // host copy
    uint8_t *ws = nullptr;
    bool owns_ws = false;
    size_t plane_bytes = 0;               // one colour plane of one lattice
    int *error = nullptr;
    cudaStream_t stream = nullptr;
    size_t smem_optin = 0;
    uint8_t *scratch = nullptr;           // device scratch kept between calls (series, download staging)
    size_t scratch_bytes = 0;
};

namespace {

int get_batch_scratch(potts_batch_t *b, size_t bytes, uint8_t **out)
{
    if (b->scratch_bytes < bytes) {
        if (b->scratch) { cudaStreamSynchronize(b->stream); cudaFree(b->scratch); b->scratch = nullptr; b->scratch_bytes = 0; }
        CUDA_TRY(cudaMalloc(&b->scratch, bytes));
        b->scratch_bytes = bytes;
    }
    *out = b->scratch;
    return POTTS_OK;
}

struct BatchPlan { bool ok = false; int tyc = 0, nthreads = 0; size_t smem = 0; const char *why = ""; };

BatchPlan plan_batch(int32_t L, int32_t q, size_t smem_optin)
{
    BatchPlan R;
    const int wpr = L / 8;                                         // one 4-site word per thread and row visit; no comm warps (one CTA = one lattice)
    // Two visits per thread where the block allows (measured 4.6 against 6.9 ps per update at L = 64 for two visits against
    // one: half the per-half-sweep bookkeeping per site, twice the CTAs per SM), in a block of at most 512 threads (up to 128
    // registers); lattices too large for that within 8 visits take a block of up to 1024 threads (64 registers).
    // An EVEN number of thread rows: a thread's rows then share one parity and its ColKeys (potts_resident.cuh).
    int tyc = 512 / wpr;
    if (tyc > L / 2) tyc = L / 2;
    tyc &= ~1;
    if (tyc < 2 || (L + tyc - 1) / tyc > 8) {
        tyc = 1024 / wpr;
        if (tyc > L / 2) tyc = L / 2;
        tyc &= ~1;
    }
    if (tyc < 2) { R.why = "no room for two thread rows in a 1024-thread block"; return R; }
    R.tyc = tyc;
    R.nthreads = (wpr * tyc + 31) / 32 * 32;
    const size_t hist = (size_t)(q <= (int)potts::HIST_LANE_QMAX ? q * 32 : q) * 4;
    R.smem = 2 * (size_t)(L + 2) * (L / 2) + hist;
    if (R.smem + STATIC_SMEM > smem_optin) { R.why = "one lattice does not fit the shared memory of a CTA"; return R; }
    R.ok = true;
    return R;
}

size_t batch_bytes_of(int32_t n, int32_t L) { return (size_t)n * 2 * align_up((size_t)L * (L / 2)) + ALIGN; }

int check_batch_shape(int32_t n, int32_t L, int32_t q)
{
    if (n < 1) return fail(POTTS_ERR_ARG, "n = %d lattices", n);
    int rc = check_shape(L, q, POTTS_LAYOUT_U8);
    if (rc) return rc;
    if (2 * (size_t)(L + 2) * (L / 2) > 200 * 1024) return fail(POTTS_ERR_UNSUPPORTED, "L = %d does not fit one CTA's shared memory", L);
    return POTTS_OK;
}

}  // namespace

extern "C" {

int potts_batch_workspace_bytes(int32_t n, int32_t L, int32_t q, size_t *bytes)
{
    if (!bytes) return fail(POTTS_ERR_ARG, "null bytes pointer");
    int rc = check_batch_shape(n, L, q);
    if (rc) return rc;
    *bytes = batch_bytes_of(n, L);
    return POTTS_OK;
}

int potts_batch_create(potts_batch_t **out, int32_t n, int32_t L, int32_t q, const uint64_t *seeds, int32_t init,
                       void *dev_workspace, size_t workspace_bytes, void *cuda_stream)
{
    if (!out || !seeds) return fail(POTTS_ERR_ARG, "null argument");
    if (init != POTTS_INIT_ORDERED && init != POTTS_INIT_RANDOM) return fail(POTTS_ERR_ARG, "bad init %d", init);
    int rc = check_batch_shape(n, L, q);
    if (rc) return rc;
    const size_t need = batch_bytes_of(n, L);
    if (dev_workspace && workspace_bytes < need) return fail(POTTS_ERR_NOMEM, "workspace of %zu bytes < %zu needed", workspace_bytes, need);
    if (dev_workspace && (uintptr_t)dev_workspace % ALIGN) return fail(POTTS_ERR_ARG, "workspace not %zu-byte aligned", ALIGN);
    int ndev = 0;
    CUDA_TRY(cudaGetDeviceCount(&ndev));
    if (ndev < 1) return fail(POTTS_ERR_CUDA, "no CUDA device");
    potts_batch_t *b = new (std::nothrow) potts_batch_s;
    if (!b) return fail(POTTS_ERR_NOMEM, "host allocation failed");
    b->n = n; b->L = L; b->q = q;
    cudaGetDevice(&b->device);
    b->stream = (cudaStream_t)cuda_stream;
    b->seeds = new (std::nothrow) uint64_t[n];
    if (!b->seeds) { delete b; return fail(POTTS_ERR_NOMEM, "host allocation failed"); }
    std::memcpy(b->seeds, seeds, sizeof(uint64_t) * n);
    if (dev_workspace) b->ws = (uint8_t *)dev_workspace;
    else {
        cudaError_t e = cudaMalloc(&b->ws, need);
        if (e != cudaSuccess) {
            delete[] b->seeds; delete b;
            return fail(POTTS_ERR_NOMEM, "cudaMalloc(%zu) failed: %s", need, cudaGetErrorString(e));
        }
        b->owns_ws = true;
    }
    b->plane_bytes = align_up((size_t)L * (L / 2));
    b->error = (int *)(b->ws + (size_t)n * 2 * b->plane_bytes);
    {
        int dev = 0, v = 0;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&v, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
        b->smem_optin = (size_t)v;
    }
    const BatchPlan R = plan_batch(L, q, b->smem_optin);
    if (!R.ok) { potts_batch_destroy(b); return fail(POTTS_ERR_UNSUPPORTED, "batch: %s", R.why); }
    cudaError_t e = cudaMemsetAsync(b->ws, 0, need, b->stream);
    if (e == cudaSuccess && init == POTTS_INIT_RANDOM) {
        const long long words = 2ll * L * (L / 8);
        for (int r = 0; r < n; ++r) {
            uint8_t *p0 = b->ws + (size_t)r * 2 * b->plane_bytes;
            potts::k_init_random_u8<<<(unsigned)((words + 255) / 256), 256, 0, b->stream>>>(
                p0, p0 + b->plane_bytes, L, L / 2, (uint32_t)q, (uint32_t)(seeds[r] & 0xFFFFFFFFull), (uint32_t)(seeds[r] >> 32));
        }
        b->launches += n;
        e = cudaGetLastError();
    }
    if (e != cudaSuccess) { potts_batch_destroy(b); return fail(POTTS_ERR_CUDA, "batch initialisation failed: %s", cudaGetErrorString(e)); }
    *out = b;
    return POTTS_OK;
}

void potts_batch_destroy(potts_batch_t *b)
{
    ON_DEVICE_OF(b);
    if (!b) return;
    if (b->scratch || (b->owns_ws && b->ws)) cudaStreamSynchronize(b->stream);
    if (b->scratch) cudaFree(b->scratch);
    if (b->owns_ws && b->ws) cudaFree(b->ws);
    delete[] b->seeds;
    delete b;
}

int potts_batch_sweep_count(potts_batch_t *b, uint64_t *t)
{
    ON_DEVICE_OF(b);
    if (!b || !t) return fail(POTTS_ERR_ARG, "null argument");
    *t = b->t;
    return POTTS_OK;
}

int potts_batch_set_stream_spec(potts_batch_t *b, int32_t spec)
{
    ON_DEVICE_OF(b);
    if (!b) return fail(POTTS_ERR_ARG, "null handle");
    if (spec != 1 && spec != 2) return fail(POTTS_ERR_ARG, "stream spec must be 1 or 2");
    b->stream_spec = spec;
    return POTTS_OK;
}

int potts_batch_launch_count(potts_batch_t *b, uint64_t *n)
{
    ON_DEVICE_OF(b);
    if (!b || !n) return fail(POTTS_ERR_ARG, "null argument");
    *n = b->launches;
    return POTTS_OK;
}

}  // extern "C"

namespace {

// nsweeps sweeps of every lattice of the batch, lattice r at temperature T[r * T_stride], enqueued on the batch's
// stream.  Device series (null = not recorded): E / hist samples of lattice r at E_dev + r * series_stride (+ k),
// hist_dev + (r * series_stride + k) * q; energy changes at dE_dev + r * delta_stride + sweep.  Advances b->t.
int batch_run(potts_batch_t *b, const double *T, int64_t T_stride, int64_t nsweeps, int64_t every, unsigned long long *E_dev,
              unsigned long long *hist_dev, int64_t series_stride, unsigned long long *dE_dev, int64_t delta_stride)
{
    if (nsweeps == 0) return POTTS_OK;
    const bool measure = E_dev || hist_dev;
    const BatchPlan R = plan_batch(b->L, b->q, b->smem_optin);
    static thread_local potts::BatchTable tab;               // 24 KB: copied into the launch parameters
    cudaError_t e = cudaSuccess;
    for (int r0 = 0; r0 < b->n && e == cudaSuccess; r0 += potts::BATCH_MAX) {
        const int m = b->n - r0 < potts::BATCH_MAX ? b->n - r0 : potts::BATCH_MAX;
        for (int r = 0; r < m; ++r) {
            tab.key[r][0] = (uint32_t)(b->seeds[r0 + r] & 0xFFFFFFFFull);
            tab.key[r][1] = (uint32_t)(b->seeds[r0 + r] >> 32);
            thresholds(T[(int64_t)(r0 + r) * T_stride], tab.thr[r]);
        }
        potts::BatchParams B = {};
        potts::ResidentParams &P = B.P;
        P.plane[0] = b->ws + (size_t)r0 * 2 * b->plane_bytes;
        P.plane[1] = P.plane[0] + b->plane_bytes;
        P.L = b->L;
        P.pitch = b->L / 2;
        P.q = (uint32_t)b->q;
        P.t0 = (uint32_t)b->t;
        P.nsweeps = (uint32_t)nsweeps;
        P.every = measure ? (uint32_t)every : 0u;
        P.E_series = E_dev ? E_dev + (size_t)r0 * series_stride : nullptr;
        P.hist_series = hist_dev ? hist_dev + (size_t)r0 * series_stride * b->q : nullptr;
        P.dE_series = dE_dev ? dE_dev + (size_t)r0 * delta_stride : nullptr;
        P.inbox = nullptr;
        P.error = b->error;
        P.rows_max = b->L;
        P.tyc = R.tyc;
        B.lattice_stride = 2ull * b->plane_bytes;
        B.series_stride = (unsigned long long)series_stride;
        B.delta_stride = (unsigned long long)delta_stride;
        e = potts::launch_batch(potts::compare_mode_of(b->q), b->stream_spec, B, tab, m, R.nthreads, R.smem, b->stream);
        b->launches += 1;
    }
    if (e != cudaSuccess) return fail(POTTS_ERR_CUDA, "batch launch failed: %s", cudaGetErrorString(e));
    b->t += (uint64_t)nsweeps;
    return POTTS_OK;
}

int check_batch_T(const potts_batch_t *b, const double *T, int64_t count)
{
    for (int64_t r = 0; r < count; ++r)
        if (!(T[r] > 0.0) || !std::isfinite(T[r])) return fail(POTTS_ERR_ARG, "T[%lld] = %g must be finite and > 0", (long long)r, T[r]);
    (void)b;
    return POTTS_OK;
}

// copy `bytes` of device series to the host and synchronise
int batch_finish(potts_batch_t *b, int rc, void *host0, const void *dev0, size_t bytes0, void *host1, const void *dev1, size_t bytes1)
{
    cudaError_t e = cudaSuccess;
    if (rc == POTTS_OK && bytes0) e = cudaMemcpyAsync(host0, dev0, bytes0, cudaMemcpyDeviceToHost, b->stream);
    if (rc == POTTS_OK && e == cudaSuccess && bytes1) e = cudaMemcpyAsync(host1, dev1, bytes1, cudaMemcpyDeviceToHost, b->stream);
    const cudaError_t e2 = cudaStreamSynchronize(b->stream);
    if (rc) return rc;
    if (e != cudaSuccess || e2 != cudaSuccess)
        return fail(POTTS_ERR_CUDA, "batch series copy / sync failed: %s", cudaGetErrorString(e != cudaSuccess ? e : e2));
    return POTTS_OK;
}

}  // namespace

extern "C" {

int potts_batch_sweep_measured(potts_batch_t *b, const double *T, int64_t nsweeps, int64_t every, int64_t *E_series,
                               int64_t *hist_series)
{
    ON_DEVICE_OF(b);
    if (!b || !T) return fail(POTTS_ERR_ARG, "null argument");
    if (nsweeps < 0 || nsweeps > (1ll << 30)) return fail(POTTS_ERR_ARG, "nsweeps = %lld outside [0, 2^30]", (long long)nsweeps);
    int rc = check_batch_T(b, T, b->n);
    if (rc) return rc;
    if (b->t + (uint64_t)nsweeps > 0xFFFFFFFFull) return fail(POTTS_ERR_ARG, "sweep counter would pass 2^32 - 1");
    const bool measure = E_series || hist_series;
    if (measure && (every < 1 || nsweeps % every != 0))
        return fail(POTTS_ERR_ARG, "every = %lld must be >= 1 and divide nsweeps = %lld", (long long)every, (long long)nsweeps);
    if (nsweeps == 0) return POTTS_OK;
    const int64_t ns = measure ? nsweeps / every : 0;
    const size_t eb = E_series ? (size_t)b->n * ns * 8 : 0, hb = hist_series ? (size_t)b->n * ns * b->q * 8 : 0;
    uint8_t *dev = nullptr;
    if (eb + hb) {
        rc = get_batch_scratch(b, eb + hb, &dev);
        if (rc) return rc;
        cudaMemsetAsync(dev, 0, eb + hb, b->stream);
    }
    rc = batch_run(b, T, 1, nsweeps, every, eb ? (unsigned long long *)dev : nullptr, hb ? (unsigned long long *)(dev + eb) : nullptr,
                   ns, nullptr, 0);
    return batch_finish(b, rc, E_series, dev, eb, hist_series, dev + eb, hb);
}

int potts_batch_sweep_measured_dev(potts_batch_t *b, const double *T, int64_t nsweeps, int64_t every, int64_t *E_series_dev,
                                   int64_t *hist_series_dev)
{
    ON_DEVICE_OF(b);
    if (!b || !T) return fail(POTTS_ERR_ARG, "null argument");
    if (nsweeps < 0 || nsweeps > (1ll << 30)) return fail(POTTS_ERR_ARG, "nsweeps = %lld outside [0, 2^30]", (long long)nsweeps);
    int rc = check_batch_T(b, T, b->n);
    if (rc) return rc;
    if (b->t + (uint64_t)nsweeps > 0xFFFFFFFFull) return fail(POTTS_ERR_ARG, "sweep counter would pass 2^32 - 1");
    const bool measure = E_series_dev || hist_series_dev;
    if (measure && (every < 1 || nsweeps % every != 0))
        return fail(POTTS_ERR_ARG, "every = %lld must be >= 1 and divide nsweeps = %lld", (long long)every, (long long)nsweeps);
    if (nsweeps == 0) return POTTS_OK;
    const int64_t ns = measure ? nsweeps / every : 0;
    if (E_series_dev) CUDA_TRY(cudaMemsetAsync(E_series_dev, 0, (size_t)b->n * ns * 8, b->stream));
    if (hist_series_dev) CUDA_TRY(cudaMemsetAsync(hist_series_dev, 0, (size_t)b->n * ns * b->q * 8, b->stream));
    return batch_run(b, T, 1, nsweeps, every, (unsigned long long *)E_series_dev, (unsigned long long *)hist_series_dev, ns, nullptr, 0);
}

int potts_batch_sweep_delta(potts_batch_t *b, const double *T, int64_t nsweeps, int64_t *dE_series)
{
    ON_DEVICE_OF(b);
    if (!b || !T || !dE_series) return fail(POTTS_ERR_ARG, "null argument");
    if (nsweeps < 0 || nsweeps > (1ll << 30)) return fail(POTTS_ERR_ARG, "nsweeps = %lld outside [0, 2^30]", (long long)nsweeps);
    int rc = check_batch_T(b, T, b->n);
    if (rc) return rc;
    if (b->t + (uint64_t)nsweeps > 0xFFFFFFFFull) return fail(POTTS_ERR_ARG, "sweep counter would pass 2^32 - 1");
    if (nsweeps == 0) return POTTS_OK;
    const size_t db = (size_t)b->n * nsweeps * 8;
    uint8_t *dev = nullptr;
    rc = get_batch_scratch(b, db, &dev);
    if (rc) return rc;
    cudaMemsetAsync(dev, 0, db, b->stream);
    rc = batch_run(b, T, 1, nsweeps, 0, nullptr, nullptr, 0, (unsigned long long *)dev, nsweeps);
    return batch_finish(b, rc, dE_series, dev, db, nullptr, nullptr, 0);
}

int potts_batch_ladder(potts_batch_t *b, const double *T, int32_t nT, int64_t t_tran, int64_t t_max, int64_t dt,
                       int64_t *E_series, int64_t *hist_series)
{
    ON_DEVICE_OF(b);
    if (!b || !T) return fail(POTTS_ERR_ARG, "null argument");
    if (nT < 0 || t_tran < 0 || t_max < 0 || t_tran > (1ll << 30) || t_max > (1ll << 30)) return fail(POTTS_ERR_ARG, "count outside [0, 2^30]");
    if (dt < 1 || t_max % dt != 0)
        return fail(POTTS_ERR_ARG, "dt = %lld must be >= 1 and divide t_max = %lld", (long long)dt, (long long)t_max);
    int rc = check_batch_T(b, T, (int64_t)b->n * nT);
    if (rc) return rc;
    if (b->t + (uint64_t)nT * (uint64_t)(t_tran + t_max) > 0xFFFFFFFFull) return fail(POTTS_ERR_ARG, "sweep counter would pass 2^32 - 1");
    const int64_t per_T = t_max / dt, ns = per_T * nT;
    const size_t eb = E_series ? (size_t)b->n * ns * 8 : 0, hb = hist_series ? (size_t)b->n * ns * b->q * 8 : 0;
    uint8_t *dev = nullptr;
    if (eb + hb) {
        rc = get_batch_scratch(b, eb + hb, &dev);
        if (rc) return rc;
        cudaMemsetAsync(dev, 0, eb + hb, b->stream);
    }
    unsigned long long *dE = eb ? (unsigned long long *)dev : nullptr, *dH = hb ? (unsigned long long *)(dev + eb) : nullptr;
    for (int32_t k = 0; k < nT && rc == POTTS_OK; ++k) {
        rc = batch_run(b, T + k, nT, t_tran, 0, nullptr, nullptr, 0, nullptr, 0);
        if (rc == POTTS_OK && per_T > 0)
            rc = batch_run(b, T + k, nT, t_max, dt, dE ? dE + k * per_T : nullptr, dH ? dH + k * per_T * b->q : nullptr, ns, nullptr, 0);
    }
    return batch_finish(b, rc, E_series, dev, eb, hist_series, dev + eb, hb);
}

int potts_batch_download(potts_batch_t *b, int32_t r, uint8_t *spins)
{
    ON_DEVICE_OF(b);
    if (!b || !spins) return fail(POTTS_ERR_ARG, "null argument");
    if (r < 0 || r >= b->n) return fail(POTTS_ERR_ARG, "lattice index %d outside [0, %d)", r, b->n);
    const int L = b->L;
    uint8_t *stage = nullptr;
    int rc = get_batch_scratch(b, (size_t)L * L, &stage);
    if (rc) return rc;
    uint8_t *p0 = b->ws + (size_t)r * 2 * b->plane_bytes;
    const long long threads = (long long)L * (L / 8);
    potts::k_planes_to_rowmajor<<<(unsigned)((threads + 255) / 256), 256, 0, b->stream>>>(p0, p0 + b->plane_bytes, stage, L, L / 2, 0, L);
    b->launches += 1;
    cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess) e = cudaMemcpyAsync(spins, stage, (size_t)L * L, cudaMemcpyDeviceToHost, b->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(b->stream);
    if (e != cudaSuccess) return fail(POTTS_ERR_CUDA, "batch download failed: %s", cudaGetErrorString(e));
    return POTTS_OK;
}

}  // extern "C"
