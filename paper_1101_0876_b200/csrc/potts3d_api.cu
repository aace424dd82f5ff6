// potts3d_api.cu -- C-ABI of the 3D generalisation (include/potts.h, section "3D"): argument checking, device
// memory, launches.  Every step runs in the kernels of potts3d.cuh; this file only marshals.
#include "../../include/potts.h"
#include "potts3d.cuh"

#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <new>

namespace potts {
int set_error(int code, const char *msg);      // potts_api.cu: the message potts_last_error() returns
}

namespace {

int fail(int code, const char *fmt, ...)
{
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    return potts::set_error(code, buf);
}

#define CUDA_TRY3(expr)                                                                         \
    do {                                                                                        \
        cudaError_t e_ = (expr);                                                                \
        if (e_ != cudaSuccess)                                                                  \
            return fail(e_ == cudaErrorMemoryAllocation ? POTTS_ERR_NOMEM : POTTS_ERR_CUDA,     \
                        "%s failed: %s", #expr, cudaGetErrorString(e_));                        \
    } while (0)

constexpr size_t ALIGN3 = 256;
size_t align_up3(size_t x) { return (x + ALIGN3 - 1) / ALIGN3 * ALIGN3; }

struct DeviceGuard3 {
    int prev = -1;
    explicit DeviceGuard3(int dev)
    {
        if (cudaGetDevice(&prev) != cudaSuccess) { prev = -1; return; }
        if (prev != dev) cudaSetDevice(dev); else prev = -1;
    }
    ~DeviceGuard3() { if (prev >= 0) cudaSetDevice(prev); }
};

}  // namespace

struct potts3_s {
    int32_t L = 0, q = 0;
    int device = 0;
    uint64_t seed = 0, t = 0, launches = 0;
    uint8_t *ws = nullptr;
    size_t plane_bytes = 0;
    uint8_t *plane[2] = {nullptr, nullptr};
    unsigned long long *acc = nullptr;     // device: [0] = E, [1..256] = histogram, [257] = upload flag, [258] = tile counter
    uint8_t *scratch = nullptr;            // device: series of a measured call / staging of up- and download
    size_t scratch_bytes = 0;
    cudaStream_t stream = nullptr;
    int num_sms = 0;
    uint32_t *tile_counter = nullptr;      // device: tile scheduler of k_sweep3_rows_u8 (returns to 0 at the end of every launch)
    int32_t opt_rows = 0, opt_words = 0;   // potts3_set_option
};

namespace {

int scratch3(potts3_t *h, size_t bytes, uint8_t **out)
{
    if (h->scratch_bytes < bytes) {
        if (h->scratch) { cudaStreamSynchronize(h->stream); cudaFree(h->scratch); h->scratch = nullptr; h->scratch_bytes = 0; }
        CUDA_TRY3(cudaMalloc(&h->scratch, bytes));
        h->scratch_bytes = bytes;
    }
    *out = h->scratch;
    return POTTS_OK;
}

int launched3(potts3_t *h, const char *what)
{
    h->launches += 1;
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(POTTS_ERR_CUDA, "launch of %s failed: %s", what, cudaGetErrorString(e));
    return POTTS_OK;
}

// the row-walking kernel: W words per lane and row, grid = the blocks resident at once
template <int CM, int COLOUR, int W, bool FAST>
void launch_rows3(const potts::Sweep3RowsParams &P, int num_sms, cudaStream_t st)
{
    auto fn = potts::k_sweep3_rows_u8<CM, COLOUR, W, FAST>;
    static int per_sm = 0;
    if (per_sm == 0) {
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, fn, 32 * potts::H3_WARPS, 0);
        if (per_sm < 1) per_sm = 1;
    }
    const unsigned long long want = (unsigned long long)per_sm * (unsigned)num_sms;
    const unsigned grid = (unsigned)(want < P.total_tiles ? want : P.total_tiles);
    fn<<<grid, dim3(32, potts::H3_WARPS), 0, st>>>(P);
}

template <int CM, int W>
void launch_rows3_cw(const potts::Sweep3RowsParams &P, uint32_t colour, int num_sms, cudaStream_t st)
{
    const bool fast = potts::accept_fast_ok3(P.thr);
    if (colour == 0) { if (fast) launch_rows3<CM, 0, W, true>(P, num_sms, st); else launch_rows3<CM, 0, W, false>(P, num_sms, st); }
    else { if (fast) launch_rows3<CM, 1, W, true>(P, num_sms, st); else launch_rows3<CM, 1, W, false>(P, num_sms, st); }
}

template <int CM>
void launch_rows3_c(const potts::Sweep3RowsParams &P, uint32_t colour, int W, int num_sms, cudaStream_t st)
{
    if (W == 4) launch_rows3_cw<CM, 4>(P, colour, num_sms, st);
    else if (W == 2) launch_rows3_cw<CM, 2>(P, colour, num_sms, st);
    else launch_rows3_cw<CM, 1>(P, colour, num_sms, st);
}

struct Thresholds3 {
    uint32_t thr[6];                       // floor(2^32 exp(-d/T)), d = 1..6 (reading R6')
    unsigned long long neg_thr[13];        // 2^64 - threshold(d), d = -6..6
};

int half_sweep3(potts3_t *h, uint32_t colour, const Thresholds3 &TH)
{
    int W = h->opt_words < 0 ? 0 : (h->opt_words > 0 ? h->opt_words : 4);
    if (h->opt_words == 0) {
        // lanes are dealt to a row in powers of two (or whole warps): with L = 3 * 2^k a quarter of them would idle,
        // and the one-chunk-per-thread kernel is the faster one (measured at L = 384: 3.40 against 3.62 ps)
        const int chunks = h->L / 32;
        int lanes = 1;
        while (lanes < 32 && lanes < chunks) lanes <<= 1;
        if (chunks > 32) lanes = (chunks + 31) / 32 * 32;
        if (10 * chunks < 9 * lanes) W = 0;
    }
    if (W > 0) {
        potts::Sweep3RowsParams P;
        P.plane_own = h->plane[colour];
        P.plane_oth = h->plane[1 - colour];
        P.L = h->L;
        P.pitch = h->L / 2;
        P.q = (uint32_t)h->q;
        P.key1 = (uint32_t)(h->seed >> 32);
        P.K = potts::half_sweep_keys((uint32_t)(h->seed & 0xFFFFFFFFull), P.key1, (uint32_t)h->t, colour);
        for (int d = 0; d < 6; ++d) P.thr[d] = TH.thr[d];
        const int chunks = P.pitch / (4 * W);                           // lanes a row takes
        P.lpr_log2 = 0;
        while (P.lpr_log2 < 5 && (1 << P.lpr_log2) < chunks) P.lpr_log2 += 1;
        const int windows_per_tile = potts::H3_WARPS << (5 - P.lpr_log2);
        P.rpw = h->opt_rows > 0 ? h->opt_rows : 16;                     // L % 32 == 0: 2 .. 32 all divide L
        const int cbs = (chunks + 31) / 32;
        for (;;) {
            P.row_groups = (h->L / P.rpw + windows_per_tile - 1) / windows_per_tile;
            P.total_tiles = (uint32_t)cbs * (uint32_t)h->L * (uint32_t)P.row_groups;
            // automatic: shorter windows until there are ~7 tiles per SM to draw (L = 256: 16 -> 4 rows, 3.92 -> 3.21 ps)
            if (h->opt_rows > 0 || P.rpw <= 2 || P.total_tiles >= 1024u) break;
            P.rpw >>= 1;
        }
        P.tile_counter = h->tile_counter;
        switch (potts::compare_mode_of(h->q)) {
        case potts::CM_7BIT: launch_rows3_c<potts::CM_7BIT>(P, colour, W, h->num_sms, h->stream); break;
        case potts::CM_8BIT: launch_rows3_c<potts::CM_8BIT>(P, colour, W, h->num_sms, h->stream); break;
        case potts::CM_NIB4: launch_rows3_c<potts::CM_NIB4>(P, colour, W, h->num_sms, h->stream); break;
        default: launch_rows3_c<potts::CM_NIB3>(P, colour, W, h->num_sms, h->stream); break;
        }
        return launched3(h, "k_sweep3_rows_u8");
    }
    potts::Sweep3Params P;
    P.plane_own = h->plane[colour];
    P.plane_oth = h->plane[1 - colour];
    P.L = h->L;
    P.pitch = h->L / 2;
    P.q = (uint32_t)h->q;
    P.colour = colour;
    P.key0 = (uint32_t)(h->seed & 0xFFFFFFFFull);
    P.key1 = (uint32_t)(h->seed >> 32);
    P.t = (uint32_t)h->t;
    for (int k = 0; k < 13; ++k) P.neg_thr[k] = TH.neg_thr[k];
    const long long chunks = (long long)h->L * h->L * (h->L / 32);
    long long blocks = (chunks + 127) / 128;
    const long long cap = (long long)h->num_sms * 8;
    if (blocks > cap) blocks = cap;
    switch (potts::compare_mode_of(h->q)) {
    case potts::CM_7BIT: potts::k_sweep3_u8<potts::CM_7BIT><<<(unsigned)blocks, 128, 0, h->stream>>>(P); break;
    case potts::CM_8BIT: potts::k_sweep3_u8<potts::CM_8BIT><<<(unsigned)blocks, 128, 0, h->stream>>>(P); break;
    case potts::CM_NIB4: potts::k_sweep3_u8<potts::CM_NIB4><<<(unsigned)blocks, 128, 0, h->stream>>>(P); break;
    default: potts::k_sweep3_u8<potts::CM_NIB3><<<(unsigned)blocks, 128, 0, h->stream>>>(P); break;
    }
    return launched3(h, "k_sweep3_u8");
}

int measure3(potts3_t *h, unsigned long long *E_out, unsigned long long *hist_out)
{
    potts::Measure3Params M;
    M.plane0 = h->plane[0];
    M.plane1 = h->plane[1];
    M.L = h->L;
    M.pitch = h->L / 2;
    M.q = (uint32_t)h->q;
    M.E_out = E_out;
    M.hist_out = hist_out;
    const long long chunks = (long long)h->L * h->L * (h->L / 32);
    long long blocks = (chunks + 255) / 256;
    if (blocks > (long long)h->num_sms * 8) blocks = (long long)h->num_sms * 8;
    const size_t smem = hist_out ? (size_t)potts::hist_words((uint32_t)h->q) * 4 : 0;
    if (h->q > 128) potts::k_measure3_u8<true><<<(unsigned)blocks, 256, smem, h->stream>>>(M);
    else potts::k_measure3_u8<false><<<(unsigned)blocks, 256, smem, h->stream>>>(M);
    return launched3(h, "k_measure3_u8");
}

// nsweeps sweeps; every > 0: after every `every`-th sweep the energy / histogram go to the device series
int run3(potts3_t *h, double T, int64_t nsweeps, int64_t every, unsigned long long *E_dev, unsigned long long *hist_dev)
{
    Thresholds3 TH;
    for (int d = -6; d <= 6; ++d) {
        // reading R6': threshold(d) = 2^32 for d <= 0, floor(ldexp(exp(-d/T), 32)) for d = 1..6
        const unsigned long long th = d <= 0 ? (1ull << 32) : (unsigned long long)(uint32_t)std::floor(std::ldexp(std::exp(-(double)d / T), 32));
        TH.neg_thr[d + 6] = 0ull - th;
        if (d > 0) TH.thr[d - 1] = (uint32_t)th;
    }
    for (int64_t n = 0; n < nsweeps; ++n) {
        int rc = half_sweep3(h, 0u, TH);
        if (rc == POTTS_OK) rc = half_sweep3(h, 1u, TH);
        if (rc) return rc;
        h->t += 1;
        if (every > 0 && (n + 1) % every == 0 && (E_dev || hist_dev)) {
            const int64_t k = (n + 1) / every - 1;
            rc = measure3(h, E_dev ? E_dev + k : nullptr, hist_dev ? hist_dev + k * h->q : nullptr);
            if (rc) return rc;
        }
    }
    return POTTS_OK;
}

int check_args3(potts3_t *h, double T, int64_t nsweeps)
{
    if (!h) return fail(POTTS_ERR_ARG, "null handle");
    if (!(T > 0.0) || !std::isfinite(T)) return fail(POTTS_ERR_ARG, "T = %g must be finite and > 0", T);
    if (nsweeps < 0) return fail(POTTS_ERR_ARG, "nsweeps = %lld < 0", (long long)nsweeps);
    if (h->t + (uint64_t)nsweeps > 0xFFFFFFFFull) return fail(POTTS_ERR_ARG, "sweep counter would pass 2^32 - 1 (Philox counter word)");
    return POTTS_OK;
}

int chunk_rows3(int L) { long long r = (32ll << 20) / L; return (int)(r < 1 ? 1 : r); }

}  // namespace

extern "C" {

int potts3_create(potts3_t **out, int32_t L, int32_t q, uint64_t seed, int32_t init, void *cuda_stream)
{
    if (!out) return fail(POTTS_ERR_ARG, "null out pointer");
    if (init != POTTS_INIT_ORDERED && init != POTTS_INIT_RANDOM) return fail(POTTS_ERR_ARG, "bad init %d", init);
    if (L < 2 || (L & 1)) return fail(POTTS_ERR_ARG, "L = %d must be even and >= 2", L);
    if (q < 2 || q > 256) return fail(POTTS_ERR_ARG, "q = %d outside [2, 256]", q);
    if (L % 32 != 0) return fail(POTTS_ERR_UNSUPPORTED, "L = %d is not a multiple of 32 (kernel vector width)", L);
    if (L > 2048) return fail(POTTS_ERR_UNSUPPORTED, "L = %d: a cubic lattice above 2048^3 does not fit the device", L);
    int ndev = 0;
    CUDA_TRY3(cudaGetDeviceCount(&ndev));
    if (ndev < 1) return fail(POTTS_ERR_CUDA, "no CUDA device");
    potts3_t *h = new (std::nothrow) potts3_s;
    if (!h) return fail(POTTS_ERR_NOMEM, "host allocation failed");
    h->L = L; h->q = q; h->seed = seed; h->stream = (cudaStream_t)cuda_stream;
    cudaGetDevice(&h->device);
    cudaDeviceGetAttribute(&h->num_sms, cudaDevAttrMultiProcessorCount, h->device);
    h->plane_bytes = align_up3((size_t)L * L * (L / 2));
    const size_t need = 2 * h->plane_bytes + align_up3(260 * sizeof(unsigned long long));
    const cudaError_t e = cudaMalloc(&h->ws, need);
    if (e != cudaSuccess) {
        delete h;
        return fail(e == cudaErrorMemoryAllocation ? POTTS_ERR_NOMEM : POTTS_ERR_CUDA, "cudaMalloc(%zu) failed: %s", need, cudaGetErrorString(e));
    }
    h->plane[0] = h->ws;
    h->plane[1] = h->ws + h->plane_bytes;
    h->acc = (unsigned long long *)(h->ws + 2 * h->plane_bytes);
    h->tile_counter = (uint32_t *)(h->acc + 258);
    cudaError_t e2 = cudaMemsetAsync(h->ws, 0, need, h->stream);
    if (e2 == cudaSuccess && init == POTTS_INIT_RANDOM) {
        const long long words = 2ll * L * L * (L / 8);
        potts::k_init_random3_u8<<<(unsigned)((words + 255) / 256), 256, 0, h->stream>>>(
            h->plane[0], h->plane[1], L, L / 2, (uint32_t)q, (uint32_t)(seed & 0xFFFFFFFFull), (uint32_t)(seed >> 32));
        h->launches += 1;
        e2 = cudaGetLastError();
    }
    if (e2 != cudaSuccess) {
        potts3_destroy(h);
        return fail(POTTS_ERR_CUDA, "initialisation failed: %s", cudaGetErrorString(e2));
    }
    *out = h;
    return POTTS_OK;
}

void potts3_destroy(potts3_t *h)
{
    if (!h) return;
    DeviceGuard3 g(h->device);
    cudaStreamSynchronize(h->stream);
    if (h->scratch) cudaFree(h->scratch);
    if (h->ws) cudaFree(h->ws);
    delete h;
}

int potts3_sweep(potts3_t *h, double T, int64_t nsweeps)
{
    int rc = check_args3(h, T, nsweeps);
    if (rc) return rc;
    DeviceGuard3 g(h->device);
    return run3(h, T, nsweeps, 0, nullptr, nullptr);
}

int potts3_sweep_measured(potts3_t *h, double T, int64_t nsweeps, int64_t every, int64_t *E_series, int64_t *hist_series)
{
    int rc = check_args3(h, T, nsweeps);
    if (rc) return rc;
    if (every < 1 || nsweeps % every != 0)
        return fail(POTTS_ERR_ARG, "every = %lld must be >= 1 and divide nsweeps = %lld", (long long)every, (long long)nsweeps);
    DeviceGuard3 g(h->device);
    const int64_t ns = nsweeps / every;
    if (ns == 0) return POTTS_OK;
    const size_t eb = E_series ? (size_t)ns * 8 : 0, hb = hist_series ? (size_t)ns * h->q * 8 : 0;
    uint8_t *dev = nullptr;
    if (eb + hb) {
        rc = scratch3(h, eb + hb, &dev);
        if (rc) return rc;
        CUDA_TRY3(cudaMemsetAsync(dev, 0, eb + hb, h->stream));
    }
    rc = run3(h, T, nsweeps, every, eb ? (unsigned long long *)dev : nullptr, hb ? (unsigned long long *)(dev + eb) : nullptr);
    cudaError_t e = cudaSuccess;
    if (rc == POTTS_OK && eb) e = cudaMemcpyAsync(E_series, dev, eb, cudaMemcpyDeviceToHost, h->stream);
    if (rc == POTTS_OK && e == cudaSuccess && hb) e = cudaMemcpyAsync(hist_series, dev + eb, hb, cudaMemcpyDeviceToHost, h->stream);
    const cudaError_t e2 = cudaStreamSynchronize(h->stream);
    if (rc) return rc;
    if (e != cudaSuccess || e2 != cudaSuccess) return fail(POTTS_ERR_CUDA, "series copy / sync failed: %s", cudaGetErrorString(e != cudaSuccess ? e : e2));
    return POTTS_OK;
}

int potts3_energy(potts3_t *h, int64_t *E)
{
    if (!h || !E) return fail(POTTS_ERR_ARG, "null argument");
    DeviceGuard3 g(h->device);
    CUDA_TRY3(cudaMemsetAsync(h->acc, 0, 8, h->stream));
    int rc = measure3(h, h->acc, nullptr);
    if (rc) return rc;
    int64_t v = 0;
    CUDA_TRY3(cudaMemcpyAsync(&v, h->acc, 8, cudaMemcpyDeviceToHost, h->stream));
    CUDA_TRY3(cudaStreamSynchronize(h->stream));
    *E = v;
    return POTTS_OK;
}

int potts3_histogram(potts3_t *h, int64_t *counts)
{
    if (!h || !counts) return fail(POTTS_ERR_ARG, "null argument");
    DeviceGuard3 g(h->device);
    CUDA_TRY3(cudaMemsetAsync(h->acc + 1, 0, 8 * (size_t)h->q, h->stream));
    int rc = measure3(h, nullptr, h->acc + 1);
    if (rc) return rc;
    CUDA_TRY3(cudaMemcpyAsync(counts, h->acc + 1, 8 * (size_t)h->q, cudaMemcpyDeviceToHost, h->stream));
    CUDA_TRY3(cudaStreamSynchronize(h->stream));
    return POTTS_OK;
}

int potts3_download(potts3_t *h, uint8_t *spins)
{
    if (!h || !spins) return fail(POTTS_ERR_ARG, "null argument");
    DeviceGuard3 g(h->device);
    const int L = h->L, rows = chunk_rows3(L);
    const long long total_rows = (long long)L * L;
    uint8_t *stage = nullptr;
    int rc = scratch3(h, (size_t)rows * L, &stage);
    if (rc) return rc;
    for (long long r0 = 0; r0 < total_rows; r0 += rows) {
        const int r = (int)(total_rows - r0 < rows ? total_rows - r0 : rows);
        const long long threads = (long long)r * (L / 8);
        potts::k_planes_to_rowmajor3<<<(unsigned)((threads + 255) / 256), 256, 0, h->stream>>>(h->plane[0], h->plane[1], stage, L, L / 2, r0, r);
        rc = launched3(h, "k_planes_to_rowmajor3");
        if (rc) return rc;
        CUDA_TRY3(cudaMemcpyAsync(spins + (size_t)r0 * L, stage, (size_t)r * L, cudaMemcpyDeviceToHost, h->stream));
        CUDA_TRY3(cudaStreamSynchronize(h->stream));
    }
    return POTTS_OK;
}

int potts3_upload(potts3_t *h, const uint8_t *spins)
{
    if (!h || !spins) return fail(POTTS_ERR_ARG, "null argument");
    DeviceGuard3 g(h->device);
    const int L = h->L, rows = chunk_rows3(L);
    const long long total_rows = (long long)L * L;
    if (h->q < 256)
        for (size_t n = 0; n < (size_t)L * L * L; ++n)
            if (spins[n] >= h->q) return fail(POTTS_ERR_ARG, "spin value %d >= q at offset %zu", (int)spins[n], n);
    uint8_t *stage = nullptr;
    int rc = scratch3(h, (size_t)rows * L, &stage);
    if (rc) return rc;
    int *flag = (int *)(h->acc + 257);
    CUDA_TRY3(cudaMemsetAsync(flag, 0, sizeof(int), h->stream));
    for (long long r0 = 0; r0 < total_rows; r0 += rows) {
        const int r = (int)(total_rows - r0 < rows ? total_rows - r0 : rows);
        CUDA_TRY3(cudaMemcpyAsync(stage, spins + (size_t)r0 * L, (size_t)r * L, cudaMemcpyHostToDevice, h->stream));
        const long long threads = (long long)r * (L / 8);
        potts::k_rowmajor_to_planes3<<<(unsigned)((threads + 255) / 256), 256, 0, h->stream>>>(stage, h->plane[0], h->plane[1], L, L / 2, r0, r,
                                                                                                (uint32_t)h->q, flag);
        rc = launched3(h, "k_rowmajor_to_planes3");
        if (rc) return rc;
        CUDA_TRY3(cudaStreamSynchronize(h->stream));
    }
    return POTTS_OK;
}

int potts3_sweep_count(potts3_t *h, uint64_t *t)
{
    if (!h || !t) return fail(POTTS_ERR_ARG, "null argument");
    *t = h->t;
    return POTTS_OK;
}

int potts3_set_sweep_count(potts3_t *h, uint64_t t)
{
    if (!h) return fail(POTTS_ERR_ARG, "null handle");
    if (t > 0xFFFFFFFFull) return fail(POTTS_ERR_ARG, "t must be < 2^32");
    h->t = t;
    return POTTS_OK;
}

int potts3_launch_count(potts3_t *h, uint64_t *n)
{
    if (!h || !n) return fail(POTTS_ERR_ARG, "null argument");
    *n = h->launches;
    return POTTS_OK;
}

int potts3_set_option(potts3_t *h, const char *key, int64_t value)
{
    if (!h || !key) return fail(POTTS_ERR_ARG, "null argument");
    if (!std::strcmp(key, "stream_words")) {
        if (value != 0 && value != 1 && value != 2 && value != 4 && value != -1) return fail(POTTS_ERR_ARG, "stream_words = %lld not in {-1, 0, 1, 2, 4}", (long long)value);
        h->opt_words = (int32_t)value;
        return POTTS_OK;
    }
    if (!std::strcmp(key, "stream_rows")) {
        if (value != 0 && value != 2 && value != 4 && value != 8 && value != 16 && value != 32) return fail(POTTS_ERR_ARG, "stream_rows = %lld not in {0, 2, 4, 8, 16, 32}", (long long)value);
        h->opt_rows = (int32_t)value;
        return POTTS_OK;
    }
    return fail(POTTS_ERR_ARG, "unknown option '%s'", key);
}

}  // extern "C"
