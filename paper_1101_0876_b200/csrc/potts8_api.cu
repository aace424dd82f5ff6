// potts8_api.cu -- C-ABI of the first + second neighbour generalisation (include/potts.h, section "first and second neighbours"): argument checking, device
// memory, launches.  Every step runs in the kernels of potts8.cuh; this file only marshals.
#include "../../include/potts.h"
#include "potts8.cuh"

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

#define CUDA_TRY8(expr)                                                                         \
    do {                                                                                        \
        cudaError_t e_ = (expr);                                                                \
        if (e_ != cudaSuccess)                                                                  \
            return fail(e_ == cudaErrorMemoryAllocation ? POTTS_ERR_NOMEM : POTTS_ERR_CUDA,     \
                        "%s failed: %s", #expr, cudaGetErrorString(e_));                        \
    } while (0)

constexpr size_t ALIGN8 = 256;
size_t align_up8(size_t x) { return (x + ALIGN8 - 1) / ALIGN8 * ALIGN8; }

struct DeviceGuard8 {
    int prev = -1;
    explicit DeviceGuard8(int dev)
    {
        if (cudaGetDevice(&prev) != cudaSuccess) { prev = -1; return; }
        if (prev != dev) cudaSetDevice(dev); else prev = -1;
    }
    ~DeviceGuard8() { if (prev >= 0) cudaSetDevice(prev); }
};

}  // namespace

struct potts8_s {
    int32_t L = 0, q = 0;
    int device = 0;
    uint64_t seed = 0, t = 0, launches = 0;
    uint8_t *ws = nullptr;
    size_t plane_bytes = 0;
    unsigned long long *acc = nullptr;     // device: [0] = E, [1..256] = histogram, [257] = upload flag
    uint8_t *scratch = nullptr;            // device: series of a measured call / staging of up- and download
    size_t scratch_bytes = 0;
    cudaStream_t stream = nullptr;
    int num_sms = 0;
    uint32_t *tile_counter = nullptr;      // device: tile scheduler of k_sweep8_rows_u8 (returns to 0 at the end of every launch)
    int32_t opt_rows = 0, opt_words = 0;   // potts8_set_option
};

namespace {

int scratch8(potts8_t *h, size_t bytes, uint8_t **out)
{
    if (h->scratch_bytes < bytes) {
        if (h->scratch) { cudaStreamSynchronize(h->stream); cudaFree(h->scratch); h->scratch = nullptr; h->scratch_bytes = 0; }
        CUDA_TRY8(cudaMalloc(&h->scratch, bytes));
        h->scratch_bytes = bytes;
    }
    *out = h->scratch;
    return POTTS_OK;
}

int launched8(potts8_t *h, const char *what)
{
    h->launches += 1;
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(POTTS_ERR_CUDA, "launch of %s failed: %s", what, cudaGetErrorString(e));
    return POTTS_OK;
}

// descriptor of the neighbour (di, dj) of the sites of sub-network c = 3 a + b
potts::Nbr8 neighbour8(uint32_t c, int di, int dj)
{
    const int a = (int)(c / 3), b = (int)(c % 3), a2 = a + di, b2 = b + dj;
    potts::Nbr8 n;
    n.dI = a2 < 0 ? -1 : (a2 > 2 ? 1 : 0);
    n.shift = b2 < 0 ? -1 : (b2 > 2 ? 1 : 0);
    n.plane = 3 * ((a2 + 3) % 3) + (b2 + 3) % 3;
    return n;
}

potts::Sweep8Params params8(const potts8_t *h, uint32_t c)
{
    potts::Sweep8Params P = {};
    P.planes = h->ws;
    P.plane_bytes = h->plane_bytes;
    P.L = h->L;
    P.pitch = P.rows = h->L / 3;
    P.q = (uint32_t)h->q;
    P.c = c;
    P.key0 = (uint32_t)(h->seed & 0xFFFFFFFFull);
    P.key1 = (uint32_t)(h->seed >> 32);
    P.t = (uint32_t)h->t;
    // the four forward directions first (k_measure8_u8 counts every bond once from them), then their opposites
    static const int dir[8][2] = {{0, 1}, {1, 0}, {1, 1}, {1, -1}, {0, -1}, {-1, 0}, {-1, -1}, {-1, 1}};
    for (int k = 0; k < 8; ++k) P.nbr[k] = neighbour8(c, dir[k][0], dir[k][1]);
    return P;
}

unsigned grid8(const potts8_t *h, int block)
{
    const long long words = (long long)(h->L / 3) * (h->L / 12);
    long long blocks = (words + block - 1) / block;
    const long long cap = (long long)h->num_sms * 8;
    return (unsigned)(blocks > cap ? cap : (blocks < 1 ? 1 : blocks));
}

struct Thresholds8 {
    uint32_t thr[8];                       // floor(2^32 exp(-d/T)), d = 1..8 (reading R6")
    unsigned long long neg_thr[17];        // 2^64 - threshold(d), d = -8..8
};

template <int CM, int B, bool FAST>
void launch_rows8(const potts::Sweep8RowsParams &P, int num_sms, cudaStream_t st)
{
    auto fn = potts::k_sweep8_rows_u8<CM, B, FAST>;
    static int per_sm = 0;
    if (per_sm == 0) {
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, fn, 32 * potts::H8_WARPS, 0);
        if (per_sm < 1) per_sm = 1;
    }
    const unsigned long long want = (unsigned long long)per_sm * (unsigned)num_sms;
    const unsigned grid = (unsigned)(want < P.total_tiles ? want : P.total_tiles);
    fn<<<grid, dim3(32, potts::H8_WARPS), 0, st>>>(P);
}

template <int CM>
void launch_rows8_c(const potts::Sweep8RowsParams &P, int num_sms, cudaStream_t st)
{
    const bool fast = potts::accept_fast_ok8(P.thr);
    switch (P.c % 3u) {
    case 0: if (fast) launch_rows8<CM, 0, true>(P, num_sms, st); else launch_rows8<CM, 0, false>(P, num_sms, st); break;
    case 1: if (fast) launch_rows8<CM, 1, true>(P, num_sms, st); else launch_rows8<CM, 1, false>(P, num_sms, st); break;
    default: if (fast) launch_rows8<CM, 2, true>(P, num_sms, st); else launch_rows8<CM, 2, false>(P, num_sms, st); break;
    }
}

int class_sweep8(potts8_t *h, uint32_t c, const Thresholds8 &TH)
{
    const potts::Sweep8Params P = [&] {
        potts::Sweep8Params p = params8(h, c);
        for (int k = 0; k < 17; ++k) p.neg_thr[k] = TH.neg_thr[k];
        return p;
    }();
    const int pitch = h->L / 3;
    // automatic: from 2^20 sites per launch on; below, a launch is a few blocks per SM and the per-block tables
    // (accept table, ColKeys) cost more than they save (measured at L = 768: 129 against 63 ps, launch latency both)
    const bool rows_kernel = h->opt_words > 0 || (h->opt_words == 0 && h->L >= 3072);
    if (rows_kernel && pitch % 16 == 0 && 9ull * h->plane_bytes < (1ull << 32)) {   // the kernel's plane offsets are 32 bit
        potts::Sweep8RowsParams R;
        R.planes = P.planes;
        R.plane_bytes = P.plane_bytes;
        R.pitch = R.rows = pitch;
        R.q = P.q;
        R.c = c;
        R.K = potts::half_sweep_keys(P.key0, P.key1, P.t, 16u + c);
        for (int k = 0; k < 8; ++k) R.nbr[k] = P.nbr[k];
        for (int d = 0; d < 8; ++d) R.thr[d] = TH.thr[d];
        const int chunks = pitch / 16;
        R.lpr_log2 = 0;
        while (R.lpr_log2 < 5 && (1 << R.lpr_log2) < chunks) R.lpr_log2 += 1;
        const int windows_per_tile = potts::H8_WARPS << (5 - R.lpr_log2);
        R.rpw = h->opt_rows > 0 ? h->opt_rows : 16;                     // pitch % 16 == 0: 2 .. 16 divide the rows
        const int cbs = (chunks + 31) / 32;
        for (;;) {
            R.row_groups = (pitch / R.rpw + windows_per_tile - 1) / windows_per_tile;
            R.total_tiles = (uint32_t)cbs * (uint32_t)R.row_groups;
            if (h->opt_rows > 0 || R.rpw <= 2 || R.total_tiles >= 1024u) break;   // automatic: ~7 tiles per SM to draw
            R.rpw >>= 1;
        }
        R.tile_counter = h->tile_counter;
        switch (potts::compare_mode_of(h->q)) {
        case potts::CM_7BIT: launch_rows8_c<potts::CM_7BIT>(R, h->num_sms, h->stream); break;
        case potts::CM_8BIT: launch_rows8_c<potts::CM_8BIT>(R, h->num_sms, h->stream); break;
        case potts::CM_NIB4: launch_rows8_c<potts::CM_NIB4>(R, h->num_sms, h->stream); break;
        default: launch_rows8_c<potts::CM_NIB3>(R, h->num_sms, h->stream); break;
        }
        return launched8(h, "k_sweep8_rows_u8");
    }
    const unsigned blocks = grid8(h, 128);
    switch (potts::compare_mode_of(h->q)) {
    case potts::CM_7BIT: potts::k_sweep8_u8<potts::CM_7BIT><<<blocks, 128, 0, h->stream>>>(P); break;
    case potts::CM_8BIT: potts::k_sweep8_u8<potts::CM_8BIT><<<blocks, 128, 0, h->stream>>>(P); break;
    case potts::CM_NIB4: potts::k_sweep8_u8<potts::CM_NIB4><<<blocks, 128, 0, h->stream>>>(P); break;
    default: potts::k_sweep8_u8<potts::CM_NIB3><<<blocks, 128, 0, h->stream>>>(P); break;
    }
    return launched8(h, "k_sweep8_u8");
}

int measure8(potts8_t *h, unsigned long long *E_out, unsigned long long *hist_out)
{
    const size_t smem = hist_out ? (size_t)potts::hist_words((uint32_t)h->q) * 4 : 0;
    for (uint32_t c = 0; c < 9; ++c) {
        const potts::Sweep8Params P = params8(h, c);
        if (h->q > 128) potts::k_measure8_u8<true><<<grid8(h, 256), 256, smem, h->stream>>>(P, E_out, hist_out);
        else potts::k_measure8_u8<false><<<grid8(h, 256), 256, smem, h->stream>>>(P, E_out, hist_out);
        const int rc = launched8(h, "k_measure8_u8");
        if (rc) return rc;
    }
    return POTTS_OK;
}

// nsweeps sweeps; every > 0: after every `every`-th sweep the energy / histogram go to the device series
int run8(potts8_t *h, double T, int64_t nsweeps, int64_t every, unsigned long long *E_dev, unsigned long long *hist_dev)
{
    Thresholds8 TH;
    for (int d = -8; d <= 8; ++d) {
        // reading R6": threshold(d) = 2^32 for d <= 0, floor(ldexp(exp(-d/T), 32)) for d = 1..8
        const unsigned long long th = d <= 0 ? (1ull << 32) : (unsigned long long)(uint32_t)std::floor(std::ldexp(std::exp(-(double)d / T), 32));
        TH.neg_thr[d + 8] = 0ull - th;
        if (d > 0) TH.thr[d - 1] = (uint32_t)th;
    }
    for (int64_t n = 0; n < nsweeps; ++n) {
        for (uint32_t c = 0; c < 9; ++c) {                                   // R2": the nine sub-networks in order
            const int rc = class_sweep8(h, c, TH);
            if (rc) return rc;
        }
        h->t += 1;
        if (every > 0 && (n + 1) % every == 0 && (E_dev || hist_dev)) {
            const int64_t k = (n + 1) / every - 1;
            const int rc = measure8(h, E_dev ? E_dev + k : nullptr, hist_dev ? hist_dev + k * h->q : nullptr);
            if (rc) return rc;
        }
    }
    return POTTS_OK;
}

int check_args8(potts8_t *h, double T, int64_t nsweeps)
{
    if (!h) return fail(POTTS_ERR_ARG, "null handle");
    if (!(T > 0.0) || !std::isfinite(T)) return fail(POTTS_ERR_ARG, "T = %g must be finite and > 0", T);
    if (nsweeps < 0) return fail(POTTS_ERR_ARG, "nsweeps = %lld < 0", (long long)nsweeps);
    if (h->t + (uint64_t)nsweeps > 0xFFFFFFFFull) return fail(POTTS_ERR_ARG, "sweep counter would pass 2^32 - 1 (Philox counter word)");
    return POTTS_OK;
}

}  // namespace

extern "C" {

int potts8_create(potts8_t **out, int32_t L, int32_t q, uint64_t seed, int32_t init, void *cuda_stream)
{
    if (!out) return fail(POTTS_ERR_ARG, "null out pointer");
    if (init != POTTS_INIT_ORDERED && init != POTTS_INIT_RANDOM) return fail(POTTS_ERR_ARG, "bad init %d", init);
    if (L < 3 || L % 3) return fail(POTTS_ERR_ARG, "L = %d must be a multiple of 3 (nine sub-networks)", L);
    if (q < 2 || q > 256) return fail(POTTS_ERR_ARG, "q = %d outside [2, 256]", q);
    if (L % 12 != 0) return fail(POTTS_ERR_UNSUPPORTED, "L = %d is not a multiple of 12 (4-site words of the nine planes)", L);
    if (L > 98304) return fail(POTTS_ERR_UNSUPPORTED, "L = %d too large", L);
    int ndev = 0;
    CUDA_TRY8(cudaGetDeviceCount(&ndev));
    if (ndev < 1) return fail(POTTS_ERR_CUDA, "no CUDA device");
    potts8_t *h = new (std::nothrow) potts8_s;
    if (!h) return fail(POTTS_ERR_NOMEM, "host allocation failed");
    h->L = L; h->q = q; h->seed = seed; h->stream = (cudaStream_t)cuda_stream;
    cudaGetDevice(&h->device);
    cudaDeviceGetAttribute(&h->num_sms, cudaDevAttrMultiProcessorCount, h->device);
    h->plane_bytes = align_up8((size_t)(L / 3) * (L / 3));
    const size_t need = 9 * h->plane_bytes + align_up8(260 * sizeof(unsigned long long));
    const cudaError_t e = cudaMalloc(&h->ws, need);
    if (e != cudaSuccess) {
        delete h;
        return fail(e == cudaErrorMemoryAllocation ? POTTS_ERR_NOMEM : POTTS_ERR_CUDA, "cudaMalloc(%zu) failed: %s", need, cudaGetErrorString(e));
    }
    h->acc = (unsigned long long *)(h->ws + 9 * h->plane_bytes);
    h->tile_counter = (uint32_t *)(h->acc + 258);
    cudaError_t e2 = cudaMemsetAsync(h->ws, 0, need, h->stream);
    if (e2 == cudaSuccess && init == POTTS_INIT_RANDOM) {
        const long long sites = (long long)L * L;
        potts::k_init_random8_u8<<<(unsigned)((sites + 255) / 256), 256, 0, h->stream>>>(
            h->ws, h->plane_bytes, L, L / 3, (uint32_t)q, (uint32_t)(seed & 0xFFFFFFFFull), (uint32_t)(seed >> 32));
        h->launches += 1;
        e2 = cudaGetLastError();
    }
    if (e2 != cudaSuccess) {
        potts8_destroy(h);
        return fail(POTTS_ERR_CUDA, "initialisation failed: %s", cudaGetErrorString(e2));
    }
    *out = h;
    return POTTS_OK;
}

void potts8_destroy(potts8_t *h)
{
    if (!h) return;
    DeviceGuard8 g(h->device);
    cudaStreamSynchronize(h->stream);
    if (h->scratch) cudaFree(h->scratch);
    if (h->ws) cudaFree(h->ws);
    delete h;
}

int potts8_sweep(potts8_t *h, double T, int64_t nsweeps)
{
    int rc = check_args8(h, T, nsweeps);
    if (rc) return rc;
    DeviceGuard8 g(h->device);
    return run8(h, T, nsweeps, 0, nullptr, nullptr);
}

int potts8_sweep_measured(potts8_t *h, double T, int64_t nsweeps, int64_t every, int64_t *E_series, int64_t *hist_series)
{
    int rc = check_args8(h, T, nsweeps);
    if (rc) return rc;
    if (every < 1 || nsweeps % every != 0)
        return fail(POTTS_ERR_ARG, "every = %lld must be >= 1 and divide nsweeps = %lld", (long long)every, (long long)nsweeps);
    DeviceGuard8 g(h->device);
    const int64_t ns = nsweeps / every;
    if (ns == 0) return POTTS_OK;
    const size_t eb = E_series ? (size_t)ns * 8 : 0, hb = hist_series ? (size_t)ns * h->q * 8 : 0;
    uint8_t *dev = nullptr;
    if (eb + hb) {
        rc = scratch8(h, eb + hb, &dev);
        if (rc) return rc;
        CUDA_TRY8(cudaMemsetAsync(dev, 0, eb + hb, h->stream));
    }
    rc = run8(h, T, nsweeps, every, eb ? (unsigned long long *)dev : nullptr, hb ? (unsigned long long *)(dev + eb) : nullptr);
    cudaError_t e = cudaSuccess;
    if (rc == POTTS_OK && eb) e = cudaMemcpyAsync(E_series, dev, eb, cudaMemcpyDeviceToHost, h->stream);
    if (rc == POTTS_OK && e == cudaSuccess && hb) e = cudaMemcpyAsync(hist_series, dev + eb, hb, cudaMemcpyDeviceToHost, h->stream);
    const cudaError_t e2 = cudaStreamSynchronize(h->stream);
    if (rc) return rc;
    if (e != cudaSuccess || e2 != cudaSuccess) return fail(POTTS_ERR_CUDA, "series copy / sync failed: %s", cudaGetErrorString(e != cudaSuccess ? e : e2));
    return POTTS_OK;
}

int potts8_energy(potts8_t *h, int64_t *E)
{
    if (!h || !E) return fail(POTTS_ERR_ARG, "null argument");
    DeviceGuard8 g(h->device);
    CUDA_TRY8(cudaMemsetAsync(h->acc, 0, 8, h->stream));
    int rc = measure8(h, h->acc, nullptr);
    if (rc) return rc;
    int64_t v = 0;
    CUDA_TRY8(cudaMemcpyAsync(&v, h->acc, 8, cudaMemcpyDeviceToHost, h->stream));
    CUDA_TRY8(cudaStreamSynchronize(h->stream));
    *E = v;
    return POTTS_OK;
}

int potts8_histogram(potts8_t *h, int64_t *counts)
{
    if (!h || !counts) return fail(POTTS_ERR_ARG, "null argument");
    DeviceGuard8 g(h->device);
    CUDA_TRY8(cudaMemsetAsync(h->acc + 1, 0, 8 * (size_t)h->q, h->stream));
    int rc = measure8(h, nullptr, h->acc + 1);
    if (rc) return rc;
    CUDA_TRY8(cudaMemcpyAsync(counts, h->acc + 1, 8 * (size_t)h->q, cudaMemcpyDeviceToHost, h->stream));
    CUDA_TRY8(cudaStreamSynchronize(h->stream));
    return POTTS_OK;
}

int potts8_download(potts8_t *h, uint8_t *spins)
{
    if (!h || !spins) return fail(POTTS_ERR_ARG, "null argument");
    DeviceGuard8 g(h->device);
    const size_t n = (size_t)h->L * h->L;
    uint8_t *stage = nullptr;
    int rc = scratch8(h, n, &stage);
    if (rc) return rc;
    potts::k_planes_to_rowmajor8<<<(unsigned)((n + 255) / 256), 256, 0, h->stream>>>(h->ws, h->plane_bytes, stage, h->L, h->L / 3);
    rc = launched8(h, "k_planes_to_rowmajor8");
    if (rc) return rc;
    CUDA_TRY8(cudaMemcpyAsync(spins, stage, n, cudaMemcpyDeviceToHost, h->stream));
    CUDA_TRY8(cudaStreamSynchronize(h->stream));
    return POTTS_OK;
}

int potts8_upload(potts8_t *h, const uint8_t *spins)
{
    if (!h || !spins) return fail(POTTS_ERR_ARG, "null argument");
    DeviceGuard8 g(h->device);
    const size_t n = (size_t)h->L * h->L;
    if (h->q < 256)
        for (size_t k = 0; k < n; ++k)
            if (spins[k] >= h->q) return fail(POTTS_ERR_ARG, "spin value %d >= q at offset %zu", (int)spins[k], k);
    uint8_t *stage = nullptr;
    int rc = scratch8(h, n, &stage);
    if (rc) return rc;
    int *flag = (int *)(h->acc + 257);
    CUDA_TRY8(cudaMemsetAsync(flag, 0, sizeof(int), h->stream));
    CUDA_TRY8(cudaMemcpyAsync(stage, spins, n, cudaMemcpyHostToDevice, h->stream));
    potts::k_rowmajor_to_planes8<<<(unsigned)((n + 255) / 256), 256, 0, h->stream>>>(stage, h->ws, h->plane_bytes, h->L, h->L / 3, (uint32_t)h->q, flag);
    rc = launched8(h, "k_rowmajor_to_planes8");
    if (rc) return rc;
    CUDA_TRY8(cudaStreamSynchronize(h->stream));
    return POTTS_OK;
}

int potts8_sweep_count(potts8_t *h, uint64_t *t)
{
    if (!h || !t) return fail(POTTS_ERR_ARG, "null argument");
    *t = h->t;
    return POTTS_OK;
}

int potts8_set_sweep_count(potts8_t *h, uint64_t t)
{
    if (!h) return fail(POTTS_ERR_ARG, "null handle");
    if (t > 0xFFFFFFFFull) return fail(POTTS_ERR_ARG, "t must be < 2^32");
    h->t = t;
    return POTTS_OK;
}

int potts8_launch_count(potts8_t *h, uint64_t *n)
{
    if (!h || !n) return fail(POTTS_ERR_ARG, "null argument");
    *n = h->launches;
    return POTTS_OK;
}

int potts8_set_option(potts8_t *h, const char *key, int64_t value)
{
    if (!h || !key) return fail(POTTS_ERR_ARG, "null argument");
    if (!std::strcmp(key, "stream_words")) {
        if (value != 0 && value != 4 && value != -1) return fail(POTTS_ERR_ARG, "stream_words = %lld not in {-1, 0, 4}", (long long)value);
        h->opt_words = (int32_t)value;
        return POTTS_OK;
    }
    if (!std::strcmp(key, "stream_rows")) {
        if (value != 0 && value != 1 && value != 2 && value != 4 && value != 8 && value != 16) return fail(POTTS_ERR_ARG, "stream_rows = %lld not in {0, 1, 2, 4, 8, 16}", (long long)value);
        h->opt_rows = (int32_t)value;
        return POTTS_OK;
    }
    return fail(POTTS_ERR_ARG, "unknown option '%s'", key);
}

}  // extern "C"
