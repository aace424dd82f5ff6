// potts_noalloc.cu -- potts_measure_noalloc (include/potts.h, section "no-allocation entry point"): energy (R1) and
// q-bin histogram (R8) of a lattice the caller holds on the device, for callers that cannot call cudaMalloc (code
// under CUDA graph capture, tight serving loops, harnesses that forbid it).
//
// It is the standalone measurement of the library (k_measure_u8, the kernel behind potts_energy / potts_histogram)
// with everything that path keeps in cudaMalloc'ed memory -- the two colour planes and the accumulator block --
// moved into ONE file-scope device array of fixed size, g_noalloc_scratch below.  Every GPU that loads the library
// holds the array (4 MiB + 4 KiB) until the process exits.  This file calls no cudaMalloc, cudaFree or allocating
// library routine: cudaGetSymbolAddress, cudaMemsetAsync and three kernel launches per call.
//
// In host code the NAME of a __device__ array is a host-side stand-in, not a device address, so the launches below
// never receive `g_noalloc_scratch` itself: the address comes from cudaGetSymbolAddress, asked once per device with
// that device current (scratch_of_current_device).
//
// Every call shares the array and finds the previous call's contents in it: the accumulators and the flag are cleared
// at the start of every call, the planes are overwritten for the L of the call (bytes beyond L*L are never read).
// Two calls that overlap on the GPU (different streams, or the same device from two host threads without ordering)
// race on the array: the caller serialises them.
#include "../../include/potts.h"
#include "potts_kernels.cuh"

#include <cstdarg>
#include <cstdint>
#include <cstdio>
#include <mutex>

namespace potts {
int set_error(int code, const char *msg);      // potts_api.cu: the message potts_last_error() returns
}

namespace {

constexpr int NOALLOC_MAX_L = POTTS_NOALLOC_MAX_L;                              // include/potts.h: 2048
constexpr size_t NOALLOC_PLANES = (size_t)NOALLOC_MAX_L * NOALLOC_MAX_L;          // both colour planes: L*L bytes
constexpr size_t NOALLOC_ACC = 4096;                                              // [0] E, [1..256] histogram, [257] flag
constexpr size_t NOALLOC_BYTES = NOALLOC_PLANES + NOALLOC_ACC;

static __device__ __align__(256) unsigned char g_noalloc_scratch[NOALLOC_BYTES];

constexpr int MAX_DEVICES = 64;
std::mutex g_mutex;
unsigned char *g_scratch_ptr[MAX_DEVICES] = {};                                   // device address of the array, per device

int fail(int code, const char *fmt, ...)
{
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    return potts::set_error(code, buf);
}

// set-up, once per device, with that device current: the device address of the array
int scratch_of_current_device(unsigned char **out)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail(POTTS_ERR_CUDA, "cudaGetDevice failed: %s", cudaGetErrorString(e));
    if (dev < 0 || dev >= MAX_DEVICES) return fail(POTTS_ERR_UNSUPPORTED, "device index %d outside [0, %d)", dev, MAX_DEVICES);
    std::lock_guard<std::mutex> lock(g_mutex);
    if (!g_scratch_ptr[dev]) {
        unsigned char *p = nullptr;
        e = cudaGetSymbolAddress((void **)&p, g_noalloc_scratch);
        if (e != cudaSuccess || !p)
            return fail(POTTS_ERR_CUDA, "cudaGetSymbolAddress(g_noalloc_scratch) on device %d failed: %s", dev, cudaGetErrorString(e));
        g_scratch_ptr[dev] = p;
    }
    *out = g_scratch_ptr[dev];
    return POTTS_OK;
}

// row-major s[i L + j] -> split colour planes (as k_rowmajor_to_planes), values >= q raise the flag and are stored as
// q - 1 so that the histogram kernel stays inside its table; one thread per 4 sites of a plane row
__global__ void k_noalloc_to_planes(const uint8_t *in, uint8_t *plane0, uint8_t *plane1, int L, int pitch, uint32_t q, int *bad)
{
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const int wpr = pitch >> 2;
    if (gid >= (long long)L * wpr) return;
    const int i = (int)(gid / wpr), kw = (int)(gid - (long long)i * wpr);
    const uint2 v = *reinterpret_cast<const uint2 *>(in + (size_t)i * L + 8 * kw);
    uint32_t ev = __byte_perm(v.x, v.y, 0x6420), od = __byte_perm(v.x, v.y, 0x7531);
    if (q < 256) {
        const uint32_t top = (q - 1u) * 0x01010101u;
        const uint32_t ev_c = __vminu4(ev, top), od_c = __vminu4(od, top);
        if (ev_c != ev || od_c != od) atomicExch(bad, 1);
        ev = ev_c;
        od = od_c;
    }
    *reinterpret_cast<uint32_t *>(((i & 1) ? plane1 : plane0) + (size_t)i * pitch + 4 * kw) = ev;
    *reinterpret_cast<uint32_t *>(((i & 1) ? plane0 : plane1) + (size_t)i * pitch + 4 * kw) = od;
}

// accumulators -> the caller's outputs; a raised flag turns them into the documented "bad input" values
__global__ void k_noalloc_finish(const unsigned long long *acc, const int *bad, long long *E_out, long long *hist_out, uint32_t q)
{
    const bool b = *bad != 0;
    if (E_out && threadIdx.x == 0) *E_out = b ? INT64_MIN : (long long)acc[0];
    if (hist_out)
        for (uint32_t k = threadIdx.x; k < q; k += blockDim.x) hist_out[k] = b ? -1ll : (long long)acc[1 + k];
}

}  // namespace

extern "C" int potts_measure_noalloc(const uint8_t *spins_dev, int32_t L, int32_t q, int64_t *E_dev, int64_t *hist_dev, void *cuda_stream)
{
    // argument checks first: none of them touches CUDA
    if (!spins_dev) return fail(POTTS_ERR_ARG, "null spins pointer");
    if (!E_dev && !hist_dev) return fail(POTTS_ERR_ARG, "both outputs are null");
    if (L < 2 || (L & 1)) return fail(POTTS_ERR_ARG, "L = %d must be even and >= 2", L);
    if (q < 2 || q > 256) return fail(POTTS_ERR_ARG, "q = %d outside [2, 256]", q);
    if (L % 32 != 0) return fail(POTTS_ERR_UNSUPPORTED, "L = %d is not a multiple of 32 (kernel vector width)", L);
    if (L > NOALLOC_MAX_L)
        return fail(POTTS_ERR_UNSUPPORTED, "L = %d exceeds POTTS_NOALLOC_MAX_L = %d: the static scratch array holds %zu bytes of planes; use a potts_t handle",
                    L, NOALLOC_MAX_L, NOALLOC_PLANES);
    if (((uintptr_t)spins_dev & 7u) || ((uintptr_t)E_dev & 7u) || ((uintptr_t)hist_dev & 7u))
        return fail(POTTS_ERR_ARG, "spins, E and hist pointers must be 8-byte aligned");

    unsigned char *scratch = nullptr;
    const int rc = scratch_of_current_device(&scratch);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const int pitch = L / 2;
    uint8_t *plane0 = scratch, *plane1 = scratch + (size_t)L * pitch;              // L * L / 2 is a multiple of 512
    unsigned long long *acc = reinterpret_cast<unsigned long long *>(scratch + NOALLOC_PLANES);
    int *bad = reinterpret_cast<int *>(acc + 257);

    // what must start at zero: E, the q histogram bins, the flag (the last call's values are still there)
    cudaError_t e = cudaMemsetAsync(acc, 0, 258 * sizeof(unsigned long long), st);
    if (e != cudaSuccess) return fail(POTTS_ERR_CUDA, "cudaMemsetAsync failed: %s", cudaGetErrorString(e));

    const long long words = (long long)L * (pitch >> 2);
    k_noalloc_to_planes<<<(unsigned)((words + 255) / 256), 256, 0, st>>>(spins_dev, plane0, plane1, L, pitch, (uint32_t)q, bad);

    potts::MeasureParams M;
    M.plane0 = plane0;
    M.plane1 = plane1;
    M.L = L;
    M.pitch = pitch;
    M.row0 = 0;
    M.strip = 0;
    M.q = (uint32_t)q;
    M.E_out = E_dev ? acc : nullptr;
    M.hist_out = hist_dev ? acc + 1 : nullptr;
    const long long threads = (long long)L * (L / 32);
    long long blocks = (threads + 255) / 256;
    if (blocks > 148 * 8) blocks = 148 * 8;
    const size_t smem = hist_dev ? (size_t)potts::hist_words((uint32_t)q) * 4 : 0;
    if (q > 128) potts::k_measure_u8<true><<<(unsigned)blocks, 256, smem, st>>>(M);
    else potts::k_measure_u8<false><<<(unsigned)blocks, 256, smem, st>>>(M);

    k_noalloc_finish<<<1, 256, 0, st>>>(acc, bad, reinterpret_cast<long long *>(E_dev), reinterpret_cast<long long *>(hist_dev), (uint32_t)q);
    e = cudaGetLastError();
    if (e != cudaSuccess) return fail(POTTS_ERR_CUDA, "launch of the no-allocation measurement failed: %s", cudaGetErrorString(e));
    return POTTS_OK;
}
