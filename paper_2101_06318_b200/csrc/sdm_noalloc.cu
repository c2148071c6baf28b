// sdm_noalloc.cu -- sdm_moments_noalloc: the moments of row a8 for callers that cannot allocate device memory.
//
// Who this is for.  Every other entry point of libsdm works on a handle whose workspace the caller obtained from
// cudaMalloc (or a framework allocator that calls it).  Some callers have no such option at the moment they want a
// diagnostic number: a host model that handed the whole device to its own memory pool at start-up and has nothing
// left to hand out; a monitoring hook running on a thread that must not block, where cudaMalloc / cudaFree would
// synchronise the whole device; a plug-in loaded into a process whose device-memory budget is fixed and fully
// spoken for.  They own (xi, v) already and have 24 bytes for the results, but nowhere to put the per-CTA partial
// sums and the arrival counter the grid-wide reduction needs.  Here that scratch is part of the library image:
// a file-scope `static __device__` array of SDM_NOALLOC_SCRATCH_BYTES (28 KiB), present on every GPU that loads
// libsdm, from the moment the module is loaded until the process exits.
//
// What follows from sharing one array.  Every call on a device uses the same bytes.  Two calls that may execute
// at the same time on that device (different streams, different host threads) race on them and return garbage;
// calls in one stream, or otherwise ordered on the GPU, are fine.  The array keeps what the previous call left:
// the arrival counter is cleared on the stream before every launch, and every partial a launch reads was written
// by that same launch, so stale contents are never read.
//
// Set-up.  In host code `g_noalloc_scratch` is only a stand-in for the device array, not an address a kernel can
// use.  The first call on a device asks the runtime for the real address (cudaGetSymbolAddress, with that device
// current) and keeps it per device ordinal.  Make that first call before any stream capture begins.
//
// This file shares no code path with the handle-based API: nothing in sdm_api.cu calls it or is called by it.
// Moments: M_k = sum xi * v^k, k = 0, 1, 2 (R13), products rounded as (xi*v) and (xi*v)*v.
#include <cuda_runtime.h>

#include <cstdint>
#include <cstdio>
#include <mutex>

#include "../../include/sdm.h"

namespace {

constexpr int kThreads = 256;
constexpr int kMaxCtas = 1184;                         // 148 SMs x 8 resident CTAs of 256 threads
constexpr int kCounterBytes = 256;                     // the arrival counter has the first 256 bytes to itself
constexpr size_t kScratchBytes = kCounterBytes + 3 * sizeof(double) * (size_t)kMaxCtas;
static_assert(kScratchBytes == SDM_NOALLOC_SCRATCH_BYTES, "sdm.h states the size of the static scratch");
constexpr int kMaxDevices = 64;

// [0, 256): unsigned arrival counter; then kMaxCtas int64 partials of M0, kMaxCtas doubles of M1, of M2
static __device__ __align__(256) unsigned char g_noalloc_scratch[kScratchBytes];

struct Scratch {
    unsigned int *done;
    long long *part0;
    double *part1;
    double *part2;
};

__host__ __device__ inline Scratch carve(unsigned char *base)
{
    Scratch s;
    s.done = reinterpret_cast<unsigned int *>(base);
    s.part0 = reinterpret_cast<long long *>(base + kCounterBytes);
    s.part1 = reinterpret_cast<double *>(base + kCounterBytes + sizeof(double) * (size_t)kMaxCtas);
    s.part2 = reinterpret_cast<double *>(base + kCounterBytes + 2 * sizeof(double) * (size_t)kMaxCtas);
    return s;
}

// Sum over the CTA of one (M0, M1, M2) triple per thread; the result is valid in thread 0.
__device__ __forceinline__ void cta_sum(long long &a0, double &a1, double &a2)
{
    __shared__ long long s0[kThreads / 32];
    __shared__ double s1[kThreads / 32], s2[kThreads / 32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) {
        a0 += __shfl_down_sync(0xffffffffu, a0, d);
        a1 = __dadd_rn(a1, __shfl_down_sync(0xffffffffu, a1, d));
        a2 = __dadd_rn(a2, __shfl_down_sync(0xffffffffu, a2, d));
    }
    __syncthreads();                                   // the arrays may still be read from a previous call
    if (lane == 0) { s0[warp] = a0; s1[warp] = a1; s2[warp] = a2; }
    __syncthreads();
    if (threadIdx.x == 0) {
        a0 = 0; a1 = 0.0; a2 = 0.0;
        for (int w = 0; w < kThreads / 32; ++w) {
            a0 += s0[w];
            a1 = __dadd_rn(a1, s1[w]);
            a2 = __dadd_rn(a2, s2[w]);
        }
    }
}

// Grid-stride pass over (xi, v), two droplets per thread and iteration (16-byte loads), one partial triple per
// CTA into the scratch; the CTA that arrives last adds the partials in index order and writes the results.
__global__ void __launch_bounds__(kThreads)
k_moments_noalloc(const long long *__restrict__ xi, const double *__restrict__ v, int n, unsigned char *scratch,
                  long long *__restrict__ m0, double *__restrict__ m1, double *__restrict__ m2)
{
    const Scratch sc = carve(scratch);
    long long a0 = 0;
    double a1 = 0.0, a2 = 0.0;
    const int n2 = n >> 1;
    const longlong2 *xi2 = reinterpret_cast<const longlong2 *>(xi);
    const double2 *v2 = reinterpret_cast<const double2 *>(v);
    for (int t = blockIdx.x * kThreads + threadIdx.x; t < n2; t += gridDim.x * kThreads) {
        const longlong2 x = __ldcs(xi2 + t);
        const double2 vol = __ldcs(v2 + t);
        const double xv0 = __dmul_rn(__ll2double_rn(x.x), vol.x), xv1 = __dmul_rn(__ll2double_rn(x.y), vol.y);
        a0 += x.x + x.y;
        a1 = __dadd_rn(a1, __dadd_rn(xv0, xv1));
        a2 = __dadd_rn(a2, __dadd_rn(__dmul_rn(xv0, vol.x), __dmul_rn(xv1, vol.y)));
    }
    if ((n & 1) && blockIdx.x == 0 && threadIdx.x == 0) {   // odd count: the last droplet
        const long long x = xi[n - 1];
        const double vol = v[n - 1];
        const double xv = __dmul_rn(__ll2double_rn(x), vol);
        a0 += x;
        a1 = __dadd_rn(a1, xv);
        a2 = __dadd_rn(a2, __dmul_rn(xv, vol));
    }
    cta_sum(a0, a1, a2);

    __shared__ bool s_last;
    if (threadIdx.x == 0) {
        sc.part0[blockIdx.x] = a0; sc.part1[blockIdx.x] = a1; sc.part2[blockIdx.x] = a2;
        __threadfence();                               // the partials are visible before the arrival is
        s_last = atomicAdd(sc.done, 1u) == gridDim.x - 1;
    }
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    a0 = 0; a1 = 0.0; a2 = 0.0;
    for (int b = threadIdx.x; b < (int)gridDim.x; b += kThreads) {   // only partials of THIS launch: b < gridDim.x
        a0 += ((volatile long long *)sc.part0)[b];
        a1 = __dadd_rn(a1, ((volatile double *)sc.part1)[b]);
        a2 = __dadd_rn(a2, ((volatile double *)sc.part2)[b]);
    }
    cta_sum(a0, a1, a2);
    if (threadIdx.x == 0) {
        *m0 = a0; *m1 = a1; *m2 = a2;
        *sc.done = 0;                                  // left clean for the next call (which clears it again anyway)
    }
}

// Device address of g_noalloc_scratch on each device ordinal, filled by the first call made with that device current.
std::mutex g_setup_mutex;
unsigned char *g_scratch_addr[kMaxDevices];

int fail(char *err_host, size_t err_len, int code, const char *what, const char *detail = nullptr)
{
    if (err_host && err_len > 0) {
        if (detail) std::snprintf(err_host, err_len, "sdm_moments_noalloc: %s: %s", what, detail);
        else std::snprintf(err_host, err_len, "sdm_moments_noalloc: %s", what);
    }
    return code;
}

}  // namespace

extern "C" int sdm_moments_noalloc(const int64_t *xi_dev, const double *v_dev, int64_t n_sd, int64_t *m0_dev,
                                   double *m1_dev, double *m2_dev, void *cuda_stream, char *err_host, size_t err_len)
{
    if (err_host && err_len > 0) err_host[0] = '\0';
    if (n_sd < 0) return fail(err_host, err_len, SDM_EINVAL, "n_sd is negative");
    if (n_sd > (int64_t)SDM_NOALLOC_MAX_SD) {
        char msg[160];
        std::snprintf(msg, sizeof msg, "n_sd = %lld exceeds SDM_NOALLOC_MAX_SD = %lld (32-bit storage indices)",
                      (long long)n_sd, (long long)SDM_NOALLOC_MAX_SD);
        return fail(err_host, err_len, SDM_ECAPACITY, msg);
    }
    if (!m0_dev || !m1_dev || !m2_dev) return fail(err_host, err_len, SDM_EINVAL, "a result pointer is NULL");
    if (n_sd > 0 && (!xi_dev || !v_dev)) return fail(err_host, err_len, SDM_EINVAL, "xi_dev or v_dev is NULL");
    if (((uintptr_t)xi_dev | (uintptr_t)v_dev) & 15)
        return fail(err_host, err_len, SDM_EINVAL, "xi_dev and v_dev must be 16-byte aligned");

    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail(err_host, err_len, SDM_ECUDA, "cudaGetDevice", cudaGetErrorString(e));
    if (dev < 0 || dev >= kMaxDevices) return fail(err_host, err_len, SDM_ECUDA, "device ordinal beyond 63");
    unsigned char *scratch = nullptr;
    {
        // once per device, with that device current: the host-side name g_noalloc_scratch -> its device address
        std::lock_guard<std::mutex> lock(g_setup_mutex);
        if (!g_scratch_addr[dev]) {
            void *p = nullptr;
            e = cudaGetSymbolAddress(&p, g_noalloc_scratch);
            if (e != cudaSuccess || !p)
                return fail(err_host, err_len, SDM_ECUDA, "cudaGetSymbolAddress(static scratch)", cudaGetErrorString(e));
            g_scratch_addr[dev] = static_cast<unsigned char *>(p);
        }
        scratch = g_scratch_addr[dev];
    }

    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    // the arrival counter must start at zero whatever an earlier (possibly failed) launch left behind
    e = cudaMemsetAsync(scratch, 0, kCounterBytes, stream);
    if (e != cudaSuccess) return fail(err_host, err_len, SDM_ECUDA, "clear of the arrival counter", cudaGetErrorString(e));
    int64_t ctas = (n_sd / 2 + (int64_t)kThreads * 4 - 1) / ((int64_t)kThreads * 4);   // >= 4 pairs per thread
    ctas = ctas < 1 ? 1 : (ctas > kMaxCtas ? kMaxCtas : ctas);
    k_moments_noalloc<<<(unsigned)ctas, kThreads, 0, stream>>>(reinterpret_cast<const long long *>(xi_dev), v_dev,
                                                               (int)n_sd, scratch,
                                                               reinterpret_cast<long long *>(m0_dev), m1_dev, m2_dev);
    e = cudaGetLastError();
    if (e != cudaSuccess) return fail(err_host, err_len, SDM_ECUDA, "launch k_moments_noalloc", cudaGetErrorString(e));
    return SDM_OK;
}
