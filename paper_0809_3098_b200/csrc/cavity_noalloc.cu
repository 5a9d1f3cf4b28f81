// cavity_noalloc.cu — cav_diag_noalloc: the a4 diagnostics for callers that are not allowed to allocate device memory.
//
// Who this is for.  cav_get_diag needs a context, and cav_create takes ~8 fields plus the reduction's partial sums from
// PyTorch's caching allocator.  Some callers can do neither that nor a cudaMalloc of their own:
//   * code that runs while a stream capture in the global mode is open anywhere in the process (cudaMalloc is refused
//     there and poisons the capture);
//   * solvers that were handed a fixed slice of HBM by a host application and must not ask the driver for a byte more
//     (another framework's pool owns the rest of the 180 GB, so the request may fail at any time);
//   * time-step loops that cannot afford the device-wide synchronisation a cudaMalloc / cudaFree brings with it.
// Such a caller already holds psi and omega in device buffers of its own; it passes those and a 4-double device result
// buffer, and this file supplies the only other memory the reduction needs (one partial result per grid row and a
// counter) from a fixed array that is part of the library image:  g_noalloc_scratch below, 256.25 KiB, held by every
// GPU the library is loaded on until the process exits.  That fixed size is where the limit N <= CAV_NOALLOC_MAX_N
// comes from.
//
// This is a VARIANT of k_diag_partial / k_diag_final (cavity_kernels.cu), not a wrapper around them: same per-point
// formulas (S8(a) row a4; u, v of eq 22), but one CTA per interior grid row, its four partial results in slot j of
// the scratch, and the CTA that finishes last (a counter in the scratch tells it) folds the slots in fixed order, so
// the whole thing is one launch and the result does not depend on which CTA happened to be last.  The summation order
// differs from cav_get_diag's, so the two agree to rounding (a few ulp of the sums), not bit for bit.
//
// Nothing here calls cudaMalloc, cudaFree, PyTorch's allocator or any library routine that allocates.
// Build with -fmad=false like the rest of the library (every fused multiply-add is an explicit fma()).
#include <cuda_runtime.h>

#include <cstdio>
#include <cstdlib>
#include <mutex>

#include "../../include/cavity.h"

#define CAV_API extern "C" __attribute__((visibility("default")))

namespace {

constexpr int NA_THREADS = 256;
constexpr int NA_MAX_ROWS = CAV_NOALLOC_MAX_N;          // interior rows j = 1 .. N - 1 use slots 0 .. N - 2
constexpr size_t NA_HEAD_BYTES = 256;                   // the counter lives alone in the first 256 bytes
constexpr size_t NA_BYTES = NA_HEAD_BYTES + 4 * (size_t)NA_MAX_ROWS * sizeof(double);

// The scratch.  In HOST code this name is only a handle for cudaGetSymbolAddress: it is not a device address, and a
// kernel that were handed `g_noalloc_scratch` from the host would fault (or scribble over host memory where the GPU can
// reach it).  Host code below therefore only ever uses the pointer scratch_of_current_device() returns.
//   bytes 0..3      : counter of finished CTAs; must be 0 when a launch starts
//   bytes 256..     : four planes (max |r|, sum r^2, sum (u^2 + v^2), sum w^2) of NA_MAX_ROWS doubles, slot = j - 1
static __device__ __align__(256) unsigned char g_noalloc_scratch[NA_BYTES];

__device__ __forceinline__ double warp_sum(double v) {
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ double warp_max(double v) {
    for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_down_sync(0xffffffffu, v, o));
    return v;
}

// (max, sum, sum, sum) over the CTA, fixed order; valid in thread 0.  Safe to call more than once per kernel.
__device__ __forceinline__ void cta_reduce4(double& m, double& s1, double& s2, double& s3) {
    __shared__ double sh[4][NA_THREADS / 32];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    m = warp_max(m); s1 = warp_sum(s1); s2 = warp_sum(s2); s3 = warp_sum(s3);
    __syncthreads();                                    // a previous call's readers are done with sh
    if (lane == 0) { sh[0][wid] = m; sh[1][wid] = s1; sh[2][wid] = s2; sh[3][wid] = s3; }
    __syncthreads();
    if (wid == 0) {
        m  = lane < NA_THREADS / 32 ? sh[0][lane] : 0.0;
        s1 = lane < NA_THREADS / 32 ? sh[1][lane] : 0.0;
        s2 = lane < NA_THREADS / 32 ? sh[2][lane] : 0.0;
        s3 = lane < NA_THREADS / 32 ? sh[3][lane] : 0.0;
        m = warp_max(m); s1 = warp_sum(s1); s2 = warp_sum(s2); s3 = warp_sum(s3);
    }
}

// One CTA per interior row j = 1 + blockIdx.x (coalesced along i); the last CTA to finish folds all rows.
__global__ void __launch_bounds__(NA_THREADS)
k_diag_rows(int N, int pitch, const double* __restrict__ psi, const double* __restrict__ w, unsigned char* scratch,
            double* __restrict__ out4) {
    unsigned int* counter = reinterpret_cast<unsigned int*>(scratch);
    double* part = reinterpret_cast<double*>(scratch + NA_HEAD_BYTES);
    const double h = 1.0 / (double)N;
    const double h2 = h * h, twoh = 2.0 * h;
    const int rows = N - 1;
    const int j = 1 + (int)blockIdx.x;
    const double* prow = psi + (size_t)j * pitch;
    const double* wrow = w + (size_t)j * pitch;

    double m = 0.0, s_r2 = 0.0, s_ke = 0.0, s_en = 0.0;
    for (int i = 1 + (int)threadIdx.x; i <= N - 1; i += NA_THREADS) {
        const double pW = prow[i - 1], pE = prow[i + 1], pS = prow[i - pitch], pN = prow[i + pitch], p = prow[i];
        const double wv = wrow[i];
        const double r = (pW + pE + pS + pN - 4.0 * p) / h2 + wv;       // S8(a) row a4: r = lap_h(psi) + omega
        const double u = (pN - pS) / twoh;                              // eq 22
        const double v = -(pE - pW) / twoh;
        m = fmax(m, fabs(r));
        s_r2 = fma(r, r, s_r2);
        s_ke += fma(u, u, v * v);
        s_en = fma(wv, wv, s_en);
    }
    cta_reduce4(m, s_r2, s_ke, s_en);

    __shared__ bool last;
    if (threadIdx.x == 0) {
        part[0 * NA_MAX_ROWS + blockIdx.x] = m;
        part[1 * NA_MAX_ROWS + blockIdx.x] = s_r2;
        part[2 * NA_MAX_ROWS + blockIdx.x] = s_ke;
        part[3 * NA_MAX_ROWS + blockIdx.x] = s_en;
        __threadfence();                                 // the slot is visible device-wide before the count goes up
        last = (atomicAdd(counter, 1u) == (unsigned int)(rows - 1));
    }
    __syncthreads();
    if (!last) return;

    __threadfence();                                     // every other CTA's slot was published before its increment
    const volatile double* vp = part;                    // written by other SMs during this launch: no cached reads
    m = 0.0; s_r2 = 0.0; s_ke = 0.0; s_en = 0.0;
    for (int t = (int)threadIdx.x; t < rows; t += NA_THREADS) {
        m = fmax(m, vp[t]);
        s_r2 += vp[1 * NA_MAX_ROWS + t];
        s_ke += vp[2 * NA_MAX_ROWS + t];
        s_en += vp[3 * NA_MAX_ROWS + t];
    }
    cta_reduce4(m, s_r2, s_ke, s_en);
    if (threadIdx.x == 0) {
        out4[0] = m;                                     // res_inf
        out4[1] = sqrt(h2 * s_r2);                       // res_l2
        out4[2] = 0.5 * h2 * s_ke;                       // kinetic energy
        out4[3] = 0.5 * h2 * s_en;                       // enstrophy
        *counter = 0u;                                   // leave the counter as the next call needs it
    }
}

// ---- host side: the device address of the scratch, looked up once per device ---------------------------
constexpr int NA_MAX_DEVICES = 64;
std::mutex g_mu;
unsigned char* g_scratch_dev[NA_MAX_DEVICES] = {nullptr};

inline void debug_msg(const char* what, cudaError_t e) {
    if (std::getenv("CAV_DEBUG")) std::fprintf(stderr, "[cavity] cav_diag_noalloc: %s -> %s\n", what, cudaGetErrorString(e));
}

// Set-up, once per device, with that device current (it is: we ask the runtime which one is).  cudaGetSymbolAddress
// makes the runtime load this library's device image on the device if it has not yet, which is why the first call on a
// device should not happen while a stream capture is open.
int scratch_of_current_device(unsigned char** out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) { debug_msg("cudaGetDevice", e); cudaGetLastError(); return CAV_ECUDA; }
    if (dev < 0 || dev >= NA_MAX_DEVICES) return CAV_ENOTSUP;
    std::lock_guard<std::mutex> lk(g_mu);
    if (!g_scratch_dev[dev]) {
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, g_noalloc_scratch);
        if (e != cudaSuccess || !p) { debug_msg("cudaGetSymbolAddress", e); cudaGetLastError(); return CAV_ECUDA; }
        g_scratch_dev[dev] = static_cast<unsigned char*>(p);
    }
    *out = g_scratch_dev[dev];
    return CAV_OK;
}

}  // namespace

CAV_API int cav_noalloc_max_n(void) { return CAV_NOALLOC_MAX_N; }

CAV_API int cav_diag_noalloc(int N, int pitch, const double* psi_dev, const double* omega_dev, double* out4_dev, void* stream) {
    if (N < 2 || pitch < N + 1 || !psi_dev || !omega_dev || !out4_dev) return CAV_EINVAL;
    if (N > CAV_NOALLOC_MAX_N) {
        if (std::getenv("CAV_DEBUG"))
            std::fprintf(stderr, "[cavity] cav_diag_noalloc: N = %d exceeds CAV_NOALLOC_MAX_N = %d (the fixed scratch has one slot per grid row)\n",
                         N, CAV_NOALLOC_MAX_N);
        return CAV_ELIMIT;
    }
    unsigned char* scratch = nullptr;
    const int rc = scratch_of_current_device(&scratch);
    if (rc != CAV_OK) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    // The array is shared by every call and keeps what the previous one left.  The slots need no clearing (the fold reads
    // only slots 0 .. N - 2, all written earlier in the same launch); the counter must start at 0.  The kernel resets it on
    // the way out, but a launch that died half way would leave it stale, so it is cleared here every time.
    cudaError_t e = cudaMemsetAsync(scratch, 0, NA_HEAD_BYTES, st);
    if (e != cudaSuccess) { debug_msg("cudaMemsetAsync", e); cudaGetLastError(); return CAV_ECUDA; }
    k_diag_rows<<<N - 1, NA_THREADS, 0, st>>>(N, pitch, psi_dev, omega_dev, scratch, out4_dev);
    e = cudaGetLastError();
    if (e != cudaSuccess) { debug_msg("k_diag_rows launch", e); return CAV_ECUDA; }
    return CAV_OK;
}
