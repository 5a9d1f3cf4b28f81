// cavity_kernels.cu — support kernels (a2, a3, a4) and the streaming sweep engine (a1) for sm_100a.
//
// Build with -fmad=false: every fused multiply-add below is an explicit fma(), so the expression
// association is exactly the one DESIGN.md "Canonical arithmetic" states (and tests compare bit for bit).
// P:n = /root/reference/PAPER.md line n.
#include "cavity_kernels.cuh"
#include "cavity_scheme.cuh"

namespace cavk {

namespace {

using namespace scheme;       // the SSPRK(5,4) table, Thom's formula, eq 8 / 22 and the stage combination: cavity_scheme.cuh

inline int cdiv(int a, int b) { return (a + b - 1) / b; }

inline int launched(int n) {
    cudaError_t e = cudaGetLastError();
    return e == cudaSuccess ? n : -(int)e;
}

// ---- q = cq * w --------------------------------------------------------------------------------------
__global__ void k_scale_rhs(int N, int pitch, double cq, const double* __restrict__ w, double* __restrict__ q) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    if (i > N || j > N) return;
    const size_t k = (size_t)j * pitch + i;
    const bool interior = (i >= 1) & (i <= N - 1) & (j >= 1) & (j <= N - 1);
    q[k] = interior ? cq * w[k] : 0.0;
}

// ---- a2: Thom ring, eq 25 P:161-169 ------------------------------------------------------------------
__global__ void k_thom_ring(int N, int pitch, double c2h2, double lid, const double* __restrict__ psi,
                            double* __restrict__ w) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t <= N) {                                    // bottom and top rows own the corners (G10)
        w[t] = thom_wall(c2h2, psi[(size_t)pitch + t]);
        w[(size_t)N * pitch + t] = thom_lid(c2h2, lid, psi[(size_t)(N - 1) * pitch + t]);
    }
    if (t >= 1 && t <= N - 1) {                      // side walls, j = 1..N-1
        w[(size_t)t * pitch] = thom_wall(c2h2, psi[(size_t)t * pitch + 1]);
        w[(size_t)t * pitch + N] = thom_wall(c2h2, psi[(size_t)t * pitch + N - 1]);
    }
}

__global__ void k_zero_ring(int N, int pitch, double* __restrict__ psi) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t <= N) {
        psi[t] = 0.0;
        psi[(size_t)N * pitch + t] = 0.0;
        psi[(size_t)t * pitch] = 0.0;
        psi[(size_t)t * pitch + N] = 0.0;
    }
}

// ---- a2 + a3: transport right-hand side and the stage combination ------------------------------------
template <int K>
__global__ void __launch_bounds__(256)
k_rk_stage(Params P, const double* __restrict__ psi, const double* __restrict__ w_in, const double* __restrict__ a,
           const double* __restrict__ b, double* __restrict__ w_out, double* __restrict__ t_out) {
    const int N = P.N, pitch = P.pitch;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    if (i > N || j > N) return;
    const size_t k = (size_t)j * pitch + i;

    if (j == 0) { w_out[k] = thom_wall(P.c2h2, psi[k + pitch]); return; }
    if (j == N) { w_out[k] = thom_lid(P.c2h2, P.lid, psi[k - pitch]); return; }
    if (i == 0) { w_out[k] = thom_wall(P.c2h2, psi[k + 1]); return; }
    if (i == N) { w_out[k] = thom_wall(P.c2h2, psi[k - 1]); return; }

    const double pW = psi[k - 1], pE = psi[k + 1], pS = psi[k - pitch], pN = psi[k + pitch];
    const double w0 = w_in[k];
    double wW, wE, wS, wN;
    if (i == 1 || i == N - 1 || j == 1 || j == N - 1) {
        // the wall value next to this point is Thom's formula applied to this point's own psi
        const double p0 = psi[k];
        wW = (i == 1) ? thom_wall(P.c2h2, p0) : w_in[k - 1];
        wE = (i == N - 1) ? thom_wall(P.c2h2, p0) : w_in[k + 1];
        wS = (j == 1) ? thom_wall(P.c2h2, p0) : w_in[k - pitch];
        wN = (j == N - 1) ? thom_lid(P.c2h2, P.lid, p0) : w_in[k + pitch];
    } else {
        wW = w_in[k - 1]; wE = w_in[k + 1]; wS = w_in[k - pitch]; wN = w_in[k + pitch];
    }
    const double dL = transport_dL(pW, pE, pS, pN, w0, wW, wE, wS, wN, P.i2h, P.ih2, P.nu, P.dt);   // eq 22, eq 8
    // eq 9-13: w0 is the stage input; a = omega^n (stages 2-4) or T (stage 5); b = omega^(2) (stage 4)
    w_out[k] = rk_stage_out(K, rk_c(K), rk_a1(K), rk_a0(K), dL, w0, K == 1 ? 0.0 : a[k]);
    if (K == 4) t_out[k] = rk_T(dL, w0, b[k]);                                       // eq 13, first three terms
}

// ---- a4: diagnostics ----------------------------------------------------------------------------------
constexpr int DIAG_BLOCKS = 296;
constexpr int DIAG_THREADS = 256;

__device__ __forceinline__ double warp_sum(double v) {
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ double warp_max(double v) {
    for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_down_sync(0xffffffffu, v, o));
    return v;
}

// block-level reduction of (max, sum, sum, sum); result valid in thread 0
__device__ __forceinline__ void block_reduce4(double& m, double& s1, double& s2, double& s3) {
    __shared__ double sh[4][DIAG_THREADS / 32];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    m = warp_max(m); s1 = warp_sum(s1); s2 = warp_sum(s2); s3 = warp_sum(s3);
    if (lane == 0) { sh[0][wid] = m; sh[1][wid] = s1; sh[2][wid] = s2; sh[3][wid] = s3; }
    __syncthreads();
    if (wid == 0) {
        const int nw = blockDim.x >> 5;
        m = lane < nw ? sh[0][lane] : 0.0;
        s1 = lane < nw ? sh[1][lane] : 0.0;
        s2 = lane < nw ? sh[2][lane] : 0.0;
        s3 = lane < nw ? sh[3][lane] : 0.0;
        m = warp_max(m); s1 = warp_sum(s1); s2 = warp_sum(s2); s3 = warp_sum(s3);
    }
}

__global__ void __launch_bounds__(DIAG_THREADS)
k_diag_partial(int N, int pitch, const double* __restrict__ psi, const double* __restrict__ w,
               double* __restrict__ scratch) {
    const double h = 1.0 / (double)N;
    const double h2 = h * h, twoh = 2.0 * h;
    const long long M = (long long)(N - 1) * (N - 1);
    double m = 0.0, s_r2 = 0.0, s_ke = 0.0, s_en = 0.0;
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < M; t += (long long)gridDim.x * blockDim.x) {
        const int j = 1 + (int)(t / (N - 1)), i = 1 + (int)(t % (N - 1));
        const size_t k = (size_t)j * pitch + i;
        const double pW = psi[k - 1], pE = psi[k + 1], pS = psi[k - pitch], pN = psi[k + pitch], p = psi[k];
        const double wv = w[k];
        const double r = (pW + pE + pS + pN - 4.0 * p) / h2 + wv;       // S8(a) row a4
        const double u = (pN - pS) / twoh;
        const double v = -(pE - pW) / twoh;
        m = fmax(m, fabs(r));
        s_r2 = fma(r, r, s_r2);
        s_ke += fma(u, u, v * v);
        s_en = fma(wv, wv, s_en);
    }
    block_reduce4(m, s_r2, s_ke, s_en);
    if (threadIdx.x == 0) {
        scratch[0 * DIAG_BLOCKS + blockIdx.x] = m;
        scratch[1 * DIAG_BLOCKS + blockIdx.x] = s_r2;
        scratch[2 * DIAG_BLOCKS + blockIdx.x] = s_ke;
        scratch[3 * DIAG_BLOCKS + blockIdx.x] = s_en;
    }
}

// second stage: one block, fixed order (deterministic; no floating-point atomics anywhere)
__global__ void __launch_bounds__(DIAG_THREADS)
k_diag_final(int N, const double* __restrict__ scratch, double* __restrict__ out4) {
    double m = 0.0, s1 = 0.0, s2 = 0.0, s3 = 0.0;
    for (int t = threadIdx.x; t < DIAG_BLOCKS; t += blockDim.x) {
        m = fmax(m, scratch[t]);
        s1 += scratch[DIAG_BLOCKS + t];
        s2 += scratch[2 * DIAG_BLOCKS + t];
        s3 += scratch[3 * DIAG_BLOCKS + t];
    }
    block_reduce4(m, s1, s2, s3);
    if (threadIdx.x == 0) {
        const double h = 1.0 / (double)N;
        const double h2 = h * h;
        out4[0] = m;
        out4[1] = sqrt(h2 * s1);
        out4[2] = 0.5 * h2 * s2;
        out4[3] = 0.5 * h2 * s3;
    }
}

// ---- a1, stream engine: one colour half-sweep over global memory --------------------------------------
// eq 15-21 P:114-138 reduced to the 5-point operator (D1-D3):
//   psi <- (1 - beta) psi + (beta/4) (psi_W + psi_E + psi_S + psi_N) + (beta/4) h^2 omega
__global__ void __launch_bounds__(256)
k_half_sweep(int N, int pitch, double cb, double omb, double* __restrict__ psi, const double* __restrict__ q,
             int colour) {
    const int j = 1 + blockIdx.y * blockDim.y + threadIdx.y;
    if (j > N - 1) return;
    const int i0 = (((1 + j) & 1) == colour) ? 1 : 2;
    const int i = i0 + 2 * (blockIdx.x * blockDim.x + threadIdx.x);
    if (i > N - 1) return;
    const size_t k = (size_t)j * pitch + i;
    const double nb = (psi[k - 1] + psi[k + 1]) + (psi[k - pitch] + psi[k + pitch]);
    psi[k] = fma(omb, psi[k], fma(cb, nb, q[k]));
}

// ---- a1, NEXT-3 variant: one damped-Jacobi sweep, old values only -------------------
// Same point formula as the red-black sweep, read from psi_in, written to psi_out (walls of psi_out are +0.0 already).
__global__ void __launch_bounds__(256)
k_jacobi_sweep(int N, int pitch, double cb, double omb, const double* __restrict__ psi_in, const double* __restrict__ q,
               double* __restrict__ psi_out) {
    const int i = 1 + blockIdx.x * blockDim.x + threadIdx.x;
    const int j = 1 + blockIdx.y * blockDim.y + threadIdx.y;
    if (i > N - 1 || j > N - 1) return;
    const size_t k = (size_t)j * pitch + i;
    const double nb = (psi_in[k - 1] + psi_in[k + 1]) + (psi_in[k - pitch] + psi_in[k + pitch]);
    psi_out[k] = fma(omb, psi_in[k], fma(cb, nb, q[k]));
}

// ---- a1, NEXT-1 variant: the paper's 4th-order compact 9-point operator, eq 14-21, four colours ----
// eq 15 collected (dx = dy = h):  psi <- (1 - beta) psi + 0.2 beta S_edge(psi) + 0.05 beta S_corner(psi) + qB,
// qB = (0.025 beta h^2) (S_edge(w) + 8 w_0)  = (3/5)(beta/a) B of eq 17; B reads the wall ring of w next to a wall.
__global__ void __launch_bounds__(256)
k_compact_rhs(int N, int pitch, double c9q, const double* __restrict__ w, double* __restrict__ qB) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    if (i > N || j > N) return;
    const size_t k = (size_t)j * pitch + i;
    const bool interior = (i >= 1) & (i <= N - 1) & (j >= 1) & (j <= N - 1);
    double v = 0.0;
    if (interior) v = c9q * (((w[k - 1] + w[k + 1]) + (w[k - pitch] + w[k + pitch])) + 8.0 * w[k]);
    qB[k] = v;
}

// one colour (i mod 2, j mod 2) = (colour & 1, colour >> 1) of a sweep; inside a colour no point reads another one of it
__global__ void __launch_bounds__(256)
k_compact_colour(int N, int pitch, double c9e, double c9c, double omb, double* __restrict__ psi, const double* __restrict__ qB,
                 int colour) {
    const int i = ((colour & 1) ? 1 : 2) + 2 * (blockIdx.x * blockDim.x + threadIdx.x);
    const int j = ((colour >> 1) ? 1 : 2) + 2 * (blockIdx.y * blockDim.y + threadIdx.y);
    if (i > N - 1 || j > N - 1) return;
    const size_t k = (size_t)j * pitch + i;
    const double se = (psi[k - 1] + psi[k + 1]) + (psi[k - pitch] + psi[k + pitch]);
    const double sc = (psi[k - pitch - 1] + psi[k - pitch + 1]) + (psi[k + pitch - 1] + psi[k + pitch + 1]);
    psi[k] = fma(omb, psi[k], fma(c9e, se, fma(c9c, sc, qB[k])));
}

// ---- NEXT-2: RES_psi, RES_omega of eq 26-27: sum over ALL grid points of |new - old| ---------
__global__ void __launch_bounds__(DIAG_THREADS)
k_res_partial(int N, int pitch, const double* __restrict__ p1, const double* __restrict__ p0, const double* __restrict__ w1,
              const double* __restrict__ w0, double* __restrict__ scratch) {
    const long long M = (long long)(N + 1) * (N + 1);
    double m = 0.0, sp = 0.0, sw = 0.0, unused = 0.0;
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < M; t += (long long)gridDim.x * blockDim.x) {
        const size_t k = (size_t)(t / (N + 1)) * pitch + (size_t)(t % (N + 1));
        sp += fabs(p1[k] - p0[k]);
        sw += fabs(w1[k] - w0[k]);
    }
    block_reduce4(m, sp, sw, unused);
    if (threadIdx.x == 0) {
        scratch[DIAG_BLOCKS + blockIdx.x] = sp;
        scratch[2 * DIAG_BLOCKS + blockIdx.x] = sw;
    }
}

__global__ void __launch_bounds__(DIAG_THREADS)
k_res_final(int N, const double* __restrict__ scratch, double* __restrict__ out2) {
    double m = 0.0, sp = 0.0, sw = 0.0, unused = 0.0;
    for (int t = threadIdx.x; t < DIAG_BLOCKS; t += blockDim.x) {
        sp += scratch[DIAG_BLOCKS + t];
        sw += scratch[2 * DIAG_BLOCKS + t];
    }
    block_reduce4(m, sp, sw, unused);
    if (threadIdx.x == 0) {
        const double npts = (double)(N + 1);     // the paper's divisor: N = n_x = n_y points per side (reading G17)
        out2[0] = sp / npts;
        out2[1] = sw / npts;
    }
}

// ---- measurement aid: the fp64 issue rate of this GPU ("the builder measures one (DFMA chain)") ----
// Every thread runs CHAINS independent chains of dependent DFMAs (enough to cover the pipe latency), every SM holds 16 warps
// (as the resident engine does).  The result is written so that nothing is optimised away.
constexpr int PEAK_CHAINS = 8;
constexpr int PEAK_UNROLL = 16;
__global__ void __launch_bounds__(512)
k_fp64_peak(int iters, double a, double b, double* __restrict__ sink) {
    double x[PEAK_CHAINS];
#pragma unroll
    for (int c = 0; c < PEAK_CHAINS; ++c) x[c] = 1.0 + 1e-9 * (threadIdx.x + c);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < PEAK_UNROLL; ++u)
#pragma unroll
            for (int c = 0; c < PEAK_CHAINS; ++c) x[c] = fma(x[c], a, b);
    }
    double s = 0.0;
#pragma unroll
    for (int c = 0; c < PEAK_CHAINS; ++c) s += x[c];
    if (s == 12345.678) sink[blockIdx.x * blockDim.x + threadIdx.x] = s;      // never true for the a, b used; keeps the chains alive
}

}  // namespace

int fp64_peak(int blocks, int iters, double* sink_dev, cudaStream_t st, double* dfma_per_thread_out) {
    k_fp64_peak<<<blocks, 512, 0, st>>>(iters, 0.999999, 1e-6, sink_dev);
    if (dfma_per_thread_out) *dfma_per_thread_out = (double)iters * PEAK_UNROLL * PEAK_CHAINS;
    return launched(1);
}

int jacobi_sweeps(const Params& P, double* psi, double* psi_tmp, const double* q, int nsweeps, cudaStream_t st) {
    dim3 b(64, 4), g(cdiv(P.N - 1, 64), cdiv(P.N - 1, 4));
    double *in = psi, *out = psi_tmp;
    for (int s = 0; s < nsweeps; ++s) {
        k_jacobi_sweep<<<g, b, 0, st>>>(P.N, P.pitch, P.cb, P.omb, in, q, out);
        double* t = in; in = out; out = t;
    }
    if (in != psi && cudaMemcpyAsync(psi, in, (size_t)P.pitch * (P.N + 1) * sizeof(double), cudaMemcpyDeviceToDevice, st) != cudaSuccess)
        return -(int)cudaGetLastError();
    return launched(nsweeps);
}

int compact_rhs(const Params& P, const double* w, double* qB, cudaStream_t st) {
    dim3 b(32, 8), g(cdiv(P.N + 1, 32), cdiv(P.N + 1, 8));
    k_compact_rhs<<<g, b, 0, st>>>(P.N, P.pitch, P.c9q, w, qB);
    return launched(1);
}

int compact_sweeps(const Params& P, double* psi, const double* qB, int nsweeps, cudaStream_t st) {
    const int half = P.N / 2 + 1;
    dim3 b(64, 4), g(cdiv(half, 64), cdiv(half, 4));
    for (int s = 0; s < nsweeps; ++s)
        for (int colour = 0; colour < 4; ++colour)             // (0,0), (1,0), (0,1), (1,1): reading N1
            k_compact_colour<<<g, b, 0, st>>>(P.N, P.pitch, P.c9e, P.c9c, P.omb, psi, qB, colour);
    return launched(4 * nsweeps);
}

int res_monitors(const Params& P, const double* psi_new, const double* psi_old, const double* w_new, const double* w_old,
                 double* scratch_dev, double* out2_dev, cudaStream_t st) {
    k_res_partial<<<DIAG_BLOCKS, DIAG_THREADS, 0, st>>>(P.N, P.pitch, psi_new, psi_old, w_new, w_old, scratch_dev);
    k_res_final<<<1, DIAG_THREADS, 0, st>>>(P.N, scratch_dev, out2_dev);
    return launched(2);
}

int scale_rhs(const Params& P, const double* w, double* q, cudaStream_t st) {
    dim3 b(32, 8), g(cdiv(P.N + 1, 32), cdiv(P.N + 1, 8));
    k_scale_rhs<<<g, b, 0, st>>>(P.N, P.pitch, P.cq, w, q);
    return launched(1);
}

int thom_ring(const Params& P, const double* psi, double* w, cudaStream_t st) {
    k_thom_ring<<<cdiv(P.N + 1, 128), 128, 0, st>>>(P.N, P.pitch, P.c2h2, P.lid, psi, w);
    return launched(1);
}

int zero_ring(const Params& P, double* psi, cudaStream_t st) {
    k_zero_ring<<<cdiv(P.N + 1, 128), 128, 0, st>>>(P.N, P.pitch, psi);
    return launched(1);
}

int rk_stage(const Params& P, int k, const double* psi, const double* w_in, const double* a, const double* b,
             double* w_out, double* t_out, cudaStream_t st) {
    dim3 bl(32, 8), g(cdiv(P.N + 1, 32), cdiv(P.N + 1, 8));
    switch (k) {
        case 1: k_rk_stage<1><<<g, bl, 0, st>>>(P, psi, w_in, a, b, w_out, t_out); break;
        case 2: k_rk_stage<2><<<g, bl, 0, st>>>(P, psi, w_in, a, b, w_out, t_out); break;
        case 3: k_rk_stage<3><<<g, bl, 0, st>>>(P, psi, w_in, a, b, w_out, t_out); break;
        case 4: k_rk_stage<4><<<g, bl, 0, st>>>(P, psi, w_in, a, b, w_out, t_out); break;
        case 5: k_rk_stage<5><<<g, bl, 0, st>>>(P, psi, w_in, a, b, w_out, t_out); break;
        default: return -(int)cudaErrorInvalidValue;
    }
    return launched(1);
}

int diag_scratch_doubles() { return DIAG_BLOCKS; }

int diagnostics(const Params& P, const double* psi, const double* w, double* scratch_dev, double* out4_dev,
                cudaStream_t st) {
    k_diag_partial<<<DIAG_BLOCKS, DIAG_THREADS, 0, st>>>(P.N, P.pitch, psi, w, scratch_dev);
    k_diag_final<<<1, DIAG_THREADS, 0, st>>>(P.N, scratch_dev, out4_dev);
    return launched(2);
}

int stream_sweeps(const Params& P, double* psi, const double* q, int nsweeps, cudaStream_t st) {
    const int per_row = (P.N - 1 + 1) / 2;
    dim3 b(64, 4), g(cdiv(per_row, 64), cdiv(P.N - 1, 4));
    for (int s = 0; s < nsweeps; ++s) {
        k_half_sweep<<<g, b, 0, st>>>(P.N, P.pitch, P.cb, P.omb, psi, q, 0);   // red = (i + j) even first (G9)
        k_half_sweep<<<g, b, 0, st>>>(P.N, P.pitch, P.cb, P.omb, psi, q, 1);
    }
    return launched(2 * nsweeps);
}

}  // namespace cavk
