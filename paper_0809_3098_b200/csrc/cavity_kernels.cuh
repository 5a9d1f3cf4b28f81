// cavity_kernels.cuh — launchers of the sm_100a kernels behind include/cavity.h.
// Plain CUDA: no torch types.  Every launcher enqueues on `st` and returns the number of kernel
// launches it made (negative = cudaError_t negated).
//
// P:n = /root/reference/PAPER.md line n.  Device layout of a field:
// element (i, j) lives at  j * pitch + i,  pitch = (N + 1) rounded up to a multiple of 4 doubles, so that
// every row starts on a 32-byte sector boundary; the base pointer is 256-byte aligned.
#pragma once
#include <cuda_runtime.h>

namespace cavk {

// Constants of one problem, computed once on the host (cavity_api.cu: make_params).
struct Params {
    int N;          // intervals per side
    int pitch;      // doubles per device row
    double cb;      // beta / 4
    double cq;      // (beta / 4) h^2                (scales omega into the sweep's right-hand side q)
    double omb;     // 1 - beta
    double i2h;     // 1 / (2h) = N / 2
    double ih2;     // 1 / h^2 = N^2
    double nu;      // 1 / Re
    double c2h2;    // 2 / h^2                       (eq 25)
    double lid;     // 2 U / h, U = 1                (eq 25, lid term)
    double dt;
    double c9e;     // 0.2 beta                      (NEXT-1 compact operator: weight of the four edge neighbours)
    double c9c;     // 0.05 beta                     (weight of the four corner neighbours)
    double c9q;     // (0.025 beta) h^2              (scales S_edge(w) + 8 w_0 into the sweep's right-hand side)
};

// ---- support kernels (both engines) ---------------------------------------------------------------
// q_ij = cq * w_ij on interior points (the per-stage right-hand side of a1; constant over the S sweeps).
int scale_rhs(const Params& P, const double* w, double* q, cudaStream_t st);

// a2: Thom ring of w from psi (eq 25; corners owned by the top/bottom rows, G10).
int thom_ring(const Params& P, const double* psi, double* w, cudaStream_t st);

// a2 + a3 fused, stage k = 1..5 (eq 8, eq 22, eq 9-13).  The wall vorticity a near-wall
// point needs is evaluated on the fly from psi by the same formula thom_ring uses; ring threads store it to
// the ring of w_out.  Pointer roles per stage:
//   k=1: w_in = w0                         -> w_out = w1
//   k=2: w_in = w1, a = w0                 -> w_out = w2
//   k=3: w_in = w2, a = w0                 -> w_out = w3
//   k=4: w_in = w3, a = w0, b = w2         -> w_out = w4, t_out = T   (first three terms of eq 13)
//   k=5: w_in = w4, a = T                  -> w_out = omega^{n+1} (may alias w0: only pointwise access to it)
int rk_stage(const Params& P, int k, const double* psi, const double* w_in, const double* a, const double* b,
             double* w_out, double* t_out, cudaStream_t st);

// a4: res_inf, res_l2, kinetic energy, enstrophy -> out4_dev[0..3] (device).  scratch_dev must hold
// 4 * diag_scratch_doubles() doubles.
int diag_scratch_doubles();
int diagnostics(const Params& P, const double* psi, const double* w, double* scratch_dev, double* out4_dev,
                cudaStream_t st);

// forces the wall ring of psi to +0.0 (cav_set_fields)
int zero_ring(const Params& P, double* psi, cudaStream_t st);

// ---- stream engine: one kernel per colour half-sweep ----------------------------------------------
// nsweeps x (red half-sweep, black half-sweep) of a1 on psi in place, right-hand side q (already scaled).
int stream_sweeps(const Params& P, double* psi, const double* q, int nsweeps, cudaStream_t st);

// ---- NEXT-3: damped-Jacobi sweeps ------------------------------------------------
// nsweeps sweeps of psi_new = fma(1 - beta, psi, fma(beta / 4, nb, q)) from OLD values only; the result is in psi
// (psi_tmp is a second field whose wall ring is +0.0; it is clobbered).
int jacobi_sweeps(const Params& P, double* psi, double* psi_tmp, const double* q, int nsweeps, cudaStream_t st);

// ---- NEXT-1: the paper's 4th-order compact 9-point operator (eq 14-21), four-colour SOR ------
// qB = c9q (S_edge(w) + 8 w_0) on interior points (reads the wall ring of w), 0 elsewhere.
int compact_rhs(const Params& P, const double* w, double* qB, cudaStream_t st);
// nsweeps x four colour passes of psi <- fma(1 - beta, psi, fma(c9e, S_edge, fma(c9c, S_corner, qB))) in place.
int compact_sweeps(const Params& P, double* psi, const double* qB, int nsweeps, cudaStream_t st);

// ---- NEXT-2: the paper's steady-state monitors (eq 26-27) ----------------------------------
// out2_dev[0] = RES_psi = (1 / (N + 1)) sum |psi_new - psi_old|, out2_dev[1] = RES_omega likewise, over all grid points.
// scratch_dev: as for diagnostics().
int res_monitors(const Params& P, const double* psi_new, const double* psi_old, const double* w_new, const double* w_old,
                 double* scratch_dev, double* out2_dev, cudaStream_t st);

// ---- measurement aid: DFMA-chain micro-kernel (one CTA of 512 threads per block, `blocks` of them; sink_dev: blocks x 512
// doubles that are never written in practice).  *dfma_per_thread_out = dependent-chain DFMAs each thread executes.
int fp64_peak(int blocks, int iters, double* sink_dev, cudaStream_t st, double* dfma_per_thread_out);

}  // namespace cavk
