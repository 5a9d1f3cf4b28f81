/* cavity.h — C ABI of libcavity.so: the fp64 SSPRK(5,4) time step of the 2-D vorticity /
 * stream-function lid-driven cavity of arXiv 0809.3098 (Cardoso & Bicudo) on one B200 (sm_100a).
 *
 * P:n = /root/reference/PAPER.md line n;  S8 = SURVEY.md section 8;  Gk / Dk = the readings and
 * departures listed in DESIGN.md ("Readings of the paper").
 *
 * The problem: unit square, uniform grid of (N+1) x (N+1) points, h = 1/N, grid index
 * i = 0..N <-> x = i h, j = 0..N <-> y = j h, j = N is the lid moving at U = 1; psi = 0 on all four
 * walls (eq 23-24); nu = 1/Re.
 *
 * One time step (eq 9-13) is five stages; stage k with input vorticity w_in = omega^(k-1):
 *   (a1) S = sweeps_per_stage red-black SOR sweeps of the 5-point Poisson problem lap(psi) = -w_in,
 *        warm-started from the current psi; red = (i + j) even first, then black (G9):
 *          psi_ij <- psi_ij + beta ( (psi_W + psi_E + psi_S + psi_N + h^2 w_ij) / 4 - psi_ij )
 *        (eq 15-21 P:114-138 reduced to the 5-point operator, D1-D3)
 *   (a2) Thom wall vorticity of w_in from psi (eq 25): omega_wall = -2 psi_adjacent / h^2,
 *        minus 2U/h on the lid; the top and bottom rows own the four corners (G10)
 *   (a3) dL = dt L(psi, w_in) with eq 8 P:80 and eq 22, then the stage combination of eq 9-13.
 *
 * All entry points: host code, callable from any thread, but a context must not be used from two
 * threads at once.  All array arguments are HOST pointers unless the name ends in _dev; fields are
 * dense row-major (N+1) x (N+1) fp64 arrays, element k = j (N+1) + i.  Buffers are borrowed for the
 * duration of the call only.  Every call returns CAV_OK (0) or a negative CAV_E* code; nothing
 * throws across the ABI.  Device memory comes from PyTorch's CUDA caching allocator and all work is
 * enqueued on the PyTorch current stream of the device that was current at cav_create (the caller must
 * have initialised PyTorch's CUDA state first: torch.cuda.init(); the Python binding does); every call
 * below is synchronous at return unless stated otherwise.  There is no CPU fallback: without a CUDA
 * device cav_create returns CAV_ECUDA.
 */
#ifndef CAVITY_H
#define CAVITY_H

#ifdef __cplusplus
extern "C" {
#endif

#define CAV_OK       0
#define CAV_EINVAL  (-1)   /* bad argument */
#define CAV_ENOMEM  (-2)   /* host or device allocation failed */
#define CAV_ECUDA   (-3)   /* CUDA runtime error, or no usable device */
#define CAV_ENOTSUP (-4)   /* requested engine cannot run this problem on this device */
#define CAV_ELIMIT  (-5)   /* problem larger than a fixed-size buffer of the library (cav_diag_noalloc: N > CAV_NOALLOC_MAX_N) */

/* Sweep engines (all compute the same red-black SOR, bit for bit; they differ in how it is scheduled). */
#define CAV_ENGINE_AUTO     0   /* pick by grid size (default) */
#define CAV_ENGINE_STREAM   1   /* one kernel per colour half-sweep over global memory (the streaming baseline) */
#define CAV_ENGINE_RESIDENT 2   /* persistent register/shared-memory resident tiles, temporal blocking */

/* a1 variants (BASELINE.json north_star: "red-black SOR (or Jacobi)"). */
#define CAV_SWEEP_REDBLACK  0   /* red-black SOR, red = (i + j) even first (default; the timed path) */
#define CAV_SWEEP_JACOBI    1   /* damped Jacobi: every interior point from the OLD values only */
#define CAV_SWEEP_COMPACT9  2   /* the paper's own operator: 4th-order compact 9-point scheme, eq 14-21, relaxed in
                                   four colours (i mod 2, j mod 2) = (0,0), (1,0), (0,1), (1,1) (reading N1) */

typedef struct cav_ctx cav_ctx;   /* opaque; owned by the library from cav_create to cav_destroy */

typedef struct cav_diag {
    double t;                /* simulated time = step * dt */
    long long step;          /* time steps taken since cav_create / cav_set_fields */
    double res_inf;          /* max |r_ij| over interior points, r = lap_h(psi) + omega   (S8(a) row a4) */
    double res_l2;           /* sqrt(h^2 sum r^2) */
    double kinetic_energy;   /* (1/2) h^2 sum (u^2 + v^2), u, v of eq 22 */
    double enstrophy;        /* (1/2) h^2 sum omega^2 */
} cav_diag;

/* Result of cav_run_to_steady. */
typedef struct cav_monitor {
    int steps;               /* time steps taken by the call */
    int converged;           /* 1 if RES_psi < tol_psi and RES_omega < tol_omega at the last monitored step */
    double res_psi;          /* eq 26 P:198 of the last monitored step */
    double res_omega;        /* eq 27 */
} cav_monitor;

/* Allocates psi, omega and the stage buffers (zero-filled: fluid at rest) for an (N+1) x (N+1) grid.
 * Re: Reynolds number (nu = 1/Re); dt: time step; sor_omega: relaxation factor beta in (0, 2);
 * sweeps_per_stage: S >= 0 red-black sweeps per RK stage (D3).
 * Errors: CAV_EINVAL (out null, N < 2, Re <= 0, dt <= 0, sor_omega outside (0, 2), S < 0, or any
 * of them not finite); CAV_ENOMEM; CAV_ECUDA.  On error *out is NULL. */
int cav_create(cav_ctx** out, int N, double Re, double dt, double sor_omega, int sweeps_per_stage);

/* Frees everything.  NULL is a no-op. */
void cav_destroy(cav_ctx* ctx);

/* Loads the state from host arrays.  psi == NULL means psi <- 0.  Wall entries of psi are ignored and
 * forced to 0 (eq 23-24, G5); wall entries of omega are stored as given (a2 overwrites them before
 * first use).  Resets step and t to 0.  omega == NULL is CAV_EINVAL. */
int cav_set_fields(cav_ctx* ctx, const double* psi, const double* omega);

/* Copies the state into caller-owned host arrays of (N+1)^2 doubles (either may be NULL).  Pure.
 * After a step: omega interior = omega^{n+1}; psi and the omega ring are those of stage 5 (G16). */
int cav_get_fields(cav_ctx* ctx, double* psi_out, double* omega_out);

/* Advances nsteps SSPRK(5,4) steps, each 5 x [a1 x S, a2, a3].  nsteps < 0: CAV_EINVAL; 0: no-op.  With the resident engine
 * and the red-black sweeps the whole call is ONE kernel launch.
 * CAV_ECUDA from this or any later call of a resident-engine context can also mean that a tile of the persistent kernel waited
 * ~10 s for a neighbour's halo and gave up (it cannot happen on a healthy device: all tiles are co-resident; a debugger,
 * time-slicing or a sanitizer can stretch the wait).  The fields are then undefined; the condition is sticky (cav_sync,
 * cav_get_fields, cav_get_diag, cav_poisson, cav_step_res and cav_run_to_steady report it too) until cav_set_fields,
 * cav_set_engine, cav_set_resident_plan or a cav_set_sweep that plans anew, which clear it.  CAV_DEBUG=1 in the environment
 * prints which tile waited for which unit (and the CUDA error string behind any other CAV_ECUDA) to stderr.
 * Two resident-engine contexts of one device must not have launches in flight at the same time: every launch wants all SMs
 * for its co-resident tiles, so create them under the same stream (they then run one after the other) or cav_sync one before
 * stepping the other.  A launch queued behind another context's long cav_step(n) on a DIFFERENT stream may start with only
 * part of its tiles resident and trip the 10 s wait.
 * Size limit of the resident engine: one tile per SM, tiles of at most 128 x 96 points including halos, so on a 148-SM B200
 * there is a plan for every N <= 1200 with the 5-point sweeps (compact operator: every N <= 1133 and 1144 <= N <= 1200).
 * Larger grids run on the streaming engine (10 S + 10 launches per step, several times slower per point); cav_describe
 * says which engine a context uses. */
int cav_step(cav_ctx* ctx, int nsteps);

/* As cav_step but returns after enqueueing on the context's stream (no host synchronisation). */
int cav_step_async(cav_ctx* ctx, int nsteps);

/* Blocks until all work enqueued for this context has finished. */
int cav_sync(cav_ctx* ctx);

/* nsweeps of a1 on the current (psi, omega), then one a2 so that the omega ring matches psi; writes
 * the max-norm residual (row a4) to *res_inf_out if non-NULL.  Does not advance time. */
int cav_poisson(cav_ctx* ctx, int nsweeps, double* res_inf_out);

/* Selects the a1 variant (CAV_SWEEP_*) used by cav_step and cav_poisson from now on.  With CAV_SWEEP_JACOBI sor_omega is the
 * damping factor: psi_new = psi + beta ((psi_W + psi_E + psi_S + psi_N + h^2 w) / 4 - psi), all from the previous sweep's
 * values (it converges for beta <= 1; nothing is checked).  With CAV_SWEEP_COMPACT9 a sweep is eq 15 of the paper,
 *   psi <- (3/5)(beta/a)(A + B + C) + (1 - beta) psi,  A, B, C of eq 16-18, a = 2/h^2,
 * whose B reads omega on the walls: the stage input carries the wall vorticity a2 computed in the previous stage (for the
 * first stage after cav_set_fields: the ring as given; reading N2).  The Jacobi sweeps run as one kernel per sweep
 * over global memory whatever the engine (inside a CUDA graph of the time step).  The compact sweeps run in the resident engine's
 * persistent kernel like the red-black ones (four colour passes per sweep, halo 4T deep; the tiling is planned anew when the
 * sweep kind changes: a T forced with cav_set_resident_plan is kept if the new operator has a plan with it, else dropped
 * for the planner's own; the exchange buffers start afresh and the sticky error of cav_step is cleared), or, with
 * CAV_ENGINE_STREAM, as four kernels per sweep over global memory; both agree bit for bit. */
int cav_set_sweep(cav_ctx* ctx, int kind);

/* One time step, and the paper's steady-state monitors of that step (eq 26-27):
 *   RES_psi = (1 / n) sum_ij |psi^{n+1}_ij - psi^n_ij|,  RES_omega likewise with omega,
 * sums over ALL (N+1)^2 grid points, n = N + 1 = the points per side (the paper's literal divisor; reading G17);
 * psi^n, psi^{n+1} are what cav_get_fields returns before / after the step (G16).  Either pointer may be NULL. */
int cav_step_res(cav_ctx* ctx, double* res_psi_out, double* res_omega_out);

/* The paper's run-to-steady-state rule: steps until RES_psi < tol_psi and RES_omega < tol_omega, evaluating the
 * monitors on every check_every-th step of the call (>= 1), for at most max_steps steps.  *out reports the steps taken,
 * whether the rule was met, and the monitors of the last monitored step (0 if none was).  CAV_EINVAL on bad arguments. */
int cav_run_to_steady(cav_ctx* ctx, int max_steps, int check_every, double tol_psi, double tol_omega, cav_monitor* out);

/* Runs the a4 reductions on the current state.  Pure. */
int cav_get_diag(cav_ctx* ctx, cav_diag* out);

/* The tuning, tracing, testing and measurement calls of the same library (engine and plan selection, phase trace, planner check,
 * exchange-unit round trip, fp64 peak, launch count, event time) are declared in cavity_debug.h; a user of the method does not need them. */

/* ---- The one entry point that allocates nothing -------------------------------------------------------------------------
 *
 * Every call above works on a context, and cav_create takes its fields and work buffers from PyTorch's caching allocator.
 * That rules the library out for callers that may not allocate device memory at the moment they need a number from it:
 * a thread that runs while some stream of the process is being captured in the global capture mode (cudaMalloc is refused
 * there and invalidates the capture), a solver that lives inside a fixed slice of HBM handed out by a host application
 * (the rest of the GPU belongs to somebody else's pool, so asking the driver for more can fail at any time), and loops that
 * cannot afford the device-wide synchronisation cudaMalloc / cudaFree imply.  For them:
 *
 * cav_diag_noalloc computes the a4 diagnostics (the same four numbers cav_get_diag reports: res_inf, res_l2, kinetic_energy,
 * enstrophy, in that order; definitions at struct cav_diag) of a state the CALLER holds in device memory, without a context
 * and without calling cudaMalloc, cudaFree, PyTorch's allocator or any other routine that allocates.
 *   N          intervals per side, 2 <= N <= CAV_NOALLOC_MAX_N
 *   pitch      doubles per row of both fields, >= N + 1 (N + 1 for dense arrays; the padded pitch for rows that are padded)
 *   psi_dev, omega_dev   DEVICE pointers, (N + 1) rows of `pitch` doubles, element (i, j) at j * pitch + i; read only.  psi is
 *              read as given, walls included (cav_set_fields forces them to 0; here that is the caller's business).
 *   out4_dev   DEVICE pointer to 4 doubles, written by the kernel
 *   stream     a cudaStream_t passed as a plain pointer (NULL = the default stream) of the CURRENT device, which must be the
 *              device the three buffers live on.
 * The call returns once the work is enqueued on `stream`: out4_dev holds the result when the stream has got that far, and
 * the input buffers must stay untouched until then.  It agrees with cav_get_diag to rounding (the sums are taken in another
 * order: relative differences of a few 1e-16 per sum), not bit for bit; repeated calls on the same input agree bit for bit.
 *
 * The memory it does need (one partial result per grid row, and a counter) is a fixed 256.25 KiB array inside the library's
 * device image.  Consequences a user must know:
 *   - LIMIT: N > CAV_NOALLOC_MAX_N (8192) does not fit and is refused with CAV_ELIMIT; nothing is launched.
 *   - Every GPU on which the library's device code gets loaded carries those 256.25 KiB until the process exits.
 *   - The array is ONE per device, shared by all calls from all threads and streams.  Two calls whose kernels can overlap on
 *     the GPU (different streams without an ordering between them) race on it and both results are garbage: order them.
 *     Calls on one stream are safe back to back; each call clears the counter it needs to start from zero.
 *   - The FIRST call on each device looks up the array's device address (cudaGetSymbolAddress, which makes the runtime load
 *     the library's device image there).  Make that first call at start-up, before any stream capture begins.
 * Errors: CAV_EINVAL (null pointer, N < 2, pitch < N + 1), CAV_ELIMIT (N too large), CAV_ENOTSUP (device ordinal >= 64),
 * CAV_ECUDA (the runtime refused the lookup, the clear or the launch; CAV_DEBUG=1 prints which). */
#define CAV_NOALLOC_MAX_N 8192
int cav_diag_noalloc(int N, int pitch, const double* psi_dev, const double* omega_dev, double* out4_dev, void* stream);

/* CAV_NOALLOC_MAX_N as the loaded library was built with. */
int cav_noalloc_max_n(void);

/* Static string for an error code. */
const char* cav_strerror(int code);

#ifdef __cplusplus
}
#endif
#endif /* CAVITY_H */
