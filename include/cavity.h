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

/* Selects the sweep engine (CAV_ENGINE_*).  CAV_ENOTSUP if that engine cannot run this grid on this
 * device.  The default is CAV_ENGINE_AUTO. */
int cav_set_engine(cav_ctx* ctx, int engine);

/* Resident engine only: forces T, the number of sweeps between two halo exchanges (1..10; the halo is 2T
 * points deep; 0 = the planner's own choice) and / or the kernel variant (0 = the only one built: one CTA of up to 16 warps per
 * SM; -1 = the planner's choice), and re-plans the tiling.  The result of every other call is unchanged bit for bit; this is a
 * tuning / testing knob.  CAV_ENOTSUP if no such plan exists (the previous plan is kept). */
int cav_set_resident_plan(cav_ctx* ctx, int sweeps_per_exchange, int variant);

/* Profiling aid, resident engine with the red-black sweeps only (CAV_ENOTSUP otherwise): runs nsweeps of a1 on the current
 * (psi, omega) like cav_poisson (without the a2 pass) and returns, for every tile, %globaltimer stamps (ns, one clock for all
 * tiles) at the phase boundaries: stamps_out is a HOST array of ntiles x slots_per_tile; slot 0 = kernel start, 1 = inputs
 * loaded, then for exchange round r: 2 + 4r = sweeps done, 3 + 4r = border strips stored (by warp 0 of the tile), 4 + 4r = ring received from the
 * neighbours, 5 + 4r = edges republished.  Unused slots are 0; *ntiles_out (if non-NULL) receives the tile count; call once
 * with the capacity of a plan's tile count (at most 1023). */
int cav_trace_sweeps(cav_ctx* ctx, int nsweeps, long long* stamps_out, int slots_per_tile, int* ntiles_out);

/* Host logic of the resident engine, no device and no context needed: plans the tiling of an (N + 1)^2 grid for a device with
 * `sms` multiprocessors, `smem_bytes` of shared memory per block and 65536 registers (sweep: CAV_SWEEP_REDBLACK or
 * CAV_SWEEP_COMPACT9; T > 0 forces the sweeps per exchange round) and checks its halo-exchange pattern: every unit of four
 * points a tile fetches must be stored by exactly one tile, every stored unit must be fetched, every tile must fit its thread
 * grid.  plan_out[9] (may be NULL) = ntx, nty, CW, CH, halo, T, warps, shared-memory bytes, EB (rows the first row of tiles owns beyond CH); counts_out[5] (may be NULL) = units
 * fetched, units stored, fetches without exactly one store, stores nobody fetches, tiles that do not fit.
 * Returns CAV_OK if the plan is consistent (also for a single-tile plan, which exchanges nothing), CAV_ENOTSUP if the grid
 * has no resident plan under these figures, CAV_EINVAL for bad arguments or an inconsistent pattern. */
int cav_plan_check(int N, int sweep, int T, int sms, int smem_bytes, int* plan_out, long long* counts_out);

/* Testing aid, resident engine (no context; current device): the exchange unit of the halo exchange (four doubles as five
 * 64-bit words, each with a 12-bit tag) as a round trip.  in_host holds nunits x 4 doubles (any bit patterns: NaN payloads, infinities,
 * denormals, signed zeros); they are packed with `tag` (1 .. 4095), stored and loaded with the accesses of the exchange, validated and
 * restored on the device into out_host, which must then equal in_host bit for bit.  *bad_out (may be NULL) = units whose five tags did not
 * validate for `tag`, or validated for a different tag.  Errors: CAV_EINVAL (null pointers, nunits < 1, tag out of range), CAV_ECUDA. */
int cav_debug_unit_roundtrip(const double* in_host, double* out_host, int nunits, unsigned int tag, int* bad_out);

/* Testing aid, resident engine: sets the host-side count of halo-exchange rounds (the 12-bit tag of a round is 1 + round mod
 * 4095, the buffer round mod 2) and clears the exchange buffers, so that a test can run across the wrap of the tags and of the
 * 32-bit counter.  Neither wrap needs any action in normal use: a reader can only ever meet the round it waits for or the one
 * two rounds earlier. */
int cav_debug_set_epoch(cav_ctx* ctx, unsigned int epoch);

/* Measurement aid (the fp64 roofline needs a MEASURED peak): runs a DFMA-chain micro-kernel on every SM
 * of the context's device (one CTA of 16 warps per SM, 8 independent dependent chains per thread, best of 4 timed launches by
 * CUDA events on the context's stream) and writes the achieved rate in fp64 FMA instructions per second, counted per thread
 * (lane), to *dfma_per_s_out; *sm_clock_mhz_out (may be NULL) receives the device's nominal SM clock.  The nominal figure for
 * B200 is 148 SMs x 64 fp64 lanes x clock.  Does not touch the state. */
int cav_measure_fp64_peak(cav_ctx* ctx, double* dfma_per_s_out, double* sm_clock_mhz_out);

/* Describes the launch plan of the current engine in `buf` (NUL-terminated, truncated to len). */
int cav_describe(cav_ctx* ctx, char* buf, int len);

/* Number of kernel launches enqueued by this context since cav_create (for bench.py's gpu_launches). */
long long cav_launch_count(cav_ctx* ctx);

/* CUDA-event time in milliseconds of the most recent cav_step / cav_step_async (the whole call) or cav_poisson (its a1
 * sweeps alone, without the a2 pass and the residual) on the context's stream (events recorded around the enqueued
 * work); blocks until that work has finished.  Writes 0 if none has run. */
int cav_last_elapsed_ms(cav_ctx* ctx, float* ms_out);

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
