/* cavity_debug.h — the tuning, tracing, testing and measurement calls of libcavity.so.
 *
 * Not part of the method's boundary (that is cavity.h: SURVEY S8(b) plus cav_step_async / cav_sync / cav_set_sweep / cav_step_res /
 * cav_run_to_steady / cav_diag_noalloc).  Same library, same conventions (host pointers unless named _dev, CAV_OK or a negative
 * CAV_E* code, nothing throws); bench.py, the tests and the profiling notes under profiles/ use them.  None of them changes a
 * result: whatever engine or plan is selected, every call of cavity.h returns the same bits.
 */
#ifndef CAVITY_DEBUG_H
#define CAVITY_DEBUG_H

#include "cavity.h"

#ifdef __cplusplus
extern "C" {
#endif

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

#ifdef __cplusplus
}
#endif
#endif /* CAVITY_DEBUG_H */
