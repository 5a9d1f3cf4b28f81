// cavity_resident.cuh — the resident engine: one persistent CTA per tile, psi and the scaled right-hand side held in
// registers, temporal blocking with a 2T-deep halo (4T: compact operator) that is refreshed through L2 every T sweeps as self-validating tagged
// data (no fence, flag or grid barrier), a2 + a3 of every stage evaluated in the tile: whole time steps in one launch.
// See DESIGN.md "Resident engine".  Plain CUDA: no torch types.
#pragma once
#include <cuda_runtime.h>

#include "cavity_kernels.cuh"

namespace cavk {

// Launch plan of the resident engine for one grid on one device (host side, computed once per context).
struct ResidentPlan {
    bool ok = false;      // false: this grid / device cannot use the resident engine
    int variant = 0;      // index into the table of compiled micro-tile shapes (cavity_resident.cu)
    int C = 0, R = 0;     // micro-tile: each thread owns C consecutive x-points times R rows, in registers
    int warps = 0;        // warps per CTA; a warp spans 32 C points in x and R rows in y
    int T = 0;            // sweeps per round (between two halo exchanges); single tile: unused
    int halo = 0;         // 2 T, compact operator 4 T (one ring is consumed per colour pass); 0 for a single tile
    int CW = 0, CH = 0;   // core (owned) points per tile in x and y: rows [bj CH, (bj+1) CH); columns [0, CW + 1), [CW + 1, 2 CW + 1), ... (CW a multiple of 4)
    int EB = 0;           // > 0: the bottom tiles own EB more rows, [0, CH + EB), the others [EB + bj CH, EB + (bj + 1) CH), the last one the rest;
                          //      the wall y = 0 then sits inside warp 0 instead of being isolated in a warp of its own (5-point operator only)
    int ntx = 0, nty = 0; // tiles in x and y
    int ntiles = 0;
    bool fixup = false;           // some tile holds both walls of one direction: the kernel variant with the wall-mask fix-up
    int smem_bytes = 0;
    int regs = 0;         // registers per thread of the chosen variant (as compiled)
    int sm_count = 0;
    int per_sm = 1;       // CTAs per SM
    int kind = 0;         // 0 = red-black sweeps of the 5-point operator (halo 2T), 1 = four-colour sweeps of the compact 9-point operator (halo 4T)
};

// T_override > 0 forces the sweeps per round (1..10; tests use it to exercise short and ragged rounds);
// variant_override >= 0 forces the micro-tile shape (index into the compiled variants).
ResidentPlan resident_plan(const Params& P, int device, int T_override = 0, int variant_override = -1, int kind = 0);
// The same planner for given device figures (no device needed: host logic, testable on CPU)
ResidentPlan resident_plan_for(int N, int kind, int T_override, int variant_override, int sms, int smem_cap, int regs_per_block);
// Host-side check of a plan's exchange pattern (every fetched unit stored by exactly one tile, every stored unit fetched);
// counts[5]: fetched, stored, unmatched fetches / double stores, stores nobody fetches, tiles that do not fit.  0 = consistent.
int resident_check_exchange(const ResidentPlan& plan, int N, long long* counts);
// Testing aid: packs nunits x 4 doubles into exchange units with `tag`, moves them through scratch_dev (>= 48 nunits + 512 bytes) with the
// accesses of the exchange, and restores them into out_dev; *bad_dev counts units whose tags did not validate (or validated for another tag).
int resident_unit_roundtrip(const double* in_dev, double* out_dev, void* scratch_dev, int nunits, unsigned int tag, unsigned int* bad_dev,
                            cudaStream_t st);
int resident_variants();
void resident_describe(const ResidentPlan& plan, char* buf, int len);

// ONE exchange buffer (the engine needs two, zero-filled before first use and whenever the plan changes): a unit per group
// of four consecutive points of a grid row (unit k = columns 4k - 3 .. 4k), stored as three planes of 16, 16 and 8 bytes per unit.
inline int resident_unit_pitch(int N) { return (N + 3) / 4 + 2; }
inline size_t resident_plane_bytes(int N, int bytes_per_unit) {
    return ((size_t)resident_unit_pitch(N) * (size_t)(N + 1) * (size_t)bytes_per_unit + 255) / 256 * 256;
}
inline size_t resident_exchange_bytes(int N) { return 2 * resident_plane_bytes(N, 16) + resident_plane_bytes(N, 8); }

// Halo-exchange rounds one launch performs (the host-side round counter advances by this).
long long resident_rounds(const ResidentPlan& plan, int nsteps, int S);

// One launch of the resident kernel.
//   nsteps > 0: nsteps whole SSPRK(5,4) time steps, each 5 x [S sweeps of a1, a2, a3].  wbase points at six fields fstride
//               doubles apart: omega^n (in: the state; out: the new state, ring = stage-5 Thom ring), omega^(1..4), T.
//   nsteps = 0: S sweeps of a1 with right-hand side cq * (field 0 of wbase); nothing but psi is written.
// Reads psi_in, writes psi_out (two different fields).  xa, xb: the two exchange buffers (may be null for a single-tile plan).  err_word: one device word, zero-filled; non-zero
// afterwards = a tile gave up waiting for a neighbour.  *epoch is the host-side count of exchange rounds, advanced by this call.
// trace_dev (profiling only, sweeps-only launches): device array of ntiles x trace_cap %globaltimer stamps (ns), slot 0 = start,
// 1 = inputs loaded, then per round r: 2 + 4r sweeps done, 3 + 4r border strips stored, 4 + 4r ring received, 5 + 4r edges republished.
// Returns the number of kernel launches (1), or a negative cudaError_t.
int resident_launch(const Params& P, const ResidentPlan& plan, const double* psi_in, double* psi_out, void* xa, void* xb,
                    double* wbase, size_t fstride, unsigned int* err_word, unsigned int* epoch,
                    int nsteps, int S, cudaStream_t st, long long* trace_dev = nullptr, int trace_cap = 0);

}  // namespace cavk
