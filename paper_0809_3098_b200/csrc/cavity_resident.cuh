// cavity_resident.cuh — the resident sweep engine (a1): one persistent CTA per tile, psi and the scaled
// right-hand side held in registers for all S sweeps of a stage, temporal blocking with a 2T-deep halo that
// is refreshed through L2 every T sweeps as self-validating tagged data (no fence, flag or grid barrier).
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
    int halo = 0;         // 2 T (one ring is consumed per colour half-sweep); 0 for a single tile
    int CW = 0, CH = 0;   // core (owned) points per tile in x and y; tile (bi, bj) owns [bi CW, (bi+1) CW) x [bj CH, (bj+1) CH)
    int ntx = 0, nty = 0; // tiles in x and y
    int ntiles = 0;
    int ns_per = 0, nr_per = 0;   // exchange units each thread stores / fetches per round (0 for a single tile)
    bool fixup = false;           // some tile holds both walls of one direction: the kernel variant with the wall-mask fix-up
    int smem_bytes = 0;
    int regs = 0;         // registers per thread of the chosen variant (as compiled)
    int sm_count = 0;
    int per_sm = 1;       // CTAs per SM the chosen kernel variant is built for
};

// T_override > 0 forces the sweeps per round (1..8; tests use it to exercise short and ragged rounds);
// variant_override >= 0 forces the micro-tile shape (index into the compiled variants).
ResidentPlan resident_plan(const Params& P, int device, int T_override = 0, int variant_override = -1);
int resident_variants();
void resident_describe(const ResidentPlan& plan, char* buf, int len);

// Doubles behind ONE exchange buffer (the engine needs two): a 16-byte unit per point of a pitch x (N+1) field.
inline size_t resident_exchange_doubles(size_t field_doubles) { return 2 * field_doubles; }

// Per-plan exchange tables (device memory, built once per plan): their size, and the kernel that fills them.
size_t resident_table_bytes(const ResidentPlan& plan);
int resident_build_tables(const Params& P, const ResidentPlan& plan, void* tables_dev, cudaStream_t st);

// nsweeps red-black sweeps of a1: reads psi_in, writes psi_out (two different fields), right-hand side cq * w (w = the
// stage's input vorticity, scaled on the fly exactly as scale_rhs does).  xa, xb: the two exchange buffers (zero-filled once
// by the caller).  tables: what resident_build_tables wrote for this plan (may be null for a single-tile plan).
// err_word: one device word, zero-filled once; non-zero afterwards = a tile gave up waiting for a neighbour.
// *epoch is the host-side tag epoch, advanced by this call (tags are unique per round and per launch).
// trace_dev (profiling only): device array of ntiles x trace_cap %globaltimer stamps (ns), slot 0 = start, 1 = inputs loaded,
// then per round r: 2 + 4r sweeps done, 3 + 4r border strips stored, 4 + 4r ring received, 5 + 4r edges republished.
// Returns the number of kernel launches (1), or a negative cudaError_t.
int resident_sweeps(const Params& P, const ResidentPlan& plan, const double* psi_in, double* psi_out, void* xa, void* xb,
                    const void* tables, const double* w, unsigned int* err_word, unsigned int* epoch, int nsweeps,
                    cudaStream_t st, long long* trace_dev = nullptr, int trace_cap = 0);

}  // namespace cavk
