// cavity_resident.cuh — the resident sweep engine (a1): one persistent CTA per tile, psi and the scaled
// right-hand side held in registers for all S sweeps of a stage, temporal blocking with a 2T-deep halo that
// is refreshed through L2 every T sweeps under neighbour-flag synchronisation.
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
    int smem_bytes = 0;
    int regs = 0;         // registers per thread of the chosen variant (as compiled)
    int sm_count = 0;
};

// T_override > 0 forces the sweeps per round (tests use it to exercise short and ragged rounds);
// variant_override >= 0 forces the micro-tile shape (index into the compiled variants).
ResidentPlan resident_plan(const Params& P, int device, int T_override = 0, int variant_override = -1);
int resident_variants();
void resident_describe(const ResidentPlan& plan, char* buf, int len);

// Flag words the engine needs (per tile, plus the error word); the caller zero-fills them once.
int resident_flag_words(const ResidentPlan& plan);

// nsweeps red-black sweeps of a1 on psi in place with right-hand side cq * w (w = the stage's input vorticity,
// scaled on the fly exactly as scale_rhs does).  xa, xb: two exchange fields of the same layout as psi.
// flags: resident_flag_words() words; *epoch is the host-side flag epoch, advanced by this call.
// trace_dev (profiling only): device array of ntiles x trace_cap clock64 stamps, slot 0 = start, 1 = inputs loaded,
// then per round r: 2 + 4r computed, 3 + 4r strips posted, 4 + 4r neighbours arrived, 5 + 4r halo reloaded.
// Returns the number of kernel launches (1), or a negative cudaError_t.
int resident_sweeps(const Params& P, const ResidentPlan& plan, double* psi, double* xa, double* xb, const double* w,
                    unsigned int* flags, unsigned int* epoch, int nsweeps, cudaStream_t st,
                    long long* trace_dev = nullptr, int trace_cap = 0);

// 0 if no tile ever timed out waiting for a neighbour (checked by the API after synchronising).
int resident_error_word_index(const ResidentPlan& plan);

}  // namespace cavk
