// cavity_resident.cuh — the resident sweep engine (a1): persistent tiles, psi in registers, temporal blocking.
// See DESIGN.md "Resident engine".  Plain CUDA: no torch types.
#pragma once
#include <cuda_runtime.h>

#include "cavity_kernels.cuh"

namespace cavk {

struct ResidentPlan {
    bool ok = false;      // false: this grid / device cannot use the resident engine
    int ntiles = 0;
};

ResidentPlan resident_plan(const Params& P, int device);
void resident_describe(const ResidentPlan& plan, char* buf, int len);

// nsweeps red-black sweeps of a1 on psi (result left in psi), right-hand side q (already scaled).
int resident_sweeps(const Params& P, const ResidentPlan& plan, double* psi, double* psi_alt, const double* q,
                    unsigned int* flags, int nsweeps, cudaStream_t st);

}  // namespace cavk
