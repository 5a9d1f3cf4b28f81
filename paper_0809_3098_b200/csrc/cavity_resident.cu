#include "cavity_resident.cuh"

#include <cstdio>

namespace cavk {

ResidentPlan resident_plan(const Params&, int) { return ResidentPlan{}; }
void resident_describe(const ResidentPlan&, char* buf, int len) { std::snprintf(buf, (size_t)len, "none"); }
int resident_sweeps(const Params&, const ResidentPlan&, double*, double*, const double*, unsigned int*, int,
                    cudaStream_t) {
    return -(int)cudaErrorNotSupported;
}

}  // namespace cavk
