// cavity_api.cu — the C ABI of include/cavity.h and include/cavity_debug.h: context, step scheduler, host <-> device copies.
//
// PyTorch is used for exactly two things (BASELINE.json north_star): device memory comes from its CUDA
// caching allocator and work is enqueued on its current stream.  No ATen operator does any arithmetic;
// every step of the path runs in the kernels of cavity_kernels.cu / cavity_resident.cu.
// There is no CPU fallback: without a CUDA device cav_create fails with CAV_ECUDA.
#include <c10/cuda/CUDACachingAllocator.h>
#include <c10/cuda/CUDAStream.h>
#include <cuda_runtime.h>
#include <nvtx3/nvToolsExt.h>      // header-only; ranges show up in Nsight timelines, cost nothing otherwise

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>
#include <utility>

#include "../../include/cavity.h"
#include "../../include/cavity_debug.h"
#include "cavity_kernels.cuh"
#include "cavity_resident.cuh"

#define CAV_API extern "C" __attribute__((visibility("default")))

struct cav_ctx {
    int N = 0, S = 0, device = 0;
    double Re = 0, dt = 0, beta = 0;
    cavk::Params P{};
    cudaStream_t st = nullptr;
    void* slab = nullptr;            // one allocation from PyTorch's caching allocator: the fields every engine needs
    double* psi = nullptr;           // stream function (current)
    double* psi2 = nullptr;          // the field the next resident launch / Jacobi sweep writes (then swapped with psi)
    void* xbuf = nullptr;            // resident engine, multi-tile plans: the two exchange buffers (allocated with the plan)
    void* xa = nullptr;              //   ... of even rounds (32-byte units)
    void* xb = nullptr;              //   ... of odd rounds
    double* q = nullptr;             // stream / Jacobi / compact sweeps: scaled right-hand side of the stage (allocated on first use)
    double* w[5] = {nullptr, nullptr, nullptr, nullptr, nullptr};   // omega^n (state), omega^(1..4): consecutive fields, then T
    double* T = nullptr;             // first three terms of eq 13
    double* prev = nullptr;          // NEXT-2 monitors: psi and omega before the monitored step (allocated on first use)
    double* psi_prev = nullptr;
    double* w_prev = nullptr;
    int sweep = CAV_SWEEP_REDBLACK;  // a1 variant
    double* scratch = nullptr;       // diagnostics partials
    double* out4 = nullptr;          // diagnostics result (device)
    unsigned int* err_word = nullptr;// resident engine: device error word (a tile gave up waiting for a neighbour)
    unsigned int epoch = 0;          // resident engine: exchange rounds done so far (host side; the tag of a round derives from it)
    bool resident_ran = false;       // a resident launch has been enqueued since the error word was last cleared
    size_t field_doubles = 0;
    long long step = 0;
    long long launches = 0;
    int forced_T = 0, forced_variant = -1;   // cav_set_resident_plan's request (0 / -1 = the planner's choice); kept across cav_set_sweep
    int engine_req = CAV_ENGINE_AUTO;
    int engine = CAV_ENGINE_STREAM;  // resolved
    cavk::ResidentPlan plan{};       // valid if plan.ok
    cudaGraphExec_t graph = nullptr; // one full time step of the current engine
    long long graph_launches = 0;    // kernel launches inside `graph`
    bool graph_tried = false;
    cudaEvent_t ev0 = nullptr, ev1 = nullptr;
    bool timed = false;
};

namespace {

struct NvtxRange {                 // one range per entry point that enqueues work (tracing)
    explicit NvtxRange(const char* name) { nvtxRangePushA(name); }
    ~NvtxRange() { nvtxRangePop(); }
};

struct DeviceGuard {
    int prev = -1;
    explicit DeviceGuard(int dev) { cudaGetDevice(&prev); if (prev != dev) cudaSetDevice(dev); else prev = -1; }
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

inline bool finite_pos(double x) { return std::isfinite(x) && x > 0.0; }

cavk::Params make_params(int N, double Re, double dt, double beta) {
    cavk::Params P;
    const double U = 1.0;                    // lid speed
    const double h = 1.0 / (double)N;        // uniform grid of the unit square
    P.N = N;
    P.pitch = ((N + 1) + 3) & ~3;
    P.cb = 0.25 * beta;
    P.cq = (0.25 * beta) * (h * h);
    P.omb = 1.0 - beta;
    P.i2h = 0.5 * (double)N;
    P.ih2 = (double)N * (double)N;
    P.nu = 1.0 / Re;
    P.c2h2 = 2.0 * ((double)N * (double)N);
    P.lid = 2.0 * U * (double)N;
    P.dt = dt;
    P.c9e = 0.2 * beta;
    P.c9c = 0.05 * beta;
    P.c9q = (0.025 * beta) * (h * h);
    return P;
}

inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

// CAV_DEBUG=1 in the environment: the CUDA error behind a CAV_ECUDA goes to stderr
inline void debug_cuda(const char* what, int code, int line) {
    static const bool on = std::getenv("CAV_DEBUG") != nullptr;
    if (on) std::fprintf(stderr, "[cavity] line %d: %s -> %s\n", line, what, cudaGetErrorString((cudaError_t)code));
}
#define CK(expr) do { cudaError_t e_ = (expr); if (e_ != cudaSuccess) { debug_cuda(#expr, (int)e_, __LINE__); cudaGetLastError(); return CAV_ECUDA; } } while (0)
#define LAUNCH(expr) do { int n_ = (expr); if (n_ < 0) { debug_cuda(#expr, -n_, __LINE__); cudaGetLastError(); return CAV_ECUDA; } nl += n_; } while (0)

void* dev_alloc(cav_ctx* c, size_t bytes) {
    try { return c10::cuda::CUDACachingAllocator::raw_alloc_with_stream(bytes, c->st); } catch (...) { cudaGetLastError(); return nullptr; }
}
void dev_free(void*& p) {
    if (p) { try { c10::cuda::CUDACachingAllocator::raw_delete(p); } catch (...) {} p = nullptr; }
}

// q: only the stream engine and the Jacobi / compact sweeps need the scaled right-hand side as a field
int need_q(cav_ctx* c) {
    if (c->q) return CAV_OK;
    c->q = (double*)dev_alloc(c, c->field_doubles * sizeof(double));
    if (!c->q) return CAV_ENOMEM;
    if (cudaMemsetAsync(c->q, 0, c->field_doubles * sizeof(double), c->st) != cudaSuccess) { cudaGetLastError(); return CAV_ECUDA; }
    return CAV_OK;
}

void drop_graph(cav_ctx* c) {
    if (c->graph) { cudaGraphExecDestroy(c->graph); c->graph = nullptr; }
    c->graph_tried = false;
    c->graph_launches = 0;
}

// (re)allocates / clears the exchange buffers of c->plan; on failure the plan is marked unusable.  Cleared buffers carry
// tag 0 = never valid, so units of another plan can never be taken for this one's.
void build_plan_buffers(cav_ctx* c) {
    if (!c->plan.ok || c->plan.ntiles <= 1) { dev_free(c->xbuf); c->xa = c->xb = nullptr; return; }
    const size_t xbytes = cavk::resident_exchange_bytes(c->N);
    if (!c->xbuf) c->xbuf = dev_alloc(c, 2 * xbytes);
    if (!c->xbuf) { c->plan.ok = false; return; }
    c->xa = c->xbuf;
    c->xb = (char*)c->xbuf + xbytes;
    if (cudaMemsetAsync(c->xbuf, 0, 2 * xbytes, c->st) != cudaSuccess) { cudaGetLastError(); c->plan.ok = false; return; }
}

// The resident engine's tiles give up (and say so) instead of spinning forever on a neighbour that never arrives.  The word
// is cleared whenever the state or the engine is set anew (cav_set_fields, cav_set_engine, cav_set_resident_plan).
int clear_resident_error(cav_ctx* c) {
    c->resident_ran = false;
    if (!c->err_word) return CAV_OK;
    if (cudaMemsetAsync(c->err_word, 0, sizeof(unsigned int), c->st) != cudaSuccess) { cudaGetLastError(); return CAV_ECUDA; }
    return CAV_OK;
}

void resolve_engine(cav_ctx* c) {
    int e = c->engine_req;
    if (e == CAV_ENGINE_AUTO) e = c->plan.ok ? CAV_ENGINE_RESIDENT : CAV_ENGINE_STREAM;
    if (e != c->engine) { c->engine = e; drop_graph(c); }
}

// the resident kernel runs the red-black sweeps (plan kind 0) and the compact operator's four-colour sweeps (kind 1)
inline int plan_kind(int sweep) { return sweep == CAV_SWEEP_COMPACT9 ? 1 : 0; }
inline bool resident_path(const cav_ctx* c) {
    return c->engine == CAV_ENGINE_RESIDENT && c->sweep != CAV_SWEEP_JACOBI && c->plan.ok && c->plan.kind == plan_kind(c->sweep);
}

// one launch of the resident kernel: nsteps whole time steps, or (nsteps = 0) S sweeps of a1 with right-hand side omega^n
int enqueue_resident(cav_ctx* c, int nsteps, int S, long long& nl, long long* trace_dev = nullptr, int trace_cap = 0) {
    if (nsteps == 0 && S <= 0) return CAV_OK;
    LAUNCH(cavk::resident_launch(c->P, c->plan, c->psi, c->psi2, c->xa, c->xb, c->w[0], c->field_doubles, c->err_word,
                                 &c->epoch, nsteps, S, c->st, trace_dev, trace_cap));
    std::swap(c->psi, c->psi2);
    c->resident_ran = true;
    drop_graph(c);                 // a captured step of another path holds the old psi / psi2
    return CAV_OK;
}

// a1: nsweeps sweeps on psi with right-hand side w_in (every path but the resident kernel's whole steps)
int enqueue_sweeps(cav_ctx* c, const double* w_in, int nsweeps, long long& nl) {
    if (nsweeps <= 0) return CAV_OK;
    if (resident_path(c) && w_in == c->w[0]) return enqueue_resident(c, 0, nsweeps, nl);
    int rc = need_q(c);
    if (rc != CAV_OK) return rc;
    if (c->sweep == CAV_SWEEP_COMPACT9) {
        LAUNCH(cavk::compact_rhs(c->P, w_in, c->q, c->st));
        LAUNCH(cavk::compact_sweeps(c->P, c->psi, c->q, nsweeps, c->st));
    } else if (c->sweep == CAV_SWEEP_JACOBI) {
        LAUNCH(cavk::scale_rhs(c->P, w_in, c->q, c->st));
        LAUNCH(cavk::jacobi_sweeps(c->P, c->psi, c->psi2, c->q, nsweeps, c->st));
    } else {
        LAUNCH(cavk::scale_rhs(c->P, w_in, c->q, c->st));
        LAUNCH(cavk::stream_sweeps(c->P, c->psi, c->q, nsweeps, c->st));
    }
    return CAV_OK;
}

int check_resident_error(cav_ctx* c) {
    if (!c->resident_ran || !c->err_word) return CAV_OK;
    unsigned int e[10] = {0};
    cudaError_t ce = cudaMemcpyAsync(e, c->err_word, sizeof e, cudaMemcpyDeviceToHost, c->st);
    if (ce == cudaSuccess) ce = cudaStreamSynchronize(c->st);
    if (ce != cudaSuccess) { debug_cuda("resident launch", (int)ce, __LINE__); cudaGetLastError(); return CAV_ECUDA; }
    if (e[0] && std::getenv("CAV_DEBUG"))
        std::fprintf(stderr, "[cavity] tile %u thread %u gave up on unit %u (row %u, group %u) in round %u: tag wanted %u, found %u %u %u %u\n",
                     e[1], e[9], e[2], e[2] / (unsigned)cavk::resident_unit_pitch(c->N), e[2] % (unsigned)cavk::resident_unit_pitch(c->N),
                     e[3], e[4], e[5], e[6], e[7], e[8]);
    return e[0] ? CAV_ECUDA : CAV_OK;
}

// one SSPRK(5,4) step, stage by stage: 5 x [a1 x S, a2 + a3] (stream engine, Jacobi and compact sweeps)
int enqueue_step(cav_ctx* c, long long& nl) {
    double* const* w = c->w;
    const double* win[5] = {w[0], w[1], w[2], w[3], w[4]};
    const double* a[5] = {nullptr, w[0], w[0], w[0], c->T};
    const double* b[5] = {nullptr, nullptr, nullptr, w[2], nullptr};
    double* wout[5] = {w[1], w[2], w[3], w[4], w[0]};
    for (int k = 0; k < 5; ++k) {
        int rc = enqueue_sweeps(c, win[k], c->S, nl);
        if (rc != CAV_OK) return rc;
        LAUNCH(cavk::rk_stage(c->P, k + 1, c->psi, win[k], a[k], b[k], wout[k], c->T, c->st));
    }
    return CAV_OK;
}

// Capture one step into a CUDA graph (the stream engine launches 10 S + 10 kernels per step).
void try_build_graph(cav_ctx* c) {
    if (c->graph_tried) return;
    c->graph_tried = true;
    if (resident_path(c)) return;     // whole time steps in one launch
    cudaGraph_t g = nullptr;
    if (cudaStreamBeginCapture(c->st, cudaStreamCaptureModeThreadLocal) != cudaSuccess) { cudaGetLastError(); return; }
    long long nl = 0;
    int rc = enqueue_step(c, nl);
    cudaError_t e = cudaStreamEndCapture(c->st, &g);
    if (rc != CAV_OK || e != cudaSuccess || !g) { cudaGetLastError(); if (g) cudaGraphDestroy(g); return; }
    cudaGraphExec_t ge = nullptr;
    if (cudaGraphInstantiate(&ge, g, 0) == cudaSuccess) { c->graph = ge; c->graph_launches = nl; }
    else cudaGetLastError();
    cudaGraphDestroy(g);
}

int step_impl(cav_ctx* c, int nsteps, bool sync) {
    if (!c || nsteps < 0) return CAV_EINVAL;
    NvtxRange nv("cav_step: SSPRK(5,4) time steps (a1 + a2 + a3)");
    DeviceGuard dg(c->device);
    if (nsteps == 0) return CAV_OK;
    resolve_engine(c);
    if (!resident_path(c)) {           // allocated here, never inside a stream capture
        const int rc = need_q(c);
        if (rc != CAV_OK) return rc;
    }
    try_build_graph(c);
    CK(cudaEventRecord(c->ev0, c->st));
    if (resident_path(c)) {
        long long nl = 0;
        int rc = enqueue_resident(c, nsteps, c->S, nl);
        c->launches += nl;
        if (rc != CAV_OK) return rc;
    } else
    for (int n = 0; n < nsteps; ++n) {
        if (c->graph) {
            CK(cudaGraphLaunch(c->graph, c->st));
            c->launches += c->graph_launches;
        } else {
            long long nl = 0;
            int rc = enqueue_step(c, nl);
            c->launches += nl;
            if (rc != CAV_OK) return rc;
        }
    }
    CK(cudaEventRecord(c->ev1, c->st));
    c->timed = true;
    c->step += nsteps;
    if (sync) {
        CK(cudaStreamSynchronize(c->st));
        return check_resident_error(c);
    }
    return CAV_OK;
}

}  // namespace

CAV_API int cav_create(cav_ctx** out, int N, double Re, double dt, double sor_omega, int sweeps_per_stage) {
    if (!out) return CAV_EINVAL;
    *out = nullptr;
    if (N < 2 || N > 32766 || !finite_pos(Re) || !finite_pos(dt) || !std::isfinite(sor_omega) || !(sor_omega > 0.0) ||
        !(sor_omega < 2.0) || sweeps_per_stage < 0)
        return CAV_EINVAL;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) { cudaGetLastError(); return CAV_ECUDA; }
    cav_ctx* c = new (std::nothrow) cav_ctx();
    if (!c) return CAV_ENOMEM;
    int rc = CAV_OK;
    try {
        if (cudaGetDevice(&c->device) != cudaSuccess) throw (int)CAV_ECUDA;
        c->N = N; c->S = sweeps_per_stage; c->Re = Re; c->dt = dt; c->beta = sor_omega;
        c->P = make_params(N, Re, dt, sor_omega);
        c->st = c10::cuda::getCurrentCUDAStream(c->device).stream();
        c->plan = cavk::resident_plan(c->P, c->device);

        const size_t fd = align_up((size_t)c->P.pitch * (size_t)(N + 1), 32);   // doubles per field, 256 B multiple
        c->field_doubles = fd;
        const size_t nfields = 8;    // psi, psi2, w0..w4, T; q, the monitors' snapshots and the exchange buffers come when needed
        const size_t scratch_d = align_up(4 * (size_t)cavk::diag_scratch_doubles(), 32);
        const size_t flags_b = 256;
        const size_t bytes = (nfields * fd + scratch_d + 32) * sizeof(double) + flags_b;
        c->slab = c10::cuda::CUDACachingAllocator::raw_alloc_with_stream(bytes, c->st);
        if (!c->slab) throw (int)CAV_ENOMEM;
        if (cudaMemsetAsync(c->slab, 0, bytes, c->st) != cudaSuccess) throw (int)CAV_ECUDA;
        double* p = (double*)c->slab;
        c->psi = p; p += fd;
        c->psi2 = p; p += fd;
        for (int k = 0; k < 5; ++k) { c->w[k] = p; p += fd; }      // the resident kernel addresses them as w[0] + k fd
        c->T = p; p += fd;
        c->scratch = p; p += scratch_d;
        c->out4 = p; p += 32;
        c->err_word = (unsigned int*)p;
        if (cudaEventCreate(&c->ev0) != cudaSuccess || cudaEventCreate(&c->ev1) != cudaSuccess) throw (int)CAV_ECUDA;
        if (cudaStreamSynchronize(c->st) != cudaSuccess) throw (int)CAV_ECUDA;
        build_plan_buffers(c);
        resolve_engine(c);
    } catch (int code) {
        rc = code;
    } catch (const std::bad_alloc&) {
        rc = CAV_ENOMEM;
    } catch (const std::exception& ex) {
        // c10 reports out-of-memory and missing-driver conditions as exceptions
        rc = (std::strstr(ex.what(), "out of memory") != nullptr) ? CAV_ENOMEM : CAV_ECUDA;
    } catch (...) {
        rc = CAV_ECUDA;
    }
    if (rc != CAV_OK) { cudaGetLastError(); cav_destroy(c); return rc; }
    *out = c;
    return CAV_OK;
}

CAV_API void cav_destroy(cav_ctx* c) {
    if (!c) return;
    {
        DeviceGuard dg(c->device);
        if (c->st || c->slab) cudaStreamSynchronize(c->st);
        drop_graph(c);
        if (c->ev0) cudaEventDestroy(c->ev0);
        if (c->ev1) cudaEventDestroy(c->ev1);
        if (c->slab) {
            try { c10::cuda::CUDACachingAllocator::raw_delete(c->slab); } catch (...) {}
        }
        dev_free(c->xbuf);
        void* qv = c->q; dev_free(qv); c->q = nullptr;
        void* pv = c->prev; dev_free(pv); c->prev = nullptr;
        cudaGetLastError();
    }
    delete c;
}

CAV_API int cav_set_fields(cav_ctx* c, const double* psi, const double* omega) {
    if (!c || !omega) return CAV_EINVAL;
    DeviceGuard dg(c->device);
    const int N = c->N;
    const size_t row = (size_t)(N + 1) * sizeof(double), dp = (size_t)c->P.pitch * sizeof(double);
    long long nl = 0;
    if (psi) CK(cudaMemcpy2DAsync(c->psi, dp, psi, row, row, N + 1, cudaMemcpyHostToDevice, c->st));
    else CK(cudaMemsetAsync(c->psi, 0, c->field_doubles * sizeof(double), c->st));
    LAUNCH(cavk::zero_ring(c->P, c->psi, c->st));                   // psi = 0 on the walls (eq 23-24)
    CK(cudaMemcpy2DAsync(c->w[0], dp, omega, row, row, N + 1, cudaMemcpyHostToDevice, c->st));
    c->launches += nl;
    c->step = 0;
    int rc = clear_resident_error(c);
    if (rc != CAV_OK) return rc;
    CK(cudaStreamSynchronize(c->st));
    return CAV_OK;
}

CAV_API int cav_get_fields(cav_ctx* c, double* psi_out, double* omega_out) {
    if (!c) return CAV_EINVAL;
    DeviceGuard dg(c->device);
    const int N = c->N;
    const size_t row = (size_t)(N + 1) * sizeof(double), dp = (size_t)c->P.pitch * sizeof(double);
    if (psi_out) CK(cudaMemcpy2DAsync(psi_out, row, c->psi, dp, row, N + 1, cudaMemcpyDeviceToHost, c->st));
    if (omega_out) CK(cudaMemcpy2DAsync(omega_out, row, c->w[0], dp, row, N + 1, cudaMemcpyDeviceToHost, c->st));
    CK(cudaStreamSynchronize(c->st));
    return check_resident_error(c);      // after cav_step_async: fields of a launch whose tile gave up are undefined, say so
}

CAV_API int cav_step(cav_ctx* c, int nsteps) { return step_impl(c, nsteps, true); }
CAV_API int cav_step_async(cav_ctx* c, int nsteps) { return step_impl(c, nsteps, false); }

CAV_API int cav_sync(cav_ctx* c) {
    if (!c) return CAV_EINVAL;
    DeviceGuard dg(c->device);
    CK(cudaStreamSynchronize(c->st));
    return check_resident_error(c);
}

CAV_API int cav_poisson(cav_ctx* c, int nsweeps, double* res_inf_out) {
    if (!c || nsweeps < 0) return CAV_EINVAL;
    NvtxRange nv("cav_poisson: a1 sweeps + a2");
    DeviceGuard dg(c->device);
    resolve_engine(c);
    long long nl = 0;
    CK(cudaEventRecord(c->ev0, c->st));
    int rc = enqueue_sweeps(c, c->w[0], nsweeps, nl);
    if (rc != CAV_OK) { c->launches += nl; return rc; }
    CK(cudaEventRecord(c->ev1, c->st));          // the timed region is the a1 sweeps alone (bench.py's roofline leg)
    c->timed = true;
    LAUNCH(cavk::thom_ring(c->P, c->psi, c->w[0], c->st));
    double r = 0.0;
    if (res_inf_out) {
        LAUNCH(cavk::diagnostics(c->P, c->psi, c->w[0], c->scratch, c->out4, c->st));
        CK(cudaMemcpyAsync(&r, c->out4, sizeof(double), cudaMemcpyDeviceToHost, c->st));
    }
    c->launches += nl;
    CK(cudaStreamSynchronize(c->st));
    if (res_inf_out) *res_inf_out = r;
    return check_resident_error(c);
}

CAV_API int cav_get_diag(cav_ctx* c, cav_diag* out) {
    if (!c || !out) return CAV_EINVAL;
    NvtxRange nv("cav_get_diag: a4 reductions");
    DeviceGuard dg(c->device);
    long long nl = 0;
    double r[4] = {0, 0, 0, 0};
    LAUNCH(cavk::diagnostics(c->P, c->psi, c->w[0], c->scratch, c->out4, c->st));
    c->launches += nl;
    CK(cudaMemcpyAsync(r, c->out4, 4 * sizeof(double), cudaMemcpyDeviceToHost, c->st));
    CK(cudaStreamSynchronize(c->st));
    { const int rc = check_resident_error(c); if (rc != CAV_OK) return rc; }
    out->t = (double)c->step * c->dt;
    out->step = c->step;
    out->res_inf = r[0]; out->res_l2 = r[1]; out->kinetic_energy = r[2]; out->enstrophy = r[3];
    return CAV_OK;
}

CAV_API int cav_set_sweep(cav_ctx* c, int kind) {
    if (!c || kind < CAV_SWEEP_REDBLACK || kind > CAV_SWEEP_COMPACT9) return CAV_EINVAL;
    DeviceGuard dg(c->device);
    CK(cudaStreamSynchronize(c->st));
    if (kind != c->sweep) {
        c->sweep = kind;
        drop_graph(c);
        if (kind != CAV_SWEEP_JACOBI && c->plan.kind != plan_kind(kind)) {       // the halo depth per sweep differs: plan anew
            c->plan = cavk::resident_plan(c->P, c->device, c->forced_T, c->forced_variant, plan_kind(kind));
            if (!c->plan.ok && (c->forced_T != 0 || c->forced_variant >= 0)) {   // no plan with the forced T for this operator: the planner's own
                c->forced_T = 0; c->forced_variant = -1;
                c->plan = cavk::resident_plan(c->P, c->device, 0, -1, plan_kind(kind));
            }
            build_plan_buffers(c);                                               // fresh exchange buffers
            resolve_engine(c);
            return clear_resident_error(c);
        }
    }
    return CAV_OK;
}

CAV_API int cav_step_res(cav_ctx* c, double* res_psi_out, double* res_omega_out) {
    if (!c) return CAV_EINVAL;
    NvtxRange nv("cav_step_res: time step + RES monitors");
    DeviceGuard dg(c->device);
    const size_t nb = c->field_doubles * sizeof(double);
    if (!c->prev) {
        c->prev = (double*)dev_alloc(c, 2 * nb);
        if (!c->prev) return CAV_ENOMEM;
        c->psi_prev = c->prev;
        c->w_prev = c->prev + c->field_doubles;
    }
    CK(cudaMemcpyAsync(c->psi_prev, c->psi, nb, cudaMemcpyDeviceToDevice, c->st));
    CK(cudaMemcpyAsync(c->w_prev, c->w[0], nb, cudaMemcpyDeviceToDevice, c->st));
    int rc = step_impl(c, 1, false);
    if (rc != CAV_OK) return rc;
    long long nl = 0;
    double r[2] = {0.0, 0.0};
    LAUNCH(cavk::res_monitors(c->P, c->psi, c->psi_prev, c->w[0], c->w_prev, c->scratch, c->out4 + 8, c->st));
    c->launches += nl;
    CK(cudaMemcpyAsync(r, c->out4 + 8, 2 * sizeof(double), cudaMemcpyDeviceToHost, c->st));
    CK(cudaStreamSynchronize(c->st));
    if (res_psi_out) *res_psi_out = r[0];
    if (res_omega_out) *res_omega_out = r[1];
    return check_resident_error(c);
}

CAV_API int cav_run_to_steady(cav_ctx* c, int max_steps, int check_every, double tol_psi, double tol_omega, cav_monitor* out) {
    if (!c || max_steps < 0 || check_every < 1 || !out) return CAV_EINVAL;
    out->steps = 0; out->converged = 0; out->res_psi = 0.0; out->res_omega = 0.0;
    int n = 0;
    while (n < max_steps) {
        const int plain = std::min(check_every - 1, max_steps - n);      // steps before the next monitored one
        if (plain > 0) {
            const int rc = step_impl(c, plain, false);
            if (rc != CAV_OK) return rc;
            n += plain;
        }
        if (n >= max_steps) break;
        const int rc = cav_step_res(c, &out->res_psi, &out->res_omega);    // step n + 1 is a multiple of check_every
        if (rc != CAV_OK) return rc;
        ++n;
        if (out->res_psi < tol_psi && out->res_omega < tol_omega) { out->converged = 1; break; }
    }
    out->steps = n;
    DeviceGuard dg(c->device);
    CK(cudaStreamSynchronize(c->st));
    return check_resident_error(c);
}

CAV_API int cav_set_engine(cav_ctx* c, int engine) {
    if (!c || engine < CAV_ENGINE_AUTO || engine > CAV_ENGINE_RESIDENT) return CAV_EINVAL;
    if (engine == CAV_ENGINE_RESIDENT && !c->plan.ok) return CAV_ENOTSUP;
    DeviceGuard dg(c->device);
    CK(cudaStreamSynchronize(c->st));
    c->engine_req = engine;
    resolve_engine(c);
    return clear_resident_error(c);
}

CAV_API int cav_set_resident_plan(cav_ctx* c, int sweeps_per_exchange, int variant) {
    if (!c || sweeps_per_exchange < 0 || variant >= cavk::resident_variants()) return CAV_EINVAL;
    DeviceGuard dg(c->device);
    CK(cudaStreamSynchronize(c->st));
    cavk::ResidentPlan pl = cavk::resident_plan(c->P, c->device, sweeps_per_exchange, variant < 0 ? -1 : variant, plan_kind(c->sweep));
    if (!pl.ok) return CAV_ENOTSUP;
    const cavk::ResidentPlan old = c->plan;
    c->plan = pl;
    build_plan_buffers(c);
    if (!c->plan.ok) { c->plan = old; build_plan_buffers(c); resolve_engine(c); return CAV_ENOMEM; }
    c->forced_T = sweeps_per_exchange;
    c->forced_variant = variant < 0 ? -1 : variant;
    return clear_resident_error(c);
}

CAV_API int cav_trace_sweeps(cav_ctx* c, int nsweeps, long long* stamps_out, int slots_per_tile, int* ntiles_out) {
    if (!c || nsweeps < 1 || !stamps_out || slots_per_tile < 2) return CAV_EINVAL;
    DeviceGuard dg(c->device);
    resolve_engine(c);
    if (!resident_path(c) || c->sweep != CAV_SWEEP_REDBLACK) return CAV_ENOTSUP;   // the red-black sweeps of the resident engine only
    const size_t n = (size_t)c->plan.ntiles * (size_t)slots_per_tile;
    long long* dev = (long long*)dev_alloc(c, n * sizeof(long long));
    if (!dev) return CAV_ENOMEM;
    int rc = CAV_OK;
    if (cudaMemsetAsync(dev, 0, n * sizeof(long long), c->st) != cudaSuccess) rc = CAV_ECUDA;
    if (rc == CAV_OK) {
        long long nl = 0;
        rc = enqueue_resident(c, 0, nsweeps, nl, dev, slots_per_tile);
        c->launches += nl;
    }
    if (rc == CAV_OK && (cudaMemcpyAsync(stamps_out, dev, n * sizeof(long long), cudaMemcpyDeviceToHost, c->st) != cudaSuccess ||
                         cudaStreamSynchronize(c->st) != cudaSuccess)) rc = CAV_ECUDA;
    if (rc != CAV_OK) cudaGetLastError();
    void* dv = dev; dev_free(dv);
    if (ntiles_out) *ntiles_out = c->plan.ntiles;
    return rc == CAV_OK ? check_resident_error(c) : rc;
}

CAV_API int cav_plan_check(int N, int sweep, int T, int sms, int smem_bytes, int* plan_out, long long* counts_out) {
    if (N < 2 || (sweep != CAV_SWEEP_REDBLACK && sweep != CAV_SWEEP_COMPACT9) || T < 0 || sms < 1 || smem_bytes < 1) return CAV_EINVAL;
    const cavk::ResidentPlan pl = cavk::resident_plan_for(N, plan_kind(sweep), T, -1, sms, smem_bytes, 65536);
    if (counts_out) for (int k = 0; k < 5; ++k) counts_out[k] = 0;
    if (!pl.ok) return CAV_ENOTSUP;
    if (plan_out) {
        plan_out[0] = pl.ntx; plan_out[1] = pl.nty; plan_out[2] = pl.CW; plan_out[3] = pl.CH; plan_out[4] = pl.halo;
        plan_out[5] = pl.ntiles > 1 ? pl.T : 0; plan_out[6] = pl.warps; plan_out[7] = pl.smem_bytes; plan_out[8] = pl.EB;
    }
    return cavk::resident_check_exchange(pl, N, counts_out) == 0 ? CAV_OK : CAV_EINVAL;
}

CAV_API int cav_debug_unit_roundtrip(const double* in_host, double* out_host, int nunits, unsigned int tag, int* bad_out) {
    if (!in_host || !out_host || nunits < 1 || tag < 1u || tag > 4095u) return CAV_EINVAL;
    const size_t nb = (size_t)nunits * 4 * sizeof(double), sb = (((size_t)nunits * 16 + 255) / 256 * 256) * 2 + (size_t)nunits * 8 + 256;
    double *din = nullptr, *dout = nullptr;
    void* scratch = nullptr;
    unsigned int* bad = nullptr;
    unsigned int hbad = 0;
    int rc = CAV_OK;
    if (cudaMalloc(&din, nb) != cudaSuccess || cudaMalloc(&dout, nb) != cudaSuccess || cudaMalloc(&scratch, sb) != cudaSuccess ||
        cudaMalloc(&bad, sizeof(unsigned int)) != cudaSuccess) rc = CAV_ECUDA;
    if (rc == CAV_OK && (cudaMemcpy(din, in_host, nb, cudaMemcpyHostToDevice) != cudaSuccess || cudaMemset(scratch, 0, sb) != cudaSuccess ||
                         cudaMemset(bad, 0, sizeof(unsigned int)) != cudaSuccess)) rc = CAV_ECUDA;
    if (rc == CAV_OK && cavk::resident_unit_roundtrip(din, dout, scratch, nunits, tag, bad, 0) < 0) rc = CAV_ECUDA;
    if (rc == CAV_OK && (cudaMemcpy(out_host, dout, nb, cudaMemcpyDeviceToHost) != cudaSuccess ||
                         cudaMemcpy(&hbad, bad, sizeof(unsigned int), cudaMemcpyDeviceToHost) != cudaSuccess)) rc = CAV_ECUDA;
    if (rc != CAV_OK) cudaGetLastError();
    cudaFree(din); cudaFree(dout); cudaFree(scratch); cudaFree(bad);
    if (bad_out) *bad_out = (int)hbad;
    return rc;
}

CAV_API int cav_debug_set_epoch(cav_ctx* c, unsigned int epoch) {
    if (!c) return CAV_EINVAL;
    DeviceGuard dg(c->device);
    CK(cudaStreamSynchronize(c->st));
    // a jump of the round counter breaks the "this round or the one two before" invariant of the tags: start from cleared buffers
    if (c->xbuf) CK(cudaMemsetAsync(c->xbuf, 0, 2 * cavk::resident_exchange_bytes(c->N), c->st));
    c->epoch = epoch;
    return CAV_OK;
}

CAV_API int cav_measure_fp64_peak(cav_ctx* c, double* dfma_per_s_out, double* sm_clock_mhz_out) {
    if (!c || !dfma_per_s_out) return CAV_EINVAL;
    DeviceGuard dg(c->device);
    int sms = 0, khz = 0;
    CK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, c->device));
    CK(cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, c->device));
    const int blocks = sms;                                         // one CTA of 16 warps per SM, like the resident engine
    double* sink = (double*)dev_alloc(c, (size_t)blocks * 512 * sizeof(double));
    if (!sink) return CAV_ENOMEM;
    int rc = CAV_OK;
    double per_thread = 0.0, best_ms = 1e30;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) rc = CAV_ECUDA;
    for (int rep = 0; rc == CAV_OK && rep < 6; ++rep) {             // the first two warm up; best of the rest
        cudaEventRecord(e0, c->st);
        const int nl = cavk::fp64_peak(blocks, 4000, sink, c->st, &per_thread);
        cudaEventRecord(e1, c->st);
        if (nl < 0 || cudaEventSynchronize(e1) != cudaSuccess) { rc = CAV_ECUDA; break; }
        c->launches += nl;
        float ms = 0.0f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (rep >= 2 && ms < best_ms) best_ms = ms;
    }
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    void* sv = sink; dev_free(sv);
    if (rc != CAV_OK) { cudaGetLastError(); return rc; }
    *dfma_per_s_out = per_thread * 512.0 * blocks / (best_ms * 1e-3);
    if (sm_clock_mhz_out) *sm_clock_mhz_out = khz / 1000.0;
    return CAV_OK;
}

CAV_API int cav_describe(cav_ctx* c, char* buf, int len) {
    if (!c || !buf || len < 1) return CAV_EINVAL;
    resolve_engine(c);
    std::string s;
    char tmp[512];
    std::snprintf(tmp, sizeof tmp, "grid %dx%d pitch %d S %d engine %s", c->N + 1, c->N + 1, c->P.pitch, c->S,
                  c->engine == CAV_ENGINE_RESIDENT ? "resident" : "stream");
    s = tmp;
    if (c->plan.ok) { cavk::resident_describe(c->plan, tmp, sizeof tmp); s += " | resident plan: "; s += tmp; }
    else s += " | resident plan: unavailable";
    std::snprintf(buf, (size_t)len, "%s", s.c_str());
    return CAV_OK;
}

CAV_API long long cav_launch_count(cav_ctx* c) { return c ? c->launches : 0; }

CAV_API int cav_last_elapsed_ms(cav_ctx* c, float* ms_out) {
    if (!c || !ms_out) return CAV_EINVAL;
    *ms_out = 0.0f;
    if (!c->timed) return CAV_OK;
    DeviceGuard dg(c->device);
    CK(cudaEventSynchronize(c->ev1));
    CK(cudaEventElapsedTime(ms_out, c->ev0, c->ev1));
    return CAV_OK;
}

CAV_API const char* cav_strerror(int code) {
    switch (code) {
        case CAV_OK: return "ok";
        case CAV_EINVAL: return "invalid argument";
        case CAV_ENOMEM: return "out of memory";
        case CAV_ECUDA: return "CUDA error or no usable CUDA device";
        case CAV_ENOTSUP: return "engine not supported for this problem on this device";
        case CAV_ELIMIT: return "problem larger than a fixed-size buffer of the library (cav_diag_noalloc: N > CAV_NOALLOC_MAX_N = 8192)";
        default: return "unknown error";
    }
}
