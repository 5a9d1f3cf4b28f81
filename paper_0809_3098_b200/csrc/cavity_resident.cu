// cavity_resident.cu — the resident sweep engine (a1) for sm_100a.  DESIGN.md "Resident engine".
//
// What it computes is exactly S red-black SOR sweeps of the 5-point Poisson problem (eq 15-21 P:114-138 reduced,
// DESIGN.md D1-D3), red = (i + j) even first (G9), with the arithmetic of DESIGN.md "Canonical arithmetic":
//     nb = (psi_W + psi_E) + (psi_S + psi_N);   psi <- fma(1 - beta, psi, fma(beta / 4, nb, q)),   q = ((beta / 4) h^2) w
// Inside one colour every update reads only the other colour, so the schedule below cannot change a bit of
// the result; the tests compare with the FMA-mode oracle bit for bit.
//
// Schedule.  The (N+1)^2 grid is cut into ntx x nty tiles; tile (bi, bj) OWNS the core [bi CW, (bi+1) CW) x
// [bj CH, (bj+1) CH) and additionally carries a halo of `halo` = 2T points on every side.  One CTA per tile,
// all CTAs co-resident (cooperative launch).  A thread owns a C x R micro-tile (C consecutive x, R rows) of
// psi AND q in registers for the whole call; a warp spans 32 C points of R rows.  Threads exchange only the
// perimeter of their micro-tile: left / right columns by warp shuffle, bottom / top rows through shared memory
// (edge arrays laid out so that every access is unit-stride over the lanes), one __syncthreads per colour half-sweep.
// Every T sweeps (2T half-sweeps, each of which invalidates one more ring of the halo) the CTAs refresh their
// halos through L2: write the 2T-wide border strips of the core to an exchange field, release a per-tile flag,
// acquire the flags of the up to 8 neighbours, reload the halo (ld.global.cg: L1 is not coherent).  Two
// exchange fields alternate, so a tile can run at most one round ahead of a neighbour without a hazard.
// Points on a wall are forced back to +0.0 after every half-sweep by the (few) threads that own any; points
// outside the walls have only zero inputs and therefore stay +0.0 by themselves.
#include "cavity_resident.cuh"

#include <algorithm>
#include <cstdio>

namespace cavk {

namespace {

constexpr long long SPIN_TIMEOUT_CYCLES = 4000000000LL;   // ~2 s: a neighbour that never arrives is a bug, not a wait

struct ResArgs {
    int N, pitch;
    double cb, omb, cq;
    const double* w;        // stage input vorticity; q = cq * w on interior points
    double* psi;            // in / out
    double* x0;             // exchange field of even rounds
    double* x1;             // exchange field of odd rounds
    unsigned int* flags;    // one word per tile (monotonic event counter) ...
    unsigned int* err;      // ... and the error word
    unsigned int base;      // flag epoch of this launch
    int nsweeps, T, halo, CW, CH, ntx, nty;
    long long* trace;       // profiling only (cav_trace_sweeps): per tile, clock64 at the phase boundaries; else null
    int trace_cap;          // slots per tile
};

__device__ __forceinline__ unsigned int ld_relaxed(const unsigned int* p) {
    unsigned int v;
    asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_release(unsigned int* p, unsigned int v) {
    asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

// All threads' earlier global stores -> visible to whoever acquires flag >= v.
__device__ __forceinline__ void post(unsigned int* flag, unsigned int v) {
    __syncthreads();
    if (threadIdx.x == 0 && threadIdx.y == 0) st_release(flag, v);     // release = fence + store: cumulative over the barrier
}

// Waits until each existing neighbour tile has posted event >= v.  Threads 0..7 of warp 0 take one direction each.
__device__ __forceinline__ void wait_neighbours(const ResArgs& a, int bi, int bj, unsigned int v) {
    if (threadIdx.y == 0 && threadIdx.x < 8) {
        const int d = threadIdx.x < 4 ? threadIdx.x : threadIdx.x + 1;     // 0..8 without the centre (4)
        const int ni = bi + d % 3 - 1, nj = bj + d / 3 - 1;
        if (ni >= 0 && ni < a.ntx && nj >= 0 && nj < a.nty && *(volatile unsigned int*)a.err == 0u) {
            const unsigned int* f = a.flags + (nj * a.ntx + ni);
            const long long t0 = clock64();
            while ((int)(ld_relaxed(f) - v) < 0) {
                if (clock64() - t0 > SPIN_TIMEOUT_CYCLES) { atomicExch(a.err, 1u); break; }
            }
        }
        __threadfence();      // one acquire fence after the relaxed polls; the barrier extends it to the CTA
    }
    __syncthreads();
}

// One colour half-sweep on the register micro-tile.  K = colour being updated; local point (ci, rj) has colour
// (ci + rj) & 1 because every tile origin is even in x and y and C, R are even (resident_plan guarantees it).
// Left / right neighbours live in the adjacent lanes and come by warp shuffle (no barrier, no shared memory);
// the rows above / below live in the adjacent warps and come through the sB / sT edge arrays.
// wallmask: bit rj * C + ci set = that point lies ON a wall and is put back to +0.0 after the update
// (eq 23-24).  Points outside the walls need nothing: all their inputs are 0, so they stay +0.0.
template <int C, int R, int K>
__device__ __forceinline__ void half_sweep(double (&p)[R][C], const double (&q)[R][C], const double cb, const double omb,
                                           double* __restrict__ sB, double* __restrict__ sT, const unsigned int wallmask,
                                           const int lane) {
    // sB / sT point at [warp][0][lane] of the bottom / top edge arrays (stride 32 per ci, C * 32 per warp)
    double Lnb[R], Rnb[R], Bnb[C], Tnb[C];
#pragma unroll
    for (int ci = 0; ci < C; ++ci) {
        if ((ci & 1) == K) Bnb[ci] = sT[ci * 32];                          // top row of the warp below (slot warp)
        if (((ci + R - 1) & 1) == K) Tnb[ci] = sB[C * 32 + ci * 32];       // bottom row of the warp above (slot warp + 1)
    }
#pragma unroll
    for (int rj = 0; rj < R; ++rj) {
        if ((rj & 1) == K) {                                               // right edge of lane - 1; nothing left of lane 0
            const double v = __shfl_up_sync(0xffffffffu, p[rj][C - 1], 1);
            Lnb[rj] = lane == 0 ? 0.0 : v;
        }
        if (((C - 1 + rj) & 1) == K) {                                     // left edge of lane + 1; nothing right of lane 31
            const double v = __shfl_down_sync(0xffffffffu, p[rj][0], 1);
            Rnb[rj] = lane == 31 ? 0.0 : v;
        }
    }
#pragma unroll
    for (int rj = 0; rj < R; ++rj) {
#pragma unroll
        for (int ci = 0; ci < C; ++ci) {
            if (((ci + rj) & 1) != K) continue;
            const double pW = ci > 0 ? p[rj][ci - 1] : Lnb[rj];
            const double pE = ci < C - 1 ? p[rj][ci + 1] : Rnb[rj];
            const double pS = rj > 0 ? p[rj - 1][ci] : Bnb[ci];
            const double pN = rj < R - 1 ? p[rj + 1][ci] : Tnb[ci];
            const double nb = (pW + pE) + (pS + pN);
            p[rj][ci] = fma(omb, p[rj][ci], fma(cb, nb, q[rj][ci]));
        }
    }
    unsigned int wm = wallmask;
    asm volatile("" : "+r"(wm));      // opaque: keeps the bit tests from being hoisted into live registers
    if (wm) {
#pragma unroll
        for (int ci = 0; ci < C; ++ci) {
            unsigned int colbits = 0;                                      // the points of column ci with colour K
#pragma unroll
            for (int rj = 0; rj < R; ++rj)
                if (((ci + rj) & 1) == K) colbits |= 1u << (rj * C + ci);
            if (wm & colbits) {
#pragma unroll
                for (int rj = 0; rj < R; ++rj)
                    if (((ci + rj) & 1) == K && ((wm >> (rj * C + ci)) & 1u)) p[rj][ci] = 0.0;
            }
        }
    }
    // publish the updated points of the bottom and top rows
#pragma unroll
    for (int ci = 0; ci < C; ++ci) {
        if ((ci & 1) == K) sB[ci * 32] = p[0][ci];
        if (((ci + R - 1) & 1) == K) sT[C * 32 + ci * 32] = p[R - 1][ci];
    }
    __syncthreads();
}

template <int C, int R>
__device__ __forceinline__ void publish_all(const double (&p)[R][C], double* __restrict__ sB, double* __restrict__ sT) {
#pragma unroll
    for (int ci = 0; ci < C; ++ci) { sB[ci * 32] = p[0][ci]; sT[C * 32 + ci * 32] = p[R - 1][ci]; }
    __syncthreads();
}

__device__ __forceinline__ void load4(const double* __restrict__ g, double (&v)[4], bool cg) {
    const double2* g2 = reinterpret_cast<const double2*>(g);
    double2 a, b;
    if (cg) { a = __ldcg(g2); b = __ldcg(g2 + 1); } else { a = g2[0]; b = g2[1]; }
    v[0] = a.x; v[1] = a.y; v[2] = b.x; v[3] = b.y;
}
__device__ __forceinline__ void store4(double* __restrict__ g, const double (&v)[4]) {
    double2* g2 = reinterpret_cast<double2*>(g);
    g2[0] = make_double2(v[0], v[1]);
    g2[1] = make_double2(v[2], v[3]);
}

__device__ __forceinline__ void mark(const ResArgs& a, int tile, int slot) {
    if (a.trace != nullptr && threadIdx.x == 0 && threadIdx.y == 0 && slot < a.trace_cap)
        a.trace[(size_t)tile * a.trace_cap + slot] = clock64();
}

// MAXW = most warps per CTA this variant is launched with: 65536 / (32 MAXW) registers per thread are available.
template <int C, int R, int MAXW>
__global__ void __launch_bounds__(32 * MAXW, 1) k_resident(const ResArgs a) {
    static_assert(C == 4, "vector loads below assume 4 consecutive x-points per thread");
    static_assert(R % 2 == 0 && R * C <= 32, "R must be even and the micro-tile must fit the 32-bit wall mask");
    extern __shared__ double sm[];
    const int lane = threadIdx.x, warp = threadIdx.y, nwarps = blockDim.y;
    const int tid = warp * 32 + lane, nthreads = nwarps * 32;
    const int N = a.N, pitch = a.pitch;

    // edge arrays; the slots no thread ever writes (warp -1, warp nwarps) stay 0
    double* const sBa = sm;                                   // [nwarps + 1][C][32]  bottom row of warp at [warp]
    double* const sTa = sBa + (nwarps + 1) * C * 32;          // [nwarps + 1][C][32]  top row of warp at [warp + 1]
    const int smem_doubles = 2 * (nwarps + 1) * C * 32;
    for (int k = tid; k < smem_doubles; k += nthreads) sm[k] = 0.0;
    double* const sB = sBa + warp * C * 32 + lane;
    double* const sT = sTa + warp * C * 32 + lane;

    const int bi = blockIdx.x, bj = blockIdx.y;
    const int cx0 = bi * a.CW, cy0 = bj * a.CH;
    const int cx1 = min(cx0 + a.CW, N + 1), cy1 = min(cy0 + a.CH, N + 1);
    const int gx0 = cx0 - a.halo + lane * C;       // multiple of 4: 32-byte aligned in every device row
    const int gy0 = cy0 - a.halo + warp * R;       // even
    const bool x_in = gx0 >= 0 && gx0 <= N;        // chunk [gx0, gx0 + 4) lies inside the padded device row
    const bool x_core = gx0 >= cx0 && gx0 < cx1;

    const int tile = bj * a.ntx + bi;
    mark(a, tile, 0);
    double p[R][C], q[R][C];
    unsigned int wallmask = 0;            // points ON a wall (psi = 0 there, eq 23-24)
#pragma unroll
    for (int rj = 0; rj < R; ++rj) {
        const int gy = gy0 + rj;
        const bool in = x_in && gy >= 0 && gy <= N;
        double pv[4] = {0.0, 0.0, 0.0, 0.0}, wv[4] = {0.0, 0.0, 0.0, 0.0};
        if (in) {
            load4(a.psi + (size_t)gy * pitch + gx0, pv, false);
            load4(a.w + (size_t)gy * pitch + gx0, wv, false);
        }
#pragma unroll
        for (int ci = 0; ci < C; ++ci) {
            const int gx = gx0 + ci;
            const bool upd = gx >= 1 && gx <= N - 1 && gy >= 1 && gy <= N - 1;
            p[rj][ci] = upd ? pv[ci] : 0.0;
            q[rj][ci] = upd ? a.cq * wv[ci] : 0.0;
            const bool wall = gx >= 0 && gx <= N && gy >= 0 && gy <= N && !upd;
            if (wall) wallmask |= 1u << (rj * C + ci);
        }
    }
    __syncthreads();                      // the zero fill of the edge arrays is complete
    publish_all<C, R>(p, sB, sT);

    const bool multi = a.ntx * a.nty > 1;
    unsigned int ev = a.base + 1;
    if (multi) post(a.flags + tile, ev);  // event base + 1: this tile has read its inputs from psi
    mark(a, tile, 1);

    const int T = a.T;
    const int nrounds = (a.nsweeps + T - 1) / T;
    for (int r = 0; r < nrounds; ++r) {
        const int ns = min(T, a.nsweeps - r * T);
        for (int s = 0; s < ns; ++s) {
            half_sweep<C, R, 0>(p, q, a.cb, a.omb, sB, sT, wallmask, lane);     // red = (i + j) even first (G9)
            half_sweep<C, R, 1>(p, q, a.cb, a.omb, sB, sT, wallmask, lane);
        }
        mark(a, tile, 2 + 4 * r);
        if (r == nrounds - 1) break;
        // ---- halo exchange through L2 ----
        double* const xb = (r & 1) ? a.x1 : a.x0;
#pragma unroll
        for (int rj = 0; rj < R; ++rj) {
            const int gy = gy0 + rj;
            if (x_core && gy >= cy0 && gy < cy1) {
                const bool strip = gy < cy0 + a.halo || gy >= cy1 - a.halo || gx0 < cx0 + a.halo || gx0 + C > cx1 - a.halo;
                if (strip) store4(xb + (size_t)gy * pitch + gx0, p[rj]);
            }
        }
        ev += 1;
        post(a.flags + tile, ev);
        mark(a, tile, 3 + 4 * r);
        wait_neighbours(a, bi, bj, ev);
        mark(a, tile, 4 + 4 * r);
        // Reload the ring.  What arrives is final as it stands: the owners keep wall points and the padding columns at +0.0.
        // Loads go straight into the micro-tile registers, so all of a thread's rows are in flight together.
        {
            const bool xr = x_in && gx0 >= cx0 - a.halo && gx0 < cx1 + a.halo;
#pragma unroll
            for (int rj = 0; rj < R; ++rj) {
                const int gy = gy0 + rj;
                const bool core = x_core && gy >= cy0 && gy < cy1;
                const bool ring = xr && !core && gy >= 0 && gy <= N && gy >= cy0 - a.halo && gy < cy1 + a.halo;
                if (ring) load4(xb + (size_t)gy * pitch + gx0, p[rj], true);
            }
        }
        publish_all<C, R>(p, sB, sT);
        mark(a, tile, 5 + 4 * r);
    }

    // every neighbour has read its halo of the INPUT psi before this tile overwrites its core
    if (multi) wait_neighbours(a, bi, bj, a.base + 1);
#pragma unroll
    for (int rj = 0; rj < R; ++rj) {
        const int gy = gy0 + rj;
        if (x_core && gy >= cy0 && gy < cy1) store4(a.psi + (size_t)gy * pitch + gx0, p[rj]);
    }
}

// ---- compiled variants ------------------------------------------------------------------------------
struct Variant {
    int C, R, maxw;
    const void* fn;
};
const Variant VARIANTS[] = {
    {4, 8, 12, (const void*)k_resident<4, 8, 12>},     // 32 points per thread, up to 170 registers
    {4, 6, 16, (const void*)k_resident<4, 6, 16>},     // 24 points per thread, up to 128 registers
};
constexpr int NVARIANTS = sizeof(VARIANTS) / sizeof(VARIANTS[0]);

int smem_bytes_for(int C, int R, int warps) {
    (void)R;
    return (int)sizeof(double) * (2 * (warps + 1) * C * 32);
}

inline int cdiv(int a, int b) { return (a + b - 1) / b; }
inline int round_up(int a, int m) { return cdiv(a, m) * m; }

}  // namespace

ResidentPlan resident_plan(const Params& P, int device, int T_override, int variant_override) {
    ResidentPlan best;
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) { cudaGetLastError(); return best; }
    int coop = 0;
    cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, device);
    if (!coop) return best;
    const int sms = prop.multiProcessorCount;
    const int G = P.N + 1;                       // points per side, walls included
    double best_cost = 1e300;

    for (int vi = 0; vi < NVARIANTS; ++vi) {
        if (variant_override >= 0 && vi != variant_override) continue;
        const Variant& v = VARIANTS[vi];
        cudaFuncAttributes fa;
        if (cudaFuncGetAttributes(&fa, v.fn) != cudaSuccess) { cudaGetLastError(); continue; }
        const int max_warps = std::min(v.maxw, std::min(fa.maxThreadsPerBlock / 32, (int)(prop.regsPerBlock / (32 * std::max(fa.numRegs, 1)))));
        const int W = 32 * v.C;                  // tile width in points
        for (int warps = 1; warps <= max_warps; ++warps) {
            const int H = warps * v.R;           // tile height in points
            const int smem = smem_bytes_for(v.C, v.R, warps);
            if (smem > (int)prop.sharedMemPerBlockOptin) continue;
            // single tile: the whole grid in one CTA, no exchange at all
            if (G <= W && G <= H) {
                const double cost = (double)H * W * 0.11 + 150.0;
                if (cost < best_cost) {
                    best_cost = cost;
                    best = ResidentPlan{};
                    best.ok = true; best.variant = vi; best.C = v.C; best.R = v.R; best.warps = warps;
                    best.T = 1 << 30; best.halo = 0; best.CW = round_up(G, v.C); best.CH = round_up(G, 2);
                    best.ntx = best.nty = best.ntiles = 1; best.smem_bytes = smem; best.regs = fa.numRegs; best.sm_count = sms;
                }
                continue;
            }
            for (int T = 2; T <= 16; T += 2) {   // halo = 2T must be a multiple of C = 4 (chunks never straddle the core edge)
                if (T_override > 0 && T != T_override) continue;
                const int halo = 2 * T;
                // x: either one tile column without an x-halo, or columns of CW <= W - 2 halo
                int CW, ntx;
                if (G + halo <= W) { CW = round_up(G, v.C); ntx = 1; }          // origin is -halo: [0, G) must still fit
                else {
                    const int cwmax = W - 2 * halo;
                    if (cwmax < halo || cwmax < v.C) continue;
                    ntx = cdiv(G, cwmax);
                    CW = round_up(cdiv(G, ntx), v.C);
                    if (CW > cwmax) continue;
                    ntx = cdiv(G, CW);
                    if (G - (ntx - 1) * CW < halo || CW < halo) continue;     // the halo must come from adjacent tiles only
                }
                int CH, nty;
                if (G + halo <= H) { CH = round_up(G, 2); nty = 1; }
                else {
                    const int chmax = H - 2 * halo;
                    if (chmax < halo || chmax < 2) continue;
                    nty = cdiv(G, chmax);
                    CH = round_up(cdiv(G, nty), 2);
                    if (CH > chmax) continue;
                    nty = cdiv(G, CH);
                    if (G - (nty - 1) * CH < halo || CH < halo) continue;
                }
                if (ntx * nty > sms) continue;
                // cost per sweep in SM cycles: shared-memory-bound compute of the whole tile + two barriers + exchange / T
                const double cost = (double)H * W * 0.11 + 150.0 + 3000.0 / T;
                if (cost < best_cost) {
                    best_cost = cost;
                    best = ResidentPlan{};
                    best.ok = true; best.variant = vi; best.C = v.C; best.R = v.R; best.warps = warps;
                    best.T = T; best.halo = halo; best.CW = CW; best.CH = CH; best.ntx = ntx; best.nty = nty;
                    best.ntiles = ntx * nty; best.smem_bytes = smem; best.regs = fa.numRegs; best.sm_count = sms;
                }
            }
        }
    }
    if (best.ok) {
        const Variant& v = VARIANTS[best.variant];
        if (cudaFuncSetAttribute(v.fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)prop.sharedMemPerBlockOptin) != cudaSuccess) {
            cudaGetLastError();
            best.ok = false;
            return best;
        }
        int per_sm = 0;
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, v.fn, 32 * best.warps, best.smem_bytes) != cudaSuccess ||
            per_sm * sms < best.ntiles) {
            cudaGetLastError();
            best.ok = false;
        }
    }
    return best;
}

void resident_describe(const ResidentPlan& pl, char* buf, int len) {
    if (!pl.ok) { std::snprintf(buf, (size_t)len, "none"); return; }
    if (pl.ntiles == 1)
        std::snprintf(buf, (size_t)len, "1 tile, %d warps x (%dx%d micro-tiles), all sweeps on chip, %d regs, %d B smem",
                      pl.warps, pl.C, pl.R, pl.regs, pl.smem_bytes);
    else
        std::snprintf(buf, (size_t)len,
                      "%dx%d tiles of %dx%d core + halo %d, T=%d sweeps per exchange, %d warps x (%dx%d micro-tiles), "
                      "%d regs, %d B smem, %d SMs",
                      pl.ntx, pl.nty, pl.CW, pl.CH, pl.halo, pl.T, pl.warps, pl.C, pl.R, pl.regs, pl.smem_bytes, pl.sm_count);
}

int resident_variants() { return NVARIANTS; }

int resident_flag_words(const ResidentPlan& plan) { return (plan.ok ? plan.ntiles : 0) + 1; }
int resident_error_word_index(const ResidentPlan& plan) { return plan.ok ? plan.ntiles : 0; }

int resident_sweeps(const Params& P, const ResidentPlan& pl, double* psi, double* xa, double* xb, const double* w,
                    unsigned int* flags, unsigned int* epoch, int nsweeps, cudaStream_t st, long long* trace_dev,
                    int trace_cap) {
    if (!pl.ok) return -(int)cudaErrorNotSupported;
    if (nsweeps <= 0) return 0;
    ResArgs a;
    a.N = P.N; a.pitch = P.pitch; a.cb = P.cb; a.omb = P.omb; a.cq = P.cq;
    a.w = w; a.psi = psi; a.x0 = xa; a.x1 = xb;
    a.flags = flags; a.err = flags + resident_error_word_index(pl);
    a.base = *epoch;
    a.nsweeps = nsweeps;
    a.T = pl.ntiles == 1 ? nsweeps : pl.T;
    a.halo = pl.halo; a.CW = pl.CW; a.CH = pl.CH; a.ntx = pl.ntx; a.nty = pl.nty;
    a.trace = trace_dev; a.trace_cap = trace_cap;
    const int nrounds = (nsweeps + a.T - 1) / a.T;
    *epoch += (unsigned int)nrounds + 1u;           // events base + 1 .. base + nrounds are used by this launch
    void* args[] = {&a};
    const dim3 grid(pl.ntx, pl.nty), block(32, pl.warps);
    const cudaError_t e = cudaLaunchCooperativeKernel(VARIANTS[pl.variant].fn, grid, block, args, (size_t)pl.smem_bytes, st);
    if (e != cudaSuccess) { cudaGetLastError(); return -(int)e; }
    return 1;
}

}  // namespace cavk
