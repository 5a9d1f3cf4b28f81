// cavity_resident.cu — the resident sweep engine (a1) for sm_100a.  DESIGN.md section 6.
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
//
// Walls cost nothing inside the sweeps.  The origin of an edge tile is shifted so that the wall column x = 0 is the LAST
// column of a lane (x = N: the FIRST column of a lane) and the wall row y = 0 the LAST row of a warp (y = N: the FIRST row
// of a warp).  Such a lane / warp owns no interior point; what it computes is never used: the adjacent lane substitutes
// 0 for what the shuffle brings (the select that the tile edge needs anyway), and the warp never publishes that edge row,
// so the shared-memory slot keeps the +0.0 it was initialised with (eq 23-24: psi = 0 on the walls).  A tile
// whose origin parity is odd sweeps its local colour 1 first.  Walls that cannot be aligned (both walls of one direction in
// the same tile: small grids) fall back to a bit mask of points that are put back to +0.0 after every half-sweep.
//
// Every T sweeps (2T half-sweeps, each of which invalidates one more ring of the halo) the CTAs refresh their
// halos through L2 WITHOUT any fence, flag or barrier between CTAs: the validity tag travels inside the data.
// A point is exchanged as one 16-byte unit {lo32(psi), tag, hi32(psi), tag} written by one st.v4.b32; each 8-byte half is
// a single-copy-atomic access carrying its own tag, so a reader that finds both tags equal to the tag of the round it waits
// for holds the two halves of that round's value, however the stores of the sender were ordered or torn.  Tags are unique
// per round and per launch (a host-side epoch).  Two exchange buffers alternate by round parity: a tile can write round
// r + 1 only after it has received round r from every neighbour, and a neighbour posts round r only after it has consumed
// round r - 1, so the buffer a tile overwrites is never still being read.
// The exchange is cooperative and coalesced: owners put the border-strip values into a shared-memory staging array, then
// ALL threads of the CTA store the strip units (consecutive threads = consecutive x) and fetch the ring units the same
// way (a few units per thread, all in flight together; a unit that does not carry the tag yet is polled), and the owners
// pick the ring values up from the staging array.  Which unit a thread moves is precomputed once per launch into
// shared-memory tables.
// The kernel reads psi_in and writes psi_out (the API ping-pongs two fields), so no tile ever overwrites input a
// neighbour has not loaded yet.
#include "cavity_resident.cuh"

#include <algorithm>
#include <cstdio>

namespace cavk {

namespace {

constexpr long long SPIN_TIMEOUT_CYCLES = 4000000000LL;   // ~2 s: a neighbour whose data never arrives is a bug, not a wait
constexpr unsigned int NO_UNIT = 0xffffffffu;
#ifndef CAV_QROWS
#define CAV_QROWS 2             // rows of the micro-tile whose q lives in shared memory instead of registers
#endif
#ifndef CAV_RECV_BATCH
#define CAV_RECV_BATCH 2        // ring units a thread keeps in flight at a time (4 registers each; more than 2 makes ptxas spill around the exchange, which costs more than the extra L2 round trips: profiles/)
#endif

struct ResArgs {
    int N, pitch;
    double cb, omb, cq;
    const double* w;        // stage input vorticity; q = cq * w on interior points
    const double* psi_in;   // stream function before the sweeps
    double* psi_out;        // ... and after (a different field)
    uint4* x0;              // exchange buffer of even rounds: one 16-byte unit per grid point, same (pitch) indexing as a field
    uint4* x1;              // exchange buffer of odd rounds
    unsigned int* err;      // error word: set if a tile gave up waiting for a neighbour
    unsigned int base;      // tag epoch of this launch: round r is tagged base + 1 + r
    int nsweeps, T, halo, CW, CH, ntx, nty;
    int ns_per, nr_per;     // table entries per thread: strip units to store / ring units to fetch
    const uint4* tables;    // per-plan exchange tables, one block per tile (k_build_tables)
    long long* trace;       // profiling only (cav_trace_sweeps): per tile, %globaltimer at the phase boundaries; else null
    int trace_cap;          // slots per tile
};

// Geometry of tile (bi, bj): owned core, origin of the thread grid, wall alignment.  Shared by the planner (host) and the
// kernel so that both agree on what fits.
struct TileGeom {
    int cx0, cx1, cy0, cy1;        // core [cx0, cx1) x [cy0, cy1)
    int ox, oy;                    // grid coordinates of local point (0, 0)
    bool left_al, right_al, bot_al, top_al;   // wall isolated in a lane / warp that owns no interior point
    bool fits;                     // the W x H thread grid covers core + halo (clipped to the grid) and the aligned walls
};

__host__ __device__ inline TileGeom tile_geom(int N, int CW, int CH, int halo, int ntx, int nty, int bi, int bj, int C, int R,
                                              int W, int H) {
    TileGeom g;
    g.cx0 = bi * CW; g.cy0 = bj * CH;
    g.cx1 = g.cx0 + CW < N + 1 ? g.cx0 + CW : N + 1;
    g.cy1 = g.cy0 + CH < N + 1 ? g.cy0 + CH : N + 1;
    g.left_al = bi == 0;
    g.right_al = bi == ntx - 1 && ntx > 1;
    g.bot_al = bj == 0;
    g.top_al = bj == nty - 1 && nty > 1;
    if (g.left_al) g.ox = -(C - 1);                                   // x = 0 is column C - 1 of lane 0
    else if (g.right_al) g.ox = g.cx0 - halo - (C - (N - g.cx0 + halo) % C) % C;      // (N - ox) % C == 0
    else g.ox = g.cx0 - halo;
    if (g.bot_al) g.oy = -(R - 1);                                    // y = 0 is row R - 1 of warp 0
    else if (g.top_al) g.oy = g.cy0 - halo - (R - (N - g.cy0 + halo) % R) % R;        // (N - oy) % R == 0
    else g.oy = g.cy0 - halo;
    const int xneed = (g.cx1 + halo < N + 1 ? g.cx1 + halo : N + 1);  // one past the last column the tile must hold
    const int yneed = (g.cy1 + halo < N + 1 ? g.cy1 + halo : N + 1);
    g.fits = g.ox + W >= xneed && g.oy + H >= yneed;
    return g;
}

// One exchanged point: {lo32, tag, hi32, tag}.  Each aligned 8-byte half is single-copy atomic and self-validating.
__device__ __forceinline__ void st_unit(uint4* p, double v, unsigned int tag) {
    const unsigned int lo = (unsigned int)__double2loint(v), hi = (unsigned int)__double2hiint(v);
    asm volatile("st.relaxed.gpu.global.v4.u32 [%0], {%1, %2, %3, %4};" ::"l"(p), "r"(lo), "r"(tag), "r"(hi), "r"(tag) : "memory");
}
__device__ __forceinline__ uint4 ld_unit(const uint4* p) {
    uint4 v;
    asm volatile("ld.relaxed.gpu.global.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ bool unit_ok(const uint4& v, unsigned int tag) { return v.y == tag && v.w == tag; }
__device__ __forceinline__ double unit_value(const uint4& v) { return __hiloint2double((int)v.z, (int)v.x); }

__device__ __forceinline__ long long globaltimer_ns() {
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return (long long)t;
}
__device__ __forceinline__ void mark(const ResArgs& a, int slot) {
    if (a.trace != nullptr && threadIdx.x == 0 && threadIdx.y == 0 && slot < a.trace_cap)
        a.trace[(size_t)(blockIdx.y * a.ntx + blockIdx.x) * a.trace_cap + slot] = globaltimer_ns();
}
// An integer zero the compiler cannot see through: values computed from special registers + opaque_zero() are
// recomputed where they are used instead of being kept live across the sweep loop (which would push q into local memory).
__device__ __forceinline__ int opaque_zero() {
    int z = 0;
    asm volatile("" : "+r"(z));
    return z;
}

// Per-thread flags of the sweep (one register): what the lane / warp must NOT take from / give to its neighbours.
constexpr unsigned int FL_ZERO_LEFT = 1u;     // the left neighbour column is a wall or the tile edge: use 0
constexpr unsigned int FL_ZERO_RIGHT = 2u;    // same on the right
constexpr unsigned int FL_PUB_BOTTOM = 4u;    // publish the bottom row of the micro-tile to the warp below
constexpr unsigned int FL_PUB_TOP = 8u;       // publish the top row to the warp above

// One colour half-sweep on the register micro-tile.  K = LOCAL colour being updated: local point (ci, rj) has local colour
// (ci + rj) & 1 (C, R even); the kernel maps the global colour to the local one through the parity of the tile origin.
// Left / right neighbours live in the adjacent lanes and come by warp shuffle (no barrier, no shared memory);
// the rows above / below live in the adjacent warps and come through the sB / sT edge arrays.
// wallmask: bit rj * C + ci set = that point lies ON a wall that could not be isolated by alignment and is put back to
// +0.0 after the update (eq 23-24).
template <int C, int R, int K, bool FIX, int TOPOFF>
__device__ __forceinline__ void half_sweep(double (&p)[R][C], const double (&q)[R][C], const double cb, const double omb,
                                           double* __restrict__ sB, const unsigned int wallmask, const unsigned int fl) {
    // sB / sT point at [warp][0][lane] of the bottom / top edge arrays (stride 32 per ci, C * 32 per warp);
    // the top array starts TOPOFF doubles after the bottom one (a compile-time distance: one address register)
    // q of the two middle rows of the micro-tile lives in shared memory, in two more arrays of the same shape 2 TOPOFF and
    // 3 TOPOFF after the bottom edge array (same address register): 16 registers fewer held across the whole kernel.
    double* const sT = sB + TOPOFF;
    constexpr int QR = CAV_QROWS, Q0 = (R - QR) / 2;
    double Lnb[R], Rnb[R], Bnb[C], Tnb[C], qs[QR][C];
#pragma unroll
    for (int ci = 0; ci < C; ++ci) {
#pragma unroll
        for (int k = 0; k < QR; ++k)
            if (((ci + Q0 + k) & 1) == K) qs[k][ci] = sB[(2 + k) * TOPOFF + ci * 32];
    }
#pragma unroll
    for (int ci = 0; ci < C; ++ci) {
        if ((ci & 1) == K) Bnb[ci] = sT[ci * 32];                          // top row of the warp below (slot warp)
        if (((ci + R - 1) & 1) == K) Tnb[ci] = sB[C * 32 + ci * 32];       // bottom row of the warp above (slot warp + 1)
    }
#pragma unroll
    for (int rj = 0; rj < R; ++rj) {
        if ((rj & 1) == K) {                                               // right edge of lane - 1
            const double v = __shfl_up_sync(0xffffffffu, p[rj][C - 1], 1);
            Lnb[rj] = (fl & FL_ZERO_LEFT) ? 0.0 : v;
        }
        if (((C - 1 + rj) & 1) == K) {                                     // left edge of lane + 1
            const double v = __shfl_down_sync(0xffffffffu, p[rj][0], 1);
            Rnb[rj] = (fl & FL_ZERO_RIGHT) ? 0.0 : v;
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
            const double qv = (rj >= Q0 && rj < Q0 + QR) ? qs[rj - Q0 < 0 ? 0 : (rj - Q0 >= QR ? QR - 1 : rj - Q0)][ci] : q[rj][ci];
            p[rj][ci] = fma(omb, p[rj][ci], fma(cb, nb, qv));
        }
    }
    unsigned int wm = FIX ? wallmask : 0u;
    if (FIX) asm volatile("" : "+r"(wm));      // opaque: keeps the bit tests from being hoisted into live registers
    if (FIX && wm) {
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
        if ((ci & 1) == K && (fl & FL_PUB_BOTTOM)) sB[ci * 32] = p[0][ci];
        if (((ci + R - 1) & 1) == K && (fl & FL_PUB_TOP)) sT[C * 32 + ci * 32] = p[R - 1][ci];
    }
    __syncthreads();
}

template <int C, int R, int TOPOFF>
__device__ __forceinline__ void publish_all(const double (&p)[R][C], double* __restrict__ sB, const unsigned int fl) {
    double* const sT = sB + TOPOFF;
#pragma unroll
    for (int ci = 0; ci < C; ++ci) {
        if (fl & FL_PUB_BOTTOM) sB[ci * 32] = p[0][ci];
        if (fl & FL_PUB_TOP) sT[C * 32 + ci * 32] = p[R - 1][ci];
    }
    __syncthreads();
}

// ---- the points a tile sends (border strips of its core) and receives (its ring): four disjoint rectangles each ----
struct Rect { int x0, x1, y0, y1; };                     // [x0, x1) x [y0, y1)
struct Region { Rect r[4]; };
__host__ __device__ inline int imax(int a, int b) { return a > b ? a : b; }
__host__ __device__ inline int imin(int a, int b) { return a < b ? a : b; }
__host__ __device__ inline int rect_count(const Rect& r) {
    const int w = r.x1 - r.x0, h = r.y1 - r.y0;
    return (w > 0 && h > 0) ? w * h : 0;
}
__device__ __forceinline__ bool region_has(const Region& g, int x, int y) {
    bool in = false;
#pragma unroll
    for (int k = 0; k < 4; ++k) in = in || (x >= g.r[k].x0 && x < g.r[k].x1 && y >= g.r[k].y0 && y < g.r[k].y1);
    return in;
}
// u-th point of the region (row-major inside each rectangle, rectangles in order); false if u is past the end
__device__ __forceinline__ bool region_point(const Region& g, int u, int& x, int& y) {
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const int n = rect_count(g.r[k]);
        if (u < n) {
            const int w = g.r[k].x1 - g.r[k].x0;
            y = g.r[k].y0 + u / w;
            x = g.r[k].x0 + u % w;
            return true;
        }
        u -= n;
    }
    return false;
}
// Interior points of the core within `halo` of a core edge that has a neighbour tile behind it (walls are never sent).
__host__ __device__ inline Region send_region(const TileGeom& t, int N, int halo, int bi, int bj, int ntx, int nty) {
    const int X0 = imax(t.cx0, 1), X1 = imin(t.cx1, N), Y0 = imax(t.cy0, 1), Y1 = imin(t.cy1, N);
    const int hb = bj > 0 ? halo : 0, ht = bj < nty - 1 ? halo : 0, wl = bi > 0 ? halo : 0, wr = bi < ntx - 1 ? halo : 0;
    const int yB = imin(Y0 + hb, Y1), yT = imax(Y1 - ht, yB), xL = imin(X0 + wl, X1), xR = imax(X1 - wr, xL);
    Region g;
    g.r[0] = Rect{X0, X1, Y0, yB};
    g.r[1] = Rect{X0, X1, yT, Y1};
    g.r[2] = Rect{X0, xL, yB, yT};
    g.r[3] = Rect{xR, X1, yB, yT};
    return g;
}
// Interior points within `halo` of the core, outside it (the ring).
__host__ __device__ inline Region recv_region(const TileGeom& t, int N, int halo) {
    const int xlo = imax(t.cx0 - halo, 1), xhi = imin(t.cx1 + halo, N), ylo = imax(t.cy0 - halo, 1), yhi = imin(t.cy1 + halo, N);
    const int yc0 = imax(t.cy0, ylo), yc1 = imin(t.cy1, yhi), xc0 = imax(t.cx0, xlo), xc1 = imin(t.cx1, xhi);
    // Order = the order in which the neighbours STORE these points (send_region: bottom strip, top strip, left, right), so
    // that what was stored first is fetched first: the ring above comes from the northern tile's bottom strip, etc.
    Region g;
    g.r[0] = Rect{xlo, xhi, yc1, yhi};      // ring above   <- bottom strips of the tiles above
    g.r[1] = Rect{xlo, xhi, ylo, yc0};      // ring below   <- top strips of the tiles below
    g.r[2] = Rect{xc1, xhi, yc0, yc1};      // ring right   <- left strip of the tile to the right
    g.r[3] = Rect{xlo, xc0, yc0, yc1};      // ring left    <- right strip of the tile to the left
    return g;
}

__host__ __device__ inline size_t xtab_bytes(int nth, int ns_per, int nr_per) {
    return (4 + 2) * (size_t)(ns_per + nr_per) * nth + 4 * 2 * (size_t)nth;      // a multiple of 64
}
// Shared-memory layout (doubles unless said otherwise), nthreads = 32 nwarps:
//   edges   4 (MAXW + 1) C 32            bottom / top rows of the micro-tiles, q of the two middle rows (sized for MAXW warps)
//   stage   R C (nthreads + 4)           one slot per thread and micro-tile point, [point][thread] (+4: the 4 points of a chunk fall in different banks)
//   offS    ns_per nthreads u32          unit offset in the exchange buffer of the strip units this thread stores (NO_UNIT: none)
//   offR    nr_per nthreads u32          same for the ring units this thread fetches
//   masks   2 nthreads u32               bit k: point k of this thread's micro-tile is in the send region / in the ring
//   slotS   ns_per nthreads u16          staging slot of each of those units
//   slotR   nr_per nthreads u16
__host__ __device__ inline size_t smem_layout_bytes(int C, int R, int maxw, int warps, int ns_per, int nr_per) {
    const size_t nth = 32 * (size_t)warps;
    return 8 * ((2 + CAV_QROWS) * (size_t)(maxw + 1) * C * 32 + (size_t)R * C * (nth + 4)) + xtab_bytes((int)nth, ns_per, nr_per);
}

// Global <-> micro-tile transfers of one warp, coalesced: the warp moves rows of 32 C consecutive doubles (lane = x), and a
// per-warp shared-memory buffer of R rows x 32 C doubles transposes between that and the C-consecutive-points-per-lane
// layout of the registers.  Points that are not interior (walls, outside, row padding) read as +0.0.
template <int C, int R>
__device__ __forceinline__ void warp_load_tile(double (&v)[R][C], const double* __restrict__ g, const int x0w, const int y0,
                                               const int N, const int pitch, double* __restrict__ wbuf, const int lane) {
#pragma unroll
    for (int rj = 0; rj < R; ++rj) {
        const int gy = y0 + rj;
#pragma unroll
        for (int j = 0; j < C; ++j) {
            const int gx = x0w + j * 32 + lane;
            const bool upd = gx >= 1 && gx <= N - 1 && gy >= 1 && gy <= N - 1;
            wbuf[rj * (32 * C) + j * 32 + lane] = upd ? g[(size_t)gy * pitch + gx] : 0.0;
        }
    }
    __syncwarp();
#pragma unroll
    for (int rj = 0; rj < R; ++rj)
#pragma unroll
        for (int ci = 0; ci < C; ci += 2) {
            const double2 d = *reinterpret_cast<const double2*>(wbuf + rj * (32 * C) + lane * C + ci);
            v[rj][ci] = d.x; v[rj][ci + 1] = d.y;
        }
    __syncwarp();
}

struct XTab {
    unsigned int *offS, *offR, *masks;
    unsigned short *slotS, *slotR;
};
__device__ __forceinline__ XTab xtab(void* base, int nth, int ns_per, int nr_per) {
    XTab t;
    t.offS = reinterpret_cast<unsigned int*>(base);
    t.offR = t.offS + ns_per * nth;
    t.masks = t.offR + nr_per * nth;
    t.slotS = reinterpret_cast<unsigned short*>(t.masks + 2 * nth);
    t.slotR = t.slotS + ns_per * nth;
    return t;
}

// Builds, once per plan, the exchange tables of every tile in global memory (one block of xtab_bytes per tile, in the
// layout the sweep kernel copies to shared memory at launch): which exchange unit each thread stores / fetches and which
// staging slot it belongs to, and each thread's masks of micro-tile points that are sent / received.
template <int C, int R>
__global__ void k_build_tables(const ResArgs a, unsigned char* __restrict__ out) {
    const int lane = threadIdx.x, warp = threadIdx.y, nwarps = blockDim.y;
    const int tid = warp * 32 + lane, nthreads = nwarps * 32;
    const int N = a.N, bi = blockIdx.x, bj = blockIdx.y;
    const TileGeom t = tile_geom(N, a.CW, a.CH, a.halo, a.ntx, a.nty, bi, bj, C, R, 32 * C, nwarps * R);
    const int gx0 = t.ox + lane * C, gy0 = t.oy + warp * R;
    const XTab xt = xtab(out + (size_t)(bj * a.ntx + bi) * xtab_bytes(nthreads, a.ns_per, a.nr_per), nthreads, a.ns_per, a.nr_per);
    const Region gs = send_region(t, N, a.halo, bi, bj, a.ntx, a.nty), gr = recv_region(t, N, a.halo);
    for (int i = 0; i < a.ns_per + a.nr_per; ++i) {
        const bool snd = i < a.ns_per;
        const int u = (snd ? i : i - a.ns_per) * nthreads + tid;
        int x = 0, y = 0;
        uint2 e = make_uint2(NO_UNIT, 0u);
        if (region_point(snd ? gs : gr, u, x, y)) {
            const int lx = x - t.ox, ly = y - t.oy;                        // owner: lane lx / C, warp ly / R
            e.x = (unsigned int)(y * a.pitch + x);                         // < 2^31: N <= 32766
            e.y = (unsigned int)(((ly % R) * C + lx % C) * (nthreads + 4) + (ly / R) * 32 + lx / C);
        }
        (snd ? xt.offS : xt.offR)[(snd ? i : i - a.ns_per) * nthreads + tid] = e.x;
        (snd ? xt.slotS : xt.slotR)[(snd ? i : i - a.ns_per) * nthreads + tid] = (unsigned short)e.y;
    }
    unsigned int smask = 0, rmask = 0;
    for (int k = 0; k < R * C; ++k) {
        if (region_has(gs, gx0 + k % C, gy0 + k / C)) smask |= 1u << k;
        if (region_has(gr, gx0 + k % C, gy0 + k / C)) rmask |= 1u << k;
    }
    xt.masks[tid] = smask;
    xt.masks[nthreads + tid] = rmask;
}

// MAXW = most warps per CTA this variant is launched with: 65536 / (32 MAXW) registers per thread are available.
// PERSM = CTAs per SM the variant is built for (two half-size CTAs per SM hide each other's exchange and barrier latency).
template <int C, int R, int MAXW, int PERSM, bool FIX>
__global__ void __launch_bounds__(32 * MAXW, PERSM) k_resident(const ResArgs a) {
    constexpr int TOPOFF = (MAXW + 1) * C * 32;
    static_assert(C % 2 == 0 && R % 2 == 0 && R * C <= 32, "even micro-tile that fits the 32-bit point masks");
    extern __shared__ __align__(16) double sm[];
    const int lane = threadIdx.x, warp = threadIdx.y, nwarps = blockDim.y;
    const int tid = warp * 32 + lane, nthreads = nwarps * 32;
    const int N = a.N, pitch = a.pitch;
    const int bi = blockIdx.x, bj = blockIdx.y;
    mark(a, 0);

    // edge arrays; the slots no thread ever writes (warp -1, warp nwarps, unpublished wall rows) stay +0.0
    constexpr int edge_doubles = (2 + CAV_QROWS) * TOPOFF;       // bottom edges, top edges, q of the CAV_QROWS middle rows
    for (int k = tid; k < edge_doubles; k += nthreads) sm[k] = 0.0;
    double* const sB = sm + warp * C * 32 + lane;      // [MAXW + 1][C][32] bottom row of warp at [warp]; top rows TOPOFF further, at [warp + 1]

    const TileGeom t = tile_geom(N, a.CW, a.CH, a.halo, a.ntx, a.nty, bi, bj, C, R, 32 * C, nwarps * R);
    const int gx0_ = t.ox + lane * C, gy0_ = t.oy + warp * R;
    const bool odd_origin = ((t.ox + t.oy) & 1) != 0;          // local colour = global colour ^ odd_origin

    unsigned int fl = FL_PUB_BOTTOM | FL_PUB_TOP;
    {
        const int lzl = t.left_al ? 1 : 0;                                     // lane 0 holds x = -(C-1) .. 0
        const int lzr = t.right_al ? (N - t.ox) / C - 1 : 31;                  // lane (N - ox) / C holds x = N .. N + C - 1
        if (lane == lzl) fl |= FL_ZERO_LEFT;
        if (lane == lzr) fl |= FL_ZERO_RIGHT;
        if (t.bot_al && warp == 0) fl &= ~FL_PUB_TOP;                          // warp 0 holds y = -(R-1) .. 0
        if (t.top_al && warp == (N - t.oy) / R) fl &= ~FL_PUB_BOTTOM;          // that warp holds y = N .. N + R - 1
    }

    // ---- exchange tables and masks (multi-tile plans only): copied from the per-plan tables in global memory ----
    if (a.ntx * a.nty > 1) {
        const int n16 = (int)(xtab_bytes(nthreads, a.ns_per, a.nr_per) / 16);
        const uint4* const src = a.tables + (size_t)(bj * a.ntx + bi) * n16;
        uint4* const dst = reinterpret_cast<uint4*>(sm + edge_doubles + R * C * (nthreads + 4));
        for (int k = tid; k < n16; k += nthreads) dst[k] = src[k];
    }

    // ---- load the micro-tile ----
    double p[R][C], q[R][C];
    unsigned int wallmask = 0;            // wall points that alignment could not isolate (psi = 0 there, eq 23-24)
    {
        double* const wbuf = sm + edge_doubles + warp * (R * 32 * C);         // inside the staging array, which is idle now
        warp_load_tile<C, R>(p, a.psi_in, t.ox, gy0_, N, pitch, wbuf, lane);
        warp_load_tile<C, R>(q, a.w, t.ox, gy0_, N, pitch, wbuf, lane);
    }
#pragma unroll
    for (int rj = 0; rj < R; ++rj)
#pragma unroll
        for (int ci = 0; ci < C; ++ci) q[rj][ci] = a.cq * q[rj][ci];          // +0.0 where the point is not interior
    if (FIX) {
#pragma unroll 1
        for (int k = 0; k < R * C; ++k) {
            const int gx = gx0_ + k % C, gy = gy0_ + k / C;
            const bool upd = gx >= 1 && gx <= N - 1 && gy >= 1 && gy <= N - 1;
            const bool wall = gx >= 0 && gx <= N && gy >= 0 && gy <= N && !upd;
            const bool isolated = (gx == 0 && t.left_al) || (gx == N && t.right_al) || (gy == 0 && t.bot_al) || (gy == N && t.top_al);
            if (wall && !isolated) wallmask |= 1u << k;
        }
    }
    __syncthreads();                      // the zero fill of the edge arrays and the tables are complete
#pragma unroll
    for (int ci = 0; ci < C; ++ci) {      // q of the two middle rows moves to shared memory (read back by this thread only)
#pragma unroll
        for (int k = 0; k < CAV_QROWS; ++k) sB[(2 + k) * TOPOFF + ci * 32] = q[(R - CAV_QROWS) / 2 + k][ci];
    }
    publish_all<C, R, TOPOFF>(p, sB, fl);
    mark(a, 1);

    const int T = a.T;
    const int nrounds = (a.nsweeps + T - 1) / T;
    for (int r = 0; r < nrounds; ++r) {
        const int ns = min(T, a.nsweeps - r * T);
        if (odd_origin) {
            for (int s = 0; s < ns; ++s) {                                    // red = (i + j) even first (G9): local colour 1 here
                half_sweep<C, R, 1, FIX, TOPOFF>(p, q, a.cb, a.omb, sB, wallmask, fl);
                half_sweep<C, R, 0, FIX, TOPOFF>(p, q, a.cb, a.omb, sB, wallmask, fl);
            }
        } else {
            for (int s = 0; s < ns; ++s) {
                half_sweep<C, R, 0, FIX, TOPOFF>(p, q, a.cb, a.omb, sB, wallmask, fl);
                half_sweep<C, R, 1, FIX, TOPOFF>(p, q, a.cb, a.omb, sB, wallmask, fl);
            }
        }
        mark(a, 2 + 4 * r);
        if (r == nrounds - 1) break;

        // ---- halo exchange through L2: tagged data, no fence, no flag ----
        // Opaque copies: everything derived from them is recomputed here every round instead of being hoisted out of
        // the round loop, where it would stay live across the sweeps and push q into local memory.
        const int z = opaque_zero();
        const int tid_o = ((int)threadIdx.y + z) * 32 + (int)threadIdx.x, nth_o = ((int)blockDim.y + z) * 32;
        double* const stage = sm + edge_doubles;
        const XTab xt = xtab(stage + R * C * (nth_o + 4), nth_o, a.ns_per, a.nr_per);
        const unsigned int* const masks = xt.masks;
        uint4* const xb = (r & 1) ? a.x1 : a.x0;
        const unsigned int tag = a.base + 1u + (unsigned int)r;

        {   // owners stage the strip values, then all threads store strip units, consecutive threads = consecutive x
            const unsigned int smask = masks[tid_o];
#pragma unroll
            for (int k = 0; k < R * C; ++k)
                if ((smask >> k) & 1u) stage[k * (nth_o + 4) + tid_o] = p[k / C][k % C];
            __syncthreads();
            for (int i = 0; i < a.ns_per; ++i) {
                const unsigned int off = xt.offS[i * nth_o + tid_o];
                if (off != NO_UNIT) st_unit(xb + off, stage[xt.slotS[i * nth_o + tid_o]], tag);
            }
        }
        mark(a, 3 + 4 * r);
        // All threads fetch ring units (4 in flight per thread), validate, and stage the values for their owners.
        // While some unit of the warp does not carry the tag yet, ONE lane polls one such unit (2 100 pollers on the whole
        // chip: waiting tiles do not load L2), then every lane fetches its missing units again.
        constexpr int NB = CAV_RECV_BATCH;
        for (int i0 = 0; i0 < a.nr_per; i0 += NB) {
            uint2 e[NB];
            uint4 v[NB];
            unsigned int bad = 0;
#pragma unroll
            for (int j = 0; j < NB; ++j)
                e[j] = i0 + j < a.nr_per ? make_uint2(xt.offR[(i0 + j) * nth_o + tid_o], xt.slotR[(i0 + j) * nth_o + tid_o])
                                         : make_uint2(NO_UNIT, 0u);
#pragma unroll
            for (int j = 0; j < NB; ++j)
                if (e[j].x != NO_UNIT) v[j] = ld_unit(xb + e[j].x);
#pragma unroll
            for (int j = 0; j < NB; ++j)
                if (e[j].x != NO_UNIT && !unit_ok(v[j], tag)) bad |= 1u << j;
            unsigned int waiting = __ballot_sync(0xffffffffu, bad != 0u);
            if (waiting) {
                const long long t0 = clock64();
                while (waiting) {
                    int giveup = 0;
                    if ((int)threadIdx.x == __ffs((int)waiting) - 1) {
                        unsigned int off = e[NB - 1].x;                // the first missing unit of this lane
#pragma unroll
                        for (int j = NB - 2; j >= 0; --j)
                            if ((bad >> j) & 1u) off = e[j].x;
                        while (!unit_ok(ld_unit(xb + off), tag)) {
                            if (*(volatile unsigned int*)a.err != 0u) { giveup = 1; break; }      // some tile gave up: do not wait again
                            if (clock64() - t0 > SPIN_TIMEOUT_CYCLES) { atomicExch(a.err, 1u); giveup = 1; break; }
                        }
                    }
                    if (__any_sync(0xffffffffu, giveup)) break;
#pragma unroll
                    for (int j = 0; j < NB; ++j)
                        if ((bad >> j) & 1u) {
                            v[j] = ld_unit(xb + e[j].x);
                            if (unit_ok(v[j], tag)) bad &= ~(1u << j);
                        }
                    waiting = __ballot_sync(0xffffffffu, bad != 0u);
                }
            }
#pragma unroll
            for (int j = 0; j < NB; ++j)
                if (e[j].x != NO_UNIT) stage[e[j].y] = unit_value(v[j]);
        }
        __syncthreads();
        {
            const unsigned int rmask = masks[nth_o + tid_o];
#pragma unroll
            for (int k = 0; k < R * C; ++k)
                if ((rmask >> k) & 1u) p[k / C][k % C] = stage[k * (nth_o + 4) + tid_o];
        }
        mark(a, 4 + 4 * r);
        publish_all<C, R, TOPOFF>(p, sB, fl);
        mark(a, 5 + 4 * r);
    }

    // ---- store the core (walls are exactly +0.0); the geometry is recomputed, not kept live across the sweeps ----
    {
        const int z = opaque_zero();
        const int nw = (int)blockDim.y + z;
        const TileGeom te = tile_geom(a.N + z, a.CW, a.CH, a.halo, a.ntx, a.nty, (int)blockIdx.x + z, (int)blockIdx.y + z, C, R,
                                      32 * C, nw * R);
        const int ln = (int)threadIdx.x + z, wp = (int)threadIdx.y + z;
        const int ex0 = te.ox + ln * C, ey0 = te.oy + wp * R, Ne = a.N + z;
        double* const wbuf = sm + (2 + CAV_QROWS) * TOPOFF + wp * (R * 32 * C);     // the staging array is idle again
#pragma unroll
        for (int rj = 0; rj < R; ++rj)
#pragma unroll
            for (int ci = 0; ci < C; ci += 2) {
                const int gy = ey0 + rj;
                const bool rowi = gy >= 1 && gy <= Ne - 1;
                double2 d;
                d.x = (rowi && ex0 + ci >= 1 && ex0 + ci <= Ne - 1) ? p[rj][ci] : 0.0;
                d.y = (rowi && ex0 + ci + 1 >= 1 && ex0 + ci + 1 <= Ne - 1) ? p[rj][ci + 1] : 0.0;
                *reinterpret_cast<double2*>(wbuf + rj * (32 * C) + ln * C + ci) = d;
            }
        __syncwarp();
#pragma unroll
        for (int rj = 0; rj < R; ++rj) {
            const int gy = ey0 + rj;
#pragma unroll
            for (int j = 0; j < C; ++j) {
                const int gx = te.ox + j * 32 + ln;
                if (gx >= te.cx0 && gx < te.cx1 && gy >= te.cy0 && gy < te.cy1)
                    a.psi_out[(size_t)gy * a.pitch + gx] = wbuf[rj * (32 * C) + j * 32 + ln];
            }
        }
    }
}

// ---- compiled variants ------------------------------------------------------------------------------
struct Variant {
    int C, R, maxw, persm;
    const void* fn;        // every wall isolated by alignment (the plans of large grids)
    const void* fn_fix;    // with the wall-mask fix-up (a tile that holds both walls of one direction)
};
const Variant VARIANTS[] = {
    // one CTA of up to 16 warps per SM (also the single-tile plans of small grids)
    {4, 6, 16, 1, (const void*)k_resident<4, 6, 16, 1, false>, (const void*)k_resident<4, 6, 16, 1, true>},
    // two CTAs of up to 8 warps per SM: while one exchanges its halo or sits in a barrier, the other computes
    {4, 6, 8, 2, (const void*)k_resident<4, 6, 8, 2, false>, (const void*)k_resident<4, 6, 8, 2, true>},
};
constexpr int NVARIANTS = sizeof(VARIANTS) / sizeof(VARIANTS[0]);

inline int cdiv(int a, int b) { return (a + b - 1) / b; }

int region_total(const Region& g) { return rect_count(g.r[0]) + rect_count(g.r[1]) + rect_count(g.r[2]) + rect_count(g.r[3]); }

// Checks that every tile of the candidate fits its thread grid and counts the exchange units per thread.
bool finish_plan(ResidentPlan& pl, int N, int max_smem) {
    const int W = 32 * pl.C, H = pl.warps * pl.R, nth = 32 * pl.warps;
    int smax = 0, rmax = 0;
    for (int bj = 0; bj < pl.nty; ++bj)
        for (int bi = 0; bi < pl.ntx; ++bi) {
            const TileGeom t = tile_geom(N, pl.CW, pl.CH, pl.halo, pl.ntx, pl.nty, bi, bj, pl.C, pl.R, W, H);
            if (!t.fits) return false;
            if (pl.ntiles > 1) {
                smax = std::max(smax, region_total(send_region(t, N, pl.halo, bi, bj, pl.ntx, pl.nty)));
                rmax = std::max(rmax, region_total(recv_region(t, N, pl.halo)));
            }
        }
    pl.ns_per = cdiv(smax, nth);
    pl.nr_per = cdiv(rmax, nth);
    const int maxw = VARIANTS[pl.variant].maxw;
    const size_t smem = pl.ntiles > 1 ? smem_layout_bytes(pl.C, pl.R, maxw, pl.warps, pl.ns_per, pl.nr_per)
                                      : 8 * (size_t)((2 + CAV_QROWS) * (maxw + 1) * pl.C * 32 + pl.R * pl.C * (nth + 4));
    pl.fixup = pl.ntx == 1 || pl.nty == 1;
    if (smem > (size_t)max_smem) return false;
    pl.smem_bytes = (int)smem;
    return true;
}

// One direction of the tiling: G points, thread grid of L points, halo h.  false if no uniform core size works.
bool split(int G, int L, int lead, int h, int& core, int& n) {
    if (G + lead <= L) { core = G; n = 1; return true; }       // one tile holds both walls (lead = alignment slack of the first wall)
    const int cmax = L - 2 * h;
    if (cmax <= h) return false;
    n = cdiv(G, cmax);
    core = cdiv(G, n);
    n = cdiv(G, core);
    // the halo must come from adjacent tiles only, and must not reach a wall through an edge tile (only an
    // edge tile isolates the wall; elsewhere nothing keeps a wall point inside the thread grid at 0)
    return core > h && G - (n - 1) * core > h;
}

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
        cudaFuncAttributes fa, fb;
        if (cudaFuncGetAttributes(&fa, v.fn) != cudaSuccess || cudaFuncGetAttributes(&fb, v.fn_fix) != cudaSuccess) { cudaGetLastError(); continue; }
        const int regs = std::max(fa.numRegs, fb.numRegs);
        const int max_threads = std::min(fa.maxThreadsPerBlock, fb.maxThreadsPerBlock);
        const int max_warps = std::min(v.maxw, std::min(max_threads / 32, (int)(prop.regsPerBlock / (32 * std::max(regs, 1)))));
        const int W = 32 * v.C;                  // tile width in points
        const int smem_cap = std::min((int)prop.sharedMemPerBlockOptin,
                                      (int)(prop.sharedMemPerMultiprocessor / v.persm) - (int)prop.reservedSharedMemPerBlock);
        for (int warps = 1; warps <= max_warps; ++warps) {
            const int H = warps * v.R;           // tile height in points
            ResidentPlan c;
            c.ok = true; c.variant = vi; c.C = v.C; c.R = v.R; c.warps = warps; c.regs = regs; c.sm_count = sms; c.per_sm = v.persm;
            // single tile: the whole grid in one CTA, no exchange at all
            if (G + v.C - 1 <= W && G + v.R - 1 <= H) {
                if (v.persm != 1) continue;
                const double cost = (double)H * W * 0.135 + 150.0;
                c.T = 1 << 30; c.halo = 0; c.CW = G; c.CH = G; c.ntx = c.nty = c.ntiles = 1;
                if (cost < best_cost && finish_plan(c, P.N, smem_cap)) { best_cost = cost; best = c; }
                continue;
            }
            for (int T = 1; T <= 8; ++T) {
                if (T_override > 0 && T != T_override) continue;
                const int halo = 2 * T;
                int CW, ntx, CH, nty;
                if (!split(G, W, v.C - 1, halo, CW, ntx) || !split(G, H, v.R - 1, halo, CH, nty)) continue;
                const int ntiles = ntx * nty;
                if (ntiles < 2 || ntiles > v.persm * sms) continue;
                // Cost per sweep in SM cycles, calibrated on B200 at 1025^2 (profiles/): 0.135 cycles per point of the thread
                // grid(s) an SM holds (the CTAs of an SM share its fp64 pipe), plus one exchange per T sweeps whose cost is
                // mostly latency (staging, store burst, L2 round trips) and grows with the halo depth.  Two CTAs per SM were
                // measured NOT to hide each other's exchange (1.95 vs 1.67 us per sweep), so they get no discount.
                const int ctas = cdiv(ntiles, sms);
                const double cost = ctas * (double)H * W * 0.135 + (5000.0 + 600.0 * T) / T;
                c.T = T; c.halo = halo; c.CW = CW; c.CH = CH; c.ntx = ntx; c.nty = nty; c.ntiles = ntiles;
                if (cost < best_cost && finish_plan(c, P.N, smem_cap)) { best_cost = cost; best = c; }
            }
        }
    }
    if (best.ok) {
        const void* fn = best.fixup ? VARIANTS[best.variant].fn_fix : VARIANTS[best.variant].fn;
        if (cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)prop.sharedMemPerBlockOptin) != cudaSuccess) {
            cudaGetLastError();
            best.ok = false;
            return best;
        }
        int per_sm = 0;
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, fn, 32 * best.warps, best.smem_bytes) != cudaSuccess ||
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
                      "%d+%d exchange units per thread, %d regs, %d B smem, up to %d CTAs per SM on %d SMs",
                      pl.ntx, pl.nty, pl.CW, pl.CH, pl.halo, pl.T, pl.warps, pl.C, pl.R, pl.ns_per, pl.nr_per, pl.regs,
                      pl.smem_bytes, pl.per_sm, pl.sm_count);
}

int resident_variants() { return NVARIANTS; }

size_t resident_table_bytes(const ResidentPlan& pl) {
    return (pl.ok && pl.ntiles > 1) ? (size_t)pl.ntiles * xtab_bytes(32 * pl.warps, pl.ns_per, pl.nr_per) : 0;
}

int resident_build_tables(const Params& P, const ResidentPlan& pl, void* tables_dev, cudaStream_t st) {
    if (!pl.ok || pl.ntiles <= 1) return 0;
    ResArgs a{};
    a.N = P.N; a.pitch = P.pitch;
    a.halo = pl.halo; a.CW = pl.CW; a.CH = pl.CH; a.ntx = pl.ntx; a.nty = pl.nty;
    a.ns_per = pl.ns_per; a.nr_per = pl.nr_per;
    const dim3 grid(pl.ntx, pl.nty), block(32, pl.warps);
    if (pl.C == 4 && pl.R == 6) k_build_tables<4, 6><<<grid, block, 0, st>>>(a, (unsigned char*)tables_dev);
    else return -(int)cudaErrorNotSupported;
    const cudaError_t e = cudaGetLastError();
    return e == cudaSuccess ? 1 : -(int)e;
}

int resident_sweeps(const Params& P, const ResidentPlan& pl, const double* psi_in, double* psi_out, void* xa, void* xb,
                    const void* tables, const double* w, unsigned int* err_word, unsigned int* epoch, int nsweeps,
                    cudaStream_t st, long long* trace_dev, int trace_cap) {
    if (!pl.ok) return -(int)cudaErrorNotSupported;
    if (nsweeps <= 0 || psi_in == psi_out || (pl.ntiles > 1 && !tables)) return -(int)cudaErrorInvalidValue;
    ResArgs a;
    a.tables = (const uint4*)tables;
    a.N = P.N; a.pitch = P.pitch; a.cb = P.cb; a.omb = P.omb; a.cq = P.cq;
    a.w = w; a.psi_in = psi_in; a.psi_out = psi_out; a.x0 = (uint4*)xa; a.x1 = (uint4*)xb;
    a.err = err_word;
    a.base = *epoch;
    a.nsweeps = nsweeps;
    a.T = pl.ntiles == 1 ? nsweeps : pl.T;
    a.halo = pl.halo; a.CW = pl.CW; a.CH = pl.CH; a.ntx = pl.ntx; a.nty = pl.nty;
    a.ns_per = pl.ns_per; a.nr_per = pl.nr_per;
    a.trace = trace_dev; a.trace_cap = trace_cap;
    const int nrounds = (nsweeps + a.T - 1) / a.T;
    *epoch += (unsigned int)nrounds;                // tags base + 1 .. base + nrounds - 1 are used by this launch
    void* args[] = {&a};
    const dim3 grid(pl.ntx, pl.nty), block(32, pl.warps);
    const void* fn = pl.fixup ? VARIANTS[pl.variant].fn_fix : VARIANTS[pl.variant].fn;
    const cudaError_t e = cudaLaunchCooperativeKernel(fn, grid, block, args, (size_t)pl.smem_bytes, st);
    if (e != cudaSuccess) { cudaGetLastError(); return -(int)e; }
    return 1;
}

}  // namespace cavk
