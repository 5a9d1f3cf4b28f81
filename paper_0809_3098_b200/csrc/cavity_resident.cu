// cavity_resident.cu — the resident engine for sm_100a: ONE persistent cooperative kernel runs whole SSPRK(5,4) time
// steps (a1 + a2 + a3 of every stage, any number of steps per launch), or a1 sweeps alone (cav_poisson).  DESIGN.md section 6.
//
// What it computes.  a1: S red-black SOR sweeps of the 5-point Poisson problem per stage (eq 15-21 P:114-138 reduced,
// DESIGN.md D1-D3), red = (i + j) even first (G9), with the arithmetic of DESIGN.md "Canonical arithmetic":
//     nb = (psi_W + psi_E) + (psi_S + psi_N);   psi <- fma(1 - beta, psi, fma(beta / 4, nb, q)),   q = ((beta / 4) h^2) w
// a2 + a3 (eq 25, eq 8, eq 22, eq 9-13): exactly the expressions of k_rk_stage in
// cavity_kernels.cu.  Inside one colour every update reads only the other colour and a3 is pointwise in its output, so the
// schedule below cannot change a bit of the result; the tests compare with the FMA-mode oracle bit for bit.
//
// Schedule.  The (N+1)^2 grid is cut into ntx x nty tiles; tile (bi, bj) OWNS a core of about CW x CH points (tile_geom)
// and additionally carries a halo of `halo` = 2T points on every side.  One CTA per tile, all CTAs
// co-resident (cooperative launch).  A thread owns a C x R micro-tile (C consecutive x, R rows) of psi AND q in
// registers for the whole launch; a warp spans 32 C points of R rows.  Threads exchange only the perimeter of their
// micro-tile: left / right columns by warp shuffle, bottom / top rows through shared memory (edge arrays laid out so
// that every access is unit-stride over the lanes), one __syncthreads per colour half-sweep.
//
// Walls cost nothing inside the sweeps.  Left wall: the origin of a tile of the first column is shifted so that x = 0 is the LAST
// column of lane 0, which then owns no interior point.  Right wall: x = N lies in column (N - 1) mod 4 of a lane of the last
// column of tiles (every tile's lanes start on a multiple of four plus one, see the exchange).  Bottom wall: y = 0 is the last row of
// warp 0 (or, plans with EB > 0, the first row of warp 0, with interior rows above it in the same warp); top wall: y = N is the
// first row of a warp.  Wherever a live point would read the wall through a register that holds something else, the pair sum
// that contains the term is written fma(m, term, other) with m = 0.0 in that one lane / warp and 1.0 elsewhere (it rounds like
// term + other, or gives other): no select, no extra fp64 instruction; the variant is picked per tile class by a uniform
// branch (half_sweep: CLS, CLSY).  A warp that holds the isolated wall row never publishes it, so the shared-memory slot keeps
// the +0.0 it was initialised with (eq 23-24: psi = 0 on the walls).  A tile whose origin parity is odd sweeps its
// local colour 1 first.  Walls that cannot be aligned (both walls of one direction in the same tile: small grids) fall back
// to a bit mask of points that are put back to +0.0 after every half-sweep (FIX variant).
//
// Halo exchange, register to register: every T sweeps (2T half-sweeps, each of which invalidates one more ring of the halo),
// after the last sweep of a stage, and once per stage for the new vorticity, the CTAs refresh their halos through L2 WITHOUT
// any fence, flag or barrier between CTAs: the validity tag travels inside the data.  A unit is four consecutive points of a
// grid row, x = 4k - 3 .. 4k: core boundaries in x and tile origins are unit boundaries, so a unit is exactly the four columns
// one lane holds of that row, in the owner tile and in every tile that has it in its halo.  It travels as five 64-bit words,
// each carrying a 12-bit tag (word i < 4: the double with the low 12 mantissa bits replaced by the tag; word 4: the four
// displaced pieces and the tag), stored in three planes of 16 + 16 + 8 bytes per unit so that the three accesses of a warp
// cover whole sectors (st / ld.relaxed.gpu.global.v2.b64 and .b64).  The PTX memory model treats a vector access as a set of
// scalar accesses of the element type; every 64-bit element is single-copy atomic and carries its own tag, so a reader that
// finds the tag it waits for in all five words holds that round's four values, however they were ordered or torn.  At a given
// location a reader can only ever find the round it waits for or the one two rounds earlier (two buffers alternate by round
// parity: a tile writes round r + 1 only after it has received round r from every neighbour, and a neighbour posts round r
// only after it has consumed round r - 1), so tags 1 + r mod 4095 never alias; 0 = never valid (freshly cleared buffers).
// A thread stores the rows of its micro-tile that lie in the border strips of the core straight from its psi registers,
// polls the last word of its last ring row until the neighbour's data is there, and loads its ring rows straight into the
// registers they replace: no shared memory, no table, no barrier inside the exchange (xchg_setup, xchg_units).
//
// NEXT-1 (KIND = 1): the same kernel runs the paper's own compact 9-point operator, relaxed in four colours (colour_pass):
// four passes per sweep, halo 4T, right-hand side qB from the image of omega including the wall vorticity.
//
// a2 + a3 in the tile.  The shared-memory image of the tile keeps the vorticity of core + halo from one stage to the next (the
// psi rounds never touch it; at launch it is loaded from omega^n).  After the last sweep of a stage and one more psi exchange
// the wall values next to the core are Thom's formula applied to the adjacent psi (which also goes to the ring of the stage
// output in global memory, G16); each thread evaluates eq 8 / 22 and the stage combination for its core points from the image,
// stores them to the global stage buffer (pointwise operands of later stages are read back from there by the same tile), the
// new vorticity is exchanged like psi, written into the image, and scaled into q for the next stage's sweeps.
//
// The kernel reads psi_in and writes psi_out (the API ping-pongs two fields), so no tile ever overwrites input a
// neighbour has not loaded yet.
#include "cavity_resident.cuh"
#include "cavity_scheme.cuh"

#include <algorithm>
#include <cstdio>
#include <vector>

namespace cavk {

namespace {

#ifndef CAV_SPIN_TIMEOUT
#define CAV_SPIN_TIMEOUT 20000000000LL      // ~10 s at 2 GHz: a neighbour whose data never arrives is a bug, not a wait
#endif
constexpr long long SPIN_TIMEOUT_CYCLES = CAV_SPIN_TIMEOUT;
#ifndef CAV_RB
#define CAV_RB 6             // rows of a thread in flight together in the psi exchange
#endif
#ifndef CAV_EDGE_FIRST
#define CAV_EDGE_FIRST 1      // half-sweep: edge rows, publish, barrier, inner rows (0: all rows, publish, barrier)
#endif
#ifndef CAV_QROWS
#define CAV_QROWS 0             // rows of the micro-tile whose q lives in shared memory instead of registers (0: the register-to-register exchange left room for all of q)
#endif

using namespace scheme;       // the SSPRK(5,4) table, Thom's formula, eq 8 / 22 and the stage combination: cavity_scheme.cuh (shared with cavity_kernels.cu)

struct ResArgs {
    int N, pitch;
    double cb, omb, cq;                 // a1
    double c9e, c9c, c9q;               // a1, compact 9-point operator (NEXT-1): 0.2 beta, 0.05 beta, (0.025 beta) h^2
    double i2h, ih2, nu, c2h2, lid, dt; // a2, a3
    const double* psi_in;   // stream function before the launch
    double* psi_out;        // ... and after (a different field)
    double* wbase;          // omega^n, omega^(1..4), T: six fields, `fstride` doubles apart; sweeps-only launches read field 0
    size_t fstride;
    char* x0;               // exchange buffer of even rounds: three planes (16 + 16 + 8 bytes per unit of four points), upitch units per grid row
    char* x1;               // exchange buffer of odd rounds
    size_t p1off, p2off;    // byte offsets of the second and third plane inside a buffer
    int upitch;
    unsigned int* err;      // error word: set if a tile gave up waiting for a neighbour
    unsigned int base;      // exchange rounds done by earlier launches (tag of round r: 1 + r mod 4095; buffer: r & 1)
    int nsteps;             // > 0: that many whole time steps (a1 + a2 + a3, five stages each); 0: S sweeps of a1 only
    int S;                  // sweeps per stage (nsteps > 0) or in total (nsteps == 0)
    int T, halo, CW, CH, EB, ntx, nty;
    int walls;              // the exchanged regions include the wall points (compact operator)
    long long* trace;       // profiling only (cav_trace_sweeps): per tile, %globaltimer at the phase boundaries; else null
    int trace_cap;          // slots per tile
};

// Geometry of tile (bi, bj): owned core, origin of the thread grid, wall alignment.  Shared by the planner (host) and the
// kernel so that both agree on what fits.
// Exchange units are groups of four consecutive points of a grid row, unit k = the columns 4k - 3 .. 4k (so that the wall
// column x = 0 is the last column of unit 0, as it is the last column of lane 0 of a left-edge tile).  With more than one tile
// in x the cores are [0, CW + 1), [CW + 1, 2 CW + 1), ... with CW a multiple of 4: every core boundary is a unit boundary (a
// unit has exactly one owner), and every tile puts its origin at a unit boundary: the four columns of a lane ARE a unit.
// A tile of the last column then finds the wall x = N in column wc = (N - 1) mod 4 of a lane: wc = 0 isolates it as on the
// other three sides; wc > 0 leaves interior points in the same lane, and the sweeps of those tiles (a uniform branch) read
// +0.0 in place of that column (WC variant of half_sweep / colour_pass).
struct TileGeom {
    int cx0, cx1, cy0, cy1;        // core [cx0, cx1) x [cy0, cy1)
    int ox, oy;                    // grid coordinates of local point (0, 0)
    int wc;                        // tiles of the last column: the column of a lane that holds x = N (0: isolated by alignment)
    bool left_al, right_al, bot_al, top_al;   // wall isolated in a lane / warp that owns no interior point, or (right, wc > 0) read as +0.0
    bool bot_in;                   // the wall y = 0 is row 0 of warp 0, read as +0.0 by row 1 (plans with EB > 0: five more rows for the core)
    bool fits;                     // the W x H thread grid covers core + halo (clipped to the grid) and the aligned walls
};
__host__ __device__ inline int round_up4(int v) { return (v + 3) / 4 * 4; }

__host__ __device__ inline TileGeom tile_geom(int N, int CW, int CH, int EB, int halo, int ntx, int nty, int bi, int bj, int C, int R,
                                              int W, int H) {
    TileGeom g;
    g.cx0 = (ntx > 1 && bi > 0) ? bi * CW + 1 : 0;
    g.cy0 = bj == 0 ? 0 : EB + bj * CH;       // EB > 0: the bottom tiles own EB more rows (see bot_in below)
    g.cx1 = (ntx > 1 && (bi + 1) * CW + 1 < N + 1) ? (bi + 1) * CW + 1 : N + 1;
    g.cy1 = (bj < nty - 1 && EB + (bj + 1) * CH < N + 1) ? EB + (bj + 1) * CH : N + 1;      // the last tile takes what is left
    g.left_al = bi == 0;
    g.right_al = bi == ntx - 1 && ntx > 1;
    g.bot_al = bj == 0 && EB == 0;
    g.bot_in = bj == 0 && EB > 0;
    g.top_al = bj == nty - 1 && nty > 1;
    g.wc = 0;
    if (g.left_al) g.ox = -(C - 1);                                   // x = 0 is column C - 1 of lane 0
    else g.ox = g.cx0 - round_up4(halo);                              // = 1 (mod 4)
    if (g.right_al) g.wc = (N - g.ox) % C;
    if (g.bot_al) g.oy = -(R - 1);                                    // y = 0 is row R - 1 of warp 0
    else if (g.bot_in) g.oy = 0;                                      // y = 0 is row 0 of warp 0, below interior rows of the same warp
    else if (g.top_al) g.oy = g.cy0 - halo - (R - (N - g.cy0 + halo) % R) % R;        // (N - oy) % R == 0
    else g.oy = g.cy0 - halo;
    const int xneed = (g.cx1 + halo < N + 1 ? g.cx1 + halo : N + 1);  // one past the last column the tile must hold
    const int yneed = (g.cy1 + halo < N + 1 ? g.cy1 + halo : N + 1);
    g.fits = g.ox + W >= xneed && g.oy + H >= yneed;
    return g;
}

// ---- one exchanged unit: four consecutive doubles d0 .. d3 of a grid row as five 64-bit words, each carrying a 12-bit tag:
//     word i (i < 4) = d_i with the low 12 bits of its mantissa replaced by the tag
//     word 4         = the four displaced 12-bit pieces in bits 0-47, the tag in bits 48-59
// Words 0, 1 live in plane 0 of the exchange buffer (16 bytes per unit), words 2, 3 in plane 1, word 4 in plane 2 (8 bytes
// per unit): the 32 lanes of a warp move 32 consecutive units with three instructions that cover 512 + 512 + 256
// contiguous bytes (whole 32-byte sectors).  They are moved with st / ld.relaxed.gpu.global.v2.b64 and .b64; the PTX memory
// model treats a vector access as a set of scalar accesses of the element type, and every 64-bit element is single-copy
// atomic and carries its own tag, so a reader that finds the tag it waits for in all five words holds that round's four values.
struct Unit { unsigned long long w0, w1, w2, w3, w4; };
__device__ __forceinline__ Unit unit_pack(double d0, double d1, double d2, double d3, unsigned int tag) {
    const unsigned int l0 = (unsigned int)__double2loint(d0), l1 = (unsigned int)__double2loint(d1);
    const unsigned int l2 = (unsigned int)__double2loint(d2), l3 = (unsigned int)__double2loint(d3);
    Unit u;
    u.w0 = ((unsigned long long)(unsigned int)__double2hiint(d0) << 32) | ((l0 & 0xfffff000u) | tag);
    u.w1 = ((unsigned long long)(unsigned int)__double2hiint(d1) << 32) | ((l1 & 0xfffff000u) | tag);
    u.w2 = ((unsigned long long)(unsigned int)__double2hiint(d2) << 32) | ((l2 & 0xfffff000u) | tag);
    u.w3 = ((unsigned long long)(unsigned int)__double2hiint(d3) << 32) | ((l3 & 0xfffff000u) | tag);
    const unsigned int m = (l0 & 0xfffu) | ((l1 & 0xfffu) << 12) | (l2 << 24);
    const unsigned int h = ((l2 >> 8) & 0xfu) | ((l3 & 0xfffu) << 4) | (tag << 16);
    u.w4 = ((unsigned long long)h << 32) | m;
    return u;
}
// The receiver loads words 0-3 into the very registers of the doubles they replace and word 4 beside them: do all five carry the tag?
__device__ __forceinline__ bool unit_tags_ok(const double d0, const double d1, const double d2, const double d3, const unsigned long long w4,
                                             const unsigned int tag) {
    const unsigned int tg = (((unsigned int)__double2loint(d0) ^ tag) | ((unsigned int)__double2loint(d1) ^ tag) |
                             ((unsigned int)__double2loint(d2) ^ tag) | ((unsigned int)__double2loint(d3) ^ tag)) & 0xfffu;
    return tg == 0u && ((unsigned int)(w4 >> 48) & 0xfffu) == tag;
}
// ... and the displaced 12-bit pieces go back in place: only the low word of each double changes
__device__ __forceinline__ void unit_restore(double& d0, double& d1, double& d2, double& d3, const unsigned long long w4) {
    const unsigned int m = (unsigned int)w4, h = (unsigned int)(w4 >> 32);
    d0 = __hiloint2double(__double2hiint(d0), (int)(((unsigned int)__double2loint(d0) & 0xfffff000u) | (m & 0xfffu)));
    d1 = __hiloint2double(__double2hiint(d1), (int)(((unsigned int)__double2loint(d1) & 0xfffff000u) | ((m >> 12) & 0xfffu)));
    d2 = __hiloint2double(__double2hiint(d2), (int)(((unsigned int)__double2loint(d2) & 0xfffff000u) | (m >> 24) | ((h & 0xfu) << 8)));
    d3 = __hiloint2double(__double2hiint(d3), (int)(((unsigned int)__double2loint(d3) & 0xfffff000u) | ((h >> 4) & 0xfffu)));
}
__device__ __forceinline__ void st_v2(void* p, unsigned long long a, unsigned long long b) {
    asm volatile("st.relaxed.gpu.global.v2.b64 [%0], {%1, %2};" ::"l"(p), "l"(a), "l"(b) : "memory");
}
__device__ __forceinline__ void st_b64(void* p, unsigned long long a) {
    asm volatile("st.relaxed.gpu.global.b64 [%0], %1;" ::"l"(p), "l"(a) : "memory");
}
__device__ __forceinline__ void ld_v2(const void* p, unsigned long long& a, unsigned long long& b) {
    asm volatile("ld.relaxed.gpu.global.v2.b64 {%0, %1}, [%2];" : "=l"(a), "=l"(b) : "l"(p) : "memory");
}
__device__ __forceinline__ void ld_b64(const void* p, unsigned long long& a) {
    asm volatile("ld.relaxed.gpu.global.b64 %0, [%1];" : "=l"(a) : "l"(p) : "memory");
}
// predicated forms that load straight into the registers of the doubles they replace (left untouched if !on)
__device__ __forceinline__ void ld_v2_if(const int on, const void* p, double& a, double& b) {
    unsigned long long x = (unsigned long long)__double_as_longlong(a), y = (unsigned long long)__double_as_longlong(b);
    asm volatile("{\n\t.reg .pred q;\n\tsetp.ne.s32 q, %3, 0;\n\t@q ld.relaxed.gpu.global.v2.b64 {%0, %1}, [%2];\n\t}" : "+l"(x), "+l"(y) : "l"(p), "r"(on) : "memory");
    a = __longlong_as_double((long long)x); b = __longlong_as_double((long long)y);
}
__device__ __forceinline__ void ld_b64_if(const int on, const void* p, unsigned long long& a) {
    asm volatile("{\n\t.reg .pred q;\n\tsetp.ne.s32 q, %2, 0;\n\t@q ld.relaxed.gpu.global.b64 %0, [%1];\n\t}" : "+l"(a) : "l"(p), "r"(on) : "memory");
}
__host__ __device__ inline unsigned int round_tag(unsigned int round) { return 1u + round % 4095u; }

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

// Per-thread flags of the sweep (one register).
constexpr unsigned int FL_ZERO_LEFT = 1u;     // the left neighbour column is a wall or the tile edge: use 0
constexpr unsigned int FL_ZERO_RIGHT = 2u;    // same on the right
constexpr unsigned int FL_PUB_BOTTOM = 4u;    // publish the bottom row of the micro-tile to the warp below
constexpr unsigned int FL_PUB_TOP = 8u;       // publish the top row to the warp above
constexpr unsigned int FL_MASK = 32u;         // 5-point sweeps: this lane reads the wall x = 0 / x = N as one of its west / east neighbours (see half_sweep, CLS)
constexpr unsigned int FL_MASKB = 64u;        // 5-point sweeps: row 0 of this warp is the wall y = 0 (bot_in tiles): row 1 reads +0.0 below it
constexpr unsigned int FL_WALL_LANE = 16u;    // this lane holds the wall x = N in column WC > 0, behind interior points: that column reads as +0.0

// One colour half-sweep on the register micro-tile.  K = LOCAL colour being updated: local point (ci, rj) has local colour
// (ci + rj) & 1 (C, R even); the kernel maps the global colour to the local one through the parity of the tile origin.
// Left / right neighbours live in the adjacent lanes and come by warp shuffle (no barrier, no shared memory);
// the rows above / below live in the adjacent warps and come through the sB / sT edge arrays.
// wallmask: bit rj * C + ci set = that point lies ON a wall that could not be isolated by alignment and is put back to
// +0.0 after the update (eq 23-24).
// CLS: where a wall column sits for the tiles of this class (a uniform branch in the kernel picks the class from blockIdx):
//   0 none; 1 x = 0 is the last column of the lane to the LEFT of the flagged lane; 2 x = N is the first column of the lane to its
//   RIGHT; 3, 4, 5 x = N is column 1, 2, 3 of the flagged lane itself, behind interior points.
// The flagged lane (FL_MASK) must read +0.0 there (eq 23-24) although the register holds something else.  No select:
// the pair sum that contains the term is written fma(m, term, other) with m = 0.0 in the flagged lane and 1.0 elsewhere, which
// rounds exactly like term + other (m = 1) or gives other (m = 0): same fp64 instruction count, no integer work in the loop.
// CLSY = 1: tiles of the first row whose wall y = 0 is row 0 of warp 0 (bot_in): the flagged warp (FL_MASKB) masks it the same way.
template <int C, int R, int K, bool FIX, int TOPOFF, int CLS, int CLSY>
__device__ __forceinline__ void half_sweep(double (&p)[R][C], const double (&q)[R][C], const double cb, const double omb,
                                           double* __restrict__ sB, const unsigned int wallmask, const unsigned int fl_, const double m,
                                           const double mb) {
    unsigned int fl = fl_;
    asm volatile("" : "+r"(fl));               // opaque: the bit tests below are redone here, not hoisted into registers of their own
    // sB / sT point at [warp][0][lane] of the bottom / top edge arrays (stride 32 per ci, C * 32 per warp);
    // the top array starts TOPOFF doubles after the bottom one (a compile-time distance: one address register)
    // q of the two middle rows of the micro-tile lives in shared memory, in two more arrays (of MAXW warps) behind the two edge
    // arrays (same address register): 16 registers fewer held across the whole kernel.
    double* const sT = sB + TOPOFF;
    constexpr int QR = CAV_QROWS, Q0 = (R - QR) / 2;
    double Lnb[R], Rnb[R], Bnb[C], Tnb[C], qs[QR > 0 ? QR : 1][C];
#pragma unroll
    for (int ci = 0; ci < C; ++ci) {
#pragma unroll
        for (int k = 0; k < QR; ++k)
            if (((ci + Q0 + k) & 1) == K) qs[k][ci] = sB[2 * TOPOFF + k * (TOPOFF - C * 32) + ci * 32];
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
            Lnb[rj] = v;
        }
        if (((C - 1 + rj) & 1) == K) {                                     // left edge of lane + 1
            const double v = __shfl_down_sync(0xffffffffu, p[rj][0], 1);
            Rnb[rj] = v;
        }
    }
    auto update_row = [&](const int rj) {
#pragma unroll
        for (int ci = 0; ci < C; ++ci) {
            if (((ci + rj) & 1) != K) continue;
            const double pW = ci > 0 ? p[rj][ci - 1] : Lnb[rj];
            const double pE = ci < C - 1 ? p[rj][ci + 1] : Rnb[rj];
            const double pS = rj > 0 ? p[rj - 1][ci] : Bnb[ci];
            const double pN = rj < R - 1 ? p[rj + 1][ci] : Tnb[ci];
            double we;
            if (CLS == 1 && ci == 0) we = fma(m, pW, pE);                      // pW is the wall x = 0 in the flagged lane
            else if ((CLS == 2 && ci == C - 1) || (CLS >= 3 && ci == CLS - 3)) we = fma(m, pE, pW);      // pE is the wall x = N there
            else we = pW + pE;
            const double sn = (CLSY == 1 && rj == 1) ? fma(mb, pS, pN) : pS + pN;      // pS is the wall y = 0 in the flagged warp
            const double nb = we + sn;
            const double qv = (rj >= Q0 && rj < Q0 + QR) ? qs[rj - Q0 < 0 ? 0 : (rj - Q0 >= QR ? QR - 1 : rj - Q0)][ci] : q[rj][ci];
            p[rj][ci] = fma(omb, p[rj][ci], fma(cb, nb, qv));
        }
    };
#if CAV_EDGE_FIRST
    if (!FIX) {
        // The two rows other warps wait for come first and are published at once; the four inner rows, which need nothing
        // from other warps, follow BEHIND the barrier: they cover its skew and the latency of the next half-sweep's edge loads.
        update_row(0);
        update_row(R - 1);
#pragma unroll
        for (int ci = 0; ci < C; ++ci) {
            if ((ci & 1) == K && (fl & FL_PUB_BOTTOM)) sB[ci * 32] = p[0][ci];
            if (((ci + R - 1) & 1) == K && (fl & FL_PUB_TOP)) sT[C * 32 + ci * 32] = p[R - 1][ci];
        }
        __syncthreads();
#pragma unroll
        for (int rj = 1; rj < R - 1; ++rj) update_row(rj);
    } else
#endif
    {
#pragma unroll
    for (int rj = 0; rj < R; ++rj) update_row(rj);
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
}

// NEXT-1: one colour pass of the paper's 4th-order compact 9-point operator (eq 14-21) relaxed in four colours
// (reading N1), on the register micro-tile.  (KX, KY) = LOCAL colour being updated: the points with ci & 1 == KX and
// rj & 1 == KY (six per thread); all eight neighbours of such a point belong to the three other colours.
//     se = (W + E) + (S + N);  sc = (SW + SE) + (NW + NE);  psi <- fma(1 - beta, psi, fma(0.2 beta, se, fma(0.05 beta, sc, qB)))
// (the expression of k_compact_colour).  From the other threads a pass needs ONE side column (the lane to the left if KX == 0, to
// the right if KX == 1: six doubles by shuffle) and ONE edge row of five values (the warp below if KY == 0, above if KY == 1: the
// edge arrays, whose neighbouring lane slots give the two diagonal values).
// CLS / CLSY and the masks m / mb as in half_sweep: the wall terms are masked inside the pair sums of se and sc.
template <int C, int R, int KX, int KY, bool FIX, int TOPOFF, int CLS, int CLSY>
__device__ __forceinline__ void colour_pass(double (&p)[R][C], const double (&q)[R][C], const double c9e, const double c9c, const double omb,
                                            double* __restrict__ sB, const unsigned int wallmask, const unsigned int fl_, const double m,
                                            const double mb) {
    static_assert(C == 4 && R == 6 && CAV_QROWS <= 2, "written for the 4 x 6 micro-tile with q of at most two middle rows in shared memory");
    constexpr int QR = CAV_QROWS, Q0 = (R - QR) / 2;
    // the row of parity KY whose q lives in shared memory (-1: none), and which of the QR arrays holds it
    constexpr int QROW = (QR >= 1 && (Q0 & 1) == KY) ? Q0 : ((QR >= 2 && ((Q0 + 1) & 1) == KY) ? Q0 + 1 : -1);
    unsigned int fl = fl_;
    asm volatile("" : "+r"(fl));               // opaque: the bit tests below are redone here, not hoisted into registers of their own
    double* const sT = sB + TOPOFF;
    double qs[C], side[R], edge[C + 2];        // edge[1 + c] = column c of the row below (KY == 0) / above (KY == 1), c = -1 .. C
#pragma unroll
    for (int ci = KX; ci < C; ci += 2) qs[ci] = QROW >= 0 ? sB[2 * TOPOFF + (QROW - Q0 < 0 ? 0 : QROW - Q0) * (TOPOFF - C * 32) + ci * 32] : 0.0;      // q of row QROW
    {
        const double* const er = KY == 0 ? sT : sB + C * 32;       // top row of the warp below (slot warp) / bottom row of the warp above
#pragma unroll
        for (int c = 0; c < C; ++c) edge[1 + c] = er[c * 32];
        if (KX == 0) {
            const double v = er[(C - 1) * 32 - 1];                  // column C - 1 of the lane to the left
            edge[0] = v;
        } else {
            const double v = er[1];                                 // column 0 of the lane to the right
            edge[C + 1] = v;
        }
    }
#pragma unroll
    for (int rj = 0; rj < R; ++rj) {
        if (KX == 0) {
            const double v = __shfl_up_sync(0xffffffffu, p[rj][C - 1], 1);
            side[rj] = v;
        } else {
            const double v = __shfl_down_sync(0xffffffffu, p[rj][0], 1);
            side[rj] = v;
        }
    }
    // value at (column c, row r) around the micro-tile, c in -1 .. C, r in -1 .. R (only what this colour needs is ever asked for)
    auto at = [&](int c, int r) -> double {
        double x;
        if (r < 0 || r >= R) x = edge[1 + c];
        else if (c < 0 || c >= C) x = side[r];
        else x = p[r][c];
        return x;
    };
    // a + b of the columns ci - 1 and ci + 1, one of which may be a wall column that must read +0.0 in the flagged lane
    auto xpair = [&](const int ci, const double a, const double b) -> double {
        if (CLS == 1 && ci == 0) return fma(m, a, b);
        if ((CLS == 2 && ci == C - 1) || (CLS >= 3 && ci == CLS - 3)) return fma(m, b, a);
        return a + b;
    };
#pragma unroll
    for (int rj = KY; rj < R; rj += 2) {
#pragma unroll
        for (int ci = KX; ci < C; ci += 2) {
            const bool wy = CLSY == 1 && rj == 1;                       // row 0 of the flagged warp is the wall y = 0
            const double we = xpair(ci, at(ci - 1, rj), at(ci + 1, rj));
            const double sn = wy ? fma(mb, at(ci, rj - 1), at(ci, rj + 1)) : at(ci, rj - 1) + at(ci, rj + 1);
            const double se = we + sn;
            const double d1 = xpair(ci, at(ci - 1, rj - 1), at(ci + 1, rj - 1)), d2 = xpair(ci, at(ci - 1, rj + 1), at(ci + 1, rj + 1));
            const double sc = wy ? fma(mb, d1, d2) : d1 + d2;
            const double qv = (rj == QROW) ? qs[ci] : q[rj][ci];
            p[rj][ci] = fma(omb, p[rj][ci], fma(c9e, se, fma(c9c, sc, qv)));
        }
    }
    unsigned int wm = FIX ? wallmask : 0u;
    if (FIX) asm volatile("" : "+r"(wm));
    if (FIX && wm) {
#pragma unroll
        for (int rj = KY; rj < R; rj += 2)
#pragma unroll
            for (int ci = KX; ci < C; ci += 2)
                if ((wm >> (rj * C + ci)) & 1u) p[rj][ci] = 0.0;
    }
#pragma unroll
    for (int ci = KX; ci < C; ci += 2) {
        if (KY == 0 && (fl & FL_PUB_BOTTOM)) sB[ci * 32] = p[0][ci];
        if (KY == 1 && (fl & FL_PUB_TOP)) sT[C * 32 + ci * 32] = p[R - 1][ci];
    }
    __syncthreads();
}

// ns sweeps on the register micro-tile.  CLS: the tile's class (half_sweep); the compact operator's passes take WC, the column of a
// lane that holds the wall x = N behind interior points (0: none), and the select flags.
template <int C, int R, bool FIX, int TOPOFF, int KIND, int CLS, int CLSY>
__device__ __forceinline__ void run_sweeps(double (&p)[R][C], const double (&q)[R][C], const double cb, const double omb, const double c9e,
                                           const double c9c, double* __restrict__ sB, const unsigned int wallmask, const unsigned int fl, const int ns,
                                           const bool odd_origin, const int par9) {
    // the masks of half_sweep (CLS, CLSY), once per round: two registers each while the sweeps run
    double m = (CLS != 0 && (fl & FL_MASK)) ? 0.0 : 1.0;
    double mb = (CLSY != 0 && (fl & FL_MASKB)) ? 0.0 : 1.0;
    if (CLS != 0) asm volatile("" : "+d"(m));          // opaque: kept in two registers, not recomputed from the flags in every half-sweep
    if (CLSY != 0) asm volatile("" : "+d"(mb));
    if (KIND == 1) {
        // four colours (i mod 2, j mod 2) in the order (0,0), (1,0), (0,1), (1,1) (reading N1); local colour = global ^ origin parity
        for (int s = ns; s > 0; --s)
            for (int g = 0; g < 4; ++g) {
                switch (g ^ par9) {
                    case 0: colour_pass<C, R, 0, 0, FIX, TOPOFF, CLS, CLSY>(p, q, c9e, c9c, omb, sB, wallmask, fl, m, mb); break;
                    case 1: colour_pass<C, R, 1, 0, FIX, TOPOFF, CLS, CLSY>(p, q, c9e, c9c, omb, sB, wallmask, fl, m, mb); break;
                    case 2: colour_pass<C, R, 0, 1, FIX, TOPOFF, CLS, CLSY>(p, q, c9e, c9c, omb, sB, wallmask, fl, m, mb); break;
                    default: colour_pass<C, R, 1, 1, FIX, TOPOFF, CLS, CLSY>(p, q, c9e, c9c, omb, sB, wallmask, fl, m, mb); break;
                }
            }
        return;
    }
    if (odd_origin) {
        for (int s = ns; s > 0; --s) {                                     // red = (i + j) even first (G9): local colour 1 here
            half_sweep<C, R, 1, FIX, TOPOFF, CLS, CLSY>(p, q, cb, omb, sB, wallmask, fl, m, mb);
            half_sweep<C, R, 0, FIX, TOPOFF, CLS, CLSY>(p, q, cb, omb, sB, wallmask, fl, m, mb);
        }
    } else {
        for (int s = ns; s > 0; --s) {
            half_sweep<C, R, 0, FIX, TOPOFF, CLS, CLSY>(p, q, cb, omb, sB, wallmask, fl, m, mb);
            half_sweep<C, R, 1, FIX, TOPOFF, CLS, CLSY>(p, q, cb, omb, sB, wallmask, fl, m, mb);
        }
    }
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

__host__ __device__ inline int imax(int a, int b) { return a > b ? a : b; }
__host__ __device__ inline int imin(int a, int b) { return a < b ? a : b; }

// Shared-memory layout (doubles unless said otherwise), nthreads = 32 nwarps, H = R nwarps, SW = 32 C:
//   edges   (2 (MAXW + 1) + 2 MAXW) C 32   bottom / top rows of the micro-tiles, q of the two middle rows (sized for MAXW warps)
//   image   (H + 1) SW                   the tile, row-major (+ one row: the compact operator's right-hand side reads one row past
//                                        the tile, values it never uses): initial load, final store; between the stages it keeps the vorticity
//                                        of core + halo (the input of the next stage's a3): the psi rounds never touch it
//   xinfo   3 nthreads u32               per thread: which rows of its micro-tile it sends / receives, and its unit index (xchg_setup);
//                                        then one word per thread: which of its 24 registers are not interior points of the grid
__host__ __device__ inline size_t smem_layout_bytes(int C, int R, int maxw, int warps) {
    const size_t nth = 32 * (size_t)warps, H = (size_t)R * warps, SW = 32 * (size_t)C;
    return 8 * ((2 * (size_t)(maxw + 1) + CAV_QROWS * (size_t)maxw) * C * 32 + (H + 1) * SW) + 4 * 3 * nth;
}

// Which units a thread moves in an exchange.  Row rj of its micro-tile is the unit (k, y = gy0 + rj), k = (ox + 3) / 4 + lane.
//   info bits 0-5:   rows whose own unit it STORES: the unit lies in the tile's core, within `halo` of a core edge that has
//                    a neighbour behind it
//   info bits 8-13:  rows whose own unit it FETCHES: the unit lies outside the core, within `halo` of it (the ring)
//   ubase:           index of the own unit of row 0 in the exchange planes (row rj: + rj upitch); may be negative for
//                    rows below the grid, which are never moved
// Points: interior rows / columns only; with `walls` (compact operator: its right-hand side reads omega ON the walls, also in
// the ring) the wall rows / columns too.  A unit counts if at least one of its columns does.
template <int C, int R>
__host__ __device__ inline void xchg_setup(const int N, const int halo, const bool walls, const int ntx, const int nty, const int upitch,
                                           const TileGeom& t, const int lane, const int warp, const int bi, const int bj,
                                           unsigned int& info, int& ubase) {
    static_assert(C == 4, "units are groups of four columns");
    const int kown = (t.ox + 3) / 4 + lane;                         // ox + 3 is a non-negative multiple of 4
    const int gy0 = t.oy + warp * R;
    const int xf = 4 * kown - 3, xl = 4 * kown, xr = imax(xf, 0);   // first / last column of the unit, its first column inside the grid
    const int lo = walls ? 0 : 1, hi = walls ? N : N - 1;           // the rows / columns that are exchanged
    const bool colok = xl >= lo && xf <= hi;
    const bool incx = xr >= t.cx0 && xr < t.cx1;
    const bool bandx = (bi > 0 && xr < t.cx0 + halo) || (bi < ntx - 1 && xl >= t.cx1 - halo);
    const bool nearx = xl >= t.cx0 - halo && xf < t.cx1 + halo;
    unsigned int send = 0, recv = 0;
    for (int rj = 0; rj < R; ++rj) {
        const int y = gy0 + rj;
        const bool rowok = y >= lo && y <= hi;
        const bool incy = y >= t.cy0 && y < t.cy1;
        const bool bandy = (bj > 0 && y < t.cy0 + halo) || (bj < nty - 1 && y >= t.cy1 - halo);
        const bool neary = y >= t.cy0 - halo && y < t.cy1 + halo;
        if (colok && rowok && incx && incy && (bandx || bandy)) send |= 1u << rj;
        if (colok && rowok && nearx && neary && !(incx && incy)) recv |= 1u << rj;
    }
    info = send | (recv << 8);
    ubase = gy0 * upitch + kown;
}

// The halo exchange of one field held in registers (psi after a round of sweeps; the new vorticity once per stage): every
// thread stores the rows of its micro-tile that lie in the border strips of the core, straight from its registers, and
// fetches its ring rows straight into them.  No shared memory, no table, no barrier.
// RB rows of a thread are in flight together; the words of a unit are loaded into the very registers of the doubles they
// replace (those ring values are dead), so that only word 4 of each row needs registers of its own.
template <int C, int R, int RB>
__device__ __forceinline__ void xchg_units(double (&v)[R][C], char* __restrict__ xb, const size_t p1off, const size_t p2off,
                                           const unsigned int round, const unsigned int info, const int ubase, const int upitch,
                                           unsigned int* __restrict__ err, long long* __restrict__ stamp, const unsigned int tile) {
    static_assert(C == 4 && R % RB == 0, "a unit is the four columns of a lane");
    const unsigned int tag = round_tag(round);
    const unsigned int send = info & 0x3fu;
#pragma unroll
    for (int rj = 0; rj < R; ++rj) {
        if ((send >> rj) & 1u) {
            const Unit u = unit_pack(v[rj][0], v[rj][1], v[rj][2], v[rj][3], tag);
            const size_t ui = (size_t)(ubase + rj * upitch);
            st_v2(xb + 16 * ui, u.w0, u.w1);
            st_v2(xb + p1off + 16 * ui, u.w2, u.w3);
            st_b64(xb + p2off + 8 * ui, u.w4);
        }
    }
    if (stamp != nullptr && threadIdx.x == 0 && threadIdx.y == 0) *stamp = globaltimer_ns();

    unsigned int pending = (info >> 8) & 0x3fu;
    long long t0 = 0;
    // The neighbours store while this tile does: fetching at once would mostly bring the previous round's bytes.  Every lane
    // that waits for anything polls the last word of its last row (what its neighbour stores last; the lanes of a warp read
    // neighbouring words: one coalesced access) until it carries the tag; only then does the warp fetch.  A heuristic for
    // WHEN to fetch: the tags decide validity.
    {
        bool need = pending != 0u;
        const char* const pw = xb + p2off + 8 * (size_t)(ubase + (need ? 31 - __clz((int)pending) : 0) * upitch);
        for (;;) {
            if (need) {
                unsigned long long w4;
                ld_b64(pw, w4);
                if (((unsigned int)(w4 >> 48) & 0xfffu) == tag) need = false;
            }
            if (!__any_sync(0xffffffffu, need)) break;
            if (t0 == 0) t0 = clock64();
            if (__any_sync(0xffffffffu, need && (*(volatile unsigned int*)err != 0u || clock64() - t0 > SPIN_TIMEOUT_CYCLES))) break;      // decided below
        }
    }
    while (__any_sync(0xffffffffu, pending != 0u)) {
#pragma unroll
        for (int b0 = 0; b0 < R; b0 += RB) {
            unsigned long long w4[RB];
#pragma unroll
            for (int j = 0; j < RB; ++j) {
                const int rj = b0 + j;
                const int on = (int)((pending >> rj) & 1u);
                const size_t ui = (size_t)(ubase + rj * upitch);
                w4[j] = 0ull;
                ld_v2_if(on, xb + 16 * ui, v[rj][0], v[rj][1]);
                ld_v2_if(on, xb + p1off + 16 * ui, v[rj][2], v[rj][3]);
                ld_b64_if(on, xb + p2off + 8 * ui, w4[j]);
            }
#pragma unroll
            for (int j = 0; j < RB; ++j) {
                const int rj = b0 + j;
                double& d0 = v[rj][0]; double& d1 = v[rj][1]; double& d2 = v[rj][2]; double& d3 = v[rj][3];
                if (((pending >> rj) & 1u) && unit_tags_ok(d0, d1, d2, d3, w4[j], tag)) {
                    pending &= ~(1u << rj);
                    unit_restore(d0, d1, d2, d3, w4[j]);
                }
            }
        }
        int gu = 0;
        if (pending != 0u) {
        if (t0 == 0) t0 = clock64();
        if (*(volatile unsigned int*)err != 0u) gu = 1;
        else if (clock64() - t0 > SPIN_TIMEOUT_CYCLES) {
            if (atomicExch(err, 1u) == 0u) {          // the first tile to give up says what it was waiting for (CAV_DEBUG)
                const int rj = __ffs((int)pending) - 1;
                const size_t ui = (size_t)(ubase + rj * upitch);
                unsigned long long f0, f1, f4;
                ld_v2(xb + 16 * ui, f0, f1);
                ld_b64(xb + p2off + 8 * ui, f4);
                err[1] = tile; err[2] = (unsigned int)ui; err[3] = round; err[4] = tag;
                err[5] = (unsigned int)f0 & 0xfffu; err[6] = (unsigned int)f1 & 0xfffu; err[7] = (unsigned int)(f4 >> 48) & 0xfffu; err[8] = pending;
                err[9] = threadIdx.y * 32 + threadIdx.x;
            }
            gu = 1;
        }
        }
        if (__any_sync(0xffffffffu, gu)) break;
    }
    __syncwarp();
}

// ---- the tile image in shared memory ----------------------------------------------------------------------------
// Row-major, SW = 32 C doubles per row.
__host__ __device__ __forceinline__ int img_ix(int row, int lx, int SW) { return row * SW + lx; }
// rows: bit rj set = row rj of the micro-tile is copied (only the rows that meet the strips / the ring need to move)
template <int C, int R>
__device__ __forceinline__ void stage_tile(const double (&v)[R][C], double* __restrict__ img, const int lane, const int warp,
                                           const unsigned int rows) {
    static_assert(C == 4, "two 16-byte chunks per micro-tile row");
    double* const d = img + (warp * R) * (32 * C) + lane * C;
#pragma unroll
    for (int rj = 0; rj < R; ++rj)
        if ((rows >> rj) & 1u) {
            *reinterpret_cast<double2*>(d + rj * (32 * C)) = make_double2(v[rj][0], v[rj][1]);
            *reinterpret_cast<double2*>(d + rj * (32 * C) + 2) = make_double2(v[rj][2], v[rj][3]);
        }
}
template <int C, int R>
__device__ __forceinline__ void read_tile(double (&v)[R][C], const double* __restrict__ img, const int lane, const int warp,
                                          const unsigned int rows) {
    static_assert(C == 4, "two 16-byte chunks per micro-tile row");
    const double* const s = img + (warp * R) * (32 * C) + lane * C;
#pragma unroll
    for (int rj = 0; rj < R; ++rj)
        if ((rows >> rj) & 1u) {
            const double2 lo = *reinterpret_cast<const double2*>(s + rj * (32 * C));
            const double2 hi = *reinterpret_cast<const double2*>(s + rj * (32 * C) + 2);
            v[rj][0] = lo.x; v[rj][1] = lo.y; v[rj][2] = hi.x; v[rj][3] = hi.y;
        }
}
// image <- field g on the interior points of [x0, x1) x [y0, y1) (grid coordinates), +0.0 everywhere else.  Coalesced: a warp
// takes whole image rows (rows warp, warp + nwarps, ...: R of them), a lane the columns lane + 32 j.  cg: the field may have been
// written by this CTA during this launch.  The loads are issued in two batches of R C / 2, all of a batch in flight together
// (an L2 round trip per element, one after the other, would cost more than the whole stage combination).
template <int C, int R, bool WALLS = false>
__device__ __forceinline__ void fill_image(double* __restrict__ img, const double* __restrict__ g, const int x0, const int x1,
                                           const int y0, const int y1, const int ox, const int oy, const int nwarps, const int N,
                                           const int pitch, const int lane, const int warp) {
    constexpr int SW = 32 * C;
    // WALLS: the wall points too (the compact operator's right-hand side reads omega on the walls)
    const int xa = imax(x0, WALLS ? 0 : 1), xb = imin(x1, WALLS ? N + 1 : N), ya = imax(y0, WALLS ? 0 : 1), yb = imin(y1, WALLS ? N + 1 : N);
    unsigned int colok = 0;
#pragma unroll
    for (int j = 0; j < C; ++j)
        if (ox + lane + 32 * j >= xa && ox + lane + 32 * j < xb) colok |= 1u << j;
    const double* const gc = g + (ox + lane);                 // column of this lane, j = 0
    double* const ic = img + lane;
#pragma unroll
    for (int half = 0; half < 2; ++half) {
        double v[R / 2][C];
#pragma unroll
        for (int i = 0; i < R / 2; ++i) {
            const int row = warp + nwarps * (half * (R / 2) + i), gy = oy + row;
            const bool rowok = gy >= ya && gy < yb;
            const double* const gr = gc + (size_t)gy * pitch;
#pragma unroll
            for (int j = 0; j < C; ++j) {
                v[i][j] = 0.0;
                if (rowok && ((colok >> j) & 1u)) v[i][j] = __ldcg(gr + 32 * j);
            }
        }
#pragma unroll
        for (int i = 0; i < R / 2; ++i) {
            const int row = warp + nwarps * (half * (R / 2) + i);
#pragma unroll
            for (int j = 0; j < C; ++j) ic[row * SW + 32 * j] = v[i][j];
        }
    }
}

// NEXT-1: the right-hand side of the compact sweeps from the image of omega (walls included):
//     qB = ((0.025 beta) h^2) (((wW + wE) + (wS + wN)) + 8 w0) on interior points, +0.0 elsewhere   (k_compact_rhs)
// The outermost ring of the tile gets a value computed from whatever lies beyond it: that ring is only ever read, never updated.
template <int C, int R>
__device__ __forceinline__ void qb_from_image(double (&q)[R][C], const double* __restrict__ img, const double c9q, const int gx0,
                                              const int gy0, const int N, const int lane, const int warp) {
    constexpr int SW = 32 * C;
    const double* const s = img + (warp * R) * SW + lane * C;
#pragma unroll
    for (int rj = 0; rj < R; ++rj) {
        double wc[C + 2];
        wc[0] = s[rj * SW - 1]; wc[C + 1] = s[rj * SW + C];
#pragma unroll
        for (int ci = 0; ci < C; ++ci) wc[1 + ci] = s[rj * SW + ci];
#pragma unroll
        for (int ci = 0; ci < C; ++ci) {
            const int gx = gx0 + ci, gy = gy0 + rj;
            const bool inter = gx >= 1 && gx <= N - 1 && gy >= 1 && gy <= N - 1;
            const double v = c9q * (((wc[ci] + wc[ci + 2]) + (s[(rj - 1) * SW + ci] + s[(rj + 1) * SW + ci])) + 8.0 * wc[1 + ci]);
            q[rj][ci] = inter ? v : 0.0;
        }
    }
}


// a2 (eq 25) for the points of this thread's micro-tile that lie next to a wall and inside the tile's core
// [X0, X1) x [Y0, Y1): the wall value goes into the image next to the point and, with TO_GLOBAL, into the ring of the stage
// output (the bottom and top rows own the corners, G10).  A thread holds at most one column next to the left / right wall and
// one row next to the bottom / top wall; which one is a run-time index, resolved by selects (most threads hold none and skip
// everything: the fully unrolled point-by-point form of this took 2500 instructions per thread and stage).
template <int C, int R, bool TO_GLOBAL>
__device__ __forceinline__ void thom_walls(const double (&pp)[R][C], double* __restrict__ img, double* __restrict__ wout, const int gx0,
                                           const int gy0, const int X0, const int X1, const int Y0, const int Y1, const int Ne,
                                           const int pitch, const int row0, const int lx0, const double c2h2, const double lid) {
    constexpr int SW = 32 * C;
    static_assert(C == 4 && R == 6, "select chains written for the 4 x 6 micro-tile");
    auto col = [&](const int rj, const int c) -> double {
        return c == 0 ? pp[rj][0] : (c == 1 ? pp[rj][1] : (c == 2 ? pp[rj][2] : pp[rj][3]));
    };
    auto row = [&](const int r, const int ci) -> double {
        return r == 0 ? pp[0][ci] : (r == 1 ? pp[1][ci] : (r == 2 ? pp[2][ci] : (r == 3 ? pp[3][ci] : (r == 4 ? pp[4][ci] : pp[5][ci]))));
    };
#pragma unroll
    for (int side = 0; side < 2; ++side) {                    // x = 1 (wall x = 0) and x = Ne - 1 (wall x = Ne)
        const int xa = side == 0 ? 1 : Ne - 1, c = xa - gx0;
        if (c < 0 || c >= C || xa < X0 || xa >= X1) continue;
#pragma unroll
        for (int rj = 0; rj < R; ++rj) {
            const int gy = gy0 + rj;
            if (gy < Y0 || gy >= Y1) continue;
            const double v = thom_wall(c2h2, col(rj, c));
            img[img_ix(row0 + rj, lx0 + c + (side == 0 ? -1 : 1), SW)] = v;
            if (TO_GLOBAL) wout[(size_t)gy * pitch + (side == 0 ? 0 : Ne)] = v;
        }
    }
#pragma unroll
    for (int side = 0; side < 2; ++side) {                    // y = 1 (wall y = 0) and y = Ne - 1 (the lid y = Ne)
        const int ya = side == 0 ? 1 : Ne - 1, r = ya - gy0;
        if (r < 0 || r >= R || ya < Y0 || ya >= Y1) continue;
#pragma unroll
        for (int ci = 0; ci < C; ++ci) {
            const int gx = gx0 + ci;
            if (gx < X0 || gx >= X1) continue;
            const double pv = row(r, ci);
            const double v = side == 0 ? thom_wall(c2h2, pv) : thom_lid(c2h2, lid, pv);
            img[img_ix(row0 + r + (side == 0 ? -1 : 1), lx0 + ci, SW)] = v;
            if (TO_GLOBAL) {
                double* const wrow = wout + (side == 0 ? (size_t)0 : (size_t)Ne * pitch);
                wrow[gx] = v;
                const double vc = side == 0 ? thom_wall(c2h2, 0.0) : thom_lid(c2h2, lid, 0.0);
                if (gx == 1) wrow[0] = vc;
                if (gx == Ne - 1) wrow[Ne] = vc;
            }
        }
    }
}

// a2 + a3 of one stage for this tile (see the file header).  pp: the thread's psi micro-tile (registers).  On return the
// image holds the NEW vorticity on core + halo (+0.0 elsewhere) and the ring copy is refreshed; the caller turns it into q.
// Inlined: with psi passed through local memory to a non-inlined version the phase took 33 us per stage instead of 24.
template <int C, int R, int MAXW, int KIND>
__device__ __forceinline__ void rhs_phase(const ResArgs& a, const double (&pp)[R][C], double* __restrict__ sm, const int stage,
                                       const unsigned int round, const unsigned int fl) {
    constexpr int TOPOFF = (MAXW + 1) * C * 32;
    constexpr int SW = 32 * C;
    constexpr int edge_doubles = 2 * TOPOFF + CAV_QROWS * (TOPOFF - C * 32);
    double* const sB = sm + (int)threadIdx.y * C * 32 + (int)threadIdx.x;
    {
    const int z = opaque_zero();
    const int ln = (int)threadIdx.x + z, wp = (int)threadIdx.y + z;
    const int nw = (int)blockDim.y + z, tid_o = wp * 32 + ln, H = nw * R;
    const int Ne = a.N + z, pitch = a.pitch;
    const TileGeom te = tile_geom(Ne, a.CW, a.CH, a.EB, a.halo, a.ntx, a.nty, (int)blockIdx.x + z, (int)blockIdx.y + z, C, R, SW, H);
    const int k = stage % 5 + 1;                                    // RK stage 1..5
    double* const wout = a.wbase + (size_t)(k % 5) * a.fstride;         // omega^(k); stage 5 writes omega^{n+1} over omega^n
    double* const tbuf = a.wbase + (size_t)(5 + z) * a.fstride;         // T: first three terms of eq 13 (+ z: not hoisted)
    const double* const w0b = a.wbase + (size_t)z * a.fstride;          // omega^n
    const double* const w2b = a.wbase + (size_t)(2 + z) * a.fstride;
    double* const img = sm + edge_doubles;
    // interior points of the core, in grid and in local coordinates
    const int X0 = imax(te.cx0, 1), X1 = imin(te.cx1, Ne), Y0 = imax(te.cy0, 1), Y1 = imin(te.cy1, Ne);
    const int lx0 = ln * C, row0 = wp * R, gx0 = te.ox + lx0, gy0 = te.oy + row0;

    // (0) the pointwise operand of the combination (omega^n for stages 2-4, T for stage 5) is requested now, for all points of
    //     the micro-tile at once, and used in (2): its L2 round trip hides behind (1).  The same registers then take the result.
    double ab[R][C];
    unsigned int rowin = 0, colin = 0;                    // rows / columns of the micro-tile that hold interior points of the core
#pragma unroll
    for (int rj = 0; rj < R; ++rj)
        if (gy0 + rj >= Y0 && gy0 + rj < Y1) rowin |= 1u << rj;
#pragma unroll
    for (int ci = 0; ci < C; ++ci)
        if (gx0 + ci >= X0 && gx0 + ci < X1) colin |= 1u << ci;
    {
        const double* const src = (k == 5 ? tbuf : w0b) + ((size_t)gy0 * pitch + gx0);
        const unsigned int rsel = k != 1 ? rowin : 0u;
#pragma unroll
        for (int rj = 0; rj < R; ++rj)
#pragma unroll
            for (int ci = 0; ci < C; ++ci) {
                ab[rj][ci] = 0.0;
                if (((rsel >> rj) & 1u) && ((colin >> ci) & 1u)) ab[rj][ci] = src[(size_t)rj * pitch + ci];
            }
    }

    // (1) the image still holds the stage input on core + halo: nothing has written it since the end of the previous stage
    //     (the psi rounds move registers only), at the first stage of a launch it holds omega^n as loaded.  Only the walls next to
    //     the core change: Thom's formula on the new psi, written by the owner of the adjacent point, who also stores it to the
    //     ring of the stage output (k_rk_stage does the same).
    thom_walls<C, R, true>(pp, img, wout, gx0, gy0, X0, X1, Y0, Y1, Ne, pitch, row0, lx0, a.c2h2, a.lid);
    __syncthreads();

    // (2) eq 8 + eq 22 and the combination of eq 9-13 for the core points of this thread, row by row
    const double c_k = rk_c(k), a1_k = rk_a1(k), a0_k = rk_a0(k);
#pragma unroll
    for (int rj = 0; rj < R; ++rj) {
        const int gy = gy0 + rj;
        if (!((rowin >> rj) & 1u)) continue;                            // the same for the whole warp
        const double* const ir = img + (row0 + rj) * SW + lx0;
        double lnb = __shfl_up_sync(0xffffffffu, pp[rj][C - 1], 1);
        double rnb = __shfl_down_sync(0xffffffffu, pp[rj][0], 1);
        if (fl & FL_ZERO_LEFT) lnb = 0.0;                               // the wall (or the end of the thread grid), as in the sweeps
        if (fl & FL_ZERO_RIGHT) rnb = 0.0;
        if (colin == 0u) continue;
        double wc[C + 2], ws[C], wn[C];
        wc[0] = img[img_ix(row0 + rj, lx0 - 1, SW)]; wc[C + 1] = img[img_ix(row0 + rj, lx0 + C, SW)];
#pragma unroll
        for (int ci = 0; ci < C; ci += 2) {
            const int o = ci;
            const double2 c2 = *reinterpret_cast<const double2*>(ir + o);
            const double2 s2 = *reinterpret_cast<const double2*>(ir - SW + o);
            const double2 n2 = *reinterpret_cast<const double2*>(ir + SW + o);
            wc[1 + ci] = c2.x; wc[2 + ci] = c2.y; ws[ci] = s2.x; ws[ci + 1] = s2.y; wn[ci] = n2.x; wn[ci + 1] = n2.y;
        }
#pragma unroll
        for (int ci = 0; ci < C; ++ci) {
            const int gx = gx0 + ci;
            if (!((colin >> ci) & 1u)) continue;
            const double pW = ci > 0 ? pp[rj][ci - 1] : lnb;
            const double pE = gx == Ne - 1 ? 0.0 : (ci < C - 1 ? pp[rj][ci + 1] : rnb);      // psi = 0 on the wall x = N, wherever it sits
            const double pS = gy == 1 ? 0.0 : (rj > 0 ? pp[rj - 1][ci] : sB[TOPOFF + ci * 32]);      // psi = 0 on the wall y = 0; else the top row of the warp below
            const double pN = rj < R - 1 ? pp[rj + 1][ci] : sB[C * 32 + ci * 32];        // bottom row of the warp above
            const double w0 = wc[1 + ci], wW = wc[ci], wE = wc[2 + ci], wS = ws[ci], wN = wn[ci];
            const double dL = transport_dL(pW, pE, pS, pN, w0, wW, wE, wS, wN, a.i2h, a.ih2, a.nu, a.dt);   // eq 22, eq 8
            const size_t gk = (size_t)gy * pitch + gx;
            const double av = ab[rj][ci];
            const double out = rk_stage_out(k, c_k, a1_k, a0_k, dL, w0, av);                 // eq 9-13 (eq 13: a0 = 1, av = T)
            if (k == 4) tbuf[gk] = rk_T(dL, w0, w2b[gk]);                                    // eq 13, first three terms
            wout[gk] = out;
            ab[rj][ci] = out;
        }
    }
    __syncthreads();              // every read of the image is done

    // (3) the new vorticity: the core from the registers, +0.0 elsewhere, then the ring from the neighbours
#pragma unroll
    for (int rj = 0; rj < R; ++rj)
#pragma unroll
        for (int ci = 0; ci < C; ++ci)
            if (!(((rowin >> rj) & 1u) && ((colin >> ci) & 1u))) ab[rj][ci] = 0.0;
    stage_tile<C, R>(ab, img, ln, wp, 0x3fu);
    if (KIND == 1) {
        // NEXT-1: B of eq 17 reads omega on the walls: the stage output carries the wall vorticity just computed (reading N2),
        // so the image of the new vorticity gets it too (neighbours fetch it with the ring; corners are never read)
        __syncthreads();              // the zeros staged by the owners of the wall points are in place
        thom_walls<C, R, false>(pp, img, nullptr, gx0, gy0, X0, X1, Y0, Y1, Ne, pitch, row0, lx0, a.c2h2, a.lid);
    }
    __syncthreads();
    if (a.ntx * a.nty > 1) {
        // the new vorticity of core + walls goes back to the registers (the walls were written into the image by the owners
        // of the adjacent points), is exchanged like psi, and the ring it brought goes into the image
        read_tile<C, R>(ab, img, ln, wp, 0x3fu);
        const unsigned int* const xi = reinterpret_cast<const unsigned int*>(img + (H + 1) * SW) + 2 * tid_o;
        const unsigned int info = xi[0];
        const int ubase = (int)xi[1];
        char* const xb = (round & 1u) ? a.x1 : a.x0;
        xchg_units<C, R, R / 2>(ab, xb, a.p1off, a.p2off, round, info, ubase, a.upitch, a.err, nullptr, blockIdx.y * a.ntx + blockIdx.x);
        stage_tile<C, R>(ab, img, ln, wp, info >> 8);
        __syncthreads();
    }
    }
}

// MAXW = most warps per CTA the kernel is launched with: 65536 / (32 MAXW) registers per thread are available.
// KIND: 0 = red-black sweeps of the 5-point operator (a1), 1 = four-colour sweeps of the compact 9-point operator (NEXT-1)
template <int C, int R, int MAXW, bool FIX, int KIND>
__global__ void __launch_bounds__(32 * MAXW, 16 / MAXW) k_resident(const __grid_constant__ ResArgs a) {
    constexpr int TOPOFF = (MAXW + 1) * C * 32;
    constexpr int SW = 32 * C;
    static_assert(C % 2 == 0 && R % 2 == 0 && R * C <= 32, "even micro-tile that fits the 32-bit point masks");
    extern __shared__ __align__(16) double sm[];
    const int lane = threadIdx.x, warp = threadIdx.y, nwarps = blockDim.y;
    const int tid = warp * 32 + lane, nthreads = nwarps * 32;
    const int N = a.N;
    const int bi = blockIdx.x, bj = blockIdx.y;
    mark(a, 0);

    // edge arrays; the slots no thread ever writes (warp -1, warp nwarps) stay +0.0
    constexpr int edge_doubles = 2 * TOPOFF + CAV_QROWS * (TOPOFF - C * 32);   // bottom edges, top edges (MAXW + 1 warps), q of the CAV_QROWS middle rows (MAXW warps)
    for (int k = tid; k < edge_doubles; k += nthreads) sm[k] = 0.0;
    double* const sB = sm + warp * C * 32 + lane;      // [MAXW + 1][C][32] bottom row of warp at [warp]; top rows TOPOFF further, at [warp + 1]

    const TileGeom t = tile_geom(N, a.CW, a.CH, a.EB, a.halo, a.ntx, a.nty, bi, bj, C, R, SW, nwarps * R);
    const int gx0_ = t.ox + lane * C, gy0_ = t.oy + warp * R;
    // local colour = global colour ^ odd_origin.  Computed from blockIdx only: the branch on it is uniform for the compiler
    // too, so the sweep loops stay convergent code (uniform registers for the coefficients, no divergence guards on the shuffles)
    const bool odd_origin = ((t.ox + t.oy) & 1) != 0;
    const int par9 = (t.ox & 1) | ((t.oy & 1) << 1);            // compact operator: parity of the origin in x and y
    unsigned int fl = FL_PUB_BOTTOM | FL_PUB_TOP;
    {
        const int lzl = t.left_al ? 1 : 0;                                     // lane 0 holds x = -(C-1) .. 0
        const int lzr = (t.right_al && t.wc == 0) ? (N - t.ox) / C - 1 : 31;   // lane (N - ox) / C holds x = N .. N + C - 1
        if (t.right_al && t.wc > 0 && lane == (N - t.ox) / C) fl |= FL_WALL_LANE;
        if (lane == lzl) fl |= FL_ZERO_LEFT;
        if (lane == lzr) fl |= FL_ZERO_RIGHT;
        // the lane of the 5-point sweeps' mask (half_sweep, CLS 1 / 2 / 3-5); a tile has one class, so one flag serves all
        if (t.left_al ? lane == 1 : (t.right_al && lane == (N - t.ox) / C - (t.wc == 0 ? 1 : 0))) fl |= FL_MASK;
        if (t.bot_in && warp == 0) fl |= FL_MASKB;
        if (t.bot_al && warp == 0) fl &= ~FL_PUB_TOP;                          // warp 0 holds y = -(R-1) .. 0
        if (t.top_al && warp == (N - t.oy) / R) fl &= ~FL_PUB_BOTTOM;          // that warp holds y = N .. N + R - 1
    }

    // ---- what this thread moves in an exchange (multi-tile plans), and which of its registers are not interior points of the grid,
    //      kept in shared memory: the sweeps have no register to spare ----
    {
        const int H = nwarps * R;
        unsigned int* const xw = reinterpret_cast<unsigned int*>(sm + edge_doubles + (H + 1) * SW);
        unsigned int info = 0u;
        int ubase = 0;
        if (a.ntx * a.nty > 1) xchg_setup<C, R>(N, a.halo, a.walls != 0, a.ntx, a.nty, a.upitch, t, lane, warp, bi, bj, info, ubase);
        xw[2 * tid] = info; xw[2 * tid + 1] = (unsigned int)ubase;
        unsigned int deadbits = 0;
        for (int k = 0; k < R * C; ++k) {
            const int gx = gx0_ + k % C, gy = gy0_ + k / C;
            if (gx <= 0 || gx >= N || gy <= 0 || gy >= N) deadbits |= 1u << k;
        }
        xw[2 * nthreads + tid] = deadbits;
    }

    // ---- load the micro-tile: psi, and the right-hand side q = cq w of the first stage ----
    double p[R][C], q[R][C];
    unsigned int wallmask = 0;            // wall points that alignment could not isolate (psi = 0 there, eq 23-24)
    {
        double* const img = sm + edge_doubles;
        fill_image<C, R>(img, a.psi_in, 0, N + 1, 0, N + 1, t.ox, t.oy, nwarps, N, a.pitch, lane, warp);
        __syncthreads();
        read_tile<C, R>(p, img, lane, warp, 0x3fu);
        __syncthreads();
        fill_image<C, R, KIND == 1>(img, a.wbase, 0, N + 1, 0, N + 1, t.ox, t.oy, nwarps, N, a.pitch, lane, warp);
        __syncthreads();
        if (KIND == 1) qb_from_image<C, R>(q, img, a.c9q, gx0_, gy0_, N, lane, warp);
        else read_tile<C, R>(q, img, lane, warp, 0x3fu);
    }
    if (KIND == 0) {
#pragma unroll
        for (int rj = 0; rj < R; ++rj)
#pragma unroll
            for (int ci = 0; ci < C; ++ci) q[rj][ci] = a.cq * q[rj][ci];      // +0.0 where the point is not interior
    }
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
    __syncthreads();                      // the zero fill of the edge arrays, the tables and the ring copy are complete
#pragma unroll
    for (int ci = 0; ci < C; ++ci) {      // q of the two middle rows moves to shared memory (read back by this thread only)
#pragma unroll
        for (int k = 0; k < CAV_QROWS; ++k) sB[2 * TOPOFF + k * (TOPOFF - C * 32) + ci * 32] = q[(R - CAV_QROWS) / 2 + k][ci];
    }
    publish_all<C, R, TOPOFF>(p, sB, fl);
    mark(a, 1);

    // Few scalars stay live across the sweeps (they would push q into local memory): the stage counter, the sweeps left in
    // the stage and the exchange round; everything else is recomputed from the kernel parameters where it is used.
    unsigned int round = a.base;          // exchange rounds done so far (all tiles count alike)
    for (int stage = 0; stage < (a.nsteps > 0 ? 5 * a.nsteps : 1); ++stage) {
        // ================= a1: S sweeps, a halo exchange after every T of them =================
        for (int rem = a.S; rem > 0; rem -= a.T) {
            {
                // the class of the tile (where a wall column sits: first column of tiles, last column, none), from blockIdx and the
                // parameters only: a uniform branch, like the colour order
                const int cls = (int)blockIdx.x == 0 ? 1 : (((int)blockIdx.x == a.ntx - 1) ? 2 + ((a.N - 1) & 3) : 0);
                const int ns = min(a.T, rem);
                if ((int)blockIdx.y == 0 && a.EB > 0) {       // bot_in tiles (uniform branch)
                    switch (cls) {
                        case 0: run_sweeps<C, R, FIX, TOPOFF, KIND, 0, 1>(p, q, a.cb, a.omb, a.c9e, a.c9c, sB, wallmask, fl, ns, odd_origin, par9); break;
                        case 1: run_sweeps<C, R, FIX, TOPOFF, KIND, 1, 1>(p, q, a.cb, a.omb, a.c9e, a.c9c, sB, wallmask, fl, ns, odd_origin, par9); break;
                        case 2: run_sweeps<C, R, FIX, TOPOFF, KIND, 2, 1>(p, q, a.cb, a.omb, a.c9e, a.c9c, sB, wallmask, fl, ns, odd_origin, par9); break;
                        case 3: run_sweeps<C, R, FIX, TOPOFF, KIND, 3, 1>(p, q, a.cb, a.omb, a.c9e, a.c9c, sB, wallmask, fl, ns, odd_origin, par9); break;
                        case 4: run_sweeps<C, R, FIX, TOPOFF, KIND, 4, 1>(p, q, a.cb, a.omb, a.c9e, a.c9c, sB, wallmask, fl, ns, odd_origin, par9); break;
                        default: run_sweeps<C, R, FIX, TOPOFF, KIND, 5, 1>(p, q, a.cb, a.omb, a.c9e, a.c9c, sB, wallmask, fl, ns, odd_origin, par9); break;
                    }
                } else {
                    switch (cls) {
                        case 0: run_sweeps<C, R, FIX, TOPOFF, KIND, 0, 0>(p, q, a.cb, a.omb, a.c9e, a.c9c, sB, wallmask, fl, ns, odd_origin, par9); break;
                        case 1: run_sweeps<C, R, FIX, TOPOFF, KIND, 1, 0>(p, q, a.cb, a.omb, a.c9e, a.c9c, sB, wallmask, fl, ns, odd_origin, par9); break;
                        case 2: run_sweeps<C, R, FIX, TOPOFF, KIND, 2, 0>(p, q, a.cb, a.omb, a.c9e, a.c9c, sB, wallmask, fl, ns, odd_origin, par9); break;
                        case 3: run_sweeps<C, R, FIX, TOPOFF, KIND, 3, 0>(p, q, a.cb, a.omb, a.c9e, a.c9c, sB, wallmask, fl, ns, odd_origin, par9); break;
                        case 4: run_sweeps<C, R, FIX, TOPOFF, KIND, 4, 0>(p, q, a.cb, a.omb, a.c9e, a.c9c, sB, wallmask, fl, ns, odd_origin, par9); break;
                        default: run_sweeps<C, R, FIX, TOPOFF, KIND, 5, 0>(p, q, a.cb, a.omb, a.c9e, a.c9c, sB, wallmask, fl, ns, odd_origin, par9); break;
                    }
                }
            }
            const int tslot = 2 + 4 * (int)(round - a.base);                    // trace slot (meaningful in sweeps-only launches)
            mark(a, tslot);
            if (a.ntx * a.nty == 1 || (a.nsteps == 0 && rem <= a.T)) continue;  // sweeps only: the last round needs no exchange

            // ---- halo exchange of psi through L2, register to register: tagged data, no fence, no flag, no barrier ----
            // Opaque copies: everything derived from them is recomputed here every round instead of being hoisted out of
            // the round loop, where it would stay live across the sweeps and push q into local memory.
            {
                const int z = opaque_zero();
                const int nw = (int)blockDim.y + z, tid_o = ((int)threadIdx.y + z) * 32 + (int)threadIdx.x;
                const unsigned int* const xi = reinterpret_cast<const unsigned int*>(sm + edge_doubles + (nw * R + 1) * SW) + 2 * tid_o;
                const unsigned int info = xi[0];
                const int ubase = (int)xi[1];
                char* const xb = (round & 1u) ? a.x1 : a.x0;
                long long* const stamp = (a.trace != nullptr && tslot + 1 < a.trace_cap) ? a.trace + (size_t)(blockIdx.y * a.ntx + blockIdx.x) * a.trace_cap + tslot + 1 : nullptr;
                const unsigned int tile = blockIdx.y * a.ntx + blockIdx.x;
                xchg_units<C, R, CAV_RB>(p, xb, a.p1off, a.p2off, round, info, ubase, a.upitch, a.err, stamp, tile);
            }
            ++round;
            mark(a, tslot + 2);
            if (a.nsteps == 0 || KIND == 1) {
                // sweeps-only launches (cav_poisson, cav_trace_sweeps) never reach the once-per-stage reset below: put the
                // registers of non-interior points back to +0.0 after every exchange round instead (outside the sweep loops).
                // The compact operator does so in time-step launches too: its four colour passes per sweep let a dead register
                // grow by up to 2.94^4 per sweep at beta -> 2, which over the sweeps of one stage reaches Inf (and 0 x Inf = NaN)
                const int z = opaque_zero();
                const unsigned int dead = reinterpret_cast<const unsigned int*>(sm + edge_doubles + (((int)blockDim.y + z) * R + 1) * SW)
                                              [2 * ((int)blockDim.y + z) * 32 + ((int)threadIdx.y + z) * 32 + (int)threadIdx.x];
                if (dead != 0u) {
#pragma unroll
                    for (int rj = 0; rj < R; ++rj)
#pragma unroll
                        for (int ci = 0; ci < C; ++ci)
                            if ((dead >> (rj * C + ci)) & 1u) p[rj][ci] = 0.0;
                }
            }
            publish_all<C, R, TOPOFF>(p, sB, fl);
            mark(a, tslot + 3);
        }
        if (a.nsteps == 0) break;

        // ================= a2 + a3: wall vorticity, transport right-hand side, stage combination =================
        {
            {   // The registers of points that are not interior to the grid (lanes / warps / columns that hold or lie beyond a wall)
                // take part in the sweeps like any other.  Live points never read them unmasked, but a masked read is 0 * value, so
                // they must stay finite; a half-sweep can grow them by at most |1 - beta| + beta < 3.  Once per stage they are put back
                // to +0.0 (they have stayed bounded over 7e8 sweeps in practice, profiles/r2c_final.md: this is a safety net).
                const int z = opaque_zero();
                const unsigned int dead = reinterpret_cast<const unsigned int*>(sm + edge_doubles + (((int)blockDim.y + z) * R + 1) * SW)
                                              [2 * ((int)blockDim.y + z) * 32 + ((int)threadIdx.y + z) * 32 + (int)threadIdx.x];
                if (dead != 0u) {
#pragma unroll
                    for (int rj = 0; rj < R; ++rj)
#pragma unroll
                        for (int ci = 0; ci < C; ++ci)
                            if ((dead >> (rj * C + ci)) & 1u) p[rj][ci] = 0.0;
                }
            }
            rhs_phase<C, R, MAXW, KIND>(a, p, sm, stage, round, fl);
            if (a.ntx * a.nty > 1) ++round;                                     // the vorticity exchange
            const int z = opaque_zero();
            const int ln = (int)threadIdx.x + z, wp = (int)threadIdx.y + z;
            double* const img = sm + edge_doubles;
            if (KIND == 1) {
                const TileGeom tq = tile_geom(a.N + z, a.CW, a.CH, a.EB, a.halo, a.ntx, a.nty, (int)blockIdx.x + z, (int)blockIdx.y + z, C, R, SW, ((int)blockDim.y + z) * R);
                qb_from_image<C, R>(q, img, a.c9q, tq.ox + ln * C, tq.oy + wp * R, a.N + z, ln, wp);
            } else {
                read_tile<C, R>(q, img, ln, wp, 0x3fu);
#pragma unroll
                for (int rj = 0; rj < R; ++rj)
#pragma unroll
                    for (int ci = 0; ci < C; ++ci) q[rj][ci] = a.cq * q[rj][ci];
            }
#pragma unroll
            for (int ci = 0; ci < C; ++ci) {
#pragma unroll
                for (int kq = 0; kq < CAV_QROWS; ++kq) sB[2 * TOPOFF + kq * (TOPOFF - C * 32) + ci * 32] = q[(R - CAV_QROWS) / 2 + kq][ci];
            }
            __syncthreads();              // the ring copy is complete before the image is staged again
        }
    }

    // ---- store the core of psi (walls are exactly +0.0); the geometry is recomputed, not kept live across the sweeps ----
    {
        const int z = opaque_zero();
        const int ln = (int)threadIdx.x + z, wp = (int)threadIdx.y + z;
        const int nw = (int)blockDim.y + z, tid_o = wp * 32 + ln, nth_o = nw * 32, H = nw * R;
        const int Ne = a.N + z;
        const TileGeom te = tile_geom(Ne, a.CW, a.CH, a.EB, a.halo, a.ntx, a.nty, (int)blockIdx.x + z, (int)blockIdx.y + z, C, R, SW, H);
        double* const img = sm + edge_doubles;
        stage_tile<C, R>(p, img, ln, wp, 0x3fu);
        __syncthreads();
        const int cw = te.cx1 - te.cx0, ch = te.cy1 - te.cy0;
        for (int k = tid_o; k < cw * ch; k += nth_o) {
            const int gy = te.cy0 + k / cw, gx = te.cx0 + k % cw;
            const bool inter = gx >= 1 && gx <= Ne - 1 && gy >= 1 && gy <= Ne - 1;
            a.psi_out[(size_t)gy * a.pitch + gx] = inter ? img[img_ix(gy - te.oy, gx - te.ox, SW)] : 0.0;
        }
    }
}

// ---- compiled variants ------------------------------------------------------------------------------
struct Variant {
    int C, R, maxw;
    const void* fn[2];        // [kind] every wall isolated by alignment (the plans of large grids)
    const void* fn_fix[2];    // [kind] with the wall-mask fix-up (a tile that holds both walls of one direction)
};
const Variant VARIANTS[] = {
    // one CTA of up to 16 warps per SM (also the single-tile plans of small grids); kind 0 = red-black 5-point, 1 = compact 9-point
    {4, 6, 16, {(const void*)k_resident<4, 6, 16, false, 0>, (const void*)k_resident<4, 6, 16, false, 1>},
               {(const void*)k_resident<4, 6, 16, true, 0>, (const void*)k_resident<4, 6, 16, true, 1>}},
};
constexpr int NVARIANTS = sizeof(VARIANTS) / sizeof(VARIANTS[0]);

inline int cdiv(int a, int b) { return (a + b - 1) / b; }
inline double sweep_cycles(int warps) { return 2.0 * (cdiv(warps, 4) * 187.0 + 40.0); }      // one sweep = two colour half-sweeps

// Checks that every tile of the candidate fits its thread grid.
bool finish_plan(ResidentPlan& pl, int N, int max_smem) {
    const int W = 32 * pl.C, H = pl.warps * pl.R;
    for (int bj = 0; bj < pl.nty; ++bj)
        for (int bi = 0; bi < pl.ntx; ++bi) {
            const TileGeom t = tile_geom(N, pl.CW, pl.CH, pl.EB, pl.halo, pl.ntx, pl.nty, bi, bj, pl.C, pl.R, W, H);
            if (!t.fits) return false;
        }
    const int maxw = VARIANTS[pl.variant].maxw;
    const size_t smem = smem_layout_bytes(pl.C, pl.R, maxw, pl.warps);
    pl.fixup = pl.ntx == 1 || pl.nty == 1;
    if (smem > (size_t)max_smem) return false;
    pl.smem_bytes = (int)smem;
    return true;
}

// Tiling in y: G points, thread grid of L rows, halo h.  false if no uniform core size works.
bool split(int G, int L, int lead, int h, int& core, int& n) {
    if (G + lead <= L) { core = G; n = 1; return true; }       // one tile holds both walls (lead = alignment slack of the first wall)
    const int cmax = L - 2 * h;
    if (cmax <= h) return false;
    for (n = cdiv(G, cmax); n <= G; ++n) {
        core = cdiv(G, n);
        if (core > cmax) continue;
        n = cdiv(G, core);
        // the halo must come from adjacent tiles only, and must not reach a wall through an edge tile (only an
        // edge tile isolates the wall; elsewhere nothing keeps a wall point inside the thread grid at 0)
        return n >= 2 && core > h && G - (n - 1) * core > h;
    }
    return false;
}
// Tiling in y with the wall y = 0 INSIDE warp 0 of the first row of tiles (tile_geom: bot_in): that row can own up to `h` more
// rows than the others (it needs no halo below and no warp to isolate the wall), the last row takes what is left (at most
// L - h - (R - 1) rows: its wall is aligned to a warp).  n tiles, cores CH + EB, CH, ..., CH, rest.  false if impossible.
bool split_wb(int G, int L, int R, int h, int n, int& core, int& eb) {
    const int cmax = L - 2 * h, ctmax = L - h - (R - 1);
    if (n < 3 || cmax <= h) return false;
    for (core = h + 1; core <= cmax; ++core) {
        // the first row takes as much of the excess as it may, the last row the remainder
        const int rest = G - (n - 1) * core;            // rows left for EB + the last core
        if (rest <= h) continue;
        eb = std::min(h, std::max(rest - core, 1));
        const int last = rest - eb;
        if (last > h && last <= ctmax && last <= core + h) return true;
    }
    return false;
}
// Tiling in x (tile_geom): cores [0, CW + 1), [CW + 1, 2 CW + 1), ..., CW a multiple of 4; an inner tile holds
// round_up4(h) + CW + h columns.
bool split_x(int N, int L, int lead, int h, int& core, int& n) {
    if (N + 1 + lead <= L) { core = N + 1; n = 1; return true; }
    const int cmax = (L - round_up4(h) - h) / 4 * 4;
    if (cmax <= h) return false;
    for (n = std::max(cdiv(N, cmax), 2); n <= N; ++n) {
        core = round_up4(cdiv(N, n));
        if (core > cmax) continue;
        n = cdiv(N, core);
        return n >= 2 && core > h && N - (n - 1) * core > h;
    }
    return false;
}

// Testing aid (cav_debug_unit_roundtrip): every thread packs four doubles into a unit with the given tag, stores it to the three planes
// with the accesses of the exchange, loads it back the way the receiver does, checks the tags and restores the doubles.
__global__ void k_unit_roundtrip(const double* __restrict__ in, double* __restrict__ out, char* __restrict__ xb, const size_t p1off,
                                 const size_t p2off, const int nunits, const unsigned int tag, unsigned int* __restrict__ bad) {
    const int u = blockIdx.x * blockDim.x + threadIdx.x;
    if (u >= nunits) return;
    const Unit w = unit_pack(in[4 * u], in[4 * u + 1], in[4 * u + 2], in[4 * u + 3], tag);
    st_v2(xb + 16 * (size_t)u, w.w0, w.w1);
    st_v2(xb + p1off + 16 * (size_t)u, w.w2, w.w3);
    st_b64(xb + p2off + 8 * (size_t)u, w.w4);
    double d0 = 0.0, d1 = 0.0, d2 = 0.0, d3 = 0.0;
    unsigned long long w4 = 0ull;
    ld_v2_if(1, xb + 16 * (size_t)u, d0, d1);
    ld_v2_if(1, xb + p1off + 16 * (size_t)u, d2, d3);
    ld_b64_if(1, xb + p2off + 8 * (size_t)u, w4);
    if (!unit_tags_ok(d0, d1, d2, d3, w4, tag) || unit_tags_ok(d0, d1, d2, d3, w4, tag == 1u ? 2u : tag - 1u)) atomicAdd(bad, 1u);
    unit_restore(d0, d1, d2, d3, w4);
    out[4 * u] = d0; out[4 * u + 1] = d1; out[4 * u + 2] = d2; out[4 * u + 3] = d3;
}

}  // namespace

int resident_unit_roundtrip(const double* in_dev, double* out_dev, void* scratch_dev, int nunits, unsigned int tag, unsigned int* bad_dev,
                             cudaStream_t st) {
    const size_t p1 = ((size_t)nunits * 16 + 255) / 256 * 256;
    k_unit_roundtrip<<<(nunits + 255) / 256, 256, 0, st>>>(in_dev, out_dev, (char*)scratch_dev, p1, 2 * p1, nunits, tag, bad_dev);
    const cudaError_t e = cudaGetLastError();
    return e == cudaSuccess ? 1 : -(int)e;
}

ResidentPlan resident_plan_for(int N, int kind, int T_override, int variant_override, int sms, int smem_cap, int regs_per_block) {
    ResidentPlan best;
    const int G = N + 1;                         // points per side, walls included
    double best_cost = 1e300;
    if (kind < 0 || kind > 1 || N < 2) return best;
    for (int vi = 0; vi < NVARIANTS; ++vi) {
        if (variant_override >= 0 && vi != variant_override) continue;
        const Variant& v = VARIANTS[vi];
        const int per_sm = 16 / v.maxw;          // CTAs per SM the variant is compiled for (__launch_bounds__(32 maxw, 16 / maxw))
        const int regs = 128;
        const int max_warps = std::min(v.maxw, regs_per_block / (32 * regs) / per_sm);
        const int smem_cta = per_sm == 1 ? smem_cap : (smem_cap + 1024) / per_sm - 1024;      // 1 KB per CTA is reserved by the system
        const int W = 32 * v.C;                  // tile width in points
        for (int warps = 1; warps <= max_warps; ++warps) {
            const int H = warps * v.R;           // tile height in points
            ResidentPlan c;
            c.ok = true; c.variant = vi; c.C = v.C; c.R = v.R; c.warps = warps; c.regs = regs; c.sm_count = sms; c.per_sm = per_sm; c.kind = kind;
            const double sweep_cost = (kind == 1 ? 2.2 : 1.0) * sweep_cycles(warps);      // four colour passes of 54 fp64 instructions instead of two of 60
            // single tile: the whole grid in one CTA, no exchange at all
            if (G + v.C - 1 <= W && G + v.R - 1 <= H) {
                const double cost = sweep_cost;
                c.T = 1 << 30; c.halo = 0; c.CW = G; c.CH = G; c.ntx = c.nty = c.ntiles = 1;
                if (per_sm == 1 && cost < best_cost && finish_plan(c, N, smem_cta)) { best_cost = cost; best = c; }
                continue;
            }
            for (int T = 1; T <= 10; ++T) {
                if (T_override > 0 && T != T_override) continue;
                const int halo = (kind == 1 ? 4 : 2) * T;      // one ring is consumed per colour pass
                int CW, ntx, CH, nty;
                if (!split_x(N, W, v.C - 1, halo, CW, ntx)) continue;
                int EB = 0;
                bool okY = split(G, H, v.R - 1, halo, CH, nty) && ntx * nty <= sms * per_sm;
                if (!okY && ntx <= sms * per_sm) {
                    // one row of tiles fewer with the wall y = 0 inside warp 0 of the first row
                    for (nty = 3; nty * ntx <= sms * per_sm && !okY; ++nty) okY = split_wb(G, H, v.R, halo, nty, CH, EB);
                    if (okY) --nty;
                }
                if (!okY) continue;
                const int ntiles = ntx * nty;
                if (ntiles < 2 || ntiles > sms * per_sm) continue;
                // Cost per sweep in SM cycles, calibrated on B200 (profiles/r2b_*.md): a colour half-sweep takes ~187 cycles per warp
                // of the busiest SM sub-partition (+ barrier), an exchange ~5000 cycles of latency + 130 per point of halo depth.
                const double cost = sweep_cost + (5000.0 + 130.0 * halo) / T;
                c.T = T; c.halo = halo; c.CW = CW; c.CH = CH; c.EB = EB; c.ntx = ntx; c.nty = nty; c.ntiles = ntiles;
                if (cost < best_cost && finish_plan(c, N, smem_cta)) { best_cost = cost; best = c; }
            }
        }
    }
    return best;
}

ResidentPlan resident_plan(const Params& P, int device, int T_override, int variant_override, int kind) {
    ResidentPlan best;
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) { cudaGetLastError(); return best; }
    int coop = 0;
    cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, device);
    if (!coop) return best;
    const int sms = prop.multiProcessorCount;
    const int smem_cap = std::min((int)prop.sharedMemPerBlockOptin, (int)prop.sharedMemPerMultiprocessor - (int)prop.reservedSharedMemPerBlock);
    best = resident_plan_for(P.N, kind, T_override, variant_override, sms, smem_cap, (int)prop.regsPerBlock);
    if (best.ok) {
        const void* fn = best.fixup ? VARIANTS[best.variant].fn_fix[kind] : VARIANTS[best.variant].fn[kind];
        cudaFuncAttributes fa;
        if (cudaFuncGetAttributes(&fa, fn) != cudaSuccess || fa.numRegs * 32 * best.warps > (int)prop.regsPerBlock ||
            cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)prop.sharedMemPerBlockOptin) != cudaSuccess) {
            cudaGetLastError();
            best.ok = false;
            return best;
        }
        best.regs = fa.numRegs;
        int per_sm = 0;
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, fn, 32 * best.warps, best.smem_bytes) != cudaSuccess ||
            per_sm * sms < best.ntiles) {
            cudaGetLastError();
            best.ok = false;
        }
    }
    return best;
}

// Host-side check of the exchange pattern of a plan (no device needed): every unit a tile fetches must be stored by
// exactly one tile, its owner, and lie in the rows / columns both agree on; every stored unit must be fetched by someone.
// counts[0] = units fetched, [1] = units stored, [2] = fetched but stored by nobody or by more than one, [3] = stored but
// fetched by nobody, [4] = tiles that do not fit their thread grid.  Returns 0 if [2] = [3] = [4] = 0.
int resident_check_exchange(const ResidentPlan& pl, int N, long long* counts) {
    long long c[5] = {0, 0, 0, 0, 0};
    if (pl.ok && pl.ntiles > 1 && pl.C == 4 && pl.R == 6) {
        const int upitch = resident_unit_pitch(N);
        const size_t nunits = (size_t)upitch * (size_t)(N + 1);
        std::vector<unsigned char> stored(nunits, 0), fetched(nunits, 0);
        const bool walls = pl.kind == 1;
        for (int bj = 0; bj < pl.nty; ++bj)
            for (int bi = 0; bi < pl.ntx; ++bi) {
                const TileGeom t = tile_geom(N, pl.CW, pl.CH, pl.EB, pl.halo, pl.ntx, pl.nty, bi, bj, 4, 6, 128, pl.warps * 6);
                if (!t.fits) ++c[4];
                for (int warp = 0; warp < pl.warps; ++warp)
                    for (int lane = 0; lane < 32; ++lane) {
                        unsigned int info; int ubase;
                        xchg_setup<4, 6>(N, pl.halo, walls, pl.ntx, pl.nty, upitch, t, lane, warp, bi, bj, info, ubase);
                        for (int rj = 0; rj < 6; ++rj) {
                            const long long u = (long long)ubase + (long long)rj * upitch;
                            if ((info >> rj) & 1u) { if (u < 0 || (size_t)u >= nunits) ++c[2]; else { ++c[1]; if (stored[(size_t)u] < 255) ++stored[(size_t)u]; } }
                            if ((info >> (8 + rj)) & 1u) { if (u < 0 || (size_t)u >= nunits) ++c[2]; else { ++c[0]; if (fetched[(size_t)u] < 255) ++fetched[(size_t)u]; } }
                        }
                    }
            }
        for (size_t u = 0; u < nunits; ++u) {
            if (fetched[u] && stored[u] != 1) ++c[2];
            if (stored[u] > 1) ++c[2];
            if (stored[u] && !fetched[u]) ++c[3];
        }
    }
    if (counts) for (int k = 0; k < 5; ++k) counts[k] = c[k];
    return (c[2] || c[3] || c[4]) ? 1 : 0;
}

void resident_describe(const ResidentPlan& pl, char* buf, int len) {
    if (!pl.ok) { std::snprintf(buf, (size_t)len, "none"); return; }
    if (pl.ntiles == 1)
        std::snprintf(buf, (size_t)len, "%s1 tile, %d warps x (%dx%d micro-tiles), whole time steps on chip, %d regs, %d B smem",
                      pl.kind == 1 ? "compact 9-point operator, " : "", pl.warps, pl.C, pl.R, pl.regs, pl.smem_bytes);
    else
        std::snprintf(buf, (size_t)len,
                      "%s%dx%d tiles of %dx%d core + halo %d, T=%d sweeps per exchange, %d warps x (%dx%d micro-tiles), "
                      "register-to-register exchange of 40-byte units of four points, %d regs, %d B smem, %d CTA(s) per SM on %d SMs",
                      pl.kind == 1 ? "compact 9-point operator, " : "", pl.ntx, pl.nty, pl.CW, pl.CH, pl.halo, pl.T, pl.warps, pl.C, pl.R, pl.regs,
                      pl.smem_bytes, pl.per_sm, pl.sm_count);
}

int resident_variants() { return NVARIANTS; }

long long resident_rounds(const ResidentPlan& pl, int nsteps, int S) {
    if (!pl.ok || pl.ntiles <= 1) return 0;
    const long long nrounds = (S + pl.T - 1) / pl.T;
    return nsteps > 0 ? (long long)nsteps * 5 * (nrounds + 1) : std::max(nrounds - 1, 0LL);
}

int resident_launch(const Params& P, const ResidentPlan& pl, const double* psi_in, double* psi_out, void* xa, void* xb,
                    double* wbase, size_t fstride, unsigned int* err_word, unsigned int* epoch,
                    int nsteps, int S, cudaStream_t st, long long* trace_dev, int trace_cap) {
    if (!pl.ok) return -(int)cudaErrorNotSupported;
    if (nsteps < 0 || S < 0 || (nsteps == 0 && S == 0) || psi_in == psi_out || (pl.ntiles > 1 && (!xa || !xb)))
        return -(int)cudaErrorInvalidValue;
    ResArgs a{};
    a.N = P.N; a.pitch = P.pitch; a.cb = P.cb; a.omb = P.omb; a.cq = P.cq;
    a.c9e = P.c9e; a.c9c = P.c9c; a.c9q = P.c9q;
    a.i2h = P.i2h; a.ih2 = P.ih2; a.nu = P.nu; a.c2h2 = P.c2h2; a.lid = P.lid; a.dt = P.dt;
    a.psi_in = psi_in; a.psi_out = psi_out; a.wbase = wbase; a.fstride = fstride;
    a.x0 = (char*)xa; a.x1 = (char*)xb; a.upitch = resident_unit_pitch(P.N);
    a.p1off = resident_plane_bytes(P.N, 16); a.p2off = 2 * resident_plane_bytes(P.N, 16);
    a.walls = pl.kind == 1;
    a.err = err_word;
    a.base = *epoch;
    a.nsteps = nsteps; a.S = S;
    a.T = pl.ntiles == 1 ? std::max(S, 1) : pl.T;
    a.halo = pl.halo; a.CW = pl.CW; a.CH = pl.CH; a.EB = pl.EB; a.ntx = pl.ntx; a.nty = pl.nty;
    a.trace = trace_dev; a.trace_cap = trace_cap;
    *epoch += (unsigned int)resident_rounds(pl, nsteps, S);      // wraps harmlessly: tags only tell round r from round r - 2
    void* args[] = {&a};
    const dim3 grid(pl.ntx, pl.nty), block(32, pl.warps);
    const void* fn = pl.fixup ? VARIANTS[pl.variant].fn_fix[pl.kind] : VARIANTS[pl.variant].fn[pl.kind];
    const cudaError_t e = cudaLaunchCooperativeKernel(fn, grid, block, args, (size_t)pl.smem_bytes, st);
    if (e != cudaSuccess) { cudaGetLastError(); return -(int)e; }
    return 1;
}

}  // namespace cavk
