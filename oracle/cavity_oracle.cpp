// ORACLE — TEST INFRASTRUCTURE ONLY.
//
// Plain, slow, single-threaded fp64 restatement of the hot path of arXiv 0809.3098
// (Cardoso & Bicudo): one SSPRK(5,4) time step of the vorticity / stream-function
// lid-driven cavity.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
// --impl reference legs may build, load or call this file.  It shares no code, header,
// constant table or helper with the CUDA path in paper_0809_3098_b200/csrc/.
//
// P:n = /root/reference/PAPER.md line n.  S8(c) = SURVEY.md section 8(c).
//
// What it computes (state psi, omega on the (N+1)x(N+1) grid, h = 1/N, nu = 1/Re, lid speed U):
//
//   step():                                                   eq 9-13
//     w0 <- omega
//     for stage k = 1..5 with w_in = w0, w1, w2, w3, w4:
//       (a1) S times: red half-sweep then black half-sweep of the 5-point SOR on psi
//            with right-hand side w_in                        eq 15-21, reduced (see sor_point)
//       (a2) Thom wall vorticity of w_in from psi             eq 25
//       (a3) dL = dt * L(psi, w_in) at interior points        eq 8, eq 22
//            then the stage combination                       eq 9-13
//     omega <- w5, ring of omega <- ring computed at k = 5;  t <- t + dt
//
// Readings of the paper used here (DESIGN.md lists them all):
//   G1  eq 10 second weight is 0.555629506348765 (printed 0.555626... is a misprint: weights must sum to 1)
//   G2  eq 9 constant is the 15-digit 0.391752226571890 of ref [23] (printed with 11 digits)
//   G7  order inside a stage: Poisson sweeps -> wall vorticity -> RHS + combination (Figure 2 is missing)
//   G9  red = (i + j) even, swept first; then black
//   G10 top and bottom walls own the four corners of omega; left/right walls cover j = 1..N-1
//   D1-D3 (BASELINE.json): 2nd-order 5-point operator, red-black order, fixed sweep count S, warm start
//
// Arithmetic modes:
//   ORC_MODE_PLAIN (default, the 1e-10 contract): every formula is written the way the paper
//     prints it (divisions by dx^2, 2 dx, no fused multiply-add; build with -ffp-contract=off).
//   ORC_MODE_FMA (S8(c) G20, Appendix A of SURVEY.md): same algorithm, expressions associated as
//     SURVEY Appendix A states, with std::fma.  A red-black sweep has no order dependence inside a
//     colour, so any implementation using that association must agree with this mode BIT FOR BIT;
//     a non-zero difference is an indexing / halo / barrier bug, not rounding.
//
// Pins (tests/test_oracle_pins.py, run with -m "not gpu"): manufactured Poisson solution and its
// closed-form discrete eigenvalue, exactness on quadratics, Thom on a quadratic wall profile,
// SSPRK(5,4) stability polynomial + 4th-order convergence, Young's SOR rate, dense direct solve
// on 9x9, wall/fixed-point invariants, and the composed whole step: bit-exact recomposition in numpy from the
// operator-level entry points (orc_sor / orc_jacobi / orc_compact, orc_thom, orc_rhs) in the order above.
// No function of this file is "parity unpinned".

#include <cmath>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

#define ORC_API extern "C" __attribute__((visibility("default")))

enum { ORC_OK = 0, ORC_EINVAL = -1, ORC_ENOMEM = -2 };
enum { ORC_MODE_PLAIN = 0, ORC_MODE_FMA = 1 };
// (a1) variants: red-black SOR of the 5-point operator (default) / damped Jacobi (NEXT-3) / the paper's own 4th-order
// compact 9-point operator relaxed in four colours (NEXT-1)
enum { ORC_SWEEP_REDBLACK = 0, ORC_SWEEP_JACOBI = 1, ORC_SWEEP_COMPACT9 = 2 };

struct orc_diag {
    double t;
    long long step;
    double res_inf;
    double res_l2;
    double kinetic_energy;
    double enstrophy;
};

struct orc_ctx {
    int N;            // intervals per side; N+1 points per side
    int S;            // SOR sweeps per stage
    int mode;
    int sweep;        // ORC_SWEEP_*
    double Re, dt, beta, U;
    double t;
    long long step;
    std::vector<double> psi, w;           // state
    std::vector<double> w1, w2, w3, w4;   // stage values, one buffer each (no aliasing: obviousness over memory)
};

namespace {

// SSPRK(5,4), Shu-Osher form, eq 9-13 P:85-108 with readings G1, G2.
const double K1_C   = 0.391752226571890;   // eq 9  (G2)
const double K2_A0  = 0.444370493651235;   // eq 10
const double K2_A1  = 0.555629506348765;   // eq 10 (G1)
const double K2_C   = 0.368410593050371;
const double K3_A0  = 0.620101851488403;   // eq 11
const double K3_A2  = 0.379898148511597;
const double K3_C   = 0.251891774271694;
const double K4_A0  = 0.178079954393132;   // eq 12
const double K4_A3  = 0.821920045606868;
const double K4_C   = 0.544974750228521;
const double K5_A2  = 0.517231671970585;   // eq 13
const double K5_A3  = 0.096059710526147;
const double K5_C3  = 0.063692468666290;
const double K5_A4  = 0.386708617503269;
const double K5_C4  = 0.226007483236906;

inline size_t idx(int N, int i, int j) { return (size_t)j * (size_t)(N + 1) + (size_t)i; }

// ---- (a1) one SOR point update -------------------------------------------------------------
// eq 15 P:116 with the 5-point operator: C = 0 (no psi_xxyy term), B = omega_ij, and the centre
// coefficient 2a instead of (5/3)a:  psi <- (beta / (2a)) (A + B) + (1 - beta) psi,
// A = b (psi_E + psi_W) + c (psi_N + psi_S)  (eq 16),  a = b + c, b = 1/dx^2, c = 1/dy^2 (eq 19-21).
inline double sor_point_plain(double pW, double pE, double pS, double pN, double p, double w,
                              double beta, double dx, double dy) {
    const double b = 1.0 / (dx * dx);
    const double c = 1.0 / (dy * dy);
    const double a = b + c;
    const double A = b * (pE + pW) + c * (pN + pS);
    const double B = w;
    return (beta / (2.0 * a)) * (A + B) + (1.0 - beta) * p;
}

// SURVEY Appendix A association: nb = (W + E) + (S + N); p = fma(1-beta, p, fma(beta/4, nb, (beta/4 h^2) w)).
inline double sor_point_fma(double pW, double pE, double pS, double pN, double p, double w,
                            double beta, int N) {
    const double h = 1.0 / (double)N;
    const double cb = 0.25 * beta;
    const double cq = (0.25 * beta) * (h * h);
    const double omb = 1.0 - beta;
    const double nb = (pW + pE) + (pS + pN);
    return std::fma(omb, p, std::fma(cb, nb, cq * w));
}

void sor_half_sweep(int N, int mode, double beta, std::vector<double>& psi, const std::vector<double>& w,
                    int colour) {
    const double h = 1.0 / (double)N;
    for (int j = 1; j <= N - 1; ++j) {
        for (int i = 1; i <= N - 1; ++i) {
            if (((i + j) & 1) != colour) continue;   // G9: colour 0 (red) = (i + j) even
            const double pW = psi[idx(N, i - 1, j)], pE = psi[idx(N, i + 1, j)];
            const double pS = psi[idx(N, i, j - 1)], pN = psi[idx(N, i, j + 1)];
            const double p = psi[idx(N, i, j)];
            const double wij = w[idx(N, i, j)];
            psi[idx(N, i, j)] = (mode == ORC_MODE_FMA) ? sor_point_fma(pW, pE, pS, pN, p, wij, beta, N)
                                                        : sor_point_plain(pW, pE, pS, pN, p, wij, beta, h, h);
        }
    }
}

void sor_sweeps(int N, int mode, double beta, std::vector<double>& psi, const std::vector<double>& w, int nsweeps) {
    for (int s = 0; s < nsweeps; ++s) {
        sor_half_sweep(N, mode, beta, psi, w, 0);   // red first (G9)
        sor_half_sweep(N, mode, beta, psi, w, 1);   // then black
    }
}

// ---- (a1, NEXT-3 variant) damped Jacobi sweeps ------------------------------------------------
// BASELINE.json north_star allows "red-black SOR (or Jacobi)"; every interior point is relaxed from the
// OLD values only,  psi_new = psi + beta ( (psi_W + psi_E + psi_S + psi_N + h^2 w) / 4 - psi ),  i.e. eq 15 P:116 without the
// "use new values when available" of P:114.  The point formula is the one of the red-black sweep (sor_point_*); only the
// data it reads differs (a second buffer).
void jacobi_sweeps(int N, int mode, double beta, std::vector<double>& psi, const std::vector<double>& w, int nsweeps) {
    const double h = 1.0 / (double)N;
    std::vector<double> old(psi.size());
    for (int s = 0; s < nsweeps; ++s) {
        old = psi;
        for (int j = 1; j <= N - 1; ++j) {
            for (int i = 1; i <= N - 1; ++i) {
                const double pW = old[idx(N, i - 1, j)], pE = old[idx(N, i + 1, j)];
                const double pS = old[idx(N, i, j - 1)], pN = old[idx(N, i, j + 1)];
                const double p = old[idx(N, i, j)], wij = w[idx(N, i, j)];
                psi[idx(N, i, j)] = (mode == ORC_MODE_FMA) ? sor_point_fma(pW, pE, pS, pN, p, wij, beta, N)
                                                            : sor_point_plain(pW, pE, pS, pN, p, wij, beta, h, h);
            }
        }
    }
}

// ---- (a1, NEXT-1 variant) the paper's fourth-order compact operator, eq 14-21 P:110-138 --------
// eq 15:  psi <- (3/5) (beta / a) (A + B + C) + (1 - beta) psi,  with (eq 16-21, dx = dy = h, a = b + c, b = c = 1/h^2)
//   A = b (psi_E + psi_W) + c (psi_N + psi_S)
//   B = (1/12) (w_E + w_N + 8 w_0 + w_W + w_S)                      (reads the wall ring of omega next to a wall)
//   C = (a/12) (psi_NE - 2 psi_N + psi_NW - 2 psi_E - 2 psi_W + psi_SE - 2 psi_S + psi_SW)
// (eq 17 is printed twice and the tags (17)/(18) are displaced, G3; C is the expression printed above tag (18).)
// ORDER (reading, N1): the paper relaxes lexicographically, "use the new values when they become available"
// (P:114); its superscripts in eq 18 fit no single order (G3).  A 9-point stencil decouples under FOUR colours
// (i mod 2, j mod 2), so both sides sweep colour (0,0), then (1,0), (0,1), (1,1), each from the latest values: inside a
// colour no point reads another point of that colour, so the result does not depend on the order inside a colour.
inline double compact_point_plain(const std::vector<double>& psi, const std::vector<double>& w, int N, int i, int j,
                                  double beta) {
    const double dx = 1.0 / (double)N, dy = 1.0 / (double)N;
    const double b = 1.0 / (dx * dx), c = 1.0 / (dy * dy), a = b + c;
    const double A = b * (psi[idx(N, i + 1, j)] + psi[idx(N, i - 1, j)]) + c * (psi[idx(N, i, j + 1)] + psi[idx(N, i, j - 1)]);
    const double B = (1.0 / 12.0) * (w[idx(N, i + 1, j)] + w[idx(N, i, j + 1)] + 8.0 * w[idx(N, i, j)] + w[idx(N, i - 1, j)] +
                                     w[idx(N, i, j - 1)]);
    const double C = (1.0 / 12.0) * a *
                     (psi[idx(N, i + 1, j + 1)] - 2.0 * psi[idx(N, i, j + 1)] + psi[idx(N, i - 1, j + 1)] - 2.0 * psi[idx(N, i + 1, j)] -
                      2.0 * psi[idx(N, i - 1, j)] + psi[idx(N, i + 1, j - 1)] - 2.0 * psi[idx(N, i, j - 1)] + psi[idx(N, i - 1, j - 1)]);
    return (3.0 / 5.0) * (beta / a) * (A + B + C) + (1.0 - beta) * psi[idx(N, i, j)];
}
// The same update collected as  psi <- (1 - beta) psi + 0.2 beta S_edge + 0.05 beta S_corner + (0.025 beta h^2) (S_edge(w) + 8 w_0)
// with the association DESIGN.md "Canonical arithmetic" states for the kernels.
inline double compact_point_fma(const std::vector<double>& psi, const std::vector<double>& w, int N, int i, int j,
                                double beta) {
    const double h = 1.0 / (double)N;
    const double c1 = 0.2 * beta, c2 = 0.05 * beta, c3 = (0.025 * beta) * (h * h), omb = 1.0 - beta;
    const double se = (psi[idx(N, i - 1, j)] + psi[idx(N, i + 1, j)]) + (psi[idx(N, i, j - 1)] + psi[idx(N, i, j + 1)]);
    const double sc = (psi[idx(N, i - 1, j - 1)] + psi[idx(N, i + 1, j - 1)]) + (psi[idx(N, i - 1, j + 1)] + psi[idx(N, i + 1, j + 1)]);
    const double sw = ((w[idx(N, i - 1, j)] + w[idx(N, i + 1, j)]) + (w[idx(N, i, j - 1)] + w[idx(N, i, j + 1)])) + 8.0 * w[idx(N, i, j)];
    const double qB = c3 * sw;
    return std::fma(omb, psi[idx(N, i, j)], std::fma(c1, se, std::fma(c2, sc, qB)));
}

void compact_sweeps(int N, int mode, double beta, std::vector<double>& psi, const std::vector<double>& w, int nsweeps) {
    for (int s = 0; s < nsweeps; ++s)
        for (int colour = 0; colour < 4; ++colour)               // (i mod 2, j mod 2) = (0,0), (1,0), (0,1), (1,1)
            for (int j = 1; j <= N - 1; ++j)
                for (int i = 1; i <= N - 1; ++i) {
                    if ((i & 1) + 2 * (j & 1) != colour) continue;
                    psi[idx(N, i, j)] = (mode == ORC_MODE_FMA) ? compact_point_fma(psi, w, N, i, j, beta)
                                                                : compact_point_plain(psi, w, N, i, j, beta);
                }
}

// NEXT-3 (oracle only): the sweep order the paper itself describes: lexicographic, "use the current estimates of
// psi when they become available" (Gauss-Seidel with relaxation factor beta, eq 15), here i inner, j outer.  A serial
// recurrence: it has no GPU counterpart (reading N1 replaces it by four colours on both sides); it exists so that the paper's
// own order and its under-relaxed range beta = 0.8 ... 0.1 can be exercised and compared with the four-colour order.
void compact_sweeps_lex(int N, int mode, double beta, std::vector<double>& psi, const std::vector<double>& w, int nsweeps) {
    for (int s = 0; s < nsweeps; ++s)
        for (int j = 1; j <= N - 1; ++j)
            for (int i = 1; i <= N - 1; ++i)
                psi[idx(N, i, j)] = (mode == ORC_MODE_FMA) ? compact_point_fma(psi, w, N, i, j, beta)
                                                            : compact_point_plain(psi, w, N, i, j, beta);
}

void poisson_sweeps(const orc_ctx* c, std::vector<double>& psi, const std::vector<double>& w, int nsweeps) {
    if (c->sweep == ORC_SWEEP_COMPACT9) compact_sweeps(c->N, c->mode, c->beta, psi, w, nsweeps);
    else if (c->sweep == ORC_SWEEP_JACOBI) jacobi_sweeps(c->N, c->mode, c->beta, psi, w, nsweeps);
    else sor_sweeps(c->N, c->mode, c->beta, psi, w, nsweeps);
}

// ---- (a2) Thom wall vorticity, eq 25 P:161-169 ----------------------------------------------
// omega_{i,1} = -2 psi_{i,2}/dx^2 ; omega_{i,ny} = -2 psi_{i,ny-1}/dx^2 - 2U/dx ;
// omega_{1,j} = -2 psi_{2,j}/dy^2 ; omega_{nx,j} = -2 psi_{nx-1,j}/dy^2   (paper is 1-based; dx = dy = h, G4)
// G10: the bottom and top rows run over i = 0..N (they own the corners); side walls over j = 1..N-1.
void thom(int N, int mode, double U, const std::vector<double>& psi, std::vector<double>& w) {
    const double h = 1.0 / (double)N;
    if (mode == ORC_MODE_FMA) {
        const double c2h2 = 2.0 * ((double)N * (double)N);
        const double lid = 2.0 * U * (double)N;
        for (int i = 0; i <= N; ++i) {
            w[idx(N, i, 0)] = -(c2h2 * psi[idx(N, i, 1)]);
            w[idx(N, i, N)] = -(c2h2 * psi[idx(N, i, N - 1)]) - lid;
        }
        for (int j = 1; j <= N - 1; ++j) {
            w[idx(N, 0, j)] = -(c2h2 * psi[idx(N, 1, j)]);
            w[idx(N, N, j)] = -(c2h2 * psi[idx(N, N - 1, j)]);
        }
        return;
    }
    const double dx = h, dy = h;
    for (int i = 0; i <= N; ++i) {
        w[idx(N, i, 0)] = -2.0 * psi[idx(N, i, 1)] / (dx * dx);
        w[idx(N, i, N)] = -2.0 * psi[idx(N, i, N - 1)] / (dx * dx) - 2.0 * U / dx;
    }
    for (int j = 1; j <= N - 1; ++j) {
        w[idx(N, 0, j)] = -2.0 * psi[idx(N, 1, j)] / (dy * dy);
        w[idx(N, N, j)] = -2.0 * psi[idx(N, N - 1, j)] / (dy * dy);
    }
}

// ---- (a3) transport right-hand side L(omega), eq 8 P:80 with eq 22 P:142 --------------------
inline double rhs_point_plain(const std::vector<double>& psi, const std::vector<double>& w, int N, int i, int j,
                              double nu) {
    const double dx = 1.0 / (double)N, dy = 1.0 / (double)N;
    const double u = (psi[idx(N, i, j + 1)] - psi[idx(N, i, j - 1)]) / (2.0 * dy);        // eq 22
    const double v = -(psi[idx(N, i + 1, j)] - psi[idx(N, i - 1, j)]) / (2.0 * dx);       // eq 22
    const double wE = w[idx(N, i + 1, j)], wW = w[idx(N, i - 1, j)];
    const double wN = w[idx(N, i, j + 1)], wS = w[idx(N, i, j - 1)];
    const double w0 = w[idx(N, i, j)];
    return -u * (wE - wW) / (2.0 * dx) - v * (wN - wS) / (2.0 * dy)
           + nu * ((wE - 2.0 * w0 + wW) / (dx * dx) + (wN - 2.0 * w0 + wS) / (dy * dy));   // eq 8
}

// SURVEY Appendix A association.
inline double rhs_point_fma(const std::vector<double>& psi, const std::vector<double>& w, int N, int i, int j,
                            double nu) {
    const double i2h = 0.5 * (double)N;
    const double ih2 = (double)N * (double)N;
    const double pN = psi[idx(N, i, j + 1)], pS = psi[idx(N, i, j - 1)];
    const double pE = psi[idx(N, i + 1, j)], pW = psi[idx(N, i - 1, j)];
    const double wE = w[idx(N, i + 1, j)], wW = w[idx(N, i - 1, j)];
    const double wN = w[idx(N, i, j + 1)], wS = w[idx(N, i, j - 1)];
    const double w0 = w[idx(N, i, j)];
    const double u = (pN - pS) * i2h;
    const double v = (pW - pE) * i2h;
    const double wx = (wE - wW) * i2h;
    const double wy = (wN - wS) * i2h;
    const double lap = (((wW + wE) + (wS + wN)) - 4.0 * w0) * ih2;
    return std::fma(nu, lap, -std::fma(u, wx, v * wy));
}

inline double rhs_point(int mode, const std::vector<double>& psi, const std::vector<double>& w, int N, int i, int j,
                        double nu) {
    return (mode == ORC_MODE_FMA) ? rhs_point_fma(psi, w, N, i, j, nu) : rhs_point_plain(psi, w, N, i, j, nu);
}

// a*x + b*y  and  (.) + c*dL in the two arithmetic modes.
inline double lin2(int mode, double a, double x, double b, double y) {
    return (mode == ORC_MODE_FMA) ? std::fma(b, y, a * x) : (a * x + b * y);
}
inline double addc(int mode, double s, double c, double dL) {
    return (mode == ORC_MODE_FMA) ? std::fma(c, dL, s) : (s + c * dL);
}

// ---- SSPRK(5,4) stage combinations, eq 9-13, applied to one scalar ----------------------------
// dL = dt * L(w_in of that stage).  Used pointwise by step() and as is by orc_ssprk54_scalar().
inline double stage1(int m, double w0, double dL)                      { return addc(m, w0, K1_C, dL); }
inline double stage2(int m, double w0, double w1, double dL)           { return addc(m, lin2(m, K2_A0, w0, K2_A1, w1), K2_C, dL); }
inline double stage3(int m, double w0, double w2, double dL)           { return addc(m, lin2(m, K3_A0, w0, K3_A2, w2), K3_C, dL); }
inline double stage4(int m, double w0, double w3, double dL)           { return addc(m, lin2(m, K4_A0, w0, K4_A3, w3), K4_C, dL); }
// eq 13 left to right: ((A2 w2 + A3 w3) + C3 dL3) + A4 w4) + C4 dL4
inline double stage5(int m, double w2, double w3, double dL3, double w4, double dL4) {
    const double T = addc(m, lin2(m, K5_A2, w2, K5_A3, w3), K5_C3, dL3);
    const double s = (m == ORC_MODE_FMA) ? std::fma(K5_A4, w4, T) : (T + K5_A4 * w4);
    return addc(m, s, K5_C4, dL4);
}

void one_step(orc_ctx* c) {
    const int N = c->N, m = c->mode;
    const double nu = 1.0 / c->Re;      // Re = U L / nu with U = L = 1
    const double dt = c->dt;
    std::vector<double>& w0 = c->w;
    std::vector<double> dL3((size_t)(N + 1) * (N + 1), 0.0);   // dt L(w3), kept for eq 13

    for (int k = 1; k <= 5; ++k) {
        std::vector<double>& win = (k == 1) ? w0 : (k == 2) ? c->w1 : (k == 3) ? c->w2 : (k == 4) ? c->w3 : c->w4;
        poisson_sweeps(c, c->psi, win, c->S);                   // (a1)
        thom(N, m, c->U, c->psi, win);                          // (a2)
        if (k <= 4) {
            // The stage output carries the wall vorticity just computed.  Nothing on the 5-point path ever reads it (a2 of
            // the next stage overwrites it first); the compact operator's B (eq 17) does, during the next stage's sweeps:
            // "the most recent wall vorticity" (reading N2; the paper is silent).
            std::vector<double>& wout = (k == 1) ? c->w1 : (k == 2) ? c->w2 : (k == 3) ? c->w3 : c->w4;
            for (int i = 0; i <= N; ++i) { wout[idx(N, i, 0)] = win[idx(N, i, 0)]; wout[idx(N, i, N)] = win[idx(N, i, N)]; }
            for (int j = 1; j <= N - 1; ++j) { wout[idx(N, 0, j)] = win[idx(N, 0, j)]; wout[idx(N, N, j)] = win[idx(N, N, j)]; }
        }
        for (int j = 1; j <= N - 1; ++j) {                      // (a3)
            for (int i = 1; i <= N - 1; ++i) {
                const size_t p = idx(N, i, j);
                const double dL = dt * rhs_point(m, c->psi, win, N, i, j, nu);
                switch (k) {
                    case 1: c->w1[p] = stage1(m, w0[p], dL); break;
                    case 2: c->w2[p] = stage2(m, w0[p], c->w1[p], dL); break;
                    case 3: c->w3[p] = stage3(m, w0[p], c->w2[p], dL); break;
                    case 4: c->w4[p] = stage4(m, w0[p], c->w3[p], dL); dL3[p] = dL; break;
                    case 5: w0[p] = stage5(m, c->w2[p], c->w3[p], dL3[p], c->w4[p], dL); break;
                }
            }
        }
    }
    // ring of omega <- ring computed at k = 5 (it sits in w4)
    for (int i = 0; i <= N; ++i) { w0[idx(N, i, 0)] = c->w4[idx(N, i, 0)]; w0[idx(N, i, N)] = c->w4[idx(N, i, N)]; }
    for (int j = 1; j <= N - 1; ++j) { w0[idx(N, 0, j)] = c->w4[idx(N, 0, j)]; w0[idx(N, N, j)] = c->w4[idx(N, N, j)]; }
    c->t += dt;
    c->step += 1;
}

// ---- (a4) diagnostics; sums in long double ------------------------------
void diagnostics(const orc_ctx* c, orc_diag* d) {
    const int N = c->N;
    const double h = 1.0 / (double)N;
    long double s_r2 = 0.0L, s_ke = 0.0L, s_en = 0.0L;
    double rmax = 0.0;
    for (int j = 1; j <= N - 1; ++j) {
        for (int i = 1; i <= N - 1; ++i) {
            const double pE = c->psi[idx(N, i + 1, j)], pW = c->psi[idx(N, i - 1, j)];
            const double pN = c->psi[idx(N, i, j + 1)], pS = c->psi[idx(N, i, j - 1)];
            const double p = c->psi[idx(N, i, j)], w = c->w[idx(N, i, j)];
            const double r = (pW + pE + pS + pN - 4.0 * p) / (h * h) + w;
            const double u = (pN - pS) / (2.0 * h);
            const double v = -(pE - pW) / (2.0 * h);
            if (std::fabs(r) > rmax) rmax = std::fabs(r);
            s_r2 += (long double)r * (long double)r;
            s_ke += (long double)u * (long double)u + (long double)v * (long double)v;
            s_en += (long double)w * (long double)w;
        }
    }
    const long double h2 = (long double)h * (long double)h;
    d->t = c->t;
    d->step = c->step;
    d->res_inf = rmax;
    d->res_l2 = (double)sqrtl(h2 * s_r2);
    d->kinetic_energy = (double)(0.5L * h2 * s_ke);
    d->enstrophy = (double)(0.5L * h2 * s_en);
}

}  // namespace

// ================================ C ABI ========================================================

ORC_API int orc_create(orc_ctx** out, int N, double Re, double dt, double sor_omega, int sweeps_per_stage) {
    if (!out) return ORC_EINVAL;
    *out = nullptr;
    if (N < 2 || !(Re > 0.0) || !(dt > 0.0) || !(sor_omega > 0.0) || !(sor_omega < 2.0) || sweeps_per_stage < 0)
        return ORC_EINVAL;
    orc_ctx* c = new (std::nothrow) orc_ctx();
    if (!c) return ORC_ENOMEM;
    try {
        const size_t G = (size_t)(N + 1) * (size_t)(N + 1);
        c->N = N; c->S = sweeps_per_stage; c->mode = ORC_MODE_PLAIN; c->sweep = ORC_SWEEP_REDBLACK;
        c->Re = Re; c->dt = dt; c->beta = sor_omega; c->U = 1.0;   // P:190 U_wall = 1
        c->t = 0.0; c->step = 0;
        c->psi.assign(G, 0.0); c->w.assign(G, 0.0);
        c->w1.assign(G, 0.0); c->w2.assign(G, 0.0); c->w3.assign(G, 0.0); c->w4.assign(G, 0.0);
    } catch (...) { delete c; return ORC_ENOMEM; }
    *out = c;
    return ORC_OK;
}

ORC_API void orc_destroy(orc_ctx* c) { delete c; }

ORC_API int orc_set_mode(orc_ctx* c, int mode) {
    if (!c || (mode != ORC_MODE_PLAIN && mode != ORC_MODE_FMA)) return ORC_EINVAL;
    c->mode = mode;
    return ORC_OK;
}

ORC_API int orc_set_sweep(orc_ctx* c, int kind) {
    if (!c || kind < ORC_SWEEP_REDBLACK || kind > ORC_SWEEP_COMPACT9) return ORC_EINVAL;
    c->sweep = kind;
    return ORC_OK;
}

// Lid speed (paper: U = 1).  Exposed only so the U = 0 fixed-point invariant can be tested.
ORC_API int orc_set_lid(orc_ctx* c, double U) {
    if (!c) return ORC_EINVAL;
    c->U = U;
    return ORC_OK;
}

// psi == NULL -> psi <- 0.  Wall entries of psi are forced to 0 (eq 23-24 "S = 0", G5).
ORC_API int orc_set_fields(orc_ctx* c, const double* psi, const double* omega) {
    if (!c || !omega) return ORC_EINVAL;
    const int N = c->N;
    const size_t G = (size_t)(N + 1) * (size_t)(N + 1);
    if (psi) std::memcpy(c->psi.data(), psi, G * sizeof(double));
    else c->psi.assign(G, 0.0);
    for (int i = 0; i <= N; ++i) { c->psi[idx(N, i, 0)] = 0.0; c->psi[idx(N, i, N)] = 0.0; }
    for (int j = 0; j <= N; ++j) { c->psi[idx(N, 0, j)] = 0.0; c->psi[idx(N, N, j)] = 0.0; }
    std::memcpy(c->w.data(), omega, G * sizeof(double));
    c->t = 0.0; c->step = 0;
    return ORC_OK;
}

ORC_API int orc_get_fields(const orc_ctx* c, double* psi_out, double* omega_out) {
    if (!c) return ORC_EINVAL;
    const size_t G = (size_t)(c->N + 1) * (size_t)(c->N + 1);
    if (psi_out) std::memcpy(psi_out, c->psi.data(), G * sizeof(double));
    if (omega_out) std::memcpy(omega_out, c->w.data(), G * sizeof(double));
    return ORC_OK;
}

ORC_API int orc_step(orc_ctx* c, int nsteps) {
    if (!c || nsteps < 0) return ORC_EINVAL;
    for (int n = 0; n < nsteps; ++n) one_step(c);
    return ORC_OK;
}

// nsweeps of (a1) on the current (psi, omega), then one (a2); max-norm residual if asked.
ORC_API int orc_poisson(orc_ctx* c, int nsweeps, double* res_inf_out) {
    if (!c || nsweeps < 0) return ORC_EINVAL;
    poisson_sweeps(c, c->psi, c->w, nsweeps);
    thom(c->N, c->mode, c->U, c->psi, c->w);
    if (res_inf_out) { orc_diag d; diagnostics(c, &d); *res_inf_out = d.res_inf; }
    return ORC_OK;
}

ORC_API int orc_get_diag(const orc_ctx* c, orc_diag* out) {
    if (!c || !out) return ORC_EINVAL;
    diagnostics(c, out);
    return ORC_OK;
}

// ---- operator-level entry points for the pins (each calls the very routine step() uses) ------

// L(omega) at interior points (walls of L_out are set to 0); omega's ring is read as given.
ORC_API int orc_rhs(int N, double Re, int mode, const double* psi, const double* omega, double* L_out) {
    if (N < 2 || !psi || !omega || !L_out) return ORC_EINVAL;
    const size_t G = (size_t)(N + 1) * (size_t)(N + 1);
    std::vector<double> p(psi, psi + G), w(omega, omega + G);
    std::memset(L_out, 0, G * sizeof(double));
    for (int j = 1; j <= N - 1; ++j)
        for (int i = 1; i <= N - 1; ++i) L_out[idx(N, i, j)] = rhs_point(mode, p, w, N, i, j, 1.0 / Re);
    return ORC_OK;
}

// Thom ring of omega (in place) from psi.
ORC_API int orc_thom(int N, double U, int mode, const double* psi, double* omega) {
    if (N < 2 || !psi || !omega) return ORC_EINVAL;
    const size_t G = (size_t)(N + 1) * (size_t)(N + 1);
    std::vector<double> p(psi, psi + G), w(omega, omega + G);
    thom(N, mode, U, p, w);
    std::memcpy(omega, w.data(), G * sizeof(double));
    return ORC_OK;
}

// nsweeps red-black SOR sweeps on psi (in place; walls taken as given) with right-hand side omega.
ORC_API int orc_sor(int N, double beta, int mode, double* psi, const double* omega, int nsweeps) {
    if (N < 2 || !psi || !omega || nsweeps < 0) return ORC_EINVAL;
    const size_t G = (size_t)(N + 1) * (size_t)(N + 1);
    std::vector<double> p(psi, psi + G), w(omega, omega + G);
    sor_sweeps(N, mode, beta, p, w, nsweeps);
    std::memcpy(psi, p.data(), G * sizeof(double));
    return ORC_OK;
}

// nsweeps damped-Jacobi sweeps on psi (in place; walls taken as given) with right-hand side omega.
ORC_API int orc_jacobi(int N, double beta, int mode, double* psi, const double* omega, int nsweeps) {
    if (N < 2 || !psi || !omega || nsweeps < 0) return ORC_EINVAL;
    const size_t G = (size_t)(N + 1) * (size_t)(N + 1);
    std::vector<double> p(psi, psi + G), w(omega, omega + G);
    jacobi_sweeps(N, mode, beta, p, w, nsweeps);
    std::memcpy(psi, p.data(), G * sizeof(double));
    return ORC_OK;
}

// nsweeps four-colour sweeps of the paper's compact operator on psi (in place; walls taken as given), RHS omega incl. its ring.
ORC_API int orc_compact(int N, double beta, int mode, double* psi, const double* omega, int nsweeps) {
    if (N < 2 || !psi || !omega || nsweeps < 0) return ORC_EINVAL;
    const size_t G = (size_t)(N + 1) * (size_t)(N + 1);
    std::vector<double> p(psi, psi + G), w(omega, omega + G);
    compact_sweeps(N, mode, beta, p, w, nsweeps);
    std::memcpy(psi, p.data(), G * sizeof(double));
    return ORC_OK;
}

// nsweeps LEXICOGRAPHIC sweeps of the compact operator (the paper's own order; NEXT-3, oracle only).
ORC_API int orc_compact_lex(int N, double beta, int mode, double* psi, const double* omega, int nsweeps) {
    if (N < 2 || !psi || !omega || nsweeps < 0) return ORC_EINVAL;
    const size_t G = (size_t)(N + 1) * (size_t)(N + 1);
    std::vector<double> p(psi, psi + G), w(omega, omega + G);
    compact_sweeps_lex(N, mode, beta, p, w, nsweeps);
    std::memcpy(psi, p.data(), G * sizeof(double));
    return ORC_OK;
}

// NEXT-2: one time step and the paper's steady-state monitors of that step, eq 26-27 P:196-202:
//   RES_psi = (1/N) sum_ij |psi^{n+1}_ij - psi^n_ij|,  RES_omega likewise, sums over ALL grid points, and N = n_x = n_y
// the number of points per side, i.e. c->N + 1 here (reading G17: the literal divisor, not N^2).
// psi^n / psi^{n+1} are the states orc_get_fields returns before / after the step (G16).  Sums in long double.
ORC_API int orc_step_res(orc_ctx* c, double* res_psi_out, double* res_omega_out) {
    if (!c) return ORC_EINVAL;
    const std::vector<double> p0 = c->psi, w0 = c->w;
    one_step(c);
    long double sp = 0.0L, sw = 0.0L;
    for (size_t k = 0; k < p0.size(); ++k) {
        sp += (long double)std::fabs(c->psi[k] - p0[k]);
        sw += (long double)std::fabs(c->w[k] - w0[k]);
    }
    const long double npts = (long double)(c->N + 1);
    if (res_psi_out) *res_psi_out = (double)(sp / npts);
    if (res_omega_out) *res_omega_out = (double)(sw / npts);
    return ORC_OK;
}

// NEXT-2 driver: steps until RES_psi < tol_psi and RES_omega < tol_omega (the paper's stopping rule), checking the
// monitors on every check_every-th step, for at most max_steps steps.  Returns the steps taken in *steps_out and the
// monitors of the last checked step; *converged_out = 1 if the rule was met.
ORC_API int orc_run_to_steady(orc_ctx* c, int max_steps, int check_every, double tol_psi, double tol_omega, int* steps_out,
                              double* res_psi_out, double* res_omega_out, int* converged_out) {
    if (!c || max_steps < 0 || check_every < 1) return ORC_EINVAL;
    double rp = 0.0, rw = 0.0;
    int n = 0, conv = 0;
    while (n < max_steps) {
        if ((n + 1) % check_every == 0) {
            orc_step_res(c, &rp, &rw);
            ++n;
            if (rp < tol_psi && rw < tol_omega) { conv = 1; break; }
        } else {
            one_step(c);
            ++n;
        }
    }
    if (steps_out) *steps_out = n;
    if (res_psi_out) *res_psi_out = rp;
    if (res_omega_out) *res_omega_out = rw;
    if (converged_out) *converged_out = conv;
    return ORC_OK;
}

// nsteps of eq 9-13 on the scalar problem y' = lambda y (the same stage routines step() applies pointwise).
ORC_API double orc_ssprk54_scalar(double lambda, double dt, double y0, int nsteps, int mode) {
    double y = y0;
    for (int n = 0; n < nsteps; ++n) {
        const double w0 = y;
        const double w1 = stage1(mode, w0, dt * (lambda * w0));
        const double w2 = stage2(mode, w0, w1, dt * (lambda * w1));
        const double w3 = stage3(mode, w0, w2, dt * (lambda * w2));
        const double dL3 = dt * (lambda * w3);
        const double w4 = stage4(mode, w0, w3, dL3);
        y = stage5(mode, w2, w3, dL3, w4, dt * (lambda * w4));
    }
    return y;
}
