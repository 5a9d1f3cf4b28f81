// cavity_scheme.cuh — the pointwise arithmetic of a2 and a3, in ONE place for every engine of the product.
//
// Included by cavity_kernels.cu (one thread per point over global memory) and cavity_resident.cu (register / shared-memory
// tiles): both evaluate eq 25 (Thom), eq 22 + eq 8 (velocities and transport right-hand side) and eq 9-13 (the SSPRK(5,4)
// combination) through the functions below, so the two engines cannot drift apart.  Product code only: the test oracle
// (oracle/) types the scheme out on its own and shares nothing with this file.
// Build with -fmad=false: the association is exactly what is written.
// P:n = /root/reference/PAPER.md line n.
#pragma once

namespace cavk {
namespace scheme {

// SSPRK(5,4) in Shu-Osher form, eq 9-13 P:85-108.  eq 9's constant is printed with 11 digits and eq 10's second weight with a
// wrong digit (0.555626...); the values below are the 15-digit ones of the paper's ref [23], which make every
// stage's weights sum to 1 (readings G1, G2).
__device__ constexpr double RK1_C  = 0.391752226571890;
__device__ constexpr double RK2_A0 = 0.444370493651235, RK2_A1 = 0.555629506348765, RK2_C = 0.368410593050371;
__device__ constexpr double RK3_A0 = 0.620101851488403, RK3_A2 = 0.379898148511597, RK3_C = 0.251891774271694;
__device__ constexpr double RK4_A0 = 0.178079954393132, RK4_A3 = 0.821920045606868, RK4_C = 0.544974750228521;
__device__ constexpr double RK5_A2 = 0.517231671970585, RK5_A3 = 0.096059710526147, RK5_C3 = 0.063692468666290;
__device__ constexpr double RK5_A4 = 0.386708617503269, RK5_C4 = 0.226007483236906;

// a2, eq 25: omega_wall = -2 psi_adjacent / h^2 (c2h2 = 2 / h^2), minus 2U/h (lid = 2U/h) on the moving wall
__device__ __forceinline__ double thom_wall(double c2h2, double p_adj) { return -(c2h2 * p_adj); }
__device__ __forceinline__ double thom_lid(double c2h2, double lid, double p_adj) { return -(c2h2 * p_adj) - lid; }

// a3: dt L(psi, omega) at one interior point.  eq 22: u = dpsi/dy, v = -dpsi/dx (second-order central differences,
// i2h = 1 / (2h));  eq 8: L = nu lap(omega) - (u omega_x + v omega_y), ih2 = 1 / h^2.
__device__ __forceinline__ double transport_dL(double pW, double pE, double pS, double pN, double w0, double wW, double wE,
                                               double wS, double wN, double i2h, double ih2, double nu, double dt) {
    const double u = (pN - pS) * i2h;
    const double v = (pW - pE) * i2h;
    const double wx = (wE - wW) * i2h;
    const double wy = (wN - wS) * i2h;
    const double lap = (((wW + wE) + (wS + wN)) - 4.0 * w0) * ih2;
    const double L = fma(nu, lap, -fma(u, wx, v * wy));
    return dt * L;
}

// eq 9-13 in one form: stage k's output = fma(c, dL, inner), inner = w0 (eq 9) or fma(a1, w0, a0 * av), where w0 is the
// stage's input vorticity and av the other operand: omega^n for k = 2..4, T for k = 5 (a0 = 1: eq 13's remaining terms).
__device__ __forceinline__ double rk_c(int k) { return k == 1 ? RK1_C : (k == 2 ? RK2_C : (k == 3 ? RK3_C : (k == 4 ? RK4_C : RK5_C4))); }
__device__ __forceinline__ double rk_a1(int k) { return k == 2 ? RK2_A1 : (k == 3 ? RK3_A2 : (k == 4 ? RK4_A3 : RK5_A4)); }
__device__ __forceinline__ double rk_a0(int k) { return k == 2 ? RK2_A0 : (k == 3 ? RK3_A0 : (k == 4 ? RK4_A0 : 1.0)); }
__device__ __forceinline__ double rk_stage_out(int k, double c, double a1, double a0, double dL, double w0, double av) {
    const double inner = k == 1 ? w0 : fma(a1, w0, a0 * av);
    return fma(c, dL, inner);
}
// stage 4 also leaves T = the first three terms of eq 13 (w2 = omega^(2)), so that L(omega^(3)) need not be kept
__device__ __forceinline__ double rk_T(double dL, double w3, double w2) { return fma(RK5_C3, dL, fma(RK5_A3, w3, RK5_A2 * w2)); }

}  // namespace scheme
}  // namespace cavk
