// math_f64.cuh -- steps S2-S6 of the hot path in double (Table I lines 6-10, PAPER.md:166;
// Eqs. (24),(25)).  Tolerance against the oracle: 1e-12 relative per component.
//
// Every step is the cancellation-free re-association listed in DESIGN.md ("Readings" R3, R7):
//   1 - U      exact, from the integer complement ~w          (PAPER.md:250 turned into an identity)
//   1 - U1^(2/3) = t1 (1+r)/(1+r+r^2),  r = cbrt(U1), t1 = 1-U1   (since 1 - r^3 = t1)
//   (..)^(-1/kappa*) - 1 = expm1(-ln(S)/kappa*)
//   root of Eq. (24): the form whose denominator/numerator adds
//   azimuth: sincospi on 2 U3 (exact in double) = quarter-turn reduction
// No data-dependent branch: selects only ("no loops or conditional statements").
#pragma once
#include <cstdint>
#include "coefs.cuh"

namespace kappagen {

__device__ __forceinline__ double speed_f64(uint32_t w0, const Coef<double>& C) {
    const double u1 = ((double)w0 + 0.5) * 0x1p-32;               // U1 in (0,1), exact
    const double t1 = ((double)(uint32_t)(~w0) + 0.5) * 0x1p-32;  // 1 - U1, exact
    const double r = cbrt(u1);
    const double p = r * r;                                        // U1^(2/3)
    const double S = t1 * (1.0 + r) / (1.0 + r + p);              // 1 - U1^(2/3)
    // ln S with relative accuracy at both ends: S -> 1 (p -> 0) wants log1p(-p), S -> 0 wants log(S)
    const double lnS = (p < 0.5) ? log1p(-p) : log(S);
    const double Y = expm1(-lnS * C.s);                            // S^(-1/kappa*) - 1 = -L/kappa*
    const double A = fma(-C.ck, Y, C.a);                           // a + cL
    const double D = sqrt(fma(A, A, C.bk4 * Y));                   // sqrt((a+cL)^2 - 4bL) > |A|
    const double T = fabs(A) + D;
    const double x = (A >= 0.0) ? (C.k2 * Y) / T : T * C.i2b;      // Eq. (24), the form that adds
    return C.theta * sqrt(x);
}

__device__ __forceinline__ void velocity_f64(uint32_t w0, uint32_t w1, uint32_t w2,
                                             const Coef<double>& C, double& vx, double& vy, double& vz) {
    const double V = speed_f64(w0, C);
    const double u2 = ((double)w1 + 0.5) * 0x1p-32;
    const double t2 = ((double)(uint32_t)(~w1) + 0.5) * 0x1p-32;                  // 1 - U2, exact
    const double mu = ((double)(int32_t)(w1 ^ 0x80000000u) + 0.5) * 0x1p-31;      // 2 U2 - 1, exact
    const double sth = 2.0 * sqrt(u2 * t2);                                        // 2 sqrt(U2 (1-U2))
    double sphi, cphi;
    sincospi(((double)w2 + 0.5) * 0x1p-31, &sphi, &cphi);                          // angle = 2 pi U3
    const double Vs = V * sth;
    vx = V * mu;
    vy = Vs * cphi;
    vz = Vs * sphi;
}

}  // namespace kappagen
