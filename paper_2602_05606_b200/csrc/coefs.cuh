// coefs.cuh -- step S0: Table I lines 1-4 (Eqs. (16),(13),(20),(17)) and the
// per-(kappa,theta) constants the per-particle math consumes.
//
// The per-particle chain is written in terms of Y = (1 - U1^(2/3))^(-1/kappa*) - 1 >= 0, so that
// L = -kappa* Y (Eq. 25) never has to be formed:
//   A    = a + cL            = a  - ck  * Y          ck  = c kappa*
//   disc = (a+cL)^2 - 4bL    = A^2 + bk4 * Y         bk4 = 4 b kappa*
//   x    = -2L / (A + sqrt(disc))   = k2 * Y / (A + D)     k2  = 2 kappa*      (A >= 0)
//        = (-A + sqrt(disc)) / (2b) = (D - A) / b2         b2  = 2b            (A <  0)
// (the two printed forms of Eq. (24)).  V = theta sqrt(x).
#pragma once
#include <cmath>

namespace kappagen {

// Table I lines 1-4 in one precision F (long double on the host, double on the device).
template <typename F>
struct TableIParams {
    F kstar, a, b, c;
};

// Per-(kappa, theta) constants in the kernel's arithmetic type: 64 bytes (double), 32 bytes (float);
// the cells path stores one per cell in the workspace.
template <typename T> struct Coef;

template <>
struct alignas(16) Coef<double> {
    double s;      // 1/kappa*
    double a;      // Eq. (13)
    double ck;     // c kappa*
    double bk4;    // 4 b kappa*
    double k2;     // 2 kappa*
    double b2;     // 2 b
    double theta;  // most probable speed; NaN marks an invalid cell
    double theta2; // 2 theta: the chain carries 2V, so that neither V + V nor 2 U2 - 1 costs an instruction
};

// The float chain returns 2V = sqrt(num/den) with
//   A >= 0: num = k2 Y, den = T;   A < 0: num = th4 T, den = b2;   T = |A| + sqrt(A^2 + bk4 Y).
// Folded (uniform parameters, theta in [2^-30, 2^30]): k2 = 8 kappa* theta^2, th4 = 4 theta^2, theta = 1,
// so the speed needs no further multiply.  Unfolded (per-cell parameters, theta = 0 or extreme):
// k2 = 8 kappa*, th4 = 4, and the kernel multiplies by theta (NaN marks an invalid cell).
template <>
struct alignas(16) Coef<float> {
    float s;      // 1/kappa*
    float a;      // Eq. (13)
    float ck;     // c kappa*
    float bk4;    // 4 b kappa*
    float k2;     // 8 kappa* [theta^2]
    float b2;     // 2 b
    float th4;    // 4 [theta^2]
    float theta;  // theta, or 1 when folded
};

// Workspace record of one cell (kappagen_sample_cells): the constants of the per-particle chain -- the two that the
// chain uses negated stored negated -- and the cell's drift: 12 values, 48 bytes (float) / 96 bytes (double), written
// once by the pre-kernel and read once per 128-bit particle group, so that the sampling kernel has neither a drift
// pointer nor a drift branch.
template <typename T> struct CellRec;
template <>
struct alignas(16) CellRec<float> {
    float s, ms, a, mck;       // 1/kappa*, -1/kappa*, a, -c kappa*
    float bk4, k2, b2, th4;    // as Coef<float>, never folded
    float theta, dx, dy, dz;   // theta (NaN marks an invalid cell), drift
};
template <>
struct alignas(16) CellRec<double> {
    Coef<double> C;
    double dx, dy, dz, pad;
};

#ifdef __CUDACC__
#define KAPPAGEN_HD __host__ __device__
#else
#define KAPPAGEN_HD
#endif

// c_approx, Eq. (20), in double without losing digits.  Both quadratics nearly vanish
// around kappa ~ 4-4.6 (denominator 0.037 at kappa = 3.95 from terms of size 31), so a plain double
// evaluation amplifies rounding by ~1e3.  The printed 3-digit decimals are exact ratios of integers:
//   c = (123 k^2 - 1120 k + 2560) / (10 (100 k^2 - 789 k + 1560)),
// and each quadratic is evaluated by Horner in double-double (error-free product/sum via fma).
KAPPAGEN_HD inline double quad_dd(double c2, double c1, double c0, double k) {
    const double ah = c2 * k, al = fma(c2, k, -ah);            // c2 k = ah + al exactly
    const double s = ah + c1, bb = s - ah;
    const double e = (ah - (s - bb)) + (c1 - bb) + al;         // (c2 k + c1) = s + e
    const double ph = s * k, pl = fma(s, k, -ph) + e * k;      // (s + e) k = ph + pl
    const double r = ph + c0, cc = r - ph;
    const double re = (ph - (r - cc)) + (c0 - cc);
    return r + (re + pl);
}
KAPPAGEN_HD inline double c_approx_f64(double kappa) {
    return quad_dd(123.0, -1120.0, 2560.0, kappa) / (10.0 * quad_dd(100.0, -789.0, 1560.0, kappa));
}

// a and b from ln B(3/2, kappa*) and c (the caller supplies both: lgammal and long double arithmetic on
// the host, lgamma and c_approx_f64 on the device; "B(a,b) = Gamma(a)Gamma(b)/Gamma(a+b)").
template <typename F>
KAPPAGEN_HD inline TableIParams<F> table1_params(F kappa, F lnB, F c) {
    using std::exp;
    using std::log;
    TableIParams<F> P;
    P.kstar = kappa - F(0.5);                                                      // Eq. (16)
    // a = (1/kappa) (2/(3B))^(2/3)                                                    Eq. (13)
    P.a = exp((F(2.0) / F(3.0)) * (log(F(2.0) / F(3.0)) - lnB)) / kappa;
    P.c = c;                                                                        // Eq. (20)
    // b = (kappa* (3/2) B)^(1/kappa*) (kappa*/kappa) c                                Eq. (17)
    P.b = exp((log(P.kstar * F(1.5)) + lnB) / P.kstar) * (P.kstar / kappa) * P.c;
    return P;
}

template <typename F>
KAPPAGEN_HD inline Coef<double> make_coef_f64(const TableIParams<F>& P, F theta) {
    Coef<double> C;
    C.s = (double)(F(1.0) / P.kstar);
    C.a = (double)P.a;
    C.ck = (double)(P.c * P.kstar);
    C.bk4 = (double)(F(4.0) * P.b * P.kstar);
    C.k2 = (double)(F(2.0) * P.kstar);
    C.b2 = (double)(F(2.0) * P.b);
    C.theta = (double)theta;
    C.theta2 = (double)(F(2.0) * theta);
    return C;
}

// fold: put theta^2 into k2/th4 (only when 4 theta^2 and everything it multiplies stay normal floats).
template <typename F>
KAPPAGEN_HD inline Coef<float> make_coef_f32(const TableIParams<F>& P, F theta, bool fold) {
    Coef<float> C;
    const F t2 = fold ? theta * theta : F(1.0);
    C.s = (float)(F(1.0) / P.kstar);
    C.a = (float)P.a;
    C.ck = (float)(P.c * P.kstar);
    C.bk4 = (float)(F(4.0) * P.b * P.kstar);
    C.k2 = (float)(F(8.0) * P.kstar * t2);
    C.b2 = (float)(F(2.0) * P.b);
    C.th4 = (float)(F(4.0) * t2);
    C.theta = fold ? 1.0f : (float)theta;
    return C;
}

KAPPAGEN_HD inline CellRec<float> make_cell_rec(const Coef<float>& C, float dx, float dy, float dz) {
    return CellRec<float>{C.s, -C.s, C.a, -C.ck, C.bk4, C.k2, C.b2, C.th4, C.theta, dx, dy, dz};
}
KAPPAGEN_HD inline CellRec<double> make_cell_rec(const Coef<double>& C, double dx, double dy, double dz) {
    return CellRec<double>{C, dx, dy, dz, 0.0};
}
KAPPAGEN_HD inline Coef<float> coef_of(const CellRec<float>& R) {
    Coef<float> C;
    C.s = R.s; C.a = R.a; C.ck = -R.mck; C.bk4 = R.bk4; C.k2 = R.k2; C.b2 = R.b2; C.th4 = R.th4; C.theta = R.theta;
    return C;
}
KAPPAGEN_HD inline Coef<double> coef_of(const CellRec<double>& R) { return R.C; }

KAPPAGEN_HD inline bool theta_folds(double theta) { return theta >= 0x1p-30 && theta <= 0x1p+30; }

}  // namespace kappagen
