// coefs.cuh -- step S0: Table I lines 1-4 (Eqs. (16),(13),(20),(17)) and the
// per-(kappa,theta) constants the per-particle math consumes.
//
// The per-particle chain is written in terms of Y = (1 - U1^(2/3))^(-1/kappa*) - 1 >= 0, so that
// L = -kappa* Y (Eq. 25) never has to be formed:
//   A    = a + cL            = a  - ck  * Y          ck  = c kappa*
//   disc = (a+cL)^2 - 4bL    = A^2 + bk4 * Y         bk4 = 4 b kappa*
//   x    = -2L / (A + sqrt(disc))   = k2 * Y / (A + D)     k2  = 2 kappa*      (A >= 0)
//        = (-A + sqrt(disc)) / (2b) = (D - A) * i2b        i2b = 1/(2b)        (A <  0)
// (the two printed forms of Eq. (24)).  V = theta sqrt(x).
#pragma once
#include <cmath>

namespace kappagen {

// Table I lines 1-4 in one precision F (long double on the host, double on the device).
template <typename F>
struct TableIParams {
    F kstar, a, b, c;
};

// Per-(kappa, theta) constants in the kernel's arithmetic type.  32 bytes (float) / 64 bytes
// (double): the cells path stores one of these per cell in the workspace.
template <typename T>
struct alignas(16) Coef {
    T s;      // 1/kappa*
    T a;      // Eq. (13)
    T ck;     // c kappa*
    T bk4;    // 4 b kappa*
    T k2;     // 2 kappa*
    T i2b;    // 1/(2b)
    T theta;  // most probable speed; NaN marks an invalid cell
    T pad;
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

template <typename T, typename F>
KAPPAGEN_HD inline Coef<T> make_coef(const TableIParams<F>& P, F theta) {
    Coef<T> C;
    C.s = (T)(F(1.0) / P.kstar);
    C.a = (T)P.a;
    C.ck = (T)(P.c * P.kstar);
    C.bk4 = (T)(F(4.0) * P.b * P.kstar);
    C.k2 = (T)(F(2.0) * P.kstar);
    C.i2b = (T)(F(1.0) / (F(2.0) * P.b));
    C.theta = (T)theta;
    C.pad = (T)0;
    return C;
}

}  // namespace kappagen
