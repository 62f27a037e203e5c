// math_f64.cuh -- steps S2-S6 of the hot path in double (Table I lines 6-10, PAPER.md:166;
// Eqs. (24),(25)).  Tolerance against the oracle: 1e-12 relative per component;
// measured 6.3e-14.
//
// The chain is the cancellation-free re-association of DESIGN.md readings R3, R7:
//   1 - U      exact: U = (w + 1/2)/2^32 has 33 significant bits, so 1 - U is the double ((~w) + 1/2)/2^32
//              (PAPER.md:250 turned into an identity)
//   1 - U1^(2/3) = t1 (1+r)/(1+r+r^2),  r = cbrt(U1), t1 = 1-U1   (since 1 - r^3 = t1)
//   (..)^(-1/kappa*) - 1 = expm1(-ln(S)/kappa*)
//   root of Eq. (24): the printed form whose denominator/numerator adds
//   azimuth: quarter-turn reduction on the integer word, polynomials on |angle| <= pi/4
// No data-dependent branch: selects only ("no loops or conditional statements").
//
// Written for the FP64 pipe of sm_100 (64 DFMA/clk/SM): ~100 FP64 instructions per particle instead of
// libdevice's ~200, and no divergent slow paths.
//   * integer -> double by the 2^52 trick: (2^52 + w) is the register pair (w, 0x43300000); one DFMA
//     scales and re-centres it exactly.  No I2F.F64 (quarter rate).
//   * 1/x, 1/sqrt(x), x^(-1/3): seed from the fp32 special-function unit (MUFU, relative error < 2^-20
//     after the seed is cut to the high word of a double), then ONE third-order correction in double
//     (residual ~ e^3 < 1e-17).  double -> float -> double never goes through F2F: the high word is
//     re-biased with integer arithmetic.
//   * ln: S = 2^k m, m in [sqrt(1/2), sqrt(2)), f = (m-1)/(m+1), ln m = 2 f P(f^2), P of degree 6
//     (2e-16); where S -> 1 the numerator m - 1 is taken as -p = -U1^(2/3), which is exact there.
//   * expm1: M = n ln2 + rho, |rho| <= ln2/2, expm1(M) = 2^n (rho Q(rho)) + (2^n - 1), Q of degree 8.
//   * sin/cos(pi q/2) on |q| <= 1/2: degrees 5 and 6 in q^2.
// Coefficients: fit_polynomials.py f64 (same directory).
#pragma once
#include <cstdint>
#include "coefs.cuh"

namespace kappagen {

// (2^52 + w) * scale + bias, exact whenever the result is representable (it is for all uses below).
__device__ __forceinline__ double u32_affine(uint32_t w, double scale, double bias) {
    return fma(__hiloint2double(0x43300000, (int)w), scale, bias);
}

// fp32 view of a positive double inside the float range: high word re-biased, mantissa cut to 20 bits.
__device__ __forceinline__ float seed_in(double x) {
    return __uint_as_float(((uint32_t)__double2hiint(x) << 3) + 0x40000000u);   // (hi - 0x38000000) << 3
}
// double view of a positive float: 20 mantissa bits kept; the low word is don't-care (< 2^-20 relative)
// and reuses the float's register so that no zero has to be materialised.
__device__ __forceinline__ double seed_out(float s) {
    return __hiloint2double((int)((__float_as_uint(s) >> 3) + 0x38000000u), (int)__float_as_uint(s));
}

// 1/d, third order: e = 1 - d z0, z = z0 (1 + e + e^2).
__device__ __forceinline__ double rcp3_f64(double d) {
    float s;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(s) : "f"(seed_in(d)));
    const double z0 = seed_out(s);
    const double e = fma(-d, z0, 1.0);
    return fma(z0, fma(e, e, e), z0);
}

// 1/sqrt(z), third order: e = 1 - z g0^2, g = g0 (1 + e/2 + 3 e^2/8).
__device__ __forceinline__ double rsqrt3_f64(double z) {
    float s;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(s) : "f"(seed_in(z)));
    const double g0 = seed_out(s);
    const double t = z * g0;
    const double e = fma(-t, g0, 1.0);
    const double q = fma(e, 0.375, 0.5);
    return fma(g0, q * e, g0);
}
// sqrt(z) by the same correction applied to t = z g0 (one multiply fewer than z * rsqrt3_f64(z)).
__device__ __forceinline__ double sqrt3_f64(double z) {
    float s;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(s) : "f"(seed_in(z)));
    const double g0 = seed_out(s);
    const double t = z * g0;
    const double e = fma(-t, g0, 1.0);
    const double q = fma(e, 0.375, 0.5);
    return fma(t, q * e, t);
}

template <bool U64 = false>
__device__ __forceinline__ double speed_f64(uint32_t w0, uint32_t w3, const Coef<double>& C) {
    double u1, t1;
    float useed;                                                                 // 2^32 U1 for the fp32 seed
    if (U64) {
        // reading R20: U1 = (w0 2^32 + w3 + 1/2)/2^64 (65 bits, rounded once); 1 - U1 from the complements
        u1 = u32_affine(w0, 0x1p-32, -0x1p20) + u32_affine(w3, 0x1p-64, -0x1p-12 + 0x1p-65);
        t1 = u32_affine(~w0, 0x1p-32, -0x1p20) + u32_affine(~w3, 0x1p-64, -0x1p-12 + 0x1p-65);
        useed = (float)w0 + fmaf((float)w3, 0x1p-32f, 0x1p-33f);
    } else {
        u1 = u32_affine(w0, 0x1p-32, -0x1p20 + 0x1p-33);                        // U1 = (w0 + 1/2)/2^32, exact
        t1 = 1.0 - u1;                                                           // exact: U1 has 33 significant bits
        useed = (float)w0 + 0.5f;
    }
    // r = U1^(1/3): fp32 seed y0 ~ U1^(-1/3) = 2^((32 - log2(w0 + 1/2))/3); r0 = u y0^2, e = 1 - u y0^3 = 1 - r0 y0,
    // r = u y^2 with y = y0 (1-e)^(-1/3):  r = r0 (1 + 2e/3 + 5e^2/9), residual ~ e^3
    float lg, ys;
    asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(lg) : "f"(useed));
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(ys) : "f"(fmaf(lg, -0x1.555556p-2f, 0x1.555556p+3f)));
    const double y0 = seed_out(ys);
    const double r0 = (y0 * y0) * u1;
    const double e = fma(-r0, y0, 1.0);
    const double r = fma(r0, fma(e, 0x1.1c71c71c71c72p-1, 0x1.5555555555555p-1) * e, r0);   // 5/9, 2/3
    const double p = r * r;                                                      // U1^(2/3)
    const double q1 = 1.0 + r;
    const double S = (t1 * q1) * rcp3_f64(q1 + p);                               // 1 - U1^(2/3), no cancellation
    // ln S = k ln2 + 2 f P(f^2), S = 2^k m, m in [sqrt(1/2), sqrt(2)); S < 1 so k <= 0
    const int hi = __double2hiint(S);
    const int k = (hi - 0x3fe6a09e) >> 20;
    const double m = __hiloint2double(hi - (k << 20), __double2loint(S));
    const double num = (k == 0) ? -p : m - 1.0;                                  // k = 0: m - 1 = S - 1 = -p, without cancellation
    const double f = num * rcp3_f64(num + 2.0);
    const double z = f * f;
    double P = 0x1.58dde2537d4c5p-4;
    P = fma(P, z, 0x1.732279c8761a8p-4);
    P = fma(P, z, 0x1.c722d1f4cf2b3p-4);
    P = fma(P, z, 0x1.249240af9d15dp-3);
    P = fma(P, z, 0x1.999999a442e0dp-3);
    P = fma(P, z, 0x1.5555555552d11p-2);
    P = fma(P, z, 0x1.0000000000001p+0);
    const int kb = k ^ (int)0x80000000;                                          // k as a double: 2^52 trick, signed
    const double kd = __hiloint2double(0x43300000, kb) - (0x1p52 + 0x1p31);      // (2^52 + 2^31 + k) - (2^52 + 2^31)
    const double lnS = fma(kd, 0x1.62e42fefa39efp-1, (f + f) * P);
    // Y = expm1(M), M = -ln(S)/kappa* >= 0:  M = n ln2 + rho,  Y = 2^n (rho Q(rho)) + (2^n - 1)
    const double M = -lnS * C.s;
    const double nb = fma(M, 0x1.71547652b82fep+0, 0x1.8p52);                    // n = rint(M log2 e) in the low word
    const double nd = nb - 0x1.8p52;
    const double rho = fma(-nd, 0x1.62e42fefa39efp-1, M);
    double Q = 0x1.72c79824255e0p-19;
    Q = fma(Q, rho, 0x1.a15af3e6562d7p-16);
    Q = fma(Q, rho, 0x1.a019ad55d1aa7p-13);
    Q = fma(Q, rho, 0x1.6c164d7dbdce2p-10);
    Q = fma(Q, rho, 0x1.1111111c5719ap-7);
    Q = fma(Q, rho, 0x1.555555745858dp-5);
    Q = fma(Q, rho, 0x1.5555555553b48p-3);
    Q = fma(Q, rho, 0x1.fffffffff70abp-2);
    Q = fma(Q, rho, 0x1.0000000000000p+0);
    const double sc = __hiloint2double((__double2loint(nb) + 1023) << 20, 0);    // 2^n, 0 <= n < 64
    const double Y = fma(sc, rho * Q, sc - 1.0);                                 // S^(-1/kappa*) - 1 = -L/kappa*
    // Eq. (24): root of b x^2 + A x - kappa* Y = 0, A = a + cL = a - c kappa* Y, in the form that adds
    const double A = fma(-C.ck, Y, C.a);
    const double disc = fma(A, A, C.bk4 * Y);                                    // (a+cL)^2 - 4bL > A^2
    const double T = fabs(A) + sqrt3_f64(disc);                                  // |A| + sqrt(disc)
    // x = num/den:  A >= 0: 2 kappa* Y / T;   A < 0: T / (2b).   V = theta sqrt(num/den) = theta num / sqrt(num den)
    const bool pos = A >= 0.0;
    const double nm = pos ? C.k2 * Y : T;
    const double dn = pos ? T : C.b2;
    return C.theta * (nm * rsqrt3_f64(nm * dn));
}

template <bool U64 = false>
__device__ __forceinline__ void velocity_f64(uint32_t w0, uint32_t w1, uint32_t w2, uint32_t w3,
                                             const Coef<double>& C, double& vx, double& vy, double& vz) {
    const double V = speed_f64<U64>(w0, w3, C);
    const double u2 = u32_affine(w1, 0x1p-32, -0x1p20 + 0x1p-33);               // U2, exact
    const double t2 = 1.0 - u2;                                                  // 1 - U2, exact
    const double mu = u2 - t2;                                                   // 2 U2 - 1, exact
    const double zz = u2 * t2;
    const double sth = sqrt3_f64(zz);                                            // sqrt(U2 (1-U2)); the 2 goes into Vs
    // 2 pi U3 = (pi/2)(k + q): k = nearest quarter turn, q = ((int32)(w2 << 2) + 2)/2^32 in (-1/2, 1/2)
    const double q = u32_affine((w2 << 2) ^ 0x80000000u, 0x1p-32, -0x1p20 - 0.5 + 0x1p-31);
    const double z = q * q;
    double sp = -0x1.dd54805f3f706p-19;
    sp = fma(sp, z, 0x1.5071ce4b47930p-13);
    sp = fma(sp, z, -0x1.32d2c644adc0bp-8);
    sp = fma(sp, z, 0x1.466bc67123fa1p-4);
    sp = fma(sp, z, -0x1.4abbce6257a2ap-1);
    sp = fma(sp, z, 0x1.921fb54442cfap+0);
    double cr = 0x1.f3dbcea61b1a4p-22;
    cr = fma(cr, z, -0x1.a6c9c1be9eb49p-16);
    cr = fma(cr, z, 0x1.e1f4fb60281f6p-11);
    cr = fma(cr, z, -0x1.55d3c7dbfd139p-6);
    cr = fma(cr, z, 0x1.03c1f081b0780p-2);
    cr = fma(cr, z, -0x1.3bd3cc9be458bp+0);
    cr = fma(cr, z, 0x1.0000000000000p+0);
    const double sr = sp * q;                                                    // sin(pi q/2), cos(pi q/2)
    const uint32_t wq = w2 + 0x20000000u;                                        // k = wq >> 30 (k = 4 wraps to 0)
    const bool odd = (wq & 0x40000000u) != 0u;                                   // k odd: swap
    const double c0 = odd ? sr : cr;
    const double s0 = odd ? cr : sr;
    // signs: sin < 0 for k = 2,3 (bit 31 of wq); cos < 0 for k = 1,2 (bit 31 of wq + 2^30)
    const double cphi = __hiloint2double(__double2hiint(c0) ^ (int)((wq + 0x40000000u) & 0x80000000u), __double2loint(c0));
    const double sphi = __hiloint2double(__double2hiint(s0) ^ (int)(wq & 0x80000000u), __double2loint(s0));
    const double Vs = (V + V) * sth;
    vx = V * mu;
    vy = Vs * cphi;
    vz = Vs * sphi;
}

}  // namespace kappagen
