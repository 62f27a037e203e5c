// math_f64.cuh -- steps S2-S6 of the hot path in double (Table I lines 6-10, PAPER.md:166;
// Eqs. (24),(25)).  Tolerance against the oracle: 1e-12 relative per component;
// measured 2.2e-13.
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
// Written for the FP64 pipe of sm_100 (64 DFMA/clk/SM): 85 FP64 instructions per particle instead of
// libdevice's ~200, and no divergent slow paths.  On sm_100 the FP64 pipe and the FMA-heavy pipe (IMAD,
// IMAD.WIDE, IMAD.MOV) do not overlap in time (profiles/r03_pipe_rates.md), so every instruction of either
// kind counts against the same budget; the choices below follow from that.
//   * integer -> double without a conversion instruction: 1 + w 2^-32 is the register pair
//     ((w >> 12) + 0x3ff00000, w << 20), two ALU instructions and no move; one exact DADD re-centres it.
//     No I2F.F64 (quarter rate, XU pipe).
//   * 1/x, 1/sqrt(x), x^(-1/3): seed from the fp32 special-function unit (MUFU, relative error < 2^-20
//     after the seed is cut to the high word of a double), then ONE third-order correction in double
//     (residual ~ e^3 < 1e-17).  double -> float -> double never goes through F2F: the high word is
//     re-biased with integer arithmetic.
//   * ln: S = N/D is never formed.  k = round(log2 S) from the high words of N and D, m = S 2^-k in
//     [2^-0.59, 2^0.59], f = (m-1)/(m+1) = (N_k - D)/(N_k + D) -- one division for quotient and atanh
//     argument -- ln m = 2 f P(f^2), P of degree 5 (1.9e-13); for k = 0 the numerator is -U1^(2/3) D, exact.
//   * expm1: M = n ln2 + rho, |rho| <= ln2/2, expm1(M) = 2^n (rho Q(rho)) + (2^n - 1), Q of degree 8 (9e-14).
//   * the two small integers k and n reach the arithmetic through shared-memory tables (-k ln2; 2^n and
//     2^n - 1) instead of integer -> double conversions: one LDS each.
//   * sin/cos(pi q/2) on |q| <= 1/2: degree 5 in q^2 each (4.7e-15, 7.8e-14).
// Coefficients: fit_polynomials.py f64 (same directory).
#pragma once
#include <cstdint>
#include "coefs.cuh"

namespace kappagen {

// (2^52 + w) * scale + bias, exact whenever the result is representable (it is for all uses below).  Used on the
// 64-bit-U1 path only: the register pair (w, 0x43300000) costs two moves on the pipe the FP64 unit shares.
__device__ __forceinline__ double u32_affine(uint32_t w, double scale, double bias) {
    return fma(__hiloint2double(0x43300000, (int)w), scale, bias);
}
// 1 + w 2^-32 in [1, 2), exact: the 32 bits of w become the top of the mantissa.  Both halves of the register pair
// are results of ALU instructions (shift-and-add, shift), so no move is needed to assemble it.
__device__ __forceinline__ double u32_unit(uint32_t w) {
    return __hiloint2double((int)((w >> 12) + 0x3ff00000u), (int)(w << 20));
}

// Per-block lookup tables in shared memory for the two small integers of the chain (k = round(log2 S) and
// n = rint(M log2 e), both in [0, 68]): -k ln2 as a double, and the pair (2^n, 2^n - 1).  A table read replaces an
// integer -> double conversion (register-pair assembly + one FP64 instruction each) by one LDS.
constexpr int kF64TabN = 72;
struct F64Tables {
    double neg_k_ln2[kF64TabN];
    double2 pow2[kF64TabN];
};
__device__ __forceinline__ F64Tables& f64_tables() {
    __shared__ F64Tables t;
    return t;
}
// Every kernel that evaluates the double chain calls this once, before its first particle (all threads of the block).
__device__ __forceinline__ void f64_tables_init() {
    F64Tables& t = f64_tables();
    for (int i = threadIdx.x; i < kF64TabN; i += blockDim.x) {
        t.neg_k_ln2[i] = -((double)i * 0x1.62e42fefa39efp-1);
        const double sc = __hiloint2double((i + 1023) << 20, 0);
        t.pow2[i] = make_double2(sc, sc - 1.0);
    }
    __syncthreads();
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
__device__ __forceinline__ double speed_f64(uint32_t w0, uint32_t w3, const Coef<double>& C, double scale) {   // scale sqrt(x)
    double u1, t1;
    float useed;                                                                 // 2^32 U1 for the fp32 seed
    if (U64) {
        // reading R20: U1 = (w0 2^32 + w3 + 1/2)/2^64 (65 bits, rounded once); 1 - U1 from the complements
        u1 = u32_affine(w0, 0x1p-32, -0x1p20) + u32_affine(w3, 0x1p-64, -0x1p-12 + 0x1p-65);
        t1 = u32_affine(~w0, 0x1p-32, -0x1p20) + u32_affine(~w3, 0x1p-64, -0x1p-12 + 0x1p-65);
        useed = (float)w0 + fmaf((float)w3, 0x1p-32f, 0x1p-33f);
    } else {
        const double x1 = u32_unit(w0);
        u1 = x1 - (1.0 - 0x1p-33);                                               // U1 = (w0 + 1/2)/2^32, exact
        t1 = (2.0 - 0x1p-33) - x1;                                               // 1 - U1, exact (33 significant bits)
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
    // S = 1 - U1^(2/3) = N/D without cancellation: N = t1 (1 + r), D = 1 + r + r^2 (since 1 - r^3 = t1); S is never formed.
    // ln S = k ln2 + 2 atanh(f), f = (m - 1)/(m + 1), m = S 2^-k = N_k/D:  f = (N_k - D)/(N_k + D) -- ONE division for
    // the quotient and the atanh argument.  k = round(log2 S) to within 0.09 from the high words of N and D (exponent
    // plus leading mantissa bits are a piecewise-linear log2), so m in [2^-0.59, 2^0.59] and f^2 <= 0.0407.
    const double N = t1 * q1;
    const double D = q1 + p;
    const int hN = __double2hiint(N);
    const int k = (hN - __double2hiint(D) + 0x80000) >> 20;                      // S < 1: k <= 0
    const double Nk = __hiloint2double(hN - (k << 20), __double2loint(N));       // N 2^-k, exact
    // k = 0: N - D = -p D exactly (N = (1 - p) D), which does not cancel as p -> 0
    const double num = (k == 0) ? -(p * D) : Nk - D;
    const double f = num * rcp3_f64(Nk + D);
    const double z = f * f;
    double P = 0x1.9d7eab5747345p-3;                                             // 2 atanh(sqrt z)/sqrt z, degree 5: 1.9e-13
    P = fma(P, z, 0x1.c530318164389p-3);                                         // (the fitted coefficients, doubled: exact)
    P = fma(P, z, 0x1.2497875fa7cb3p-2);
    P = fma(P, z, 0x1.99998cbcc9384p-2);
    P = fma(P, z, 0x1.5555555b16753p-1);
    P = fma(P, z, 0x1.ffffffffff957p+0);
    const F64Tables& Tb = f64_tables();
    const double lnS = fma(f, P, Tb.neg_k_ln2[-k]);                              // k ln2 + 2 f P(z): P holds 2 P
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
    const double2 sc = Tb.pow2[__double2loint(nb)];                              // (2^n, 2^n - 1), 0 <= n <= 68
    const double Y = fma(sc.x, rho * Q, sc.y);                                   // S^(-1/kappa*) - 1 = -L/kappa*
    // Eq. (24): root of b x^2 + A x - kappa* Y = 0, A = a + cL = a - c kappa* Y, in the form that adds
    const double A = fma(-C.ck, Y, C.a);
    const double disc = fma(A, A, C.bk4 * Y);                                    // (a+cL)^2 - 4bL > A^2
    const double T = fabs(A) + sqrt3_f64(disc);                                  // |A| + sqrt(disc)
    // x = num/den:  A >= 0: 2 kappa* Y / T;   A < 0: T / (2b).   V = theta sqrt(num/den) = theta num / sqrt(num den)
    const bool pos = A >= 0.0;
    const double nm = pos ? C.k2 * Y : T;
    const double dn = pos ? T : C.b2;
    return scale * (nm * rsqrt3_f64(nm * dn));
}

// DRIFT: the cell's drift as the addend of the last multiply (one rounding), as in velocity_f32.
template <bool U64 = false, bool DRIFT = false>
__device__ __forceinline__ void velocity_f64(uint32_t w0, uint32_t w1, uint32_t w2, uint32_t w3,
                                             const Coef<double>& C, double& vx, double& vy, double& vz,
                                             double dx = 0.0, double dy = 0.0, double dz = 0.0) {
    const double V2 = speed_f64<U64>(w0, w3, C, C.theta2);                       // 2V: the factor 2 of Table I lines 9-10
    const double x2 = u32_unit(w1);
    const double u2 = x2 - (1.0 - 0x1p-33);                                      // U2, exact
    const double t2 = (2.0 - 0x1p-33) - x2;                                      // 1 - U2, exact
    const double muh = x2 - (1.5 - 0x1p-33);                                     // U2 - 1/2 = (2 U2 - 1)/2, exact
    const double zz = u2 * t2;
    const double sth = sqrt3_f64(zz);                                            // sqrt(U2 (1-U2)); the 2 goes into Vs
    // 2 pi U3 = (pi/2)(k + q): k = nearest quarter turn, q = ((int32)(w2 << 2) + 2)/2^32 in (-1/2, 1/2)
    const double q = u32_unit((w2 << 2) ^ 0x80000000u) - (1.5 - 0x1p-31);
    const double z = q * q;
    double sp = -0x1.dd54805f3f706p-19;
    sp = fma(sp, z, 0x1.5071ce4b47930p-13);
    sp = fma(sp, z, -0x1.32d2c644adc0bp-8);
    sp = fma(sp, z, 0x1.466bc67123fa1p-4);
    sp = fma(sp, z, -0x1.4abbce6257a2ap-1);
    sp = fma(sp, z, 0x1.921fb54442cfap+0);
    double cr = -0x1.a0ee132c60c1fp-16;                                          // cos(pi q/2), degree 5 in z: 7.8e-14
    cr = fma(cr, z, 0x1.e1e7ccccb387ap-11);
    cr = fma(cr, z, -0x1.55d3ba300cd50p-6);
    cr = fma(cr, z, 0x1.03c1f074ded21p-2);
    cr = fma(cr, z, -0x1.3bd3cc9bd2c35p+0);
    cr = fma(cr, z, 0x1.ffffffffffe0bp-1);
    const double sr = sp * q;                                                    // sin(pi q/2), cos(pi q/2)
    const uint32_t wq = w2 + 0x20000000u;                                        // k = wq >> 30 (k = 4 wraps to 0)
    const bool odd = (wq & 0x40000000u) != 0u;                                   // k odd: swap
    const double c0 = odd ? sr : cr;
    const double s0 = odd ? cr : sr;
    // signs: sin < 0 for k = 2,3 (bit 31 of wq); cos < 0 for k = 1,2 (bit 31 of wq + 2^30)
    const double cphi = __hiloint2double(__double2hiint(c0) ^ (int)((wq + 0x40000000u) & 0x80000000u), __double2loint(c0));
    const double sphi = __hiloint2double(__double2hiint(s0) ^ (int)(wq & 0x80000000u), __double2loint(s0));
    const double Vs = V2 * sth;
    if (DRIFT) {
        vx = fma(V2, muh, dx);
        vy = fma(Vs, cphi, dy);
        vz = fma(Vs, sphi, dz);
    } else {
        vx = V2 * muh;
        vy = Vs * cphi;
        vz = Vs * sphi;
    }
}

}  // namespace kappagen
