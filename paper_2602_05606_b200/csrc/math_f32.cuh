// math_f32.cuh -- steps S2-S6 of the hot path in float (Table I lines 6-10, PAPER.md:166;
// Eqs. (24),(25)).  Tolerance against the oracle: 4e-6 relative per component.
//
// Written for the instruction budget of DESIGN.md section "fp32 kernel": the SM's special-function
// unit (MUFU lg2/ex2/rcp/rsq/sqrt, ~2^-22 relative) does the transcendentals, short polynomials take
// over exactly where a MUFU result would cancel, and every choice is a select -- no data-dependent
// branch, no loop ("no loops or conditional statements").  9 MUFU + ~75 other
// instructions per particle.
//
// A 32-bit uniform (w + 1/2)/2^32 is not representable in float, so everything that would cancel is
// taken from the integer word before the conversion (readings R3, R5, R7):
//   U1, 1-U1   : float(w0), float(~w0)                 (each rounded once, relative 2^-24)
//   2U2-1      : float(int32(w1 ^ 0x80000000))
//   U2(1-U2)   : e(1-e), e = min(U2, 1-U2) from min(w1, ~w1)
//   azimuth    : quarter turn k and signed remainder taken from w2; polynomials on |angle| <= pi/4
//   1 - U1^(2/3) = t1 (1+r)/(1+r+r^2), r = cbrt(U1), t1 = 1-U1        (since 1 - r^3 = t1)
// Speed, with Y = (1-U1^(2/3))^(-1/kappa*) - 1 = -L/kappa* (Eq. 25) and m = log2(1+Y):
//   m = -log2(S)/kappa*            MUFU.LG2 when p = U1^(2/3) >= 1/4, else p G(p)/kappa* (degree-5 G)
//   Y = 2^m - 1                    MUFU.EX2 when m >= 1/2, else m R(m) (degree-4 R)
//   x = positive root of Eq. (24)  the printed form that adds, V = theta sqrt(x) = num rsqrt(num den)/2
// The polynomial coefficients are the near-minimax fits printed by `fit_polynomials.py f32` (same directory).
#pragma once
#include <cstdint>
#include "coefs.cuh"

namespace kappagen {

__device__ __forceinline__ float mufu_lg2(float x) { float y; asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float mufu_ex2(float x) { float y; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float mufu_rcp(float x) { float y; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float mufu_rsq(float x) { float y; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float mufu_sqrt(float x) { float y; asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }

// 2^32 U1 and 1 - U1 as floats with RELATIVE accuracy at both ends.  U64 (reading R20): U1 = (w0 2^32 + w3 +
// 1/2)/2^64; the low word only matters where the high word (or its complement) is small.
template <bool U64>
__device__ __forceinline__ void uniform1_f32(uint32_t w0, uint32_t w3, float& u_scaled, float& t1) {
    if (U64) {
        u_scaled = (float)w0 + fmaf((float)w3, 0x1p-32f, 0x1p-33f);
        t1 = fmaf((float)(uint32_t)(~w0), 0x1p-32f, fmaf((float)(uint32_t)(~w3), 0x1p-64f, 0x1p-65f));
    } else {
        u_scaled = (float)w0 + 0.5f;
        t1 = fmaf((float)(uint32_t)(~w0), 0x1p-32f, 0x1p-33f);               // 1 - U1 from the integer
    }
}

// 2V = 2 theta sqrt(x) (times 1/theta when the coefficients are not folded, see Coef<float>).
template <bool U64 = false>
__device__ __forceinline__ float speed2_f32(uint32_t w0, uint32_t w3, const Coef<float>& C) {
    // r = U1^(1/3) = 2^((log2(2^32 U1) - 32)/3); only p = r^2 small needs it to relative accuracy
    float us, t1;
    uniform1_f32<U64>(w0, w3, us, t1);
    const float lg = mufu_lg2(us);
    const float r = mufu_ex2(fmaf(lg, 0x1.555556p-2f, -0x1.555556p+3f));
    const float p = r * r;                                                    // U1^(2/3)
    const float q1 = r + 1.0f;
    const float S = (t1 * q1) * mufu_rcp(q1 + p);                             // 1 - U1^(2/3), no cancellation
    // m = -log2(S)/kappa*.  For p < 1/4 (S -> 1) the MUFU result would carry only absolute accuracy:
    // -log2(1-p) = p G(p), G of degree 5, relative error of the fit 5.7e-8 on [0, 1/4].
    float G = 0x1.f448fp-2f;
    G = fmaf(G, p, 0x1.ab553ap-3f);
    G = fmaf(G, p, 0x1.7c9f74p-2f);
    G = fmaf(G, p, 0x1.ebc184p-2f);
    G = fmaf(G, p, 0x1.71565ep-1f);
    G = fmaf(G, p, 0x1.715476p+0f);
    const float m_small = (p * C.s) * G;
    const float m_large = mufu_lg2(S) * -C.s;                                 // s = 1/kappa*
    const float m = (p < 0.25f) ? m_small : m_large;
    // Y = 2^m - 1.  For m < 1/2 the subtraction would cancel: 2^m - 1 = m R(m), R of degree 4 (2.7e-8).
    float R = 0x1.945094p-10f;
    R = fmaf(R, m, 0x1.3817fcp-7f);
    R = fmaf(R, m, 0x1.c6d414p-5f);
    R = fmaf(R, m, 0x1.ebfb52p-3f);
    R = fmaf(R, m, 0x1.62e43p-1f);
    const float Y = (m < 0.5f) ? m * R : mufu_ex2(m) - 1.0f;
    // Eq. (24): root of b x^2 + A x - kappa* Y = 0, A = a + cL = a - c kappa* Y, in the form that adds
    const float A = fmaf(-C.ck, Y, C.a);
    const float D = mufu_sqrt(fmaf(A, A, C.bk4 * Y));                         // sqrt((a+cL)^2 - 4bL) > |A|
    const float T = fabsf(A) + D;
    // (2 theta)^2 x = num/den:  A >= 0: 4 theta^2 2 kappa* Y / T;   A < 0: 4 theta^2 T / (2b)
    const bool pos = A >= 0.0f;
    const float num = pos ? C.k2 * Y : C.th4 * T;
    const float den = pos ? T : C.b2;
    return num * mufu_rsq(num * den);                                         // sqrt(num/den)
}

// Direction, halved: muh = (2U2-1)/2, sth = sqrt(U2(1-U2)), (cphi, sphi) = (cos, sin)(2 pi U3).
__device__ __forceinline__ void direction_f32(uint32_t w1, uint32_t w2, float& muh, float& sth, float& cphi, float& sphi) {
    muh = fmaf((float)(int32_t)(w1 ^ 0x80000000u), 0x1p-32f, 0x1p-33f);
    const uint32_t wm = min(w1, ~w1);
    const float e = fmaf((float)wm, 0x1p-32f, 0x1p-33f);                     // min(U2, 1-U2), relative accuracy
    sth = mufu_sqrt(fmaf(-e, e, e));                                          // sqrt(U2 (1-U2))
    // 2 pi U3 = (pi/2)(k + q): k = nearest quarter turn, q in (-1/2, 1/2).  (w2 + 2^29) << 2, read as a
    // signed integer and re-centred, is simply (int32)(w2 << 2): q = ((int32)(w2 << 2) + 2) / 2^32.
    const float q = fmaf((float)(int32_t)(w2 << 2), 0x1p-32f, 0x1p-31f);
    const float z = q * q;
    float sp = -0x1.2d9b4p-8f;                                               // sin(pi q/2)/q, degree 3 in z (3.5e-8)
    sp = fmaf(sp, z, 0x1.465ec4p-4f);
    sp = fmaf(sp, z, -0x1.4abbbap-1f);
    sp = fmaf(sp, z, 0x1.921fb6p+0f);
    float cr = -0x1.4e5e06p-6f;                                               // cos(pi q/2), degree 3 in z (6.0e-8)
    cr = fmaf(cr, z, 0x1.03af58p-2f);
    cr = fmaf(cr, z, -0x1.3bd392p+0f);
    cr = fmaf(cr, z, 0x1.0p+0f);
    const float sr = sp * q;
    const uint32_t wq = w2 + 0x20000000u;                                     // k = wq >> 30 (k = 4 wraps to 0)
    const bool odd = (wq & 0x40000000u) != 0u;                                // k odd: swap
    const float c0 = odd ? sr : cr;
    const float s0 = odd ? cr : sr;
    // signs: sin < 0 for k = 2,3 (bit 31 of wq); cos < 0 for k = 1,2 (bit 31 of wq + 2^30)
    cphi = __uint_as_float(__float_as_uint(c0) ^ ((wq + 0x40000000u) & 0x80000000u));
    sphi = __uint_as_float(__float_as_uint(s0) ^ (wq & 0x80000000u));
}

// FOLD: theta is already inside C.k2 / C.th4 (uniform-parameter kernels); otherwise multiply by C.theta
// (per-cell parameters, theta = 0, or theta outside [2^-30, 2^30]).  DRIFT: the cell's drift (dx, dy, dz) enters as the
// addend of the last multiply (one rounding), in every code path alike, so that a particle's value does not
// depend on which path produced it.
template <bool FOLD, bool U64 = false, bool DRIFT = false>
__device__ __forceinline__ void velocity_f32(uint32_t w0, uint32_t w1, uint32_t w2, uint32_t w3,
                                             const Coef<float>& C, float& vx, float& vy, float& vz,
                                             float dx = 0.0f, float dy = 0.0f, float dz = 0.0f) {
    float V2 = speed2_f32<U64>(w0, w3, C);             // 2V
    if (!FOLD) V2 *= C.theta;
    float muh, sth, cphi, sphi;
    direction_f32(w1, w2, muh, sth, cphi, sphi);
    const float Vs = V2 * sth;
    if (DRIFT) {
        vx = fmaf(V2, muh, dx);
        vy = fmaf(Vs, cphi, dy);
        vz = fmaf(Vs, sphi, dz);
    } else {
        vx = V2 * muh;
        vy = Vs * cphi;
        vz = Vs * sphi;
    }
}

}  // namespace kappagen
