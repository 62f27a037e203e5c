// math_f32.cuh -- steps S2-S6 of the hot path in float (Table I lines 6-10, PAPER.md:166;
// Eqs. (24),(25)).  Tolerance against the oracle: 4e-6 relative per component.
//
// A 32-bit uniform (w + 1/2)/2^32 is not representable in float, so everything that would cancel is
// taken from the integer word before the conversion (readings R3, R5, R7):
//   U1, 1-U1   : float(w0), float(~w0)                 (each rounded once, relative 2^-24)
//   2U2-1      : float(int32(w1 ^ 0x80000000))
//   azimuth    : quarter turn k and signed remainder d taken from w2; sin/cos on |angle| <= pi/4
//   1 - U1^(2/3) = t1 (1+r)/(1+r+r^2), r = cbrt(U1)
// No data-dependent branch: selects only ("no loops or conditional statements").
#pragma once
#include <cstdint>
#include "coefs.cuh"

namespace kappagen {

__device__ __forceinline__ float speed_f32(uint32_t w0, const Coef<float>& C) {
    const float u1 = fmaf((float)w0, 0x1p-32f, 0x1p-33f);               // U1
    const float t1 = fmaf((float)(uint32_t)(~w0), 0x1p-32f, 0x1p-33f);  // 1 - U1
    const float r = cbrtf(u1);
    const float p = r * r;                                               // U1^(2/3)
    const float S = t1 * (1.0f + r) / (1.0f + r + p);                    // 1 - U1^(2/3)
    const float lnS = (p < 0.5f) ? log1pf(-p) : logf(S);
    const float Y = expm1f(-lnS * C.s);                                  // S^(-1/kappa*) - 1
    const float A = fmaf(-C.ck, Y, C.a);                                 // a + cL
    const float D = sqrtf(fmaf(A, A, C.bk4 * Y));                        // sqrt((a+cL)^2 - 4bL)
    const float T = fabsf(A) + D;
    const float x = (A >= 0.0f) ? (C.k2 * Y) / T : T * C.i2b;            // Eq. (24), the form that adds
    return C.theta * sqrtf(x);
}

__device__ __forceinline__ void direction_f32(uint32_t w1, uint32_t w2, float& mu, float& ny, float& nz) {
    const float u2 = fmaf((float)w1, 0x1p-32f, 0x1p-33f);
    const float t2 = fmaf((float)(uint32_t)(~w1), 0x1p-32f, 0x1p-33f);
    mu = fmaf((float)(int32_t)(w1 ^ 0x80000000u), 0x1p-31f, 0x1p-32f);   // 2 U2 - 1
    const float sth = 2.0f * sqrtf(u2 * t2);                             // 2 sqrt(U2 (1-U2))
    // 2 pi U3 = (pi/2) (k + q): k = nearest quarter turn, q in (-1/2, 1/2) quarter turns
    const uint32_t wq = w2 + 0x20000000u;                                // wraps: k = 4 is k = 0
    const uint32_t k = wq >> 30;
    const int32_t d = (int32_t)(wq & 0x3FFFFFFFu) - 0x20000000;
    const float q = fmaf((float)d, 0x1p-30f, 0x1p-31f);
    float sr, cr;
    sincospif(0.5f * q, &sr, &cr);                                       // |angle| <= pi/4
    const float c0 = (k & 1u) ? sr : cr;
    const float s0 = (k & 1u) ? cr : sr;
    const float cphi = ((k + 1u) & 2u) ? -c0 : c0;                       // k = 1,2: cos < 0
    const float sphi = (k & 2u) ? -s0 : s0;                              // k = 2,3: sin < 0
    ny = sth * cphi;
    nz = sth * sphi;
}

__device__ __forceinline__ void velocity_f32(uint32_t w0, uint32_t w1, uint32_t w2,
                                             const Coef<float>& C, float& vx, float& vy, float& vz) {
    const float V = speed_f32(w0, C);
    float mu, ny, nz;
    direction_f32(w1, w2, mu, ny, nz);
    vx = V * mu;
    vy = V * ny;
    vz = V * nz;
}

}  // namespace kappagen
