// math_f32x2.cuh -- the float chain of math_f32.cuh for TWO particles at a time on Blackwell's packed
// fp32 instructions (PTX fma/mul/add.rn.f32x2 -> SASS FFMA2/FMUL2/FADD2, sm_100+).
//
// Why: the fp32 sampler is bound by instruction issue and by the FMA pipe (Philox's IMAD.WIDE alone holds
// that pipe 4 cycles each); a packed instruction does two particles' FMA in one
// issue slot.  MUFU, integer->float conversions and selects have no packed form and stay scalar on the two
// halves of the register pair (no data movement: a f32x2 value IS two adjacent 32-bit registers).
// Same arithmetic, same polynomials, same selects as math_f32.cuh -- results are bit-identical to it.
#pragma once
#include <cstdint>
#include "coefs.cuh"
#include "math_f32.cuh"

namespace kappagen {

typedef unsigned long long f32x2;

__device__ __forceinline__ f32x2 pk2(float lo, float hi) { f32x2 r; asm("mov.b64 %0, {%1,%2};" : "=l"(r) : "f"(lo), "f"(hi)); return r; }
__device__ __forceinline__ f32x2 splat2(float c) { return pk2(c, c); }
__device__ __forceinline__ void up2(f32x2 r, float& lo, float& hi) { asm("mov.b64 {%0,%1}, %2;" : "=f"(lo), "=f"(hi) : "l"(r)); }
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c) { f32x2 d; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c)); return d; }
__device__ __forceinline__ f32x2 mul2(f32x2 a, f32x2 b) { f32x2 d; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }
__device__ __forceinline__ f32x2 add2(f32x2 a, f32x2 b) { f32x2 d; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }
#define KG_MAP2(fn, v) ([&] { float a_, b_; up2((v), a_, b_); return pk2(fn(a_), fn(b_)); }())

// The chain's constants as packed pairs (x, x).  Uniform parameters: splat once per kernel from the Coef in the
// constant bank; per-cell parameters: the pairs are what the cells kernel stages in shared memory (no move needed).
struct Coef2 {
    f32x2 s, ms, a, mck, bk4, k2, b2, th4, theta;
};
__device__ __forceinline__ Coef2 splat_coef(const Coef<float>& C) {
    return Coef2{splat2(C.s), splat2(-C.s), splat2(C.a), splat2(-C.ck), splat2(C.bk4), splat2(C.k2), splat2(C.b2),
                 splat2(C.th4), splat2(C.theta)};
}

// Selects as predicated arithmetic on one half of a pair: "if the chain is on its MUFU side, overwrite the polynomial
// side's value" -- the product / sum is formed by a predicated scalar instruction (as many FMA-pipe cycles as the packed
// one it replaces) and the two FSELs per pair (ALU pipe) disappear.  .rn: no contraction, same bits as the packed
// and the scalar chain.  The comparisons are the unordered complements of the scalar chain's (NaN takes the same side).
__device__ __forceinline__ void mul_if_geu(float& dst, float x, float bound, float a, float b) {
    asm("{ .reg .pred q; setp.geu.f32 q, %1, %2; @q mul.rn.f32 %0, %3, %4; }" : "+f"(dst) : "f"(x), "f"(bound), "f"(a), "f"(b));
}
__device__ __forceinline__ void add_if_geu(float& dst, float x, float bound, float a, float b) {
    asm("{ .reg .pred q; setp.geu.f32 q, %1, %2; @q add.rn.f32 %0, %3, %4; }" : "+f"(dst) : "f"(x), "f"(bound), "f"(a), "f"(b));
}
__device__ __forceinline__ void mul_mov_if_ltu(float& num, float& den, float x, float a, float b, float c) {   // x < 0 or NaN
    asm("{ .reg .pred q; setp.ltu.f32 q, %2, 0f00000000; @q mul.rn.f32 %0, %3, %4; @q mov.f32 %1, %5; }"
        : "+f"(num), "+f"(den) : "f"(x), "f"(a), "f"(b), "f"(c));
}

// 2V for two particles (see speed2_f32).
template <bool U64>
__device__ __forceinline__ f32x2 speed2_f32x2(uint32_t w0a, uint32_t w0b, uint32_t w3a, uint32_t w3b, const Coef2& C) {
    // 2^32 U1 and 1 - U1 (uniform1_f32, packed); U64: the fourth word refines both where the first is small
    const f32x2 ulo = U64 ? fma2(pk2((float)w3a, (float)w3b), splat2(0x1p-32f), splat2(0x1p-33f)) : splat2(0.5f);
    const f32x2 tlo = U64 ? fma2(pk2((float)(uint32_t)(~w3a), (float)(uint32_t)(~w3b)), splat2(0x1p-64f), splat2(0x1p-65f))
                          : splat2(0x1p-33f);
    const f32x2 lg = KG_MAP2(mufu_lg2, add2(pk2((float)w0a, (float)w0b), ulo));
    const f32x2 r = KG_MAP2(mufu_ex2, fma2(lg, splat2(0x1.555556p-2f), splat2(-0x1.555556p+3f)));
    const f32x2 t1 = fma2(pk2((float)(uint32_t)(~w0a), (float)(uint32_t)(~w0b)), splat2(0x1p-32f), tlo);
    const f32x2 p = mul2(r, r);
    const f32x2 q1 = add2(r, splat2(1.0f));
    const f32x2 S = mul2(mul2(t1, q1), KG_MAP2(mufu_rcp, add2(q1, p)));
    f32x2 G = fma2(splat2(0x1.f448fp-2f), p, splat2(0x1.ab553ap-3f));
    G = fma2(G, p, splat2(0x1.7c9f74p-2f));
    G = fma2(G, p, splat2(0x1.ebc184p-2f));
    G = fma2(G, p, splat2(0x1.71565ep-1f));
    G = fma2(G, p, splat2(0x1.715476p+0f));
    const f32x2 m_small = mul2(mul2(p, C.s), G);
    float pa, pb, ma, mb;
    up2(p, pa, pb);
    {
        float Sa, Sb, msa, msb;
        up2(S, Sa, Sb); up2(C.ms, msa, msb); up2(m_small, ma, mb);
        mul_if_geu(ma, pa, 0.25f, mufu_lg2(Sa), msa);
        mul_if_geu(mb, pb, 0.25f, mufu_lg2(Sb), msb);
    }
    const f32x2 m = pk2(ma, mb);
    f32x2 R = fma2(splat2(0x1.945094p-10f), m, splat2(0x1.3817fcp-7f));
    R = fma2(R, m, splat2(0x1.c6d414p-5f));
    R = fma2(R, m, splat2(0x1.ebfb52p-3f));
    R = fma2(R, m, splat2(0x1.62e43p-1f));
    const f32x2 y_small = mul2(m, R);
    float Ya, Yb;
    up2(y_small, Ya, Yb);
    add_if_geu(Ya, ma, 0.5f, mufu_ex2(ma), -1.0f);
    add_if_geu(Yb, mb, 0.5f, mufu_ex2(mb), -1.0f);
    const f32x2 Y = pk2(Ya, Yb);
    const f32x2 A = fma2(Y, C.mck, C.a);
    const f32x2 D = KG_MAP2(mufu_sqrt, fma2(A, A, mul2(Y, C.bk4)));
    float Aa, Ab, Da, Db;
    up2(A, Aa, Ab); up2(D, Da, Db);
    const float Ta = fabsf(Aa) + Da, Tb = fabsf(Ab) + Db;
    float b2a, b2b;
    up2(C.b2, b2a, b2b);
    float na, nb, da = Ta, db = Tb, t4a, t4b;
    up2(mul2(Y, C.k2), na, nb); up2(C.th4, t4a, t4b);
    mul_mov_if_ltu(na, da, Aa, Ta, t4a, b2a);
    mul_mov_if_ltu(nb, db, Ab, Tb, t4b, b2b);
    const f32x2 num = pk2(na, nb), den = pk2(da, db);
    return mul2(num, KG_MAP2(mufu_rsq, mul2(num, den)));
}

template <bool U64>
__device__ __forceinline__ f32x2 speed2_f32x2(uint32_t w0a, uint32_t w0b, uint32_t w3a, uint32_t w3b, const Coef<float>& C) {
    return speed2_f32x2<U64>(w0a, w0b, w3a, w3b, splat_coef(C));
}

__device__ __forceinline__ void quadrant_f32(uint32_t w2, float sr, float cr, float& cphi, float& sphi) {
    const uint32_t wq = w2 + 0x20000000u;
    const bool odd = (wq & 0x40000000u) != 0u;
    const float c0 = odd ? sr : cr;
    const float s0 = odd ? cr : sr;
    cphi = __uint_as_float(__float_as_uint(c0) ^ ((wq + 0x40000000u) & 0x80000000u));
    sphi = __uint_as_float(__float_as_uint(s0) ^ (wq & 0x80000000u));
}

// DRIFT: (dx, dy, dz) as pairs, added by the last multiply-add (see velocity_f32).
template <bool FOLD, bool U64 = false, bool DRIFT = false>
__device__ __forceinline__ void velocity_pair_f32(const uint32_t (&w0)[2], const uint32_t (&w1)[2], const uint32_t (&w2)[2],
                                                  const uint32_t (&w3)[2], const Coef2& C, float (&vx)[2],
                                                  float (&vy)[2], float (&vz)[2], f32x2 dx = 0ull, f32x2 dy = 0ull,
                                                  f32x2 dz = 0ull) {
    f32x2 V2 = speed2_f32x2<U64>(w0[0], w0[1], w3[0], w3[1], C);
    if (!FOLD) V2 = mul2(V2, C.theta);
    const f32x2 muh = fma2(pk2((float)(int32_t)(w1[0] ^ 0x80000000u), (float)(int32_t)(w1[1] ^ 0x80000000u)),
                           splat2(0x1p-32f), splat2(0x1p-33f));
    const f32x2 ef = pk2((float)min(w1[0], ~w1[0]), (float)min(w1[1], ~w1[1]));
    const f32x2 e = fma2(ef, splat2(0x1p-32f), splat2(0x1p-33f));
    const f32x2 ne = fma2(ef, splat2(-0x1p-32f), splat2(-0x1p-33f));
    const f32x2 sth = KG_MAP2(mufu_sqrt, fma2(ne, e, e));
    const f32x2 q = fma2(pk2((float)(int32_t)(w2[0] << 2), (float)(int32_t)(w2[1] << 2)), splat2(0x1p-32f), splat2(0x1p-31f));
    const f32x2 z = mul2(q, q);
    f32x2 sp = fma2(splat2(-0x1.2d9b4p-8f), z, splat2(0x1.465ec4p-4f));
    sp = fma2(sp, z, splat2(-0x1.4abbbap-1f));
    sp = fma2(sp, z, splat2(0x1.921fb6p+0f));
    f32x2 cr = fma2(splat2(-0x1.4e5e06p-6f), z, splat2(0x1.03af58p-2f));
    cr = fma2(cr, z, splat2(-0x1.3bd392p+0f));
    cr = fma2(cr, z, splat2(0x1.0p+0f));
    const f32x2 sr = mul2(sp, q);
    float sra, srb, cra, crb, ca, cb, sa, sb;
    up2(sr, sra, srb); up2(cr, cra, crb);
    quadrant_f32(w2[0], sra, cra, ca, sa);
    quadrant_f32(w2[1], srb, crb, cb, sb);
    const f32x2 Vs = mul2(V2, sth);
    if (DRIFT) {
        up2(fma2(V2, muh, dx), vx[0], vx[1]);
        up2(fma2(Vs, pk2(ca, cb), dy), vy[0], vy[1]);
        up2(fma2(Vs, pk2(sa, sb), dz), vz[0], vz[1]);
    } else {
        up2(mul2(V2, muh), vx[0], vx[1]);
        up2(mul2(Vs, pk2(ca, cb)), vy[0], vy[1]);
        up2(mul2(Vs, pk2(sa, sb)), vz[0], vz[1]);
    }
}
template <bool FOLD, bool U64 = false>
__device__ __forceinline__ void velocity_pair_f32(const uint32_t (&w0)[2], const uint32_t (&w1)[2], const uint32_t (&w2)[2],
                                                  const uint32_t (&w3)[2], const Coef<float>& C, float (&vx)[2],
                                                  float (&vy)[2], float (&vz)[2]) {
    velocity_pair_f32<FOLD, U64, false>(w0, w1, w2, w3, splat_coef(C), vx, vy, vz);
}

}  // namespace kappagen
