// pipe_probe.cuh -- issue-rate probe of the sm_100 pipes the kappagen kernels are bound by (kappagen_pipe_probe,
// include/kappagen.h).  Not on the hot path: it is the tracked source of the per-instruction cycle figures that
// DESIGN.md section 5 and profiles/r03_pipe_rates.md quote (the "alu" roofline peaks of bench.py).
//
// Each mix is a register-only loop body of N instructions per kind, eight independent dependency chains per kind so
// that latency never binds; inline PTX, one SASS instruction each:
//   wide   mul.wide.u32   -> IMAD.WIDE.U32   (Philox's 32x32->64 product)
//   lop3   lop3.b32       -> LOP3.LUT        (Philox's three-input xor; the ALU pipe)
//   ffma2  fma.rn.f32x2   -> FFMA2           (the packed float chain)
//   mufu   ex2.approx.f32 -> MUFU.EX2        (special-function unit)
//   dfma   fma.rn.f64     -> DFMA            (the double chain)
//   imad   mad.lo.u32     -> IMAD            (32-bit multiply-add)
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace kappagen {

template <int NW, int NL, int NP, int NM, int ND, int NI, bool kSpread>
__global__ void __launch_bounds__(1024) pipe_probe_kernel(int iters, uint32_t seed, uint32_t* sink, long long* cycles) {
    uint32_t w[8], l[8], im[8];
    float m[8];
    unsigned long long p[8];
    double d[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        w[i] = seed + threadIdx.x * 8u + (uint32_t)i;
        l[i] = seed ^ ((uint32_t)i * 77u + threadIdx.x);
        im[i] = l[i] * 5u;
        m[i] = 0.5f + 0.01f * (float)i;
        p[i] = ((unsigned long long)__float_as_uint(1.0f + 1e-3f * (float)i) << 32) | __float_as_uint(1.0f + 2e-3f * (float)i);
        d[i] = 1.0 + 1e-3 * (double)i + 1e-9 * (double)seed;
    }
    const float fa = 0.999f + 1e-9f * (float)seed, fb = 1e-3f;
    const double da = 0.999 + 1e-9 * (double)seed, db = 1e-3;
    const unsigned long long pa = ((unsigned long long)__float_as_uint(fa) << 32) | __float_as_uint(fa);
    const unsigned long long pb = ((unsigned long long)__float_as_uint(fb) << 32) | __float_as_uint(fb);
    constexpr int kMax = NW > NL ? (NW > NP ? NW : NP) : (NL > NP ? NL : NP);
    constexpr int kMax2 = NM > ND ? (NM > NI ? NM : NI) : (ND > NI ? ND : NI);
    constexpr int kRounds = ((kMax > kMax2 ? kMax : kMax2) + 7) / 8;
    // kSpread = false (mixes 0-20, laid out as in round 2): each kind fills the body's slots from the front.  kSpread = true
    // (the kernels' exact proportions, mixes 21 on): each kind is spread evenly over the 8 * kRounds slots of the body.
    constexpr int kSlots = 8 * kRounds;
#define KG_PROBE_EMIT(N, s) (kSpread ? (((s) + 1) * (N) / kSlots > (s) * (N) / kSlots) : ((s) < (N)))
    const long long t0 = clock64();
#pragma unroll 1
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < kRounds; ++r) {
#pragma unroll
            for (int k = 0; k < 8; ++k) {
                if (KG_PROBE_EMIT(NW, r * 8 + k)) {
                    unsigned long long q;
                    uint32_t lo, hi;
                    asm volatile("mul.wide.u32 %0, %1, 0xD2511F53;" : "=l"(q) : "r"(w[k]));
                    asm volatile("mov.b64 {%0,%1}, %2;" : "=r"(lo), "=r"(hi) : "l"(q));
                    w[k] = hi;
                }
                if (KG_PROBE_EMIT(NL, r * 8 + k)) asm volatile("lop3.b32 %0, %0, %1, 0x9E3779B9, 0x96;" : "+r"(l[k]) : "r"(l[(k + 1) & 7]));
                if (KG_PROBE_EMIT(NP, r * 8 + k)) asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(p[k]) : "l"(pa), "l"(pb));
                if (KG_PROBE_EMIT(NM, r * 8 + k)) asm volatile("ex2.approx.ftz.f32 %0, %0;" : "+f"(m[k]));
                if (KG_PROBE_EMIT(ND, r * 8 + k)) asm volatile("fma.rn.f64 %0, %0, %1, %2;" : "+d"(d[k]) : "d"(da), "d"(db));
                if (KG_PROBE_EMIT(NI, r * 8 + k)) asm volatile("mad.lo.u32 %0, %0, 0xD2511F53, %1;" : "+r"(im[k]) : "r"(seed));
            }
        }
    }
#undef KG_PROBE_EMIT
    const long long t1 = clock64();
    uint32_t acc = 0u;
#pragma unroll
    for (int i = 0; i < 8; ++i)
        acc ^= w[i] ^ l[i] ^ im[i] ^ __float_as_uint(m[i]) ^ (uint32_t)p[i] ^ (uint32_t)(p[i] >> 32) ^
               (uint32_t)__double2loint(d[i]) ^ (uint32_t)__double2hiint(d[i]);
    if (acc == 0x12345678u) sink[threadIdx.x] = acc;                 // keeps every chain alive; practically never taken
    if (threadIdx.x == 0) cycles[blockIdx.x] = t1 - t0;
}

struct PipeMix {
    int wide, lop3, ffma2, mufu, dfma, imad;
    bool spread = false;
};
// The table kappagen_pipe_probe indexes.  Single kinds first (the pipe rates), then pairs (which pipes overlap),
// then the kernels' own proportions.
constexpr PipeMix kPipeMixes[] = {
    {8, 0, 0, 0, 0, 0},  {0, 8, 0, 0, 0, 0},  {0, 0, 8, 0, 0, 0},  {0, 0, 0, 8, 0, 0},  {0, 0, 0, 0, 8, 0},   // 0-4
    {0, 0, 0, 0, 0, 8},  {8, 8, 0, 0, 0, 0},  {8, 16, 0, 0, 0, 0}, {8, 24, 0, 0, 0, 0}, {8, 0, 8, 0, 0, 0},   // 5-9
    {8, 0, 0, 4, 0, 0},  {8, 0, 0, 0, 8, 0},  {8, 0, 0, 0, 16, 0}, {4, 0, 0, 0, 16, 0}, {0, 8, 0, 0, 16, 0},  // 10-14
    {0, 0, 0, 0, 16, 8}, {0, 16, 8, 4, 0, 0}, {8, 16, 8, 4, 0, 0}, {8, 16, 0, 4, 0, 0}, {4, 8, 0, 2, 16, 0},  // 15-19
    {0, 8, 0, 2, 16, 0},                                                                                      // 20
    // 21: the double sampler's own instruction mix per particle (cuobjdump -sass, whole-tile body of
    // sample_kernel<double,1,0,0>, profiles/r03_fp64_limit.md): 85 FP64, 18 wide multiplies, 56 ALU-pipe, 6 MUFU, 9 IMAD;
    // 22: the same without the wide multiplies (the mix of kappagen_math_planes); 23: FP64 + ALU only
    {18, 56, 0, 6, 85, 9, true}, {0, 56, 0, 6, 85, 9, true}, {0, 56, 0, 0, 85, 0, true},                                        // 21-23
};
constexpr int kPipeMixCount = (int)(sizeof(kPipeMixes) / sizeof(kPipeMixes[0]));

typedef void (*PipeProbeFn)(int, uint32_t, uint32_t*, long long*);
template <int I> struct PipeProbeTable {
    static void fill(PipeProbeFn* t) {
        constexpr PipeMix M = kPipeMixes[I];
        t[I] = pipe_probe_kernel<M.wide, M.lop3, M.ffma2, M.mufu, M.dfma, M.imad, M.spread>;
        PipeProbeTable<I + 1>::fill(t);
    }
};
template <> struct PipeProbeTable<kPipeMixCount> {
    static void fill(PipeProbeFn*) {}
};

}  // namespace kappagen
