// philox.cuh -- register-resident Philox4x32-10 for the kappagen kernels (step S1 of DESIGN.md).
//
// The RNG is fixed by BASELINE.json's north_star (the paper says only "generate U1,U2,U3 ~
// Uniform(0,1)", Table I line 5).  Algorithm: Salmon, Moraes, Dror, Shaw, "Parallel
// random numbers: as easy as 1, 2, 3" (SC'11).  Written from that description for this kernel; no
// code is shared with oracle/.
//
// Layout (reading R6): particle g uses counter (lo32 g, hi32 g, c2, c3) and key
// (lo32 seed, hi32 seed); the samplers use c2 = c3 = 0, the rejection baseline uses c2 = trial
// number and c3 = stream id.  The ten round keys depend only on the seed, so the host expands them
// once (PhiloxKeys) and they reach the kernel through the constant bank: the per-particle cost is
// 10 rounds x (2 IMAD.WIDE + 2 LOP3), less what constant propagation removes when c2 = c3 = 0.
#pragma once
#include <cstdint>

namespace kappagen {

struct PhiloxKeys {
    uint32_t k0[10];
    uint32_t k1[10];
};

constexpr uint32_t kPhiloxM0 = 0xD2511F53u;  // multiplies counter word 0
constexpr uint32_t kPhiloxM1 = 0xCD9E8D57u;  // multiplies counter word 2
constexpr uint32_t kPhiloxW0 = 0x9E3779B9u;  // key schedule: golden ratio
constexpr uint32_t kPhiloxW1 = 0xBB67AE85u;  // key schedule: sqrt(3) - 1

inline PhiloxKeys philox_expand_keys(uint64_t seed) {
    PhiloxKeys K;
    uint32_t a = (uint32_t)seed, b = (uint32_t)(seed >> 32);
    for (int r = 0; r < 10; ++r) {
        K.k0[r] = a;
        K.k1[r] = b;
        a += kPhiloxW0;
        b += kPhiloxW1;
    }
    return K;
}

#ifdef __CUDACC__
// One Philox4x32-10 block.  w3 is computed only if the caller uses it (dead code otherwise).
__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                              const PhiloxKeys& K, uint32_t& w0, uint32_t& w1,
                                              uint32_t& w2, uint32_t& w3) {
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint64_t p0 = (uint64_t)kPhiloxM0 * (uint64_t)c0;  // IMAD.WIDE.U32
        const uint64_t p1 = (uint64_t)kPhiloxM1 * (uint64_t)c2;
        const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ K.k0[r];  // LOP3
        const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ K.k1[r];
        c1 = (uint32_t)p1;
        c3 = (uint32_t)p0;
        c0 = n0;
        c2 = n2;
    }
    w0 = c0; w1 = c1; w2 = c2; w3 = c3;
}

// Counters that share their high word.  With ctr = (c0, c1, 0, 0) round 1 multiplies M1 by zero, so
// after it the new word 0 is c1 ^ k0[0] -- the same for every particle with the same hi32(g) -- and
// round 2's product M0 * (c1 ^ k0[0]) is shared too.  A thread computes this head once per 128-bit
// group and each particle then needs 18 wide multiplies instead of 19 (+1 shared) and no 64-bit add.
struct PhiloxHead {
    uint32_t hi, lo;   // M0 * (hi32(g) ^ k0[0])
};
__device__ __forceinline__ PhiloxHead philox_head(uint32_t g_hi, const PhiloxKeys& K) {
    const uint64_t p = (uint64_t)kPhiloxM0 * (uint64_t)(g_hi ^ K.k0[0]);
    return PhiloxHead{(uint32_t)(p >> 32), (uint32_t)p};
}
// Same words as particle_words(g, ...) for g = (g_hi << 32) | g_lo, given H = philox_head(g_hi, K).
// q0 = M0 * lo32(g), round 1's only product, supplied by the caller: for counters a compile-time distance
// apart it is one multiply plus 64-bit additions of constants (M0 (g + d) = M0 g + M0 d).
__device__ __forceinline__ void particle_words_q0(uint64_t q0, const PhiloxHead& H, const PhiloxKeys& K,
                                                  uint32_t& w0, uint32_t& w1, uint32_t& w2, uint32_t& w3);
__device__ __forceinline__ void particle_words_head(uint32_t g_lo, const PhiloxHead& H, const PhiloxKeys& K,
                                                    uint32_t& w0, uint32_t& w1, uint32_t& w2, uint32_t& w3) {
    particle_words_q0((uint64_t)kPhiloxM0 * (uint64_t)g_lo, H, K, w0, w1, w2, w3);
}
__device__ __forceinline__ void particle_words_q0(uint64_t q0, const PhiloxHead& H, const PhiloxKeys& K,
                                                  uint32_t& w0, uint32_t& w1, uint32_t& w2, uint32_t& w3) {
    // round 1 (c2 = c3 = 0): c = (g_hi ^ k0[0], 0, hi(M0 g_lo) ^ k1[0], lo(M0 g_lo))
    // round 2: the M0 product is the shared head; c1 = 0
    const uint64_t q1 = (uint64_t)kPhiloxM1 * (uint64_t)((uint32_t)(q0 >> 32) ^ K.k1[0]);
    uint32_t c0 = (uint32_t)(q1 >> 32) ^ K.k0[1];
    uint32_t c1 = (uint32_t)q1;
    uint32_t c2 = H.hi ^ (uint32_t)q0 ^ K.k1[1];
    uint32_t c3 = H.lo;
#pragma unroll
    for (int r = 2; r < 10; ++r) {
        const uint64_t p0 = (uint64_t)kPhiloxM0 * (uint64_t)c0;
        const uint64_t p1 = (uint64_t)kPhiloxM1 * (uint64_t)c2;
        const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ K.k0[r];
        const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ K.k1[r];
        c1 = (uint32_t)p1;
        c3 = (uint32_t)p0;
        c0 = n0;
        c2 = n2;
    }
    w0 = c0; w1 = c1; w2 = c2; w3 = c3;
}

// The words of particle g.  The samplers consume w0, w1, w2; w3 is drawn and discarded (DESIGN.md reading
// R4) unless the caller asks for the 64-bit U1 (reading R20), and is dead code when unused.
__device__ __forceinline__ void particle_words(uint64_t g, const PhiloxKeys& K, uint32_t& w0,
                                               uint32_t& w1, uint32_t& w2, uint32_t& w3) {
    philox4x32_10((uint32_t)g, (uint32_t)(g >> 32), 0u, 0u, K, w0, w1, w2, w3);
}
__device__ __forceinline__ void particle_words(uint64_t g, const PhiloxKeys& K, uint32_t& w0,
                                               uint32_t& w1, uint32_t& w2) {
    uint32_t w3;
    particle_words(g, K, w0, w1, w2, w3);
    (void)w3;
}
#endif  // __CUDACC__

}  // namespace kappagen
