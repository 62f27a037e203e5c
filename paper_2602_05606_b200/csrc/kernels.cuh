// kernels.cuh -- the kappagen kernels (sm_100a).  Launchers and the C ABI are in kappagen_api.cu.
//
// Mapping.  A thread produces G = 16/sizeof(T) consecutive particles per group, so that each of its
// three stores is one 128-bit st.global (a warp writes 512 contiguous bytes per plane), and NG groups
// per tile for instruction-level parallelism.  Blocks walk the index range in a grid-stride loop; the
// output is a pure function of the particle index, so the mapping never shows in the result.
// The path is write-only: 0 bytes read, 3*sizeof(T) bytes written per particle (12 fp32 / 24 fp64).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>
#include "coefs.cuh"
#include "math_f32.cuh"
#include "math_f32x2.cuh"
#include "math_f64.cuh"
#include "philox.cuh"

namespace kappagen {

constexpr int kThreads = 256;
constexpr int kGroups = 2;  // 128-bit groups per thread per tile
// Tile shape of the sample kernels, measured on B200 (the macros are sweep knobs).
// double: 4 groups (8 particles) per thread generated in one straight line -- whole tiles inside one 2^32
// block of counters only, one Philox head per tile, no branch between the groups, stores last -- 384 threads,
// one block per SM (156 registers): the chains are long and share 64-bit constants, which the compiler keeps
// resident.  1.29e11 particles/s; 64-1024 threads x 1-6 groups all lie between 2.08 and 2.43 ms per 2^28, this
// shape is the minimum.  float: the same straight-line tile with 2 groups (8 particles, 98 registers, 2 blocks
// per SM): 2.32e11 particles/s; 1, 3 or 4 groups and min-blocks 2-4 are within 3 % below it.
#ifndef KG_JOINT_F64
#define KG_JOINT_F64 1
#endif
#ifndef KG_F64_GROUPS
#define KG_F64_GROUPS 4
#endif
#ifndef KG_F64_MINB
#define KG_F64_MINB 1
#endif
#ifndef KG_F64_THREADS
#define KG_F64_THREADS 384
#endif
#ifndef KG_JOINT_F32
#define KG_JOINT_F32 1
#endif
#ifndef KG_F32_GROUPS
#define KG_F32_GROUPS 2
#endif
#ifndef KG_F32_MINB
#define KG_F32_MINB 1
#endif
template <typename T> struct TileTraits {
    static constexpr bool joint = (sizeof(T) == 8) ? KG_JOINT_F64 : KG_JOINT_F32;
    static constexpr int groups = sizeof(T) == 8 ? KG_F64_GROUPS : KG_F32_GROUPS;   // of the sample kernel
    static constexpr int minb = sizeof(T) == 8 ? KG_F64_MINB : KG_F32_MINB;
    static constexpr int threads = sizeof(T) == 8 ? KG_F64_THREADS : kThreads;
    // round 1's product M0 * lo32(g) of the thread's 2nd..8th particle by adding the constant M0 * distance to the
    // first one's: two ALU adds instead of a quarter-rate multiply.  Pays where the FMA-heavy pipe is the
    // bound (float: +1 %), costs where it is not (double: -5 %).
    static constexpr bool round1_add = sizeof(T) == 4;
};

// Shared-memory lookup tables of the double chain (math_f64.cuh); nothing for float.  Called once per block, by all
// its threads, before the first particle.
template <typename T> __device__ __forceinline__ void math_tables_init() {
    if constexpr (sizeof(T) == 8) f64_tables_init();
}

template <typename T> struct Vec128;
template <> struct Vec128<float> { using type = float4; };
template <> struct Vec128<double> { using type = double2; };

// FOLD (float only): theta is folded into the coefficients, see coefs.cuh.  U64: U1 takes 64 bits from
// (w0, w3) instead of 32 from w0 (reading R20); w3 is ignored otherwise.
template <bool FOLD, bool U64 = false>
__device__ __forceinline__ void velocity(uint32_t w0, uint32_t w1, uint32_t w2, uint32_t w3, const Coef<float>& C,
                                         float& x, float& y, float& z) { velocity_f32<FOLD, U64>(w0, w1, w2, w3, C, x, y, z); }
template <bool FOLD, bool U64 = false>
__device__ __forceinline__ void velocity(uint32_t w0, uint32_t w1, uint32_t w2, uint32_t w3, const Coef<double>& C,
                                         double& x, double& y, double& z) { velocity_f64<U64>(w0, w1, w2, w3, C, x, y, z); }

// The Philox words of G consecutive particles starting at global counter g0.  Unless the low counter
// word wraps inside the group (one group in 2^32 particles; a uniform branch everywhere else) the
// particles share hi32(g) and with it the head of the Philox block (philox.cuh).
template <int G>
__device__ __forceinline__ void group_words(uint64_t g0, const PhiloxKeys& K, uint32_t (&w0)[G], uint32_t (&w1)[G],
                                            uint32_t (&w2)[G], uint32_t (&w3)[G]) {
    const uint32_t lo = (uint32_t)g0, hi = (uint32_t)(g0 >> 32);
    if (lo <= 0xFFFFFFFFu - (uint32_t)(G - 1)) {
        const PhiloxHead H = philox_head(hi, K);
#pragma unroll
        for (int e = 0; e < G; ++e) particle_words_head(lo + (uint32_t)e, H, K, w0[e], w1[e], w2[e], w3[e]);
    } else {
#pragma unroll
        for (int e = 0; e < G; ++e) particle_words(g0 + (uint64_t)e, K, w0[e], w1[e], w2[e], w3[e]);
    }
}

// Velocities of one 128-bit group from its words.  float: two packed pairs (math_f32x2.cuh, bit-identical
// to the scalar chain); double: two scalar chains.
template <bool FOLD, bool U64>
__device__ __forceinline__ void words_to_velocities(const uint32_t (&w0)[4], const uint32_t (&w1)[4], const uint32_t (&w2)[4],
                                                    const uint32_t (&w3)[4], const Coef<float>& C, float (&ox)[4],
                                                    float (&oy)[4], float (&oz)[4]) {
#pragma unroll
    for (int e = 0; e < 4; e += 2) {
        const uint32_t p0[2] = {w0[e], w0[e + 1]}, p1[2] = {w1[e], w1[e + 1]}, p2[2] = {w2[e], w2[e + 1]};
        const uint32_t p3[2] = {w3[e], w3[e + 1]};
        float a[2], b[2], c[2];
        velocity_pair_f32<FOLD, U64>(p0, p1, p2, p3, C, a, b, c);
        ox[e] = a[0]; ox[e + 1] = a[1];
        oy[e] = b[0]; oy[e + 1] = b[1];
        oz[e] = c[0]; oz[e + 1] = c[1];
    }
}
template <bool FOLD, bool U64>
__device__ __forceinline__ void words_to_velocities(const uint32_t (&w0)[2], const uint32_t (&w1)[2], const uint32_t (&w2)[2],
                                                    const uint32_t (&w3)[2], const Coef<double>& C, double (&ox)[2],
                                                    double (&oy)[2], double (&oz)[2]) {
#pragma unroll
    for (int e = 0; e < 2; ++e) velocity_f64<U64>(w0[e], w1[e], w2[e], w3[e], C, ox[e], oy[e], oz[e]);
}

// One 128-bit group: G consecutive particles starting at global counter g0.
template <bool FOLD, bool U64 = false, typename T, int G>
__device__ __forceinline__ void group_velocities(uint64_t g0, const PhiloxKeys& K, const Coef<T>& C,
                                                 T (&ox)[G], T (&oy)[G], T (&oz)[G]) {
    uint32_t w0[G], w1[G], w2[G], w3[G];
    group_words<G>(g0, K, w0, w1, w2, w3);
    words_to_velocities<FOLD, U64>(w0, w1, w2, w3, C, ox, oy, oz);
}
// Words of group j of a WHOLE tile (all of it inside one 2^32 block of counters): shared Philox head, no branch.
// lo_first = lo32(counter of the thread's first particle in the tile), q_first = M0 * lo_first; group j starts
// j * threads * G particles later.  Where TileTraits<T>::round1_add holds, round 1's product of every particle is
// q_first plus a compile-time constant instead of a multiply.  This is the ONE function through which the
// samplers, the histogram kernel and the kappagen_words_tile test hook draw the words of a whole tile.
template <typename T, int G, int THREADS = TileTraits<T>::threads>
__device__ __forceinline__ void tile_group_words(uint32_t lo_first, uint64_t q_first, int j, const PhiloxHead& H, const PhiloxKeys& K,
                                                 uint32_t (&w0)[G], uint32_t (&w1)[G], uint32_t (&w2)[G], uint32_t (&w3)[G]) {
    const uint32_t delta = (uint32_t)(j * (THREADS * G));                   // THREADS = the calling kernel's block size
#pragma unroll
    for (int e = 0; e < G; ++e) {
        if constexpr (TileTraits<T>::round1_add)
            particle_words_q0(q_first + (uint64_t)kPhiloxM0 * (uint64_t)(delta + (uint32_t)e), H, K, w0[e], w1[e], w2[e], w3[e]);
        else
            particle_words_head(lo_first + delta + (uint32_t)e, H, K, w0[e], w1[e], w2[e], w3[e]);
    }
}
// True when the tile starting at global counter g_tile may take the whole-tile path.
__device__ __forceinline__ bool tile_in_one_block(uint64_t g_tile, int64_t tile) {
    return (uint32_t)g_tile <= 0xFFFFFFFFu - (uint32_t)tile;
}

// Streaming (evict-first) 128-bit store: the planes are never re-read by this library.
__device__ __forceinline__ void store_group(float* p, const float (&v)[4]) {
    __stcs(reinterpret_cast<float4*>(p), make_float4(v[0], v[1], v[2], v[3]));
}
__device__ __forceinline__ void store_group(double* p, const double (&v)[2]) {
    __stcs(reinterpret_cast<double2*>(p), make_double2(v[0], v[1]));
}

template <typename T, bool VEC, int G>
__device__ __forceinline__ void store_planes(int64_t i, int64_t n, T* __restrict__ vx, T* __restrict__ vy,
                                             T* __restrict__ vz, const T (&ox)[G], const T (&oy)[G], const T (&oz)[G]) {
    if (VEC && i + G <= n) {
        store_group(vx + i, ox);
        store_group(vy + i, oy);
        store_group(vz + i, oz);
    } else {
#pragma unroll
        for (int e = 0; e < G; ++e) {
            if (i + e < n) {
                vx[i + e] = ox[e];
                vy[i + e] = oy[e];
                vz[i + e] = oz[e];
            }
        }
    }
}

// ---------------------------------------------------------------- kappagen_sample
// Group j of the tile at `base`, bounds-checked (ragged tail, unaligned planes).
template <typename T, bool VEC, bool FOLD, bool U64>
__device__ __forceinline__ void tile_group(int64_t base, int j, int64_t n, uint64_t offset, const PhiloxKeys& K, const Coef<T>& C,
                                           T* __restrict__ vx, T* __restrict__ vy, T* __restrict__ vz) {
    constexpr int G = 16 / sizeof(T);
    constexpr int kT = TileTraits<T>::threads;
    const int64_t i = base + (int64_t)j * (kT * G) + (int64_t)threadIdx.x * G;
    if (i < n) {
        T ox[G], oy[G], oz[G];
        group_velocities<FOLD, U64>(offset + (uint64_t)i, K, C, ox, oy, oz);
        store_planes<T, VEC, G>(i, n, vx, vy, vz, ox, oy, oz);
    }
}

template <typename T, bool VEC, bool FOLD, bool U64>
__global__ void __launch_bounds__(TileTraits<T>::threads, TileTraits<T>::minb)
sample_kernel(int64_t n, uint64_t offset, const __grid_constant__ PhiloxKeys K, const __grid_constant__ Coef<T> C,
              T* __restrict__ vx, T* __restrict__ vy, T* __restrict__ vz) {
    constexpr int G = 16 / sizeof(T);
    constexpr int NG = TileTraits<T>::groups;
    constexpr int kT = TileTraits<T>::threads;
    constexpr int64_t kTile = (int64_t)kT * G * NG;
    math_tables_init<T>();
    for (int64_t base = (int64_t)blockIdx.x * kTile; base < n; base += (int64_t)gridDim.x * kTile) {
        const uint64_t g_tile = offset + (uint64_t)base;
        if (VEC && TileTraits<T>::joint && base + kTile <= n && tile_in_one_block(g_tile, kTile)) {
            // whole tile in range and inside one 2^32 block of counters: one Philox head for the tile and all
            // groups of the thread in one straight line -- no branch between them, so their independent chains
            // interleave and share the materialised constants; stores last
            const PhiloxHead H = philox_head((uint32_t)(g_tile >> 32), K);
            const uint32_t lo_first = (uint32_t)g_tile + threadIdx.x * (uint32_t)G;
            const uint64_t q_first = (uint64_t)kPhiloxM0 * (uint64_t)lo_first;
            T ox[NG][G], oy[NG][G], oz[NG][G];
#pragma unroll
            for (int j = 0; j < NG; ++j) {
                uint32_t w0[G], w1[G], w2[G], w3[G];
                tile_group_words<T, G>(lo_first, q_first, j, H, K, w0, w1, w2, w3);
                words_to_velocities<FOLD, U64>(w0, w1, w2, w3, C, ox[j], oy[j], oz[j]);
            }
#pragma unroll
            for (int j = 0; j < NG; ++j) {
                const int64_t i = base + (int64_t)j * (kT * G) + (int64_t)threadIdx.x * G;
                store_group(vx + i, ox[j]);
                store_group(vy + i, oy[j]);
                store_group(vz + i, oz[j]);
            }
            continue;
        }
        if constexpr (TileTraits<T>::joint) {
#pragma unroll 1
            for (int j = 0; j < NG; ++j) tile_group<T, VEC, FOLD, U64>(base, j, n, offset, K, C, vx, vy, vz);
        } else {
#pragma unroll
            for (int j = 0; j < NG; ++j) tile_group<T, VEC, FOLD, U64>(base, j, n, offset, K, C, vx, vy, vz);
        }
    }
}

// ---------------------------------------------------------------- kappagen_sample_cells
template <typename T> __device__ __forceinline__ Coef<T> cell_coef(const TableIParams<double>& P, double theta);
template <> __device__ __forceinline__ Coef<float> cell_coef<float>(const TableIParams<double>& P, double theta) {
    return make_coef_f32<double>(P, theta, false);                     // per-cell theta: never folded
}
template <> __device__ __forceinline__ Coef<double> cell_coef<double>(const TableIParams<double>& P, double theta) {
    return make_coef_f64<double>(P, theta);
}

// Pre-kernel: Table I lines 1-4 per cell, in double, and the cell's drift, into the workspace (one CellRec<T> per cell).
template <typename T>
__global__ void __launch_bounds__(kThreads)
cell_coef_kernel(int64_t ncell, const T* __restrict__ kappa, const T* __restrict__ theta, const T* __restrict__ drift,
                 int64_t drift_stride, CellRec<T>* __restrict__ W, T* __restrict__ mom_to_zero) {
    const int64_t cell = (int64_t)blockIdx.x * kThreads + threadIdx.x;
    if (cell >= ncell) return;
    if (mom_to_zero != nullptr) {                                      // atomic moment modes accumulate into zeros
#pragma unroll
        for (int q = 0; q < 4; ++q) mom_to_zero[4 * cell + q] = T(0);
    }
    const double kap = (double)kappa[cell], th = (double)theta[cell];
    const bool ok = isfinite(kap) && isfinite(th) && kap > 1.5 && th >= 0.0;
    const double ks = ok ? kap - 0.5 : 1.0;
    const double lnB = lgamma(1.5) + lgamma(ks) - lgamma(ks + 1.5);   // ln B(3/2, kappa*)
    const TableIParams<double> P = table1_params<double>(ok ? kap : 2.5, lnB, c_approx_f64(ok ? kap : 2.5));
    // an invalid cell becomes NaN in all its particles: poison theta at the source, so that every constant derived
    // from it (theta for float, theta and 2 theta for double) carries the NaN into the chain
    const Coef<T> C = cell_coef<T>(P, ok ? th : nan(""));
    T dx = T(0), dy = T(0), dz = T(0);
    if (drift != nullptr) {
        const T* d = drift + 3 * cell * drift_stride;
        dx = d[0]; dy = d[1]; dz = d[2];
    }
    W[cell] = make_cell_rec(C, dx, dy, dz);
}

// floor(i / ppc) without a 64-bit division.  magic < 64: ppc = 2^magic, a shift.  Otherwise magic =
// floor(2^64 / ppc) + 1, exact for i * ppc < 2^64 (the launcher checks n * ppc < 2^64 and passes magic = ~0
// otherwise, which selects the plain division).
__device__ __forceinline__ int64_t cell_of(int64_t i, uint32_t ppc, uint64_t magic) {
    if (magic < 64ull) return i >> (int)magic;
    return magic != ~0ull ? (int64_t)__umul64hi((uint64_t)i, magic) : i / (int64_t)ppc;
}

// Whole cells between a tile's first particle and the particle o places after the first particle's cell began
// (o < tile + ppc).  magic32 = ceil(2^32 / ppc) where the launcher found it exact for these o; magic32 == 0 means
// ppc >= tile (the launcher's cells_magics() guarantees it), so o < 2 ppc and the answer is 0 or 1.
__device__ __forceinline__ uint32_t cells_ahead(uint32_t o, uint32_t ppc, uint32_t magic32) {
    return magic32 != 0u ? __umulhi(o, magic32) : (uint32_t)(o >= ppc);
}

// How the fused moments (kappagen_sample_cells_moments) leave the kernel.  All sums are in T.
//   kMomDirect : ppc = G * L, L a power of two <= 32: the L lanes of a cell sit side by side in one warp; an
//                xor-shuffle butterfly leaves each of the cell's four sums in one lane, which stores it.
//                No atomics, fixed summation order (bit-reproducible).
//   kMomWarp   : ppc a multiple of 32 G: a warp lies inside one cell; shuffle tree over the warp, then one
//                atomicAdd per sum per warp into the zeroed buffer.
//   kMomAtomic : any ppc: per group (or per particle where a group straddles two cells) atomicAdd.
enum MomMode : int { kMomNone = 0, kMomDirect = 1, kMomWarp = 2, kMomAtomic = 3 };

// mask: the lanes that take part.  Whole tiles: every lane of the warp; the guarded path hands in the ballot of
// its own condition (with n = ncell * ppc a cell's lanes are in range together, so the shuffle modes only ever
// see full segments).
template <typename T>
__device__ __forceinline__ void moments_out(T (&ps)[4], int64_t cell, int mode, int lanes, T* __restrict__ mom, unsigned mask) {
    if (mode == kMomAtomic) {
#pragma unroll
        for (int q = 0; q < 4; ++q) atomicAdd(mom + 4 * cell + q, ps[q]);
        return;
    }
    const unsigned lane = threadIdx.x & (unsigned)(lanes - 1);         // lane inside the cell's segment
    if (lanes >= 4) {
        // Transposing butterfly: after two exchange steps each lane of a quad owns ONE of the four sums over
        // its quad (5 shuffles for 16 lanes instead of 16); then a plain tree across quads on that one value.
        const bool b0 = (lane & 1u) != 0u, b1 = (lane & 2u) != 0u;
        const T r0 = (b0 ? ps[2] : ps[0]) + __shfl_xor_sync(mask, b0 ? ps[0] : ps[2], 1);
        const T r1 = (b0 ? ps[3] : ps[1]) + __shfl_xor_sync(mask, b0 ? ps[1] : ps[3], 1);
        T s = (b1 ? r1 : r0) + __shfl_xor_sync(mask, b1 ? r0 : r1, 2);  // lane%4 = 0,2,1,3 holds sum 0,1,2,3
        for (int d = 4; d < lanes; d <<= 1) s += __shfl_xor_sync(mask, s, d);
        if (lane < 4u) {
            const int q = (int)((lane & 1u) * 2u + (lane >> 1));
            if (mode == kMomDirect) mom[4 * cell + q] = s;
            else atomicAdd(mom + 4 * cell + q, s);
        }
        return;
    }
    for (int d = 1; d < lanes; d <<= 1) {
#pragma unroll
        for (int q = 0; q < 4; ++q) ps[q] += __shfl_xor_sync(mask, ps[q], d);
    }
    if (lane == 0u) {
        if (mode == kMomDirect) {
#pragma unroll
            for (int q = 0; q < 4; ++q) mom[4 * cell + q] = ps[q];
        } else {
#pragma unroll
            for (int q = 0; q < 4; ++q) atomicAdd(mom + 4 * cell + q, ps[q]);
        }
    }
}
template <typename T, int G>
__device__ __forceinline__ void group_moments(const T (&ox)[G], const T (&oy)[G], const T (&oz)[G], T (&ps)[4]) {
    ps[0] = ps[1] = ps[2] = ps[3] = T(0);
#pragma unroll
    for (int e = 0; e < G; ++e) {
        ps[0] += ox[e];
        ps[1] += oy[e];
        ps[2] += oz[e];
        ps[3] = fma(ox[e], ox[e], fma(oy[e], oy[e], fma(oz[e], oz[e], ps[3])));
    }
}

// One cell's record through the read-only path: 128-bit loads (16 lanes of a warp share a cell at ppc = 64, so a
// warp instruction touches a handful of sectors, resident in L1/L2).
template <typename T> struct RecRegs;
template <> struct RecRegs<float> { float4 q[3]; };
template <> struct RecRegs<double> { ulonglong2 q[6]; };
__device__ __forceinline__ void load_rec(const CellRec<float>* __restrict__ W, int64_t cell, RecRegs<float>& r) {
    const float4* src = reinterpret_cast<const float4*>(W + cell);
#pragma unroll
    for (int u = 0; u < 3; ++u) r.q[u] = __ldg(src + u);
}
__device__ __forceinline__ void load_rec(const CellRec<double>* __restrict__ W, int64_t cell, RecRegs<double>& r) {
    const ulonglong2* src = reinterpret_cast<const ulonglong2*>(W + cell);
#pragma unroll
    for (int u = 0; u < 6; ++u) r.q[u] = __ldg(src + u);
}
// Velocities of one 128-bit group with per-cell constants and drift, from the cell's record.  The drift enters
// through the last multiply-add of the chain (velocity_f32 / velocity_f64, DRIFT), the same in every path.
__device__ __forceinline__ void rec_velocities(const uint32_t (&w0)[4], const uint32_t (&w1)[4], const uint32_t (&w2)[4],
                                               const RecRegs<float>& r, float (&ox)[4], float (&oy)[4], float (&oz)[4]) {
    const float4 q0 = r.q[0], q1 = r.q[1], q2 = r.q[2];                  // the order of CellRec<float>
    const Coef2 C{splat2(q0.x), splat2(q0.y), splat2(q0.z), splat2(q0.w), splat2(q1.x), splat2(q1.y), splat2(q1.z),
                  splat2(q1.w), splat2(q2.x)};
    const f32x2 dx = splat2(q2.y), dy = splat2(q2.z), dz = splat2(q2.w);
#pragma unroll
    for (int e = 0; e < 4; e += 2) {
        const uint32_t p0[2] = {w0[e], w0[e + 1]}, p1[2] = {w1[e], w1[e + 1]}, p2[2] = {w2[e], w2[e + 1]}, p3[2] = {0u, 0u};
        float a[2], b[2], c[2];
        velocity_pair_f32<false, false, true>(p0, p1, p2, p3, C, a, b, c, dx, dy, dz);
        ox[e] = a[0]; ox[e + 1] = a[1];
        oy[e] = b[0]; oy[e + 1] = b[1];
        oz[e] = c[0]; oz[e + 1] = c[1];
    }
}
__device__ __forceinline__ double as_f64(unsigned long long b) { return __longlong_as_double((long long)b); }
__device__ __forceinline__ void rec_velocities(const uint32_t (&w0)[2], const uint32_t (&w1)[2], const uint32_t (&w2)[2],
                                               const RecRegs<double>& r, double (&ox)[2], double (&oy)[2], double (&oz)[2]) {
    const ulonglong2 (&q)[6] = r.q;
    Coef<double> C;                                                    // the order of CellRec<double>
    C.s = as_f64(q[0].x); C.a = as_f64(q[0].y); C.ck = as_f64(q[1].x); C.bk4 = as_f64(q[1].y);
    C.k2 = as_f64(q[2].x); C.b2 = as_f64(q[2].y); C.theta = as_f64(q[3].x); C.theta2 = as_f64(q[3].y);
#pragma unroll
    for (int e = 0; e < 2; ++e)
        velocity_f64<false, true>(w0[e], w1[e], w2[e], 0u, C, ox[e], oy[e], oz[e], as_f64(q[4].x), as_f64(q[4].y), as_f64(q[5].x));
}
// one particle (a group that straddles two cells): the scalar chain, bit-identical to the packed one
__device__ __forceinline__ void rec_velocity(uint32_t w0, uint32_t w1, uint32_t w2, const CellRec<float>& R, float& x, float& y, float& z) {
    velocity_f32<false, false, true>(w0, w1, w2, 0u, coef_of(R), x, y, z, R.dx, R.dy, R.dz);
}
__device__ __forceinline__ void rec_velocity(uint32_t w0, uint32_t w1, uint32_t w2, const CellRec<double>& R, double& x, double& y, double& z) {
    velocity_f64<false, true>(w0, w1, w2, 0u, R.C, x, y, z, R.dx, R.dy, R.dz);
}

// Particle g = cell * ppc + j (cell-major).  A 128-bit group of G particles that lies inside one cell -- every
// group when ppc is a multiple of G -- reads that cell's record once and runs the same packed / shared-head
// code as the uniform sampler; a group that straddles a cell boundary takes the per-particle path.
// Whole tiles (in range, inside one 2^32 block of counters) run in one straight line, as in the uniform sampler;
// a group finds its cell with one 32-bit multiply-high from its offset inside the tile (magic32 = ceil(2^32 / ppc),
// exact for those offsets; 0: ppc >= tile, one compare instead -- cells_ahead()) and the tile's first cell, which the block carries from tile to
// tile by addition.
// STORE: write the velocity planes.  MOM: also reduce (sum vx, sum vy, sum vz, sum |v|^2) per cell into
// mom[ncell][4] -- the loader fused with its first consumer: with STORE = false
// no velocity ever reaches HBM.
template <typename T, bool VEC, bool STORE, bool MOM>
__global__ void __launch_bounds__(kThreads, 2)
sample_cells_kernel(int64_t n, uint32_t ppc, uint64_t magic, uint32_t magic32, uint64_t offset,
                    const __grid_constant__ PhiloxKeys K, const CellRec<T>* __restrict__ W, T* __restrict__ vx,
                    T* __restrict__ vy, T* __restrict__ vz, T* __restrict__ mom, int mom_mode, int mom_lanes) {
    constexpr int G = 16 / sizeof(T);
    constexpr int64_t kTile = (int64_t)kThreads * G * kGroups;
    const bool whole_groups = ppc % (uint32_t)G == 0u;                 // every 128-bit group inside one cell
    math_tables_init<T>();
    const int64_t stride = (int64_t)gridDim.x * kTile;
    int64_t base = (int64_t)blockIdx.x * kTile;
    // first cell of the tile and the tile's offset inside it, advanced by (stride / ppc, stride % ppc) per tile
    int64_t cell_first = base < n ? cell_of(base, ppc, magic) : 0;
    uint32_t rem_first = (uint32_t)(base - cell_first * (int64_t)ppc);
    const int64_t dcell = cell_of(stride, ppc, magic);
    const uint32_t drem = (uint32_t)(stride - dcell * (int64_t)ppc);
    for (; base < n; base += stride) {
        const uint64_t g_tile = offset + (uint64_t)base;
        if (VEC && whole_groups && base + kTile <= n && tile_in_one_block(g_tile, kTile)) {
            // the straight-line tile of the uniform sampler (one Philox head; float: round-1 products by constant additions)
            const PhiloxHead H = philox_head((uint32_t)(g_tile >> 32), K);
            const uint32_t lo_first = (uint32_t)g_tile + threadIdx.x * (uint32_t)G;
            const uint64_t q_first = (uint64_t)kPhiloxM0 * (uint64_t)lo_first;
            T ox[kGroups][G], oy[kGroups][G], oz[kGroups][G];
            int64_t cell[kGroups];
            RecRegs<T> rec[kGroups];
#pragma unroll
            for (int j = 0; j < kGroups; ++j) {
                cell[j] = cell_first + (int64_t)cells_ahead(rem_first + (uint32_t)(j * (kThreads * G)) + threadIdx.x * (uint32_t)G, ppc, magic32);
                load_rec(W, cell[j], rec[j]);
            }
#pragma unroll
            for (int j = 0; j < kGroups; ++j) {
                uint32_t w0[G], w1[G], w2[G], w3[G];
                tile_group_words<T, G, kThreads>(lo_first, q_first, j, H, K, w0, w1, w2, w3);
                rec_velocities(w0, w1, w2, rec[j], ox[j], oy[j], oz[j]);
                if (MOM) {
                    T ps[4];
                    group_moments<T, G>(ox[j], oy[j], oz[j], ps);
                    moments_out(ps, cell[j], mom_mode, mom_lanes, mom, 0xffffffffu);
                }
            }
            if (STORE) {
#pragma unroll
                for (int j = 0; j < kGroups; ++j) {
                    const int64_t i = base + (int64_t)j * (kThreads * G) + (int64_t)threadIdx.x * G;
                    store_group(vx + i, ox[j]);
                    store_group(vy + i, oy[j]);
                    store_group(vz + i, oz[j]);
                }
            }
        } else {
#pragma unroll 1
            for (int j = 0; j < kGroups; ++j) {
                const int64_t i = base + (int64_t)j * (kThreads * G) + (int64_t)threadIdx.x * G;
                const bool in_range = i < n;
                const int64_t cell0 = in_range ? cell_of(i, ppc, magic) : 0;
                const uint32_t rem = (uint32_t)(i - cell0 * (int64_t)ppc);
                const bool one_cell = in_range && rem + (uint32_t)G <= ppc && i + G <= n;
                const unsigned one_cell_mask = __ballot_sync(0xffffffffu, one_cell);
                T ox[G], oy[G], oz[G];
                if (one_cell) {
                    RecRegs<T> rec;
                    load_rec(W, cell0, rec);
                    uint32_t w0[G], w1[G], w2[G], w3[G];
                    group_words<G>(offset + (uint64_t)i, K, w0, w1, w2, w3);
                    rec_velocities(w0, w1, w2, rec, ox, oy, oz);
                    if (MOM) {
                        T ps[4];
                        group_moments<T, G>(ox, oy, oz, ps);
                        moments_out(ps, cell0, mom_mode, mom_lanes, mom, one_cell_mask);
                    }
                } else if (in_range) {
#pragma unroll
                    for (int e = 0; e < G; ++e) {
                        int64_t cell = cell0 + (int64_t)((rem + (uint32_t)e) / ppc);
                        if (i + e >= n) cell = cell0;                 // lanes past the end: stay in bounds
                        const CellRec<T> R = W[cell];
                        uint32_t w0, w1, w2;
                        particle_words(offset + (uint64_t)(i + e), K, w0, w1, w2);
                        rec_velocity(w0, w1, w2, R, ox[e], oy[e], oz[e]);
                        if (MOM && i + e < n) {                       // only reached in kMomAtomic mode
                            T ps[4] = {ox[e], oy[e], oz[e], fma(ox[e], ox[e], fma(oy[e], oy[e], oz[e] * oz[e]))};
                            moments_out(ps, cell, kMomAtomic, 1, mom, 0u);
                        }
                    }
                }
                if (STORE && in_range) store_planes<T, VEC, G>(i, n, vx, vy, vz, ox, oy, oz);
            }
        }
        cell_first += dcell;
        rem_first += drem;
        if (rem_first >= ppc) {
            rem_first -= ppc;
            ++cell_first;
        }
    }
}

// ---------------------------------------------------------------- kappagen_speed_histogram (paper test 2)
// S1-S4 only: |v|/theta of each particle, binned with width dv; no velocity is written.  Counts go to
// per-warp-slot replicas of the histogram in shared memory (most particles fall into the few bins around
// |v| = theta, so one copy per block would serialise on a handful of addresses) and are flushed to the
// caller's 64-bit counters once per block.  speed_over_theta: float: half of the packed chain's 2V with
// theta = 1 folded in; double: speed_f64 with theta = 1.
constexpr int kHistMaxBins = 4096;

template <bool U64>
__device__ __forceinline__ void group_speeds(uint64_t g0, const PhiloxKeys& K, const Coef<float>& C, float (&s)[4]) {
    uint32_t w0[4], w1[4], w2[4], w3[4];
    group_words<4>(g0, K, w0, w1, w2, w3);
#pragma unroll
    for (int e = 0; e < 4; e += 2) up2(speed2_f32x2<U64>(w0[e], w0[e + 1], w3[e], w3[e + 1], C), s[e], s[e + 1]);   // 2V
}
template <bool U64>
__device__ __forceinline__ void group_speeds(uint64_t g0, const PhiloxKeys& K, const Coef<double>& C, double (&s)[2]) {
    uint32_t w0[2], w1[2], w2[2], w3[2];
    group_words<2>(g0, K, w0, w1, w2, w3);
#pragma unroll
    for (int e = 0; e < 2; ++e) s[e] = speed_f64<U64>(w0[e], w3[e], C, C.theta);
}
// Speeds of one group of a whole tile (words through tile_group_words, as in sample_kernel).
template <bool U64, typename T, int G>
__device__ __forceinline__ void group_speeds_tile(uint32_t lo_first, uint64_t q_first, int j, const PhiloxHead& H,
                                                  const PhiloxKeys& K, const Coef<T>& C, T (&s)[G]) {
    uint32_t w0[G], w1[G], w2[G], w3[G];
    tile_group_words<T, G>(lo_first, q_first, j, H, K, w0, w1, w2, w3);
    if constexpr (sizeof(T) == 4) {
#pragma unroll
        for (int e = 0; e < G; e += 2) up2(speed2_f32x2<U64>(w0[e], w0[e + 1], w3[e], w3[e + 1], C), s[e], s[e + 1]);
    } else {
#pragma unroll
        for (int e = 0; e < G; ++e) s[e] = speed_f64<U64>(w0[e], w3[e], C, C.theta);
    }
}
__device__ __forceinline__ int bin_of(float s, float inv) { return __float2int_rz(s * inv); }     // saturating
__device__ __forceinline__ int bin_of(double s, double inv) { return __double2int_rz(s * inv); }

// inv = 1/dv (double) or 1/(2 dv) (float, whose chain returns 2V), rounded to T.
template <typename T, bool U64>
__global__ void __launch_bounds__(TileTraits<T>::threads, TileTraits<T>::minb)
speed_histogram_kernel(int64_t n, uint64_t offset, const __grid_constant__ PhiloxKeys K, const __grid_constant__ Coef<T> C,
                       T inv, int nbins, int replicas, unsigned long long* __restrict__ hist) {
    extern __shared__ uint32_t sh_hist[];
    constexpr int G = 16 / sizeof(T);
    constexpr int NG = TileTraits<T>::groups;            // the sample kernel's tile shape: same chains, same trade-off
    constexpr int kT = TileTraits<T>::threads;
    constexpr int64_t kTile = (int64_t)kT * G * NG;
    for (int b = threadIdx.x; b < nbins * replicas; b += kT) sh_hist[b] = 0u;
    math_tables_init<T>();
    __syncthreads();
    uint32_t* mine = sh_hist + ((threadIdx.x >> 5) % (unsigned)replicas) * nbins;
    for (int64_t base = (int64_t)blockIdx.x * kTile; base < n; base += (int64_t)gridDim.x * kTile) {
        const uint64_t g_tile = offset + (uint64_t)base;
        if (base + kTile <= n && tile_in_one_block(g_tile, kTile)) {
            // whole tile in range and inside one 2^32 block of counters: straight line, one Philox head
            const PhiloxHead H = philox_head((uint32_t)(g_tile >> 32), K);
            const uint32_t lo_first = (uint32_t)g_tile + threadIdx.x * (uint32_t)G;
            const uint64_t q_first = (uint64_t)kPhiloxM0 * (uint64_t)lo_first;
            T s[NG][G];
#pragma unroll
            for (int j = 0; j < NG; ++j)
                group_speeds_tile<U64>(lo_first, q_first, j, H, K, C, s[j]);
#pragma unroll
            for (int j = 0; j < NG; ++j) {
#pragma unroll
                for (int e = 0; e < G; ++e) atomicAdd(mine + min(bin_of(s[j][e], inv), nbins - 1), 1u);
            }
            continue;
        }
#pragma unroll
        for (int j = 0; j < NG; ++j) {
            const int64_t i = base + (int64_t)j * (kT * G) + (int64_t)threadIdx.x * G;
            if (i < n) {
                T s[G];
                group_speeds<U64>(offset + (uint64_t)i, K, C, s);
#pragma unroll
                for (int e = 0; e < G; ++e) {
                    if (i + e < n) atomicAdd(mine + min(bin_of(s[e], inv), nbins - 1), 1u);
                }
            }
        }
    }
    __syncthreads();
    for (int b = threadIdx.x; b < nbins; b += kT) {
        unsigned long long c = 0ull;
        for (int r = 0; r < replicas; ++r) c += sh_hist[r * nbins + b];
        if (c != 0ull) atomicAdd(hist + b, c);
    }
}

// ---------------------------------------------------------------- test hooks
__global__ void __launch_bounds__(kThreads)
words_kernel(int64_t n, uint64_t offset, const __grid_constant__ PhiloxKeys K, uint32_t* __restrict__ o0,
             uint32_t* __restrict__ o1, uint32_t* __restrict__ o2, uint32_t* __restrict__ o3) {
    // four consecutive particles per thread through group_words, exactly as the fp32 sampler draws them
    for (int64_t i = ((int64_t)blockIdx.x * kThreads + threadIdx.x) * 4; i < n; i += (int64_t)gridDim.x * kThreads * 4) {
        uint32_t w0[4], w1[4], w2[4], w3[4];
        group_words<4>(offset + (uint64_t)i, K, w0, w1, w2, w3);
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            if (i + e < n) {
                o0[i + e] = w0[e];
                o1[i + e] = w1[e];
                o2[i + e] = w2[e];
                if (o3 != nullptr) o3[i + e] = w3[e];
            }
        }
    }
}

template <typename T, bool FOLD, bool U64>
__global__ void __launch_bounds__(kThreads)
velocity_of_words_kernel(int64_t n, const uint32_t* __restrict__ w0, const uint32_t* __restrict__ w1,
                         const uint32_t* __restrict__ w2, const uint32_t* __restrict__ w3, const __grid_constant__ Coef<T> C,
                         T* __restrict__ vx, T* __restrict__ vy, T* __restrict__ vz) {
    math_tables_init<T>();
    for (int64_t i = (int64_t)blockIdx.x * kThreads + threadIdx.x; i < n; i += (int64_t)gridDim.x * kThreads) {
        T x, y, z;
        velocity<FOLD, U64>(w0[i], w1[i], w2[i], U64 ? w3[i] : 0u, C, x, y, z);
        vx[i] = x;
        vy[i] = y;
        vz[i] = z;
    }
}

// The words exactly as sample_kernel<T> draws them: the same tile walk, the same whole-tile test, on the
// whole-tile path tile_group_words (shared head, constant-addition round 1 for float), elsewhere group_words
// (per-group head, per-particle counters where the low word wraps).  kappagen_words_tile.
template <typename T>
__global__ void __launch_bounds__(TileTraits<T>::threads)
words_tile_kernel(int64_t n, uint64_t offset, const __grid_constant__ PhiloxKeys K, uint32_t* __restrict__ o0,
                  uint32_t* __restrict__ o1, uint32_t* __restrict__ o2, uint32_t* __restrict__ o3) {
    constexpr int G = 16 / sizeof(T);
    constexpr int NG = TileTraits<T>::groups;
    constexpr int kT = TileTraits<T>::threads;
    constexpr int64_t kTile = (int64_t)kT * G * NG;
    for (int64_t base = (int64_t)blockIdx.x * kTile; base < n; base += (int64_t)gridDim.x * kTile) {
        const uint64_t g_tile = offset + (uint64_t)base;
        const bool whole = base + kTile <= n && tile_in_one_block(g_tile, kTile);
        const PhiloxHead H = philox_head((uint32_t)(g_tile >> 32), K);
        const uint32_t lo_first = (uint32_t)g_tile + threadIdx.x * (uint32_t)G;
        const uint64_t q_first = (uint64_t)kPhiloxM0 * (uint64_t)lo_first;
#pragma unroll
        for (int j = 0; j < NG; ++j) {
            const int64_t i = base + (int64_t)j * (kT * G) + (int64_t)threadIdx.x * G;
            uint32_t w0[G], w1[G], w2[G], w3[G];
            if (whole) tile_group_words<T, G>(lo_first, q_first, j, H, K, w0, w1, w2, w3);
            else if (i < n) group_words<G>(offset + (uint64_t)i, K, w0, w1, w2, w3);
#pragma unroll
            for (int e = 0; e < G; ++e) {
                if (i + e < n) {
                    o0[i + e] = w0[e];
                    o1[i + e] = w1[e];
                    o2[i + e] = w2[e];
                    o3[i + e] = w3[e];
                }
            }
        }
    }
}

// kappagen_philox_planes: S1 and S6 of sample_kernel<float> with S2-S5 stripped -- the same tile walk, the same
// whole-tile test and word functions, the three words stored as three uint32 planes with 128-bit streaming stores
// (12 bytes per particle, like the float sampler).  The measured ceiling of the float sampler.
template <bool VEC>
__global__ void __launch_bounds__(TileTraits<float>::threads, TileTraits<float>::minb)
philox_planes_kernel(int64_t n, uint64_t offset, const __grid_constant__ PhiloxKeys K, uint32_t* __restrict__ o0,
                     uint32_t* __restrict__ o1, uint32_t* __restrict__ o2) {
    constexpr int G = 4;
    constexpr int NG = TileTraits<float>::groups;
    constexpr int kT = TileTraits<float>::threads;
    constexpr int64_t kTile = (int64_t)kT * G * NG;
    for (int64_t base = (int64_t)blockIdx.x * kTile; base < n; base += (int64_t)gridDim.x * kTile) {
        const uint64_t g_tile = offset + (uint64_t)base;
        if (VEC && base + kTile <= n && tile_in_one_block(g_tile, kTile)) {
            const PhiloxHead H = philox_head((uint32_t)(g_tile >> 32), K);
            const uint32_t lo_first = (uint32_t)g_tile + threadIdx.x * (uint32_t)G;
            const uint64_t q_first = (uint64_t)kPhiloxM0 * (uint64_t)lo_first;
            uint32_t w0[NG][G], w1[NG][G], w2[NG][G];
#pragma unroll
            for (int j = 0; j < NG; ++j) {
                uint32_t w3[G];
                tile_group_words<float, G>(lo_first, q_first, j, H, K, w0[j], w1[j], w2[j], w3);
            }
#pragma unroll
            for (int j = 0; j < NG; ++j) {
                const int64_t i = base + (int64_t)j * (kT * G) + (int64_t)threadIdx.x * G;
                __stcs(reinterpret_cast<uint4*>(o0 + i), make_uint4(w0[j][0], w0[j][1], w0[j][2], w0[j][3]));
                __stcs(reinterpret_cast<uint4*>(o1 + i), make_uint4(w1[j][0], w1[j][1], w1[j][2], w1[j][3]));
                __stcs(reinterpret_cast<uint4*>(o2 + i), make_uint4(w2[j][0], w2[j][1], w2[j][2], w2[j][3]));
            }
            continue;
        }
#pragma unroll 1
        for (int j = 0; j < NG; ++j) {
            const int64_t i = base + (int64_t)j * (kT * G) + (int64_t)threadIdx.x * G;
            if (i < n) {
                uint32_t w0[G], w1[G], w2[G], w3[G];
                group_words<G>(offset + (uint64_t)i, K, w0, w1, w2, w3);
#pragma unroll
                for (int e = 0; e < G; ++e) {
                    if (i + e < n) {
                        o0[i + e] = w0[e];
                        o1[i + e] = w1[e];
                        o2[i + e] = w2[e];
                    }
                }
            }
        }
    }
}

// ---------------------------------------------------------------- kappagen_math_planes (measurement hook)
// The other side of kappagen_philox_planes: steps S2-S6 of the sampler's whole-tile body -- the same words_to_velocities,
// the same tile shape, launch bounds and 128-bit streaming stores -- with S1 (Philox) replaced by one 32-bit
// multiply-add per word, w_k = lo32(g) * kMathPlanesMul<k> + kMathPlanesAdd<k>: what the math and the stores cost
// when the random words are (almost) free.  Not a generator: the words are a fixed affine map of the index.
constexpr uint32_t kMathPlanesMul0 = 0x9E3779B1u, kMathPlanesMul1 = 0x85EBCA77u, kMathPlanesMul2 = 0xC2B2AE3Du;
constexpr uint32_t kMathPlanesAdd0 = 0x7F4A7C15u, kMathPlanesAdd1 = 0x165667B1u, kMathPlanesAdd2 = 0x27D4EB2Fu;

template <int G>
__device__ __forceinline__ void affine_words(uint32_t lo, uint32_t (&w0)[G], uint32_t (&w1)[G], uint32_t (&w2)[G], uint32_t (&w3)[G]) {
#pragma unroll
    for (int e = 0; e < G; ++e) {
        const uint32_t g = lo + (uint32_t)e;
        w0[e] = g * kMathPlanesMul0 + kMathPlanesAdd0;
        w1[e] = g * kMathPlanesMul1 + kMathPlanesAdd1;
        w2[e] = g * kMathPlanesMul2 + kMathPlanesAdd2;
        w3[e] = 0u;
    }
}

template <typename T, bool FOLD>
__global__ void __launch_bounds__(TileTraits<T>::threads, TileTraits<T>::minb)
math_planes_kernel(int64_t n, uint64_t offset, const __grid_constant__ Coef<T> C, T* __restrict__ vx, T* __restrict__ vy,
                   T* __restrict__ vz) {
    constexpr int G = 16 / sizeof(T);
    constexpr int NG = TileTraits<T>::groups;
    constexpr int kT = TileTraits<T>::threads;
    constexpr int64_t kTile = (int64_t)kT * G * NG;
    math_tables_init<T>();
    for (int64_t base = (int64_t)blockIdx.x * kTile; base < n; base += (int64_t)gridDim.x * kTile) {
        const uint32_t lo_first = (uint32_t)(offset + (uint64_t)base) + threadIdx.x * (uint32_t)G;
        if (base + kTile <= n) {
            T ox[NG][G], oy[NG][G], oz[NG][G];
#pragma unroll
            for (int j = 0; j < NG; ++j) {
                uint32_t w0[G], w1[G], w2[G], w3[G];
                affine_words<G>(lo_first + (uint32_t)(j * (kT * G)), w0, w1, w2, w3);
                words_to_velocities<FOLD, false>(w0, w1, w2, w3, C, ox[j], oy[j], oz[j]);
            }
#pragma unroll
            for (int j = 0; j < NG; ++j) {
                const int64_t i = base + (int64_t)j * (kT * G) + (int64_t)threadIdx.x * G;
                store_group(vx + i, ox[j]);
                store_group(vy + i, oy[j]);
                store_group(vz + i, oz[j]);
            }
            continue;
        }
#pragma unroll 1
        for (int j = 0; j < NG; ++j) {
            const int64_t i = base + (int64_t)j * (kT * G) + (int64_t)threadIdx.x * G;
            if (i < n) {
                uint32_t w0[G], w1[G], w2[G], w3[G];
                T ox[G], oy[G], oz[G];
                affine_words<G>(lo_first + (uint32_t)(j * (kT * G)), w0, w1, w2, w3);
                words_to_velocities<FOLD, false>(w0, w1, w2, w3, C, ox, oy, oz);
                store_planes<T, false, G>(i, n, vx, vy, vz, ox, oy, oz);
            }
        }
    }
}

// S2-S6 on caller-chosen words through the code sample_kernel<T> ships: every thread takes the NG groups of
// a tile in one straight line through words_to_velocities (float: the packed pairs of math_f32x2.cuh; double:
// the 2 NG interleaved chains), exactly as the whole-tile path instantiates them -- only the source of the
// words differs (memory instead of Philox).  Past the end the last word is repeated and nothing is stored.
// kappagen_velocity_of_words_tile.
template <typename T, bool FOLD, bool U64>
__global__ void __launch_bounds__(TileTraits<T>::threads, TileTraits<T>::minb)
velocity_of_words_tile_kernel(int64_t n, const uint32_t* __restrict__ p0, const uint32_t* __restrict__ p1,
                              const uint32_t* __restrict__ p2, const uint32_t* __restrict__ p3, const __grid_constant__ Coef<T> C,
                              T* __restrict__ vx, T* __restrict__ vy, T* __restrict__ vz) {
    constexpr int G = 16 / sizeof(T);
    constexpr int NG = TileTraits<T>::groups;
    constexpr int kT = TileTraits<T>::threads;
    constexpr int64_t kTile = (int64_t)kT * G * NG;
    math_tables_init<T>();
    for (int64_t base = (int64_t)blockIdx.x * kTile; base < n; base += (int64_t)gridDim.x * kTile) {
        T ox[NG][G], oy[NG][G], oz[NG][G];
#pragma unroll
        for (int j = 0; j < NG; ++j) {
            const int64_t i = base + (int64_t)j * (kT * G) + (int64_t)threadIdx.x * G;
            uint32_t w0[G], w1[G], w2[G], w3[G];
#pragma unroll
            for (int e = 0; e < G; ++e) {
                const int64_t k = i + e < n ? i + e : n - 1;
                w0[e] = p0[k];
                w1[e] = p1[k];
                w2[e] = p2[k];
                w3[e] = U64 ? p3[k] : 0u;
            }
            words_to_velocities<FOLD, U64>(w0, w1, w2, w3, C, ox[j], oy[j], oz[j]);
        }
#pragma unroll
        for (int j = 0; j < NG; ++j) {
            const int64_t i = base + (int64_t)j * (kT * G) + (int64_t)threadIdx.x * G;
#pragma unroll
            for (int e = 0; e < G; ++e) {
                if (i + e < n) {
                    vx[i + e] = ox[j][e];
                    vy[i + e] = oy[j][e];
                    vz[i + e] = oz[j][e];
                }
            }
        }
    }
}

}  // namespace kappagen
