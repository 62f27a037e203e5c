// baseline_mt.cuh -- GPU BASELINE, not the paper's method: the "standard method" the paper compares
// itself with.  Kappa = 3-D multivariate t: three normal variates
// divided by the square root of one gamma variate, the gamma by Marsaglia & Tsang's rejection method
// (ref. 11), shape k = kappa - 1/2:
//     v = theta sqrt(kappa / (2 g)) (n1, n2, n3),   g ~ Gamma(kappa - 1/2, 1),  n_j ~ N(0,1)
// (scaling derived in DESIGN.md: Eq. (1) is a t-distribution with 2 kappa - 1 degrees of freedom and
// scale^2 = kappa theta^2 / (2 kappa - 1); check: <v^2> = (3 kappa theta^2 / 2) E[1/g] = Eq. (5)).
// Marsaglia-Tsang: d = k - 1/3, c' = 1/sqrt(9d); repeat { z ~ N(0,1); t = (1 + c'z)^3; if t <= 0
// retry; u ~ U(0,1); accept if u < 1 - 0.0331 z^4 or ln u < z^2/2 + d (1 - t + ln t) }; g = d t.
// Per trial: one normal and one uniform.  Normals by Box-Muller.
//
// The data-dependent do/while is the point: on SIMT hardware a warp waits for its slowest lane
// (PAPER.md:236), so the loop body is issued mu_1(1-p1, 32) times per warp (Eq. 30) although a lane
// needs only 1/p1 trips.  trip_counters measures exactly that.
// Random numbers: Philox block (lo g, hi g, 0, 2) gives the three direction normals; block
// (lo g, hi g, j, 1) gives trial j's normal and uniform.  Reproducible, but only the DISTRIBUTION is
// specified: validated statistically (exact Kappa CDF, Eq. 3), never bit-compared.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>
#include "philox.cuh"

namespace kappagen {

template <typename T>
struct MtParams {
    T d;       // k - 1/3
    T cp;      // 1/sqrt(9 d)
    T scale;   // theta sqrt(kappa/2)
};

__device__ __forceinline__ float bm_uniform(uint32_t w, float) { return fmaf((float)w, 0x1p-32f, 0x1p-33f); }
__device__ __forceinline__ double bm_uniform(uint32_t w, double) { return ((double)w + 0.5) * 0x1p-32; }
__device__ __forceinline__ void bm_sincos2pi(float u, float& s, float& c) { sincospif(2.0f * u, &s, &c); }
__device__ __forceinline__ void bm_sincos2pi(double u, double& s, double& c) { sincospi(2.0 * u, &s, &c); }
__device__ __forceinline__ float bm_log(float x) { return logf(x); }
__device__ __forceinline__ double bm_log(double x) { return log(x); }
__device__ __forceinline__ float bm_sqrt(float x) { return sqrtf(x); }
__device__ __forceinline__ double bm_sqrt(double x) { return sqrt(x); }

// Box-Muller: two words -> two independent N(0,1).
template <typename T>
__device__ __forceinline__ void box_muller(uint32_t wa, uint32_t wb, T& n1, T& n2) {
    const T R = bm_sqrt(T(-2) * bm_log(bm_uniform(wa, T())));
    T s, c;
    bm_sincos2pi(bm_uniform(wb, T()), s, c);
    n1 = R * c;
    n2 = R * s;
}

template <typename T>
__global__ void __launch_bounds__(256)
baseline_mt_kernel(int64_t n, uint64_t offset, const __grid_constant__ PhiloxKeys K,
                   const __grid_constant__ MtParams<T> P, T* __restrict__ vx, T* __restrict__ vy,
                   T* __restrict__ vz, unsigned long long* __restrict__ trip_counters) {
    unsigned long long lane_trips = 0, warp_trips = 0;
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    // warp-uniform trip count of the outer loop so that the warp reductions below see whole warps
    for (int64_t base = (int64_t)blockIdx.x * blockDim.x; base < n; base += stride) {
        const int64_t i = base + threadIdx.x;
        const bool live = i < n;
        const uint64_t g = offset + (uint64_t)i;
        const uint32_t glo = (uint32_t)g, ghi = (uint32_t)(g >> 32);
        uint32_t a0, a1, a2, a3;
        philox4x32_10(glo, ghi, 0u, 2u, K, a0, a1, a2, a3);
        T n1, n2, n3, unused;
        box_muller<T>(a0, a1, n1, n2);
        box_muller<T>(a2, a3, n3, unused);
        // Marsaglia-Tsang rejection loop: the divergent part
        T t = T(1);
        uint32_t trips = 0;
        bool done = !live;
        while (!done) {
            uint32_t b0, b1, b2, b3;
            philox4x32_10(glo, ghi, trips, 1u, K, b0, b1, b2, b3);
            ++trips;
            T z, z2;
            box_muller<T>(b0, b1, z, z2);
            const T q = T(1) + P.cp * z;
            if (q > T(0)) {
                t = q * q * q;
                const T u = bm_uniform(b2, T());
                const T zz = z * z;
                if (u < T(1) - T(0.0331) * zz * zz) {
                    done = true;
                } else if (bm_log(u) < T(0.5) * zz + P.d * (T(1) - t + bm_log(t))) {
                    done = true;
                }
            }
        }
        if (live) {
            const T f = P.scale / bm_sqrt(P.d * t);      // theta sqrt(kappa / (2 g)), g = d t
            vx[i] = f * n1;
            vy[i] = f * n2;
            vz[i] = f * n3;
        }
        if (trip_counters != nullptr) {
            lane_trips += trips;
            warp_trips += 32ull * __reduce_max_sync(0xffffffffu, trips);
        }
    }
    if (trip_counters != nullptr) {
        for (int o = 16; o > 0; o >>= 1) lane_trips += __shfl_xor_sync(0xffffffffu, lane_trips, o);
        if ((threadIdx.x & 31) == 0) {
            atomicAdd(&trip_counters[0], lane_trips);
            atomicAdd(&trip_counters[1], warp_trips);
        }
    }
}

}  // namespace kappagen
