// kappagen_api.cu -- the C ABI of include/kappagen.h: argument checks and kernel launches.
// Every step of the hot path runs in the kernels of kernels.cuh; nothing here computes a velocity,
// and there is no CPU fallback: without a CUDA device the calls return KAPPAGEN_ECUDA.
#include <cmath>
#include <cstdint>
#include <cstdio>
#include <atomic>
#include <mutex>

#include <cuda_runtime.h>

#include "../../include/kappagen.h"
#include "baseline_mt.cuh"
#include "host_params.hpp"
#include "kernels.cuh"
#include "load_cells.cuh"
#include "pipe_probe.cuh"

namespace kappagen {

#define KG_CUDA(call)                                                                    \
    do {                                                                                 \
        cudaError_t e_ = (call);                                                         \
        if (e_ != cudaSuccess) {                                                         \
            set_error("%s: %s failed: %s", __func__, #call, cudaGetErrorString(e_));     \
            return KAPPAGEN_ECUDA;                                                       \
        }                                                                                \
    } while (0)

static inline bool aligned_to(const void* p, size_t a) { return (reinterpret_cast<uintptr_t>(p) % a) == 0; }
static inline size_t elem_size(int dtype) { return dtype == KAPPAGEN_F32 ? 4 : 8; }

// Grid for a grid-stride kernel: enough blocks to fill every SM at the kernel's occupancy, never more
// than there are tiles.  The (SM count, blocks per SM) pair is queried once per kernel instantiation, device and
// launch shape (a function-local cache: the kernel is a template argument, so there is one cache per kernel instantiation), not on every launch --
// small calls are launch-bound.
template <auto Kernel>
static int grid_for(int64_t tiles, int* grid_out, int threads = kThreads, size_t dyn_smem = 0) {
    constexpr int kMaxDev = 64;
    struct Entry { int sms, per_sm, threads; size_t smem; };
    static thread_local Entry cache[kMaxDev] = {};
    int dev = 0;
    KG_CUDA(cudaGetDevice(&dev));
    Entry local = {};
    Entry& e = (dev >= 0 && dev < kMaxDev) ? cache[dev] : local;
    if (e.sms == 0 || e.threads != threads || e.smem != dyn_smem) {
        int sms = 0, per_sm = 0;
        KG_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
        KG_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, Kernel, threads, dyn_smem));
        e = Entry{sms, per_sm < 1 ? 1 : per_sm, threads, dyn_smem};
    }
    const int64_t full = (int64_t)e.sms * e.per_sm;
    *grid_out = (int)(tiles < full ? tiles : full);
    return KAPPAGEN_OK;
}

static int check_planes(const char* fn, int64_t n, int dtype, const void* vx, const void* vy, const void* vz,
                        bool* vec) {
    if (dtype != KAPPAGEN_F32 && dtype != KAPPAGEN_F64) {
        set_error("%s: dtype %d is neither KAPPAGEN_F32 nor KAPPAGEN_F64", fn, dtype);
        return KAPPAGEN_EINVAL;
    }
    if (n < 0) {
        set_error("%s: negative particle count %lld", fn, (long long)n);
        return KAPPAGEN_EINVAL;
    }
    if (n == 0) return KAPPAGEN_OK;
    if (!vx || !vy || !vz) {
        set_error("%s: NULL output plane", fn);
        return KAPPAGEN_ENULL;
    }
    const size_t es = elem_size(dtype);
    if (!aligned_to(vx, es) || !aligned_to(vy, es) || !aligned_to(vz, es)) {
        set_error("%s: output plane not aligned to its element size (%zu)", fn, es);
        return KAPPAGEN_EALIGN;
    }
    *vec = aligned_to(vx, 16) && aligned_to(vy, 16) && aligned_to(vz, 16);
    return KAPPAGEN_OK;
}

template <typename T, bool VEC, bool FOLD, bool U64>
static int launch_sample_as(int64_t n, uint64_t offset, const PhiloxKeys& K, const Coef<T>& C, T* vx, T* vy, T* vz,
                            cudaStream_t st) {
    constexpr int threads = TileTraits<T>::threads;
    constexpr int64_t tile = (int64_t)threads * (16 / sizeof(T)) * TileTraits<T>::groups;
    int grid = 0, rc;
    if ((rc = grid_for<sample_kernel<T, VEC, FOLD, U64>>((n + tile - 1) / tile, &grid, threads)) != KAPPAGEN_OK) return rc;
    sample_kernel<T, VEC, FOLD, U64><<<grid, threads, 0, st>>>(n, offset, K, C, vx, vy, vz);
    KG_CUDA(cudaGetLastError());
    return KAPPAGEN_OK;
}

template <typename T, bool U64>
static int launch_sample_u(int64_t n, uint64_t offset, const PhiloxKeys& K, const Coef<T>& C, bool vec, bool fold, T* vx, T* vy,
                           T* vz, cudaStream_t st) {
    if (vec) return fold ? launch_sample_as<T, true, true, U64>(n, offset, K, C, vx, vy, vz, st)
                         : launch_sample_as<T, true, false, U64>(n, offset, K, C, vx, vy, vz, st);
    return fold ? launch_sample_as<T, false, true, U64>(n, offset, K, C, vx, vy, vz, st)
                : launch_sample_as<T, false, false, U64>(n, offset, K, C, vx, vy, vz, st);
}

static int launch_sample(int64_t n, uint64_t offset, const PhiloxKeys& K, double kappa, double theta, bool vec, bool u64,
                         float* vx, float* vy, float* vz, cudaStream_t st) {
    const bool fold = theta_folds(theta);
    const Coef<float> C = host_coef_f32(kappa, theta, fold);
    return u64 ? launch_sample_u<float, true>(n, offset, K, C, vec, fold, vx, vy, vz, st)
               : launch_sample_u<float, false>(n, offset, K, C, vec, fold, vx, vy, vz, st);
}

static int launch_sample(int64_t n, uint64_t offset, const PhiloxKeys& K, double kappa, double theta, bool vec, bool u64,
                         double* vx, double* vy, double* vz, cudaStream_t st) {
    const Coef<double> C = host_coef_f64(kappa, theta);           // FOLD is a float-only notion: always false here
    if (u64) return vec ? launch_sample_as<double, true, false, true>(n, offset, K, C, vx, vy, vz, st)
                        : launch_sample_as<double, false, false, true>(n, offset, K, C, vx, vy, vz, st);
    return vec ? launch_sample_as<double, true, false, false>(n, offset, K, C, vx, vy, vz, st)
               : launch_sample_as<double, false, false, false>(n, offset, K, C, vx, vy, vz, st);
}

static int sample_on_stream(const char* fn, int64_t n, double kappa, double theta, uint64_t seed, uint64_t offset,
                            int dtype, uint32_t flags, void* vx, void* vy, void* vz, cudaStream_t st) {
    bool vec = false;
    int rc = check_planes(fn, n, dtype, vx, vy, vz, &vec);
    if (rc != KAPPAGEN_OK) return rc;
    if (!domain_ok(kappa, theta)) {
        set_error("%s: need finite kappa > 3/2 and theta >= 0 (got kappa = %g, theta = %g)", fn, kappa, theta);
        return KAPPAGEN_EINVAL;
    }
    if (flags & ~(uint32_t)KAPPAGEN_U1_64) {
        set_error("%s: unknown flag bits 0x%x", fn, flags);
        return KAPPAGEN_EINVAL;
    }
    if (n == 0) return KAPPAGEN_OK;
    const PhiloxKeys K = philox_expand_keys(seed);
    const bool u64 = (flags & KAPPAGEN_U1_64) != 0;
    if (dtype == KAPPAGEN_F32) return launch_sample(n, offset, K, kappa, theta, vec, u64, (float*)vx, (float*)vy, (float*)vz, st);
    return launch_sample(n, offset, K, kappa, theta, vec, u64, (double*)vx, (double*)vy, (double*)vz, st);
}

template <typename T, bool VEC, bool STORE, bool MOM>
static int launch_cells_as(int64_t n, int32_t ppc, uint64_t magic, uint32_t magic32, uint64_t offset, const PhiloxKeys& K,
                           const CellRec<T>* W, T* vx, T* vy, T* vz, T* mom, int mode, int lanes, cudaStream_t st) {
    constexpr int64_t tile = (int64_t)kThreads * (16 / sizeof(T)) * kGroups;
    int grid = 0, rc;
    if ((rc = grid_for<sample_cells_kernel<T, VEC, STORE, MOM>>((n + tile - 1) / tile, &grid)) != KAPPAGEN_OK) return rc;
    sample_cells_kernel<T, VEC, STORE, MOM><<<grid, kThreads, 0, st>>>(n, (uint32_t)ppc, magic, magic32, offset, K, W, vx, vy, vz,
                                                                      mom, mode, lanes);
    KG_CUDA(cudaGetLastError());
    return KAPPAGEN_OK;
}

// The two constants that replace the division by ppc in the per-cell kernels (sample_cells_kernel, load_cells_kernel).
//  magic  : cell_of(): a shift count when ppc is a power of two; else floor(i/ppc) = mulhi64(i, floor(2^64/ppc) + 1), exact
//           for every i with i * ppc < 2^64 (i < n; the value is >= 2^32 > 64 for every ppc < 2^31); else ~0: the plain
//           64-bit division.
//  magic32: inside a tile, floor(o/ppc) = mulhi32(o, ceil(2^32/ppc)), exact while o * ppc < 2^32 (o < tile + ppc).
//           0 = no such constant: ppc == 1, or ppc so large ((tile + ppc) * ppc >= 2^32, i.e. ppc > 6.4e4 >= tile) that a
//           tile touches at most two cells and the kernels compare instead (cells_ahead()).
static void cells_magics(int64_t n, int32_t ppc, int64_t tile, uint64_t* magic, uint32_t* magic32) {
    const uint64_t up = (uint64_t)ppc;
    *magic = ~0ull;
    if ((up & (up - 1)) == 0) {
        *magic = 0;
        while ((1ull << *magic) < up) ++*magic;
    } else if ((uint64_t)n <= (~0ull) / up) {
        *magic = (~0ull) / up + 1;
    }
    *magic32 = 0;
    if (up >= 2 && ((uint64_t)tile + up) * up < (1ull << 32)) *magic32 = (uint32_t)(((1ull << 32) + up - 1) / up);
}

// store: write the planes; mom != nullptr: fused per-cell moments (at least one of the two).
template <typename T>
static int launch_cells(int64_t ncell, int32_t ppc, const T* kappa, const T* theta, const T* drift,
                        int64_t drift_stride, uint64_t offset, const PhiloxKeys& K, bool vec, bool store, T* vx, T* vy,
                        T* vz, T* mom, CellRec<T>* W, cudaStream_t st, bool prepare = true, bool sample = true) {
    constexpr int G = 16 / sizeof(T);
    constexpr int64_t tile = (int64_t)kThreads * G * kGroups;
    int mode = kMomNone, lanes = 1;
    if (mom != nullptr) {
        const int L = ppc / G;
        if (ppc % G == 0 && L <= 32 && (L & (L - 1)) == 0) { mode = kMomDirect; lanes = L; }
        else if (ppc % (32 * G) == 0) { mode = kMomWarp; lanes = 32; }
        else mode = kMomAtomic;
    }
    if (prepare) {
        const int64_t cgrid = (ncell + kThreads - 1) / kThreads;
        cell_coef_kernel<T><<<(unsigned)cgrid, kThreads, 0, st>>>(ncell, kappa, theta, drift, drift_stride, W,
                                                                  (mode == kMomWarp || mode == kMomAtomic) ? mom : nullptr);
        KG_CUDA(cudaGetLastError());
    }
    if (!sample) return KAPPAGEN_OK;
    const int64_t n = ncell * (int64_t)ppc;
    uint64_t magic;
    uint32_t magic32;
    cells_magics(n, ppc, tile, &magic, &magic32);
#define KG_CELLS(V, S, M) launch_cells_as<T, V, S, M>(n, ppc, magic, magic32, offset, K, W, vx, vy, vz, mom, mode, lanes, st)
    if (mom == nullptr) return vec ? KG_CELLS(true, true, false) : KG_CELLS(false, true, false);
    if (!store) return KG_CELLS(true, false, true);
    return vec ? KG_CELLS(true, true, true) : KG_CELLS(false, true, true);
#undef KG_CELLS
}

template <typename T>
static int launch_mt(int64_t n, double kappa, double theta, uint64_t offset, const PhiloxKeys& K, T* vx, T* vy,
                     T* vz, unsigned long long* trips, cudaStream_t st) {
    MtParams<T> P;
    const double d = (kappa - 0.5) - 1.0 / 3.0;
    P.d = (T)d;
    P.cp = (T)(1.0 / sqrt(9.0 * d));
    P.scale = (T)(theta * sqrt(0.5 * kappa));
    int grid = 0, rc;
    if ((rc = grid_for<baseline_mt_kernel<T>>((n + kThreads - 1) / kThreads, &grid)) != KAPPAGEN_OK) return rc;
    baseline_mt_kernel<T><<<grid, kThreads, 0, st>>>(n, offset, K, P, vx, vy, vz, trips);
    KG_CUDA(cudaGetLastError());
    return KAPPAGEN_OK;
}

}  // namespace kappagen

using namespace kappagen;

extern "C" int kappagen_sample(int64_t n, double kappa, double theta, uint64_t seed, uint64_t offset, int dtype,
                               void* vx, void* vy, void* vz, void* stream) {
    return sample_on_stream("kappagen_sample", n, kappa, theta, seed, offset, dtype, 0u, vx, vy, vz, (cudaStream_t)stream);
}

extern "C" int kappagen_sample_flags(int64_t n, double kappa, double theta, uint64_t seed, uint64_t offset, int dtype,
                                     uint32_t flags, void* vx, void* vy, void* vz, void* stream) {
    return sample_on_stream("kappagen_sample_flags", n, kappa, theta, seed, offset, dtype, flags, vx, vy, vz,
                            (cudaStream_t)stream);
}

extern "C" size_t kappagen_cells_workspace_bytes(int64_t ncell, int dtype) {
    if (ncell <= 0 || (dtype != KAPPAGEN_F32 && dtype != KAPPAGEN_F64)) return 0;
    return (size_t)ncell * (dtype == KAPPAGEN_F32 ? sizeof(CellRec<float>) : sizeof(CellRec<double>));
}

static int cells_impl(const char* fn, int64_t ncell, int32_t ppc, const void* kappa, const void* theta, const void* drift,
                      int64_t drift_stride, uint64_t seed, uint64_t offset, int dtype, void* vx, void* vy, void* vz,
                      void* moments, bool want_moments, void* workspace, size_t workspace_bytes, void* stream) {
    if (ncell < 0 || ppc < 0) {
        set_error("%s: negative ncell or ppc", fn);
        return KAPPAGEN_EINVAL;
    }
    if (ncell > 0 && ppc > 0 && ncell > INT64_MAX / ppc) {
        set_error("%s: ncell*ppc overflows", fn);
        return KAPPAGEN_EINVAL;
    }
    if (dtype != KAPPAGEN_F32 && dtype != KAPPAGEN_F64) {
        set_error("%s: dtype %d is neither KAPPAGEN_F32 nor KAPPAGEN_F64", fn, dtype);
        return KAPPAGEN_EINVAL;
    }
    bool vec = false;
    const int64_t n = ncell * (int64_t)ppc;
    const bool store = !(want_moments && !vx && !vy && !vz);          // moments only: all three planes NULL
    if (store) {
        int rc = check_planes(fn, n, dtype, vx, vy, vz, &vec);
        if (rc != KAPPAGEN_OK) return rc;
    }
    if (drift != nullptr && drift_stride != 0 && drift_stride != 1) {
        set_error("%s: drift_stride must be 0 (shared) or 1 (per cell), got %lld", fn, (long long)drift_stride);
        return KAPPAGEN_EINVAL;
    }
    if (n == 0) return KAPPAGEN_OK;
    if (!kappa || !theta) {
        set_error("%s: NULL kappa or theta array", fn);
        return KAPPAGEN_ENULL;
    }
    if (want_moments && !moments) {
        set_error("%s: NULL moments array", fn);
        return KAPPAGEN_ENULL;
    }
    const size_t es = elem_size(dtype);
    if (!aligned_to(kappa, es) || !aligned_to(theta, es) || (drift && !aligned_to(drift, es))) {
        set_error("%s: kappa/theta/drift not aligned to the element size", fn);
        return KAPPAGEN_EALIGN;
    }
    if (want_moments && !aligned_to(moments, 16)) {
        set_error("%s: moments not 16-byte aligned", fn);
        return KAPPAGEN_EALIGN;
    }
    if (!workspace || workspace_bytes < kappagen_cells_workspace_bytes(ncell, dtype) || !aligned_to(workspace, 16)) {
        set_error("%s: workspace NULL, misaligned or smaller than %zu bytes", fn, kappagen_cells_workspace_bytes(ncell, dtype));
        return KAPPAGEN_EWORKSPACE;
    }
    const PhiloxKeys K = philox_expand_keys(seed);
    cudaStream_t st = (cudaStream_t)stream;
    if (dtype == KAPPAGEN_F32)
        return launch_cells<float>(ncell, ppc, (const float*)kappa, (const float*)theta, (const float*)drift, drift_stride,
                                   offset, K, vec, store, (float*)vx, (float*)vy, (float*)vz, (float*)moments,
                                   (CellRec<float>*)workspace, st);
    return launch_cells<double>(ncell, ppc, (const double*)kappa, (const double*)theta, (const double*)drift, drift_stride,
                                offset, K, vec, store, (double*)vx, (double*)vy, (double*)vz, (double*)moments,
                                (CellRec<double>*)workspace, st);
}

extern "C" int kappagen_sample_cells(int64_t ncell, int32_t ppc, const void* kappa, const void* theta,
                                     const void* drift, int64_t drift_stride, uint64_t seed, uint64_t offset,
                                     int dtype, void* vx, void* vy, void* vz, void* workspace,
                                     size_t workspace_bytes, void* stream) {
    return cells_impl("kappagen_sample_cells", ncell, ppc, kappa, theta, drift, drift_stride, seed, offset, dtype, vx, vy, vz,
                      nullptr, false, workspace, workspace_bytes, stream);
}

extern "C" int kappagen_sample_cells_moments(int64_t ncell, int32_t ppc, const void* kappa, const void* theta,
                                             const void* drift, int64_t drift_stride, uint64_t seed, uint64_t offset,
                                             int dtype, void* vx, void* vy, void* vz, void* moments, void* workspace,
                                             size_t workspace_bytes, void* stream) {
    return cells_impl("kappagen_sample_cells_moments", ncell, ppc, kappa, theta, drift, drift_stride, seed, offset, dtype, vx,
                      vy, vz, moments, true, workspace, workspace_bytes, stream);
}

// ---- kappagen_sample_cells_static: kappagen_sample_cells for callers that have no device memory to hand over as
// workspace and may not ask the driver for any (see include/kappagen.h).  The per-cell records live in the array
// below, which is part of the library's device image: it is reserved on every GPU that loads libkappagen and stays
// reserved until the process exits, so it is kept small.  The kernels are the ones kappagen_sample_cells launches;
// only the place the records are kept differs.
static __device__ __align__(256) unsigned char g_static_cells_scratch[KAPPAGEN_STATIC_SCRATCH_BYTES];

// Where g_static_cells_scratch sits on the CURRENT device.  On the host the array's name is only a handle for the
// runtime, not somewhere a kernel can write: the address a kernel may use comes from cudaGetSymbolAddress, differs
// from GPU to GPU, and is looked up once per device (under a lock: two host threads may arrive here first together).
static int static_cells_scratch(const char* fn, void** out) {
    constexpr int kMaxDev = 64;
    static std::mutex mu;
    static void* addr[kMaxDev] = {};
    int dev = -1;
    KG_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kMaxDev) {
        set_error("%s: device ordinal %d is outside the %d this call keeps an address for", fn, dev, kMaxDev);
        return KAPPAGEN_ECUDA;
    }
    std::lock_guard<std::mutex> lock(mu);
    if (addr[dev] == nullptr) {
        void* p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&p, g_static_cells_scratch);
        if (e != cudaSuccess || p == nullptr) {
            set_error("%s: cudaGetSymbolAddress of the built-in scratch failed on device %d: %s", fn, dev, cudaGetErrorString(e));
            return KAPPAGEN_ECUDA;
        }
        addr[dev] = p;
    }
    *out = addr[dev];
    return KAPPAGEN_OK;
}

extern "C" int kappagen_sample_cells_static(int64_t ncell, int32_t ppc, const void* kappa, const void* theta,
                                            const void* drift, int64_t drift_stride, uint64_t seed, uint64_t offset,
                                            int dtype, void* vx, void* vy, void* vz, void* stream) {
    const char* fn = "kappagen_sample_cells_static";
    if (dtype != KAPPAGEN_F32 && dtype != KAPPAGEN_F64) {
        set_error("%s: dtype %d is neither KAPPAGEN_F32 nor KAPPAGEN_F64", fn, dtype);
        return KAPPAGEN_EINVAL;
    }
    const size_t rec = dtype == KAPPAGEN_F32 ? sizeof(CellRec<float>) : sizeof(CellRec<double>);
    const int64_t most = (int64_t)(KAPPAGEN_STATIC_SCRATCH_BYTES / rec);
    if (ncell > most) {                                               // before anything touches the device
        set_error("%s: %lld cells need %zu bytes of per-cell records, the built-in scratch holds %d bytes (at most %lld cells "
                  "of this dtype per call): split the call, or use kappagen_sample_cells with a workspace of your own",
                  fn, (long long)ncell, (size_t)ncell * rec, (int)KAPPAGEN_STATIC_SCRATCH_BYTES, (long long)most);
        return KAPPAGEN_EWORKSPACE;
    }
    void* scratch = nullptr;
    if (ncell > 0 && ppc > 0) {                                       // nothing to launch otherwise: cells_impl only checks
        const int rc = static_cells_scratch(fn, &scratch);
        if (rc != KAPPAGEN_OK) return rc;
    }
    // every record of cells 0 .. ncell-1 is rewritten in full by the pre-kernel before the sampler reads it, so what an
    // earlier call left in the array is never seen and nothing needs clearing
    return cells_impl(fn, ncell, ppc, kappa, theta, drift, drift_stride, seed, offset, dtype, vx, vy, vz, nullptr, false,
                      scratch, KAPPAGEN_STATIC_SCRATCH_BYTES, stream);
}

extern "C" int kappagen_baseline_mt(int64_t n, double kappa, double theta, uint64_t seed, uint64_t offset, int dtype,
                                    void* vx, void* vy, void* vz, void* stream, unsigned long long* trip_counters) {
    const char* fn = "kappagen_baseline_mt";
    bool vec = false;
    int rc = check_planes(fn, n, dtype, vx, vy, vz, &vec);
    if (rc != KAPPAGEN_OK) return rc;
    if (!domain_ok(kappa, theta)) {
        set_error("%s: need finite kappa > 3/2 and theta >= 0 (got kappa = %g, theta = %g)", fn, kappa, theta);
        return KAPPAGEN_EINVAL;
    }
    if (n == 0) return KAPPAGEN_OK;
    const PhiloxKeys K = philox_expand_keys(seed);
    cudaStream_t st = (cudaStream_t)stream;
    if (dtype == KAPPAGEN_F32)
        return launch_mt<float>(n, kappa, theta, offset, K, (float*)vx, (float*)vy, (float*)vz, trip_counters, st);
    return launch_mt<double>(n, kappa, theta, offset, K, (double*)vx, (double*)vy, (double*)vz, trip_counters, st);
}

static int words_impl(const char* fn, int64_t n, uint64_t seed, uint64_t offset, uint32_t* w0, uint32_t* w1, uint32_t* w2,
                      uint32_t* w3, bool want_w3, void* stream) {
    if (n < 0) {
        set_error("%s: negative count", fn);
        return KAPPAGEN_EINVAL;
    }
    if (n == 0) return KAPPAGEN_OK;
    if (!w0 || !w1 || !w2 || (want_w3 && !w3)) {
        set_error("%s: NULL output", fn);
        return KAPPAGEN_ENULL;
    }
    if (!aligned_to(w0, 4) || !aligned_to(w1, 4) || !aligned_to(w2, 4) || !aligned_to(w3, 4)) {
        set_error("%s: outputs must be 4-byte aligned", fn);
        return KAPPAGEN_EALIGN;
    }
    int grid = 0, rc;
    if ((rc = grid_for<words_kernel>((n + 4 * kThreads - 1) / (4 * kThreads), &grid)) != KAPPAGEN_OK) return rc;
    words_kernel<<<grid, kThreads, 0, (cudaStream_t)stream>>>(n, offset, philox_expand_keys(seed), w0, w1, w2, w3);
    KG_CUDA(cudaGetLastError());
    return KAPPAGEN_OK;
}

template <typename T, bool U64>
static int launch_hist(int64_t n, uint64_t offset, const PhiloxKeys& K, const Coef<T>& C, T inv, int nbins,
                       unsigned long long* hist, cudaStream_t st) {
    constexpr int threads = TileTraits<T>::threads;                  // the sample kernel's block and tile shape
    constexpr int64_t tile = (int64_t)threads * (16 / sizeof(T)) * TileTraits<T>::groups;
    constexpr int warps = threads / 32;
    int replicas = (40 * 1024) / (nbins * 4);                        // (+ the double chain's tables: static shared memory)
    if (replicas > warps) replicas = warps;
    if (replicas < 1) replicas = 1;
    const size_t smem = (size_t)replicas * nbins * 4;
    int grid = 0, rc;
    // The block counts into 32-bit shared-memory replicas and flushes them once at its end.  A replica sees the
    // particles of ceil(warps/replicas) of the block's warps, so per launch a block may process at most
    // 2^32 / that share of its particles: split larger calls into launches of `cap` particles (whatever the
    // device's SM count or the occupancy), each flushing into the caller's 64-bit counters.
    const int64_t tiles_all = (n + tile - 1) / tile;
    if ((rc = grid_for<speed_histogram_kernel<T, U64>>(tiles_all, &grid, threads, smem)) != KAPPAGEN_OK) return rc;
    const int share = (warps + replicas - 1) / replicas;
    const int64_t per_block = (((int64_t)1 << 32) - 1) / share * warps / tile * tile;     // particles, whole tiles
    const int64_t cap = per_block * (int64_t)(grid < 1 ? 1 : grid) / 2;                   // factor 2: uneven tile counts per block
    for (int64_t done = 0; done < n;) {
        const int64_t m = (n - done) < cap ? (n - done) : cap;
        int g = 0;
        if ((rc = grid_for<speed_histogram_kernel<T, U64>>((m + tile - 1) / tile, &g, threads, smem)) != KAPPAGEN_OK) return rc;
        speed_histogram_kernel<T, U64><<<g, threads, smem, st>>>(m, offset + (uint64_t)done, K, C, inv, nbins, replicas, hist);
        KG_CUDA(cudaGetLastError());
        done += m;
    }
    return KAPPAGEN_OK;
}

extern "C" int kappagen_speed_histogram(int64_t n, double kappa, uint64_t seed, uint64_t offset, int dtype, uint32_t flags,
                                        double dv, int32_t nbins, unsigned long long* hist, void* stream) {
    const char* fn = "kappagen_speed_histogram";
    if (dtype != KAPPAGEN_F32 && dtype != KAPPAGEN_F64) {
        set_error("%s: dtype %d is neither KAPPAGEN_F32 nor KAPPAGEN_F64", fn, dtype);
        return KAPPAGEN_EINVAL;
    }
    if (n < 0 || n > ((int64_t)1 << 40) || nbins < 2 || nbins > kHistMaxBins || !(dv > 0.0) || !std::isfinite(dv) ||
        !domain_ok(kappa, 0.0) || (flags & ~(uint32_t)KAPPAGEN_U1_64)) {
        set_error("%s: need 0 <= n <= 2^40, 2 <= nbins <= %d, dv > 0, kappa > 3/2, flags in {0, KAPPAGEN_U1_64}", fn, kHistMaxBins);
        return KAPPAGEN_EINVAL;
    }
    if (n == 0) return KAPPAGEN_OK;
    if (!hist) {
        set_error("%s: NULL histogram", fn);
        return KAPPAGEN_ENULL;
    }
    if (!aligned_to(hist, 8)) {
        set_error("%s: histogram not 8-byte aligned", fn);
        return KAPPAGEN_EALIGN;
    }
    const PhiloxKeys K = philox_expand_keys(seed);
    const bool u64 = (flags & KAPPAGEN_U1_64) != 0;
    cudaStream_t st = (cudaStream_t)stream;
    if (dtype == KAPPAGEN_F32) {
        const Coef<float> C = host_coef_f32(kappa, 1.0, true);        // theta = 1 folded: the chain returns 2 |v|/theta
        const float inv = (float)(0.5 / dv);
        return u64 ? launch_hist<float, true>(n, offset, K, C, inv, nbins, hist, st)
                   : launch_hist<float, false>(n, offset, K, C, inv, nbins, hist, st);
    }
    const Coef<double> C = host_coef_f64(kappa, 1.0);
    return u64 ? launch_hist<double, true>(n, offset, K, C, 1.0 / dv, nbins, hist, st)
               : launch_hist<double, false>(n, offset, K, C, 1.0 / dv, nbins, hist, st);
}

extern "C" int kappagen_words(int64_t n, uint64_t seed, uint64_t offset, uint32_t* w0, uint32_t* w1, uint32_t* w2,
                              void* stream) {
    return words_impl("kappagen_words", n, seed, offset, w0, w1, w2, nullptr, false, stream);
}

extern "C" int kappagen_words4(int64_t n, uint64_t seed, uint64_t offset, uint32_t* w0, uint32_t* w1, uint32_t* w2,
                               uint32_t* w3, void* stream) {
    return words_impl("kappagen_words4", n, seed, offset, w0, w1, w2, w3, true, stream);
}

template <bool U64>
static int velocity_of_words_impl(const char* fn, int64_t n, const uint32_t* w0, const uint32_t* w1, const uint32_t* w2,
                                  const uint32_t* w3, double kappa, double theta, int dtype, void* vx, void* vy, void* vz,
                                  void* stream) {
    bool vec = false;
    int rc = check_planes(fn, n, dtype, vx, vy, vz, &vec);
    if (rc != KAPPAGEN_OK) return rc;
    if (!domain_ok(kappa, theta)) {
        set_error("%s: need finite kappa > 3/2 and theta >= 0 (got kappa = %g, theta = %g)", fn, kappa, theta);
        return KAPPAGEN_EINVAL;
    }
    if (n == 0) return KAPPAGEN_OK;
    if (!w0 || !w1 || !w2 || (U64 && !w3)) {
        set_error("%s: NULL word array", fn);
        return KAPPAGEN_ENULL;
    }
    int grid = 0;
    cudaStream_t st = (cudaStream_t)stream;
    const int64_t tiles = (n + kThreads - 1) / kThreads;
    if (dtype == KAPPAGEN_F32) {
        const bool fold = theta_folds(theta);              // the same choice kappagen_sample makes
        const Coef<float> C = host_coef_f32(kappa, theta, fold);
        if (fold) {
            if ((rc = grid_for<velocity_of_words_kernel<float, true, U64>>(tiles, &grid)) != KAPPAGEN_OK) return rc;
            velocity_of_words_kernel<float, true, U64><<<grid, kThreads, 0, st>>>(n, w0, w1, w2, w3, C, (float*)vx, (float*)vy, (float*)vz);
        } else {
            if ((rc = grid_for<velocity_of_words_kernel<float, false, U64>>(tiles, &grid)) != KAPPAGEN_OK) return rc;
            velocity_of_words_kernel<float, false, U64><<<grid, kThreads, 0, st>>>(n, w0, w1, w2, w3, C, (float*)vx, (float*)vy, (float*)vz);
        }
    } else {
        if ((rc = grid_for<velocity_of_words_kernel<double, false, U64>>(tiles, &grid)) != KAPPAGEN_OK) return rc;
        velocity_of_words_kernel<double, false, U64><<<grid, kThreads, 0, st>>>(n, w0, w1, w2, w3, host_coef_f64(kappa, theta),
                                                                                (double*)vx, (double*)vy, (double*)vz);
    }
    KG_CUDA(cudaGetLastError());
    return KAPPAGEN_OK;
}

extern "C" int kappagen_velocity_of_words(int64_t n, const uint32_t* w0, const uint32_t* w1, const uint32_t* w2,
                                          double kappa, double theta, int dtype, void* vx, void* vy, void* vz,
                                          void* stream) {
    return velocity_of_words_impl<false>("kappagen_velocity_of_words", n, w0, w1, w2, nullptr, kappa, theta, dtype, vx, vy, vz,
                                         stream);
}

extern "C" int kappagen_velocity_of_words_u64(int64_t n, const uint32_t* w0, const uint32_t* w1, const uint32_t* w2,
                                              const uint32_t* w3, double kappa, double theta, int dtype, void* vx, void* vy,
                                              void* vz, void* stream) {
    return velocity_of_words_impl<true>("kappagen_velocity_of_words_u64", n, w0, w1, w2, w3, kappa, theta, dtype, vx, vy, vz,
                                        stream);
}

// ---- test hooks that go through the code the samplers ship (whole-tile path), include/kappagen.h
template <typename T>
static int launch_words_tile(int64_t n, uint64_t seed, uint64_t offset, uint32_t* w0, uint32_t* w1, uint32_t* w2, uint32_t* w3,
                             cudaStream_t st) {
    constexpr int threads = TileTraits<T>::threads;
    constexpr int64_t tile = (int64_t)threads * (16 / sizeof(T)) * TileTraits<T>::groups;
    int grid = 0, rc;
    if ((rc = grid_for<words_tile_kernel<T>>((n + tile - 1) / tile, &grid, threads)) != KAPPAGEN_OK) return rc;
    words_tile_kernel<T><<<grid, threads, 0, st>>>(n, offset, philox_expand_keys(seed), w0, w1, w2, w3);
    KG_CUDA(cudaGetLastError());
    return KAPPAGEN_OK;
}

extern "C" int kappagen_words_tile(int64_t n, uint64_t seed, uint64_t offset, int dtype, uint32_t* w0, uint32_t* w1,
                                   uint32_t* w2, uint32_t* w3, void* stream) {
    const char* fn = "kappagen_words_tile";
    if (n < 0 || (dtype != KAPPAGEN_F32 && dtype != KAPPAGEN_F64)) {
        set_error("%s: negative count or bad dtype", fn);
        return KAPPAGEN_EINVAL;
    }
    if (n == 0) return KAPPAGEN_OK;
    if (!w0 || !w1 || !w2 || !w3) {
        set_error("%s: NULL output", fn);
        return KAPPAGEN_ENULL;
    }
    if (!aligned_to(w0, 4) || !aligned_to(w1, 4) || !aligned_to(w2, 4) || !aligned_to(w3, 4)) {
        set_error("%s: outputs must be 4-byte aligned", fn);
        return KAPPAGEN_EALIGN;
    }
    return dtype == KAPPAGEN_F32 ? launch_words_tile<float>(n, seed, offset, w0, w1, w2, w3, (cudaStream_t)stream)
                                 : launch_words_tile<double>(n, seed, offset, w0, w1, w2, w3, (cudaStream_t)stream);
}

template <typename T, bool FOLD, bool U64>
static int launch_vow_tile(int64_t n, const uint32_t* w0, const uint32_t* w1, const uint32_t* w2, const uint32_t* w3,
                           const Coef<T>& C, T* vx, T* vy, T* vz, cudaStream_t st) {
    constexpr int threads = TileTraits<T>::threads;
    constexpr int64_t tile = (int64_t)threads * (16 / sizeof(T)) * TileTraits<T>::groups;
    int grid = 0, rc;
    if ((rc = grid_for<velocity_of_words_tile_kernel<T, FOLD, U64>>((n + tile - 1) / tile, &grid, threads)) != KAPPAGEN_OK) return rc;
    velocity_of_words_tile_kernel<T, FOLD, U64><<<grid, threads, 0, st>>>(n, w0, w1, w2, w3, C, vx, vy, vz);
    KG_CUDA(cudaGetLastError());
    return KAPPAGEN_OK;
}

extern "C" int kappagen_velocity_of_words_tile(int64_t n, const uint32_t* w0, const uint32_t* w1, const uint32_t* w2,
                                               const uint32_t* w3, double kappa, double theta, int dtype, uint32_t flags,
                                               void* vx, void* vy, void* vz, void* stream) {
    const char* fn = "kappagen_velocity_of_words_tile";
    bool vec = false;
    int rc = check_planes(fn, n, dtype, vx, vy, vz, &vec);
    if (rc != KAPPAGEN_OK) return rc;
    if (!domain_ok(kappa, theta) || (flags & ~(uint32_t)KAPPAGEN_U1_64)) {
        set_error("%s: need finite kappa > 3/2, theta >= 0, flags in {0, KAPPAGEN_U1_64}", fn);
        return KAPPAGEN_EINVAL;
    }
    if (n == 0) return KAPPAGEN_OK;
    const bool u64 = (flags & KAPPAGEN_U1_64) != 0;
    if (!w0 || !w1 || !w2 || (u64 && !w3)) {
        set_error("%s: NULL word array", fn);
        return KAPPAGEN_ENULL;
    }
    cudaStream_t st = (cudaStream_t)stream;
    if (dtype == KAPPAGEN_F32) {
        const bool fold = theta_folds(theta);              // the same choice kappagen_sample makes
        const Coef<float> C = host_coef_f32(kappa, theta, fold);
        float *x = (float*)vx, *y = (float*)vy, *z = (float*)vz;
        if (fold) return u64 ? launch_vow_tile<float, true, true>(n, w0, w1, w2, w3, C, x, y, z, st)
                             : launch_vow_tile<float, true, false>(n, w0, w1, w2, w3, C, x, y, z, st);
        return u64 ? launch_vow_tile<float, false, true>(n, w0, w1, w2, w3, C, x, y, z, st)
                   : launch_vow_tile<float, false, false>(n, w0, w1, w2, w3, C, x, y, z, st);
    }
    const Coef<double> C = host_coef_f64(kappa, theta);
    double *x = (double*)vx, *y = (double*)vy, *z = (double*)vz;
    return u64 ? launch_vow_tile<double, false, true>(n, w0, w1, w2, w3, C, x, y, z, st)
               : launch_vow_tile<double, false, false>(n, w0, w1, w2, w3, C, x, y, z, st);
}

// End-to-end path: host destination, chunked, double-buffered (the copy of chunk c overlaps the kernel
// of chunk c+1 on the other stream).
static constexpr int64_t kHostChunk = (int64_t)1 << 22;              // particles: 48 / 96 MiB of output per chunk
static size_t host_plane_bytes(int64_t n, int dtype) {
    const int64_t chunk = n < kHostChunk ? n : kHostChunk;
    return (((size_t)chunk * elem_size(dtype)) + 255) & ~(size_t)255;
}
extern "C" size_t kappagen_sample_host_workspace_bytes(int64_t n, int dtype) {
    if (n <= 0 || (dtype != KAPPAGEN_F32 && dtype != KAPPAGEN_F64)) return 0;
    return 6 * host_plane_bytes(n, dtype);
}

// dev: 6 planes of host_plane_bytes; st[0], st[1]: the two streams; both synchronised on return.
static int sample_host_on(const char* fn, int64_t n, double kappa, double theta, uint64_t seed, uint64_t offset, int dtype,
                          void* vx_host, void* vy_host, void* vz_host, char* dev, cudaStream_t* st) {
    const size_t es = elem_size(dtype);
    const int64_t chunk = n < kHostChunk ? n : kHostChunk;
    const size_t plane = host_plane_bytes(n, dtype);
    int status = KAPPAGEN_OK;
    int64_t done = 0;
    for (int c = 0; done < n && status == KAPPAGEN_OK; ++c) {
        const int b = c & 1;
        const int64_t m = (n - done) < chunk ? (n - done) : chunk;
        char* d = dev + (size_t)b * 3 * plane;
        status = sample_on_stream(fn, m, kappa, theta, seed, offset + (uint64_t)done, dtype, 0u, d, d + plane, d + 2 * plane, st[b]);
        if (status != KAPPAGEN_OK) break;
        char* hv[3] = {(char*)vx_host, (char*)vy_host, (char*)vz_host};
        for (int q = 0; q < 3; ++q) {
            if (cudaMemcpyAsync(hv[q] + (size_t)done * es, d + (size_t)q * plane, (size_t)m * es, cudaMemcpyDeviceToHost,
                                st[b]) != cudaSuccess) {
                set_error("%s: cudaMemcpyAsync failed: %s", fn, cudaGetErrorString(cudaGetLastError()));
                status = KAPPAGEN_ECUDA;
            }
        }
        done += m;
    }
    for (int b = 0; b < 2; ++b) {
        if (cudaStreamSynchronize(st[b]) != cudaSuccess && status == KAPPAGEN_OK) {
            set_error("%s: stream synchronize failed: %s", fn, cudaGetErrorString(cudaGetLastError()));
            status = KAPPAGEN_ECUDA;
        }
    }
    return status;
}

static int sample_host_checks(const char* fn, int64_t n, double kappa, double theta, int dtype, void* vx, void* vy, void* vz) {
    bool vec = false;
    int rc = check_planes(fn, n, dtype, vx, vy, vz, &vec);
    if (rc != KAPPAGEN_OK) return rc;
    if (!domain_ok(kappa, theta)) {
        set_error("%s: need finite kappa > 3/2 and theta >= 0 (got kappa = %g, theta = %g)", fn, kappa, theta);
        return KAPPAGEN_EINVAL;
    }
    return KAPPAGEN_OK;
}

extern "C" int kappagen_sample_host(int64_t n, double kappa, double theta, uint64_t seed, uint64_t offset, int dtype,
                                    void* vx_host, void* vy_host, void* vz_host) {
    const char* fn = "kappagen_sample_host";
    int rc = sample_host_checks(fn, n, kappa, theta, dtype, vx_host, vy_host, vz_host);
    if (rc != KAPPAGEN_OK || n == 0) return rc;
    char* dev = nullptr;
    cudaStream_t st[2] = {nullptr, nullptr};
    KG_CUDA(cudaMalloc(&dev, kappagen_sample_host_workspace_bytes(n, dtype)));
    int status = KAPPAGEN_OK;
    for (int b = 0; b < 2 && status == KAPPAGEN_OK; ++b)
        if (cudaStreamCreateWithFlags(&st[b], cudaStreamNonBlocking) != cudaSuccess) {
            set_error("%s: cudaStreamCreate failed", fn);
            status = KAPPAGEN_ECUDA;
        }
    if (status == KAPPAGEN_OK) status = sample_host_on(fn, n, kappa, theta, seed, offset, dtype, vx_host, vy_host, vz_host, dev, st);
    for (int b = 0; b < 2; ++b)
        if (st[b]) cudaStreamDestroy(st[b]);
    cudaFree(dev);
    return status;
}

extern "C" int kappagen_sample_host_ws(int64_t n, double kappa, double theta, uint64_t seed, uint64_t offset, int dtype,
                                       void* vx_host, void* vy_host, void* vz_host, void* workspace, size_t workspace_bytes,
                                       void* stream_a, void* stream_b) {
    const char* fn = "kappagen_sample_host_ws";
    int rc = sample_host_checks(fn, n, kappa, theta, dtype, vx_host, vy_host, vz_host);
    if (rc != KAPPAGEN_OK || n == 0) return rc;
    if (stream_a == stream_b) {
        set_error("%s: the two streams must differ (the chunks alternate between them)", fn);
        return KAPPAGEN_EINVAL;
    }
    if (!workspace || workspace_bytes < kappagen_sample_host_workspace_bytes(n, dtype) || !aligned_to(workspace, 256)) {
        set_error("%s: workspace NULL, not 256-byte aligned or smaller than %zu bytes", fn, kappagen_sample_host_workspace_bytes(n, dtype));
        return KAPPAGEN_EWORKSPACE;
    }
    cudaStream_t st[2] = {(cudaStream_t)stream_a, (cudaStream_t)stream_b};
    return sample_host_on(fn, n, kappa, theta, seed, offset, dtype, vx_host, vy_host, vz_host, (char*)workspace, st);
}

// ---- Table I lines 1-4 "are required only once": the two halves of kappagen_sample_cells as calls of their own
extern "C" int kappagen_cells_prepare(int64_t ncell, const void* kappa, const void* theta, const void* drift,
                                      int64_t drift_stride, int dtype, void* workspace, size_t workspace_bytes, void* stream) {
    const char* fn = "kappagen_cells_prepare";
    if (ncell < 0 || (dtype != KAPPAGEN_F32 && dtype != KAPPAGEN_F64)) {
        set_error("%s: negative ncell or bad dtype", fn);
        return KAPPAGEN_EINVAL;
    }
    if (drift != nullptr && drift_stride != 0 && drift_stride != 1) {
        set_error("%s: drift_stride must be 0 (shared) or 1 (per cell), got %lld", fn, (long long)drift_stride);
        return KAPPAGEN_EINVAL;
    }
    if (ncell == 0) return KAPPAGEN_OK;
    if (!kappa || !theta) {
        set_error("%s: NULL kappa or theta array", fn);
        return KAPPAGEN_ENULL;
    }
    const size_t es = elem_size(dtype);
    if (!aligned_to(kappa, es) || !aligned_to(theta, es) || (drift && !aligned_to(drift, es))) {
        set_error("%s: kappa/theta/drift not aligned to the element size", fn);
        return KAPPAGEN_EALIGN;
    }
    if (!workspace || workspace_bytes < kappagen_cells_workspace_bytes(ncell, dtype) || !aligned_to(workspace, 16)) {
        set_error("%s: workspace NULL, misaligned or smaller than %zu bytes", fn, kappagen_cells_workspace_bytes(ncell, dtype));
        return KAPPAGEN_EWORKSPACE;
    }
    const PhiloxKeys K = philox_expand_keys(0);
    cudaStream_t st = (cudaStream_t)stream;
    if (dtype == KAPPAGEN_F32)
        return launch_cells<float>(ncell, 1, (const float*)kappa, (const float*)theta, (const float*)drift, drift_stride, 0, K, false,
                                   true, nullptr, nullptr, nullptr, nullptr, (CellRec<float>*)workspace, st, true, false);
    return launch_cells<double>(ncell, 1, (const double*)kappa, (const double*)theta, (const double*)drift, drift_stride, 0, K, false,
                                true, nullptr, nullptr, nullptr, nullptr, (CellRec<double>*)workspace, st, true, false);
}

extern "C" int kappagen_sample_cells_prepared(int64_t ncell, int32_t ppc, uint64_t seed, uint64_t offset, int dtype, void* vx,
                                              void* vy, void* vz, const void* workspace, size_t workspace_bytes, void* stream) {
    const char* fn = "kappagen_sample_cells_prepared";
    if (ncell < 0 || ppc < 0 || (ncell > 0 && ppc > 0 && ncell > INT64_MAX / ppc)) {
        set_error("%s: negative ncell or ppc, or ncell*ppc overflows", fn);
        return KAPPAGEN_EINVAL;
    }
    bool vec = false;
    const int64_t n = ncell * (int64_t)ppc;
    int rc = check_planes(fn, n, dtype, vx, vy, vz, &vec);
    if (rc != KAPPAGEN_OK || n == 0) return rc;
    if (!workspace || workspace_bytes < kappagen_cells_workspace_bytes(ncell, dtype) || !aligned_to(workspace, 16)) {
        set_error("%s: workspace NULL, misaligned or smaller than %zu bytes", fn, kappagen_cells_workspace_bytes(ncell, dtype));
        return KAPPAGEN_EWORKSPACE;
    }
    const PhiloxKeys K = philox_expand_keys(seed);
    cudaStream_t st = (cudaStream_t)stream;
    if (dtype == KAPPAGEN_F32)
        return launch_cells<float>(ncell, ppc, nullptr, nullptr, nullptr, 0, offset, K, vec, true, (float*)vx, (float*)vy, (float*)vz,
                                   nullptr, (CellRec<float>*)const_cast<void*>(workspace), st, false, true);
    return launch_cells<double>(ncell, ppc, nullptr, nullptr, nullptr, 0, offset, K, vec, true, (double*)vx, (double*)vy, (double*)vz,
                                nullptr, (CellRec<double>*)const_cast<void*>(workspace), st, false, true);
}

// ---- kappagen_load_cells: per-cell velocities and positions as one AoS record per particle (load_cells.cuh)
template <typename T, bool HASW>
static int launch_load_as(int64_t n, int32_t ppc, uint64_t offset, const PhiloxKeys& K, const CellRec<T>* W, const T* weight,
                          int64_t cell_base, T* out, cudaStream_t st) {
    constexpr int64_t tile = (int64_t)kThreads * (16 / sizeof(T)) * kGroups;
    {   // the opt-in to the kernel's dynamic shared memory is per device and sticks: once per device and instantiation,
        // not on every launch (small calls are launch-bound)
        constexpr int kMaxDev = 64;
        static std::atomic<bool> opted_in[kMaxDev] = {};
        int dev = 0;
        KG_CUDA(cudaGetDevice(&dev));
        const bool cached = dev >= 0 && dev < kMaxDev;
        if (!cached || !opted_in[dev].load(std::memory_order_acquire)) {
            KG_CUDA(cudaFuncSetAttribute(load_cells_kernel<T, HASW>, cudaFuncAttributeMaxDynamicSharedMemorySize, kLoadSmemBytes));
            if (cached) opted_in[dev].store(true, std::memory_order_release);
        }
    }
    uint64_t magic;
    uint32_t magic32;
    cells_magics(n, ppc, tile, &magic, &magic32);
    PhiloxKeys Kpos = K;
    Kpos.k1[0] ^= 2u;                                                 // counter word 3 = 2: the position block (reading R22)
    int grid = 0, rc;
    if ((rc = grid_for<load_cells_kernel<T, HASW>>((n + tile - 1) / tile, &grid, kThreads, kLoadSmemBytes)) != KAPPAGEN_OK) return rc;
    load_cells_kernel<T, HASW><<<grid, kThreads, kLoadSmemBytes, st>>>(n, (uint32_t)ppc, magic, magic32, offset, K, Kpos, W, weight,
                                                                      cell_base, out);
    KG_CUDA(cudaGetLastError());
    return KAPPAGEN_OK;
}

template <typename T>
static int launch_load(int64_t ncell, int32_t ppc, const T* kappa, const T* theta, const T* drift, int64_t drift_stride,
                       const T* weight, int64_t cell_base, uint64_t offset, const PhiloxKeys& K, T* out, CellRec<T>* W,
                       cudaStream_t st) {
    const int64_t cgrid = (ncell + kThreads - 1) / kThreads;
    cell_coef_kernel<T><<<(unsigned)cgrid, kThreads, 0, st>>>(ncell, kappa, theta, drift, drift_stride, W, nullptr);
    KG_CUDA(cudaGetLastError());
    const int64_t n = ncell * (int64_t)ppc;
    return weight ? launch_load_as<T, true>(n, ppc, offset, K, W, weight, cell_base, out, st)
                  : launch_load_as<T, false>(n, ppc, offset, K, W, weight, cell_base, out, st);
}

extern "C" int kappagen_load_cells(int64_t ncell, int32_t ppc, const void* kappa, const void* theta, const void* drift,
                                   int64_t drift_stride, const void* weight, int64_t cell_base, uint64_t seed, uint64_t offset,
                                   int dtype, void* records, void* workspace, size_t workspace_bytes, void* stream) {
    const char* fn = "kappagen_load_cells";
    if (ncell < 0 || ppc < 0 || cell_base < 0) {
        set_error("%s: negative ncell, ppc or cell_base", fn);
        return KAPPAGEN_EINVAL;
    }
    if (ncell > 0 && ppc > 0 && ncell > INT64_MAX / 8 / ppc) {
        set_error("%s: ncell*ppc*8 overflows", fn);
        return KAPPAGEN_EINVAL;
    }
    if (dtype != KAPPAGEN_F32 && dtype != KAPPAGEN_F64) {
        set_error("%s: dtype %d is neither KAPPAGEN_F32 nor KAPPAGEN_F64", fn, dtype);
        return KAPPAGEN_EINVAL;
    }
    if (cell_base > INT64_MAX - ncell || (dtype == KAPPAGEN_F32 && cell_base + ncell > ((int64_t)1 << 31))) {
        set_error("%s: cell_base + ncell does not fit the record's integer (int32 for float records)", fn);
        return KAPPAGEN_EINVAL;
    }
    if (drift != nullptr && drift_stride != 0 && drift_stride != 1) {
        set_error("%s: drift_stride must be 0 (shared) or 1 (per cell), got %lld", fn, (long long)drift_stride);
        return KAPPAGEN_EINVAL;
    }
    if (ncell == 0 || ppc == 0) return KAPPAGEN_OK;
    if (!kappa || !theta || !records) {
        set_error("%s: NULL kappa, theta or records", fn);
        return KAPPAGEN_ENULL;
    }
    const size_t es = elem_size(dtype);
    if (!aligned_to(kappa, es) || !aligned_to(theta, es) || (drift && !aligned_to(drift, es)) || (weight && !aligned_to(weight, es)) ||
        !aligned_to(records, 16)) {
        set_error("%s: kappa/theta/drift/weight not aligned to the element size, or records not 16-byte aligned", fn);
        return KAPPAGEN_EALIGN;
    }
    if (!workspace || workspace_bytes < kappagen_cells_workspace_bytes(ncell, dtype) || !aligned_to(workspace, 16)) {
        set_error("%s: workspace NULL, misaligned or smaller than %zu bytes", fn, kappagen_cells_workspace_bytes(ncell, dtype));
        return KAPPAGEN_EWORKSPACE;
    }
    const PhiloxKeys K = philox_expand_keys(seed);
    cudaStream_t st = (cudaStream_t)stream;
    if (dtype == KAPPAGEN_F32)
        return launch_load<float>(ncell, ppc, (const float*)kappa, (const float*)theta, (const float*)drift, drift_stride,
                                  (const float*)weight, cell_base, offset, K, (float*)records, (CellRec<float>*)workspace, st);
    return launch_load<double>(ncell, ppc, (const double*)kappa, (const double*)theta, (const double*)drift, drift_stride,
                               (const double*)weight, cell_base, offset, K, (double*)records, (CellRec<double>*)workspace, st);
}

// ---- measurement hooks (include/kappagen.h): the Philox + store ceiling and the pipe issue-rate probe
extern "C" int kappagen_philox_planes(int64_t n, uint64_t seed, uint64_t offset, uint32_t* w0, uint32_t* w1, uint32_t* w2,
                                      void* stream) {
    const char* fn = "kappagen_philox_planes";
    if (n < 0) {
        set_error("%s: negative count", fn);
        return KAPPAGEN_EINVAL;
    }
    if (n == 0) return KAPPAGEN_OK;
    if (!w0 || !w1 || !w2) {
        set_error("%s: NULL output", fn);
        return KAPPAGEN_ENULL;
    }
    if (!aligned_to(w0, 4) || !aligned_to(w1, 4) || !aligned_to(w2, 4)) {
        set_error("%s: outputs must be 4-byte aligned", fn);
        return KAPPAGEN_EALIGN;
    }
    const bool vec = aligned_to(w0, 16) && aligned_to(w1, 16) && aligned_to(w2, 16);
    constexpr int threads = TileTraits<float>::threads;
    constexpr int64_t tile = (int64_t)threads * 4 * TileTraits<float>::groups;
    const PhiloxKeys K = philox_expand_keys(seed);
    cudaStream_t st = (cudaStream_t)stream;
    int grid = 0, rc;
    if (vec) {
        if ((rc = grid_for<philox_planes_kernel<true>>((n + tile - 1) / tile, &grid, threads)) != KAPPAGEN_OK) return rc;
        philox_planes_kernel<true><<<grid, threads, 0, st>>>(n, offset, K, w0, w1, w2);
    } else {
        if ((rc = grid_for<philox_planes_kernel<false>>((n + tile - 1) / tile, &grid, threads)) != KAPPAGEN_OK) return rc;
        philox_planes_kernel<false><<<grid, threads, 0, st>>>(n, offset, K, w0, w1, w2);
    }
    KG_CUDA(cudaGetLastError());
    return KAPPAGEN_OK;
}

template <typename T, bool FOLD>
static int launch_math_planes(int64_t n, uint64_t offset, const Coef<T>& C, T* vx, T* vy, T* vz, cudaStream_t st) {
    constexpr int threads = TileTraits<T>::threads;
    constexpr int64_t tile = (int64_t)threads * (16 / sizeof(T)) * TileTraits<T>::groups;
    int grid = 0, rc;
    if ((rc = grid_for<math_planes_kernel<T, FOLD>>((n + tile - 1) / tile, &grid, threads)) != KAPPAGEN_OK) return rc;
    math_planes_kernel<T, FOLD><<<grid, threads, 0, st>>>(n, offset, C, vx, vy, vz);
    KG_CUDA(cudaGetLastError());
    return KAPPAGEN_OK;
}

extern "C" int kappagen_math_planes(int64_t n, double kappa, double theta, uint64_t offset, int dtype, void* vx, void* vy,
                                    void* vz, void* stream) {
    const char* fn = "kappagen_math_planes";
    bool vec = false;
    int rc = check_planes(fn, n, dtype, vx, vy, vz, &vec);
    if (rc != KAPPAGEN_OK) return rc;
    if (!domain_ok(kappa, theta)) {
        set_error("%s: need finite kappa > 3/2 and theta >= 0 (got kappa = %g, theta = %g)", fn, kappa, theta);
        return KAPPAGEN_EINVAL;
    }
    if (n == 0) return KAPPAGEN_OK;
    if (!vec) {
        set_error("%s: the planes must be 16-byte aligned (this hook has the vector-store path only)", fn);
        return KAPPAGEN_EALIGN;
    }
    cudaStream_t st = (cudaStream_t)stream;
    if (dtype == KAPPAGEN_F64)
        return launch_math_planes<double, false>(n, offset, host_coef_f64(kappa, theta), (double*)vx, (double*)vy, (double*)vz, st);
    const bool fold = theta_folds(theta);
    const Coef<float> C = host_coef_f32(kappa, theta, fold);
    return fold ? launch_math_planes<float, true>(n, offset, C, (float*)vx, (float*)vy, (float*)vz, st)
                : launch_math_planes<float, false>(n, offset, C, (float*)vx, (float*)vy, (float*)vz, st);
}

extern "C" int kappagen_pipe_probe_count(void) { return kPipeMixCount; }

extern "C" int kappagen_pipe_probe(int mix, int warps_per_scheduler, int iters, double* cycles_per_iter, int* counts) {
    const char* fn = "kappagen_pipe_probe";
    if (mix < 0 || mix >= kPipeMixCount || warps_per_scheduler < 1 || warps_per_scheduler > 8 || iters < 1) {
        set_error("%s: need 0 <= mix < %d, 1 <= warps_per_scheduler <= 8, iters >= 1", fn, kPipeMixCount);
        return KAPPAGEN_EINVAL;
    }
    if (!cycles_per_iter) {
        set_error("%s: NULL result pointer", fn);
        return KAPPAGEN_ENULL;
    }
    static PipeProbeFn table[kPipeMixCount] = {};
    static std::once_flag table_once;                                 // two host threads may make the first call together
    std::call_once(table_once, [] { PipeProbeTable<0>::fill(table); });
    if (counts) {
        const PipeMix M = kPipeMixes[mix];
        counts[0] = M.wide; counts[1] = M.lop3; counts[2] = M.ffma2; counts[3] = M.mufu; counts[4] = M.dfma; counts[5] = M.imad;
    }
    int dev = 0, sms = 0;
    KG_CUDA(cudaGetDevice(&dev));
    KG_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    const int threads = warps_per_scheduler * 4 * 32;                 // one block per SM, 4 sub-partitions
    uint32_t* sink = nullptr;
    long long* cyc = nullptr;
    KG_CUDA(cudaMalloc(&sink, 1024 * sizeof(uint32_t)));
    if (cudaMalloc(&cyc, (size_t)sms * sizeof(long long)) != cudaSuccess) {
        cudaFree(sink);
        set_error("%s: cudaMalloc failed", fn);
        return KAPPAGEN_ECUDA;
    }
    int status = KAPPAGEN_OK;
    long long* host = new long long[sms];
    cudaError_t launched = cudaSuccess;
    for (int pass = 0; pass < 2 && launched == cudaSuccess; ++pass) {                           // the second pass is timed warm
        table[mix]<<<sms, threads>>>(iters, 1u, sink, cyc);
        launched = cudaGetLastError();
    }
    cudaError_t copied = cudaSuccess;
    if (launched != cudaSuccess) {
        set_error("%s: launch of mix %d failed: %s", fn, mix, cudaGetErrorString(launched));
        status = KAPPAGEN_ECUDA;
    } else if ((copied = cudaMemcpy(host, cyc, (size_t)sms * sizeof(long long), cudaMemcpyDeviceToHost)) != cudaSuccess) {
        set_error("%s: kernel or copy failed: %s", fn, cudaGetErrorString(copied));
        status = KAPPAGEN_ECUDA;
    } else {
        double mean = 0.0;
        for (int b = 0; b < sms; ++b) mean += (double)host[b];
        *cycles_per_iter = mean / sms / iters / warps_per_scheduler;
    }
    delete[] host;
    cudaFree(sink);
    cudaFree(cyc);
    return status;
}
