// load_cells.cuh -- kappagen_load_cells: the PIC particle loader (second half): per-cell
// Kappa velocities (exactly kappagen_sample_cells') written together with positions as one array-of-structures
// record per particle, { fx, fy, fz, cell_id, vx, vy, vz, weight }, 8 elements of T (32 B float / 64 B double).
//
// Positions (reading R22; they are not in the paper): a second Philox4x32-10 block of the same particle with
// counter (lo32 g, hi32 g, 0, 2).  Counter word 3 enters round 1 only through the xor with round key k1[0], so the
// block is the velocity block's code with k1[0] ^ 2 -- shared head, constant-addition round 1 and all.
//
// Stores.  A thread's G particles are 128 contiguous bytes, a warp's 4 KB; written lane by lane with 128-bit stores
// every instruction would touch 32 lines and fill a quarter of each.  Whole tiles instead assemble the warp's 4 KB in
// shared memory and hand it to the bulk-copy engine (cp.async.bulk shared -> global, one instruction per warp and
// group; one fence and one commit per tile), which drains it while the warp computes its next tile.
#pragma once
#include "kernels.cuh"

namespace kappagen {

constexpr int kRecElems = 8;                                          // elements of T per particle record
constexpr int kRecWarpBytes = 32 * 16 * 8;                            // 32 lanes x 128 bytes: one warp, one group
constexpr int kLoadSmemBytes = (kThreads / 32) * kGroups * kRecWarpBytes;   // a tile of every warp: 64 KB per block

__device__ __forceinline__ float pos_offset(uint32_t w, float) {      // ((w >> 9) + 1/2) / 2^23, exact in float
    return fmaf((float)(w >> 9), 0x1p-23f, 0x1p-24f);
}
__device__ __forceinline__ double pos_offset(uint32_t w, double) {    // (w + 1/2) / 2^32, exact in double
    return u32_unit(w) - (1.0 - 0x1p-33);
}
__device__ __forceinline__ float id_bits(int64_t id, float) { return __int_as_float((int)id); }
__device__ __forceinline__ double id_bits(int64_t id, double) { return __longlong_as_double((long long)id); }

// The record of one particle as 16-byte pieces: float 2 pieces, double 4.
__device__ __forceinline__ void record_pieces(float fx, float fy, float fz, float id, float vx, float vy, float vz, float w,
                                              float4 (&pc)[2]) {
    pc[0] = make_float4(fx, fy, fz, id);
    pc[1] = make_float4(vx, vy, vz, w);
}
__device__ __forceinline__ void record_pieces(double fx, double fy, double fz, double id, double vx, double vy, double vz,
                                              double w, double2 (&pc)[4]) {
    pc[0] = make_double2(fx, fy);
    pc[1] = make_double2(fz, id);
    pc[2] = make_double2(vx, vy);
    pc[3] = make_double2(vz, w);
}

// Two copies (the warp's two groups, kRecWarpBytes each, adjacent in shared memory) behind one fence, one commit.
__device__ __forceinline__ void bulk_store_warp2(void* g0, void* g1, const void* ssrc, uint32_t bytes) {
    // generic-proxy writes to shared memory made visible to the async proxy, then the bulk copies of the warp
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    __syncwarp();
    if ((threadIdx.x & 31u) == 0u) {
        const uint32_t s = (uint32_t)__cvta_generic_to_shared(ssrc);
        asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(g0), "r"(s), "r"(bytes) : "memory");
        asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(g1), "r"(s + bytes), "r"(bytes) : "memory");
        asm volatile("cp.async.bulk.commit_group;" ::: "memory");
    }
}
// The warp's buffer may be overwritten once the copies issued from it have READ it.
__device__ __forceinline__ void bulk_wait_reuse() {
    if ((threadIdx.x & 31u) == 0u) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
    __syncwarp();
}
__device__ __forceinline__ void bulk_wait_all() {
    if ((threadIdx.x & 31u) == 0u) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
    __syncwarp();
}

template <typename T> struct Piece;
template <> struct Piece<float> { using type = float4; static constexpr int per_particle = 2; };
template <> struct Piece<double> { using type = double2; static constexpr int per_particle = 4; };

// Kpos: the keys with k1[0] ^ 2 (the position block).  HASW: a per-cell weight array is given.
template <typename T, bool HASW>
__global__ void __launch_bounds__(kThreads, 2)
load_cells_kernel(int64_t n, uint32_t ppc, uint64_t magic, uint32_t magic32, uint64_t offset, const __grid_constant__ PhiloxKeys K,
                  const __grid_constant__ PhiloxKeys Kpos, const CellRec<T>* __restrict__ W, const T* __restrict__ weight,
                  int64_t cell_base, T* __restrict__ out) {
    extern __shared__ __align__(128) unsigned char stage_raw[];
    using P = typename Piece<T>::type;
    constexpr int G = 16 / sizeof(T);
    constexpr int PP = Piece<T>::per_particle;                        // G * PP = 8 pieces = 128 bytes per thread and group
    constexpr int64_t kTile = (int64_t)kThreads * G * kGroups;
    const bool whole_groups = ppc % (uint32_t)G == 0u;
    math_tables_init<T>();
    const unsigned warp = threadIdx.x >> 5, lane = threadIdx.x & 31u;
    P* my_stage = reinterpret_cast<P*>(stage_raw + (size_t)warp * kGroups * kRecWarpBytes);   // [group][32 lanes][8 pieces]
    const int64_t stride = (int64_t)gridDim.x * kTile;
    int64_t base = (int64_t)blockIdx.x * kTile;
    int64_t cell_first = base < n ? cell_of(base, ppc, magic) : 0;
    uint32_t rem_first = (uint32_t)(base - cell_first * (int64_t)ppc);
    const int64_t dcell = cell_of(stride, ppc, magic);
    const uint32_t drem = (uint32_t)(stride - dcell * (int64_t)ppc);
    for (; base < n; base += stride) {
        const uint64_t g_tile = offset + (uint64_t)base;
        if (whole_groups && base + kTile <= n && tile_in_one_block(g_tile, kTile)) {
            const PhiloxHead H = philox_head((uint32_t)(g_tile >> 32), K);
            const uint32_t lo_first = (uint32_t)g_tile + threadIdx.x * (uint32_t)G;
            const uint64_t q_first = (uint64_t)kPhiloxM0 * (uint64_t)lo_first;
            // the records of both groups first: their loads fly during the first group's Philox rounds (the bulk-copy
            // fences below are barriers for the compiler, it would not hoist them itself)
            int64_t cells[kGroups];
            RecRegs<T> recs[kGroups];
            T wgts[kGroups];
#pragma unroll
            for (int j = 0; j < kGroups; ++j) {
                cells[j] = cell_first + (int64_t)cells_ahead(rem_first + (uint32_t)(j * (kThreads * G)) + threadIdx.x * (uint32_t)G, ppc, magic32);
                load_rec(W, cells[j], recs[j]);
                wgts[j] = HASW ? __ldg(weight + cells[j]) : T(1);
            }
#pragma unroll
            for (int j = 0; j < kGroups; ++j) {
                const int64_t cell = cells[j];
                const RecRegs<T>& rec = recs[j];
                const T wgt = wgts[j];
                uint32_t w0[G], w1[G], w2[G], w3[G], p0[G], p1[G], p2[G], p3[G];
                tile_group_words<T, G, kThreads>(lo_first, q_first, j, H, K, w0, w1, w2, w3);
                tile_group_words<T, G, kThreads>(lo_first, q_first, j, H, Kpos, p0, p1, p2, p3);
                T ox[G], oy[G], oz[G];
                rec_velocities(w0, w1, w2, rec, ox, oy, oz);
                const T id = id_bits(cell_base + cell, T(0));
                if (j == 0) bulk_wait_reuse();                        // the previous tile's copies have read the buffer
                P* dst = my_stage + (size_t)j * (kRecWarpBytes / sizeof(P)) + lane * 8u;
#pragma unroll
                for (int e = 0; e < G; ++e) {
                    P pc[PP];
                    record_pieces(pos_offset(p0[e], T(0)), pos_offset(p1[e], T(0)), pos_offset(p2[e], T(0)), id, ox[e], oy[e],
                                  oz[e], wgt, pc);
#pragma unroll
                    for (int u = 0; u < PP; ++u) dst[e * PP + u] = pc[u];
                }
            }
            // one fence and one commit per tile: both groups' 4 KB leave together
            const int64_t i_warp = base + (int64_t)(warp * 32u) * G;
            bulk_store_warp2(out + i_warp * kRecElems, out + (i_warp + (int64_t)kThreads * G) * kRecElems, my_stage,
                             (uint32_t)kRecWarpBytes);
        } else {
            // ragged tail, tile across a 2^32 counter boundary, ppc not a multiple of G: particle by particle, the
            // scalar chain (bit-identical to the packed one), plain 128-bit stores
#pragma unroll 1
            for (int j = 0; j < kGroups; ++j) {
#pragma unroll 1
                for (int e = 0; e < G; ++e) {
                    const int64_t i = base + (int64_t)j * (kThreads * G) + (int64_t)threadIdx.x * G + e;
                    if (i < n) {
                        const int64_t cell = cell_of(i, ppc, magic);
                        const CellRec<T> R = W[cell];
                        uint32_t w0, w1, w2, p0, p1, p2;
                        particle_words(offset + (uint64_t)i, K, w0, w1, w2);
                        particle_words(offset + (uint64_t)i, Kpos, p0, p1, p2);
                        T x, y, z;
                        rec_velocity(w0, w1, w2, R, x, y, z);
                        P pc[PP];
                        record_pieces(pos_offset(p0, T(0)), pos_offset(p1, T(0)), pos_offset(p2, T(0)), id_bits(cell_base + cell, T(0)),
                                      x, y, z, HASW ? weight[cell] : T(1), pc);
                        P* g = reinterpret_cast<P*>(out + i * kRecElems);
#pragma unroll
                        for (int u = 0; u < PP; ++u) g[u] = pc[u];
                    }
                }
            }
        }
        cell_first += dcell;
        rem_first += drem;
        if (rem_first >= ppc) {
            rem_first -= ppc;
            ++cell_first;
        }
    }
    bulk_wait_all();                                                  // shared memory must outlive the copies that read it
}

}  // namespace kappagen
