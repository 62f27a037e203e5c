/* kappagen.h -- C ABI of libkappagen: the hot path of arXiv 2602.05606 (Zenitani & Umeda,
 * "An approximate Kappa generator for particle simulations") for NVIDIA B200 (sm_100a).
 *
 * The operation (paper Table I; Eqs. (22)-(25)).  For the
 * particle with global index g = offset + i:
 *   (w0,w1,w2,w3) = Philox4x32-10(counter = (lo32 g, hi32 g, 0, 0), key = (lo32 seed, hi32 seed))
 *   U1,U2,U3 = (w0+1/2)/2^32, (w1+1/2)/2^32, (w2+1/2)/2^32        "generate U1,U2,U3 ~ Uniform(0,1)"
 *   L  = -kappa* {(1 - U1^(2/3))^(-1/kappa*) - 1}                  Eq. (25)
 *   V  = theta sqrt(x),  x = positive root of b x^2 + (a + cL) x + L = 0      Eq. (24)
 *   vx = V (2U2-1);  vy = 2V sqrt(U2(1-U2)) cos(2 pi U3);  vz = 2V sqrt(U2(1-U2)) sin(2 pi U3)
 * with kappa* = kappa - 1/2, a, b, c from Table I lines 1-4 (Eqs. (16),(13),(17),(20)).
 * The output is a pure function of the arguments: independent of launch shape, of chunking
 * through `offset`, and of how many GPUs share the index range.
 *
 * Conventions for every call:
 *  - "device" pointers are CUDA device memory owned by the caller (e.g. torch tensor.data_ptr());
 *    "host" pointers are ordinary host memory.  The library keeps no state and no RNG state,
 *    and allocates nothing that outlives a call (kappagen_sample_cells_static keeps its scratch in
 *    a fixed array inside the library image instead: see there).
 *  - `stream` is a cudaStream_t passed as void* (NULL = legacy default stream).  Device-buffer
 *    calls enqueue on `stream` and return without synchronising; argument errors are returned
 *    at once, asynchronous CUDA errors surface at the caller's next synchronisation.  They
 *    allocate nothing and only launch kernels, so they may be recorded by stream capture into a
 *    CUDA graph (kappagen_sample_host may not: it allocates staging buffers and synchronises).
 *  - Output planes are SoA: vx[i], vy[i], vz[i]; element type float (KAPPAGEN_F32) or double
 *    (KAPPAGEN_F64).  Planes must be aligned to the element size; 16-byte aligned planes take
 *    the vector-store path, others a scalar-store path that writes the same values.
 *  - Return value: KAPPAGEN_OK (0) or a negative kappagen_status.  kappagen_last_error()
 *    returns a thread-local, human-readable description of the last failure.
 *  - n == 0 (or ncell == 0, ppc == 0) is KAPPAGEN_OK and launches nothing.
 */
#ifndef KAPPAGEN_H_
#define KAPPAGEN_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum { KAPPAGEN_F32 = 0, KAPPAGEN_F64 = 1 } kappagen_dtype;

typedef enum {
    KAPPAGEN_OK = 0,
    KAPPAGEN_EINVAL = -1,     /* kappa <= 3/2, theta < 0, non-finite, n < 0, bad dtype, bad stride */
    KAPPAGEN_ENULL = -2,      /* a required pointer is NULL while there is work to do               */
    KAPPAGEN_EALIGN = -3,     /* a plane is not aligned to its element size                         */
    KAPPAGEN_EWORKSPACE = -4, /* workspace NULL or smaller than kappagen_cells_workspace_bytes()    */
    KAPPAGEN_ECUDA = -5       /* a CUDA runtime call or the launch failed                           */
} kappagen_status;

/* Table I lines 5-10 with uniform parameters (S1-S6 of DESIGN.md).
 * n >= 0 particles; kappa > 3/2, theta >= 0 (theta == 0 writes zeros); particle i
 * uses counter offset + i (64-bit, wraps).  vx, vy, vz: device, [n] elements of `dtype`. */
int kappagen_sample(int64_t n, double kappa, double theta, uint64_t seed, uint64_t offset,
                    int dtype, void* vx, void* vy, void* vz, void* stream);

/* kappagen_sample with options.  flags = 0 is kappagen_sample.
 *  KAPPAGEN_U1_64: U1 takes 64 bits, U1 = (w0 2^32 + w3 + 1/2)/2^64, from the first and the otherwise
 *  discarded fourth word of the particle's Philox block (reading R20).  The paper fixes neither
 *  the generator nor its width ("generate U1 ~ Uniform(0,1)", Table I line 5); with 32 bits
 *  the largest speed is x_max = G^-1(1 - 2^-33) -- v/theta = 5.0e4 at kappa = 1.6, where the tail beyond
 *  carries 12 % of <v^2> -- and 64 bits move it to G^-1(1 - 2^-65), 2^(32/kappa*) further in v^2, at no
 *  extra random-number cost.  U2, U3 and the Philox stream are unchanged; a different (finer) generator,
 *  not bit-compatible with flags = 0.  Unknown flag bits: KAPPAGEN_EINVAL. */
enum { KAPPAGEN_U1_64 = 1 };
int kappagen_sample_flags(int64_t n, double kappa, double theta, uint64_t seed, uint64_t offset,
                          int dtype, uint32_t flags, void* vx, void* vy, void* vz, void* stream);

/* Same generator with PIC-style per-cell parameters ("10^2-10^3 particles in a grid cell",
 * PAPER.md:215).  Cell-major: particle g = cell*ppc + j (0 <= j < ppc) uses counter offset + g,
 * kappa[cell], theta[cell]; the cell's drift velocity is added last, in the output type.
 *  kappa, theta : device, [ncell] elements of `dtype`.  A cell with kappa <= 3/2, theta < 0 or a
 *                 non-finite value gets NaN in all its particles (it cannot be reported synchronously).
 *  drift        : device, elements of `dtype`, or NULL (no drift).  drift_stride == 0: one shared
 *                 (dx,dy,dz) at drift[0..2]; drift_stride == 1: per cell at drift[3*cell + 0..2].
 *  workspace    : device scratch of at least kappagen_cells_workspace_bytes(ncell, dtype) bytes
 *                 (48 bytes per cell for float, 96 for double), 16-byte aligned; holds one record per cell:
 *                 the per-cell Table I lines 1-4 (computed on the device in double by a small pre-kernel
 *                 on the same stream) and the cell's drift.  Contents are unspecified after.
 *  vx, vy, vz   : device, [ncell*ppc] elements of `dtype`. */
int kappagen_sample_cells(int64_t ncell, int32_t ppc, const void* kappa, const void* theta,
                          const void* drift, int64_t drift_stride, uint64_t seed, uint64_t offset,
                          int dtype, void* vx, void* vy, void* vz,
                          void* workspace, size_t workspace_bytes, void* stream);
size_t kappagen_cells_workspace_bytes(int64_t ncell, int dtype);

/* kappagen_sample_cells for callers that cannot hand over a workspace because they cannot get device memory at
 * all: a particle-injection routine called every time step inside a simulation whose framework took the whole
 * GPU into its own pool at start-up and forbids cudaMalloc afterwards (it stalls every stream of the device and
 * may simply fail once the pool holds everything), or a plug-in that is given output arrays but no handle to
 * that pool.  This call allocates nothing -- no cudaMalloc, no cudaFree, no library routine that allocates --
 * and the caller passes only inputs and outputs.  The per-cell records that kappagen_sample_cells keeps in
 * `workspace` are kept instead in an array of KAPPAGEN_STATIC_SCRATCH_BYTES bytes built into the library's
 * device code.  That array costs its size on every GPU that loads libkappagen, from load until the process
 * ends, whether or not this call is ever made; hence the modest limit:
 *     ncell <= KAPPAGEN_STATIC_SCRATCH_BYTES / 48 = 65536 cells per call (float), / 96 = 32768 (double).
 * More cells: KAPPAGEN_EWORKSPACE, reported before anything touches the device, with the limit in
 * kappagen_last_error(); split the call (cells c0 .. c1-1 on their own: kappa + c0, theta + c0, the planes
 * + c0*ppc and offset + c0*ppc give the same particles) or use kappagen_sample_cells.
 *  - First call on each device: it asks the CUDA runtime where the array lives on the current device and
 *    remembers the answer (per device, thread-safe).  Make that first call with the device you mean to use
 *    current, in ordinary execution, before any stream capture is begun.  Later calls only launch kernels.
 *  - One array per GPU, shared by every call from every thread and stream.  Calls that can run on the GPU at the
 *    same time (different streams, or the same stream from two unsynchronised threads) overwrite each other's
 *    records and produce garbage: order them on one stream, or by events.  The array keeps the last call's
 *    records; this call rewrites every record it reads, so nothing has to be cleared and nothing leaks from one
 *    call into the next.
 * Values are bit-identical to kappagen_sample_cells with the same arguments; all other arguments, the NaN
 * convention for invalid cells and the other error codes are as there. */
#define KAPPAGEN_STATIC_SCRATCH_BYTES 3145728 /* 3 MiB */
int kappagen_sample_cells_static(int64_t ncell, int32_t ppc, const void* kappa, const void* theta,
                                 const void* drift, int64_t drift_stride, uint64_t seed, uint64_t offset,
                                 int dtype, void* vx, void* vy, void* vz, void* stream);

/* The two halves of kappagen_sample_cells as calls of their own: "The first four lines [of Table I] are required
 * only once".  kappagen_cells_prepare fills the workspace with the per-cell records (Table I
 * lines 1-4 and the drift); kappagen_sample_cells_prepared draws velocities from a workspace so prepared -- as often
 * as wanted, with any seed, offset and ppc, for the SAME ncell and dtype -- and writes exactly what
 * kappagen_sample_cells writes.  The workspace contents are then the caller's to keep: nothing else writes them. */
int kappagen_cells_prepare(int64_t ncell, const void* kappa, const void* theta, const void* drift,
                           int64_t drift_stride, int dtype, void* workspace, size_t workspace_bytes, void* stream);
int kappagen_sample_cells_prepared(int64_t ncell, int32_t ppc, uint64_t seed, uint64_t offset, int dtype,
                                   void* vx, void* vy, void* vz,
                                   const void* workspace, size_t workspace_bytes, void* stream);

/* The loader fused with its first consumer (the step after the path in a PIC code: "initialization stage",
 * PAPER.md:15; 10^2-10^3 particles per cell): kappagen_sample_cells that ALSO reduces, per
 * cell and inside the generating kernel, the velocity moments of the cell's ppc particles (drift included)
 *     moments[4*cell + 0..2] = sum (vx, vy, vz)        (momentum density / m)
 *     moments[4*cell + 3]    = sum (vx^2 + vy^2 + vz^2)  (2/m x the energy density whose expectation is
 *                                                        Eq. (5): 3 kappa theta^2/(2 kappa - 3) each)
 * so that the consumer never re-reads the 12/24 B per particle.
 *  moments : device, [ncell][4] elements of `dtype`, 16-byte aligned; overwritten (no need to zero it).
 *  vx,vy,vz: as in kappagen_sample_cells, or ALL THREE NULL: moments only, no velocity is written to HBM.
 * Sums are formed in `dtype`: within a thread over its 128-bit group, then across the cell's lanes by a
 * shuffle tree (fixed order, bit-reproducible) when ppc = G*2^k <= 32 G (G = 4 float / 2 double), otherwise
 * through atomicAdd (order not fixed; values agree to rounding).  Other arguments, errors and workspace as
 * kappagen_sample_cells. */
int kappagen_sample_cells_moments(int64_t ncell, int32_t ppc, const void* kappa, const void* theta,
                                  const void* drift, int64_t drift_stride, uint64_t seed, uint64_t offset,
                                  int dtype, void* vx, void* vy, void* vz, void* moments,
                                  void* workspace, size_t workspace_bytes, void* stream);

/* Host-buffer variant of kappagen_sample (the end-to-end path): vx, vy, vz are HOST arrays of
 * [n] elements (pinned memory makes the copies asynchronous and fast; pageable memory works).
 * Generates on the current device in chunks, double-buffered so that the device-to-host copy of
 * one chunk overlaps the kernel of the next; allocates its staging buffers, frees them, and
 * returns only when the host arrays are complete (synchronous).  Same values as kappagen_sample. */
int kappagen_sample_host(int64_t n, double kappa, double theta, uint64_t seed, uint64_t offset,
                         int dtype, void* vx_host, void* vy_host, void* vz_host);

/* kappagen_sample_host without any allocation or stream creation inside the call (many small batches pay
 * neither): the caller supplies the device staging workspace and the two streams the chunks alternate on.
 *  workspace : device, at least kappagen_sample_host_workspace_bytes(n, dtype) bytes, 256-byte aligned
 *              (two buffers of three chunk planes; a chunk is min(n, 2^22) particles).
 *  stream_a, stream_b : two distinct cudaStream_t (as void*); both are synchronised before the call returns,
 *              so the host arrays are complete on return.  KAPPAGEN_EINVAL if they are equal.
 * Values, chunking and errors as kappagen_sample_host. */
int kappagen_sample_host_ws(int64_t n, double kappa, double theta, uint64_t seed, uint64_t offset,
                            int dtype, void* vx_host, void* vy_host, void* vz_host,
                            void* workspace, size_t workspace_bytes, void* stream_a, void* stream_b);
size_t kappagen_sample_host_workspace_bytes(int64_t n, int dtype);

/* The PIC particle loader (second half; "initialization stage", PAPER.md:15;
 * 10^2-10^3 particles per cell): kappagen_sample_cells that writes, instead of three SoA planes,
 * one array-of-structures RECORD per particle, position and velocity together, 8 elements of `dtype`
 * (32 bytes float / 64 bytes double):
 *     { fx, fy, fz, cell_id, vx, vy, vz, weight }
 *  fx,fy,fz : the particle's offset inside its cell in units of the cell size, uniform in (0,1).  Positions are not
 *             in the paper; reading R22: they come from a SECOND Philox4x32-10 block of the same particle,
 *             counter (lo32 g, hi32 g, 0, 2), same key (the velocity block has counter word 3 = 0, the rejection
 *             baseline 1), words 0,1,2 -> x,y,z as midpoint uniforms that the element type holds exactly:
 *             float ((w >> 9) + 1/2)/2^23, double (w + 1/2)/2^32.  Bit-exact against the oracle.
 *  cell_id  : cell_base + cell as a signed integer of the element's width (int32 / int64), stored in the
 *             element's bits (reinterpret, not convert).  float: cell_base + ncell <= 2^31.
 *  vx,vy,vz : exactly kappagen_sample_cells' values (drift included).
 *  weight   : weight[cell] (device, [ncell] elements of `dtype`) or 1 when weight == NULL.
 *  records  : device, [ncell*ppc][8] elements of `dtype`, 16-byte aligned.
 * Whole tiles leave the SM as bulk asynchronous copies (cp.async.bulk) out of shared memory, 4 KB (float) per warp
 * and instruction, so that the interleaved record is still written in full lines.
 * kappa, theta, drift, drift_stride, seed, offset, workspace, errors: as kappagen_sample_cells. */
int kappagen_load_cells(int64_t ncell, int32_t ppc, const void* kappa, const void* theta,
                        const void* drift, int64_t drift_stride, const void* weight, int64_t cell_base,
                        uint64_t seed, uint64_t offset, int dtype, void* records,
                        void* workspace, size_t workspace_bytes, void* stream);

/* Measurement hook: steps S1 and S6 alone -- the three Philox words each particle consumes, written as three uint32
 * planes (12 bytes per particle) by the float sampler's tile walk with 128-bit stores, S2-S5 stripped.  Its rate is
 * the ceiling of kappagen_sample(F32) on this device (bench.py reports the sampler as a fraction of it).
 * w0,w1,w2: device, [n] uint32, 4-byte aligned (16-byte aligned planes take the vector path).  Same words as
 * kappagen_words. */
int kappagen_philox_planes(int64_t n, uint64_t seed, uint64_t offset,
                           uint32_t* w0, uint32_t* w1, uint32_t* w2, void* stream);

/* Measurement hook, the counterpart of kappagen_philox_planes: steps S2-S6 alone.  The sampler's whole-tile body for
 * `dtype` (same device functions, tile shape, launch bounds and 128-bit streaming stores) with step S1 replaced by one
 * 32-bit multiply-add per word: particle g = offset + i takes
 *     w_k = lo32(g) * M_k + A_k  (mod 2^32),   M = (0x9E3779B1, 0x85EBCA77, 0xC2B2AE3D),  A = (0x7F4A7C15, 0x165667B1, 0x27D4EB2F)
 * and writes the velocity kappagen_velocity_of_words_tile gives for (w_0, w_1, w_2) (bit-identical; flags = 0).  Its
 * rate is what the math and the stores cost when the random words are almost free: the ceiling of kappagen_sample from
 * the side opposite to kappagen_philox_planes (bench.py times both).  NOT a random-number generator.
 * vx, vy, vz: device, [n] elements of `dtype`, 16-byte aligned (KAPPAGEN_EALIGN otherwise).  kappa, theta: as
 * kappagen_sample. */
int kappagen_math_planes(int64_t n, double kappa, double theta, uint64_t offset, int dtype,
                         void* vx, void* vy, void* vz, void* stream);

/* Measurement hook: issue-rate probe behind the "alu" rooflines of DESIGN.md section 5 and profiles/r03_pipe_rates.md.
 * Runs a register-only loop of a fixed instruction mix (eight independent chains per kind: IMAD.WIDE.U32, LOP3, FFMA2,
 * MUFU.EX2, DFMA, IMAD) on every SM with `warps_per_scheduler` warps per SM sub-partition and reports the mean
 * cycles per loop iteration per warp (clock64 around the loop, averaged over blocks).
 *  mix   : 0 .. kappagen_pipe_probe_count()-1; the instruction counts of that mix come back in counts[6]
 *          (host, order as above; may be NULL).
 *  iters : loop trips (>= 1).   cycles_per_iter: host pointer, required.   Synchronous; runs on the legacy stream. */
int kappagen_pipe_probe(int mix, int warps_per_scheduler, int iters, double* cycles_per_iter, int* counts);
int kappagen_pipe_probe_count(void);

/* GPU baseline, NOT the paper's method: the "standard method" it is compared with (PAPER.md:17,
 * :180, :219-224): v = theta sqrt(kappa/(2g)) (n1,n2,n3), n_j ~ N(0,1) by Box-Muller, g ~
 * Gamma(kappa-1/2) by the Marsaglia-Tsang rejection loop.  Samples the EXACT Kappa distribution;
 * validated statistically only.  Same output contract as kappagen_sample.  trip_counters
 * (device, 2 x uint64, optional, caller zeroes it): [0] += sum over lanes of loop trips,
 * [1] += sum over warps of 32 x (trips of the slowest lane), to compare with Eq. (30). */
int kappagen_baseline_mt(int64_t n, double kappa, double theta, uint64_t seed, uint64_t offset,
                         int dtype, void* vx, void* vy, void* vz, void* stream,
                         unsigned long long* trip_counters);

/* Test hook for the "uniforms bit-exact" gate: the Philox words particle i consumes, produced by
 * the same device function the samplers call.  w0, w1, w2: device, [n] uint32 each. */
int kappagen_words(int64_t n, uint64_t seed, uint64_t offset,
                   uint32_t* w0, uint32_t* w1, uint32_t* w2, void* stream);

/* As kappagen_words, plus the fourth word (consumed only under KAPPAGEN_U1_64).  w3: device, [n] uint32. */
int kappagen_words4(int64_t n, uint64_t seed, uint64_t offset,
                    uint32_t* w0, uint32_t* w1, uint32_t* w2, uint32_t* w3, void* stream);

/* Test hook: velocities from caller-chosen words instead of Philox (same device math as
 * kappagen_sample, S2-S6), so parity can be driven through the extreme words.  w0,w1,w2: device. */
int kappagen_velocity_of_words(int64_t n, const uint32_t* w0, const uint32_t* w1, const uint32_t* w2,
                               double kappa, double theta, int dtype,
                               void* vx, void* vy, void* vz, void* stream);

/* As kappagen_velocity_of_words under KAPPAGEN_U1_64: U1 from (w0, w3). */
int kappagen_velocity_of_words_u64(int64_t n, const uint32_t* w0, const uint32_t* w1, const uint32_t* w2,
                                   const uint32_t* w3, double kappa, double theta, int dtype,
                                   void* vx, void* vy, void* vz, void* stream);

/* Test hooks through the code the samplers SHIP.  kappagen_sample runs whole tiles (256 threads x 8 particles per
 * thread inside one 2^32 block of counters) through a path of its own: one shared Philox head per tile, round 1's
 * product by constant additions (float), packed pairs of particles (float) / eight interleaved chains (double).
 *  kappagen_words_tile: the four words of particles offset .. offset+n-1 drawn by the same tile walk, the same
 *    whole-tile test and the same device functions as kappagen_sample's kernel for `dtype` (the two dtypes use
 *    different tile shapes); w0..w3: device, [n] uint32 each, all required.
 *  kappagen_velocity_of_words_tile: S2-S6 on caller-chosen words through that kernel's straight-line tile body
 *    (same instantiation, words read from memory instead of drawn); flags = 0 or KAPPAGEN_U1_64 (then w3 is
 *    required, otherwise ignored and may be NULL).  Any n; planes need only element alignment. */
int kappagen_words_tile(int64_t n, uint64_t seed, uint64_t offset, int dtype,
                        uint32_t* w0, uint32_t* w1, uint32_t* w2, uint32_t* w3, void* stream);
int kappagen_velocity_of_words_tile(int64_t n, const uint32_t* w0, const uint32_t* w1, const uint32_t* w2,
                                    const uint32_t* w3, double kappa, double theta, int dtype, uint32_t flags,
                                    void* vx, void* vy, void* vz, void* stream);

/* Paper test 2 on the device: generate n particles and count
 * their speeds |v|/theta in bins of width dv ("Delta v = 1/5") WITHOUT writing a velocity: S1-S4 only, in
 * the arithmetic of `dtype`, so 2^34 particles and more are a matter of milliseconds per 2^28.
 *   bin(i) = min(floor((|v|/theta) / dv), nbins - 1): the last bin is open-ended (reading R21).
 *   hist : device, [nbins] unsigned 64-bit counters, ACCUMULATED into (the caller zeroes them once and may
 *          call repeatedly with consecutive offsets).  theta does not enter (speeds are in units of theta).
 *   flags: 0 or KAPPAGEN_U1_64.   2 <= nbins <= 4096, dv > 0, n <= 2^40 per call. */
int kappagen_speed_histogram(int64_t n, double kappa, uint64_t seed, uint64_t offset, int dtype, uint32_t flags,
                             double dv, int32_t nbins, unsigned long long* hist, void* stream);

/* The discrete relative entropy of Eqs. (26)-(27), of a HOST copy of such a histogram:
 *   D(P||Q) = sum_i (P(i) + eps) ln((P(i) + eps)/(Q(i) + eps)),  Q(i) = hist[i]/N,  eps = 1e-10 in the paper,
 * P(i) = the baseline distribution integrated over bin i: which = KAPPAGEN_ENTROPY_VS_EXACT: the Kappa
 * distribution through its CDF Eq. (3), I_{x/(x+kappa)}(3/2, kappa-1/2); KAPPAGEN_ENTROPY_VS_APPROX: the
 * generator's own CDF G, Eq. (7).  Host arithmetic only (long double); hist and D_out are host pointers. */
enum { KAPPAGEN_ENTROPY_VS_EXACT = 0, KAPPAGEN_ENTROPY_VS_APPROX = 1 };
int kappagen_relative_entropy(const unsigned long long* hist, int32_t nbins, double dv, double kappa,
                              double eps, int which, double* D_out);

/* Table I lines 1-4 on the host in double, exactly as kappagen_sample computes them before launch.
 * All four outputs are host pointers and required. */
int kappagen_params(double kappa, double* kappa_star, double* a, double* b, double* c);

const char* kappagen_last_error(void);
int kappagen_version(void);

#ifdef __cplusplus
}
#endif
#endif /* KAPPAGEN_H_ */
