// kappagen_oracle.cpp -- CPU ORACLE for arXiv 2602.05606 (Zenitani & Umeda), Table I generator.
//
// THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
// bench.py's cpu_baseline / --impl reference legs may build, load or call it.  It shares no
// code, header, table or constant generator with the CUDA path (paper_2602_05606_b200/csrc).
//
// What it is: a plain, slow, single-threaded C++17 implementation, in x87 `long double`
// (64-bit significand, eps = 5.4e-20), of what the hot path computes per particle:
//
//   S1  Philox4x32-10 words (w0,w1,w2,w3)      -- RNG fixed by BASELINE.json north_star;
//                                                 the paper says only "generate U1,U2,U3 ~
//                                                 Uniform(0,1)" (Table I line 5)
//   S2  U_j = (w_{j-1} + 1/2) / 2^32            -- open interval
//   S0  kappa*, a, c, b                         -- Table I lines 1-4,
//                                                 Eqs. (16),(13),(20),(17)
//   S3  L = -kappa* {(1-U1^{2/3})^{-1/kappa*} - 1}            -- Eq. (25)
//   S4  V = theta sqrt(x), x the positive root of
//       b x^2 + (a + cL) x + L = 0                            -- Eq. (22)->(24)
//   S5  vx = V(2U2-1); vy = 2V sqrt(U2(1-U2)) cos(2 pi U3);
//       vz = 2V sqrt(U2(1-U2)) sin(2 pi U3)                   -- Table I lines 8-10
//
// Two evaluators of that same real number are provided:
//   * oracle_sample_literal : Table I typed in verbatim, in the paper's order and notation
//     (powl, 1-p, ...-1, the -2L/((a+cL)+sqrt(...)) form).  Checkable against the paper by
//     eye.  It loses digits by cancellation at both ends of U1 (DESIGN.md "Readings" R7).
//   * oracle_sample         : the same quantities, same order of steps, but each step written
//     in its cancellation-free form (1-U from the integer complement, log1p/expm1, the root
//     of the quadratic taken from whichever of the two printed forms of Eq. (24) does not
//     cancel, the azimuth reduced to |angle| <= pi/4 on the integer word).  This is the
//     function GPU parity is measured against.
// tests/test_oracle_*.py pin both to the paper (Philox KATs, printed parameter facts, round
// trip through Eq. (A11), exact CDF Eq. (3), Eq. (5), 50-digit mpmath evaluation of Table I);
// the literal evaluator (x_literal, dir_literal, oracle_sample_literal) in tests/test_oracle_literal.py
// (Table I lines 5-10 typed once more in 50-digit mpmath; agreement with oracle_sample in the bulk;
// polar axis and the (cos, sin) assignment from the top bits of the words); oracle_positions in
// tests/test_oracle_positions.py (an independent pure-Python Philox checked against the published vectors, the
// distinctness of the position block, exact representability, uniformity and independence of the velocity stream).
//
// Parity status: every exported function below is pinned; none is "parity unpinned".

#include <cfloat>
#include <cmath>
#include <cstdint>

static_assert(LDBL_MANT_DIG == 64, "oracle needs x87 80-bit long double");

typedef long double ld;

namespace {

// ---------------------------------------------------------------- S1: Philox4x32-10
// Salmon et al. 2011 "Parallel random numbers: as easy as 1, 2, 3": multipliers M0, M1 and
// Weyl key increments W0, W1; 10 rounds; key bumped between rounds.
const uint32_t PHILOX_M0 = 0xD2511F53u;
const uint32_t PHILOX_M1 = 0xCD9E8D57u;
const uint32_t PHILOX_W0 = 0x9E3779B9u;
const uint32_t PHILOX_W1 = 0xBB67AE85u;

void philox4x32_10(const uint32_t ctr_in[4], const uint32_t key_in[2], uint32_t out[4]) {
    uint32_t c0 = ctr_in[0], c1 = ctr_in[1], c2 = ctr_in[2], c3 = ctr_in[3];
    uint32_t k0 = key_in[0], k1 = key_in[1];
    for (int round = 0; round < 10; ++round) {
        if (round > 0) {
            k0 += PHILOX_W0;
            k1 += PHILOX_W1;
        }
        const uint64_t p0 = (uint64_t)PHILOX_M0 * (uint64_t)c0;
        const uint64_t p1 = (uint64_t)PHILOX_M1 * (uint64_t)c2;
        const uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
        const uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
        const uint32_t n0 = hi1 ^ c1 ^ k0;
        const uint32_t n1 = lo1;
        const uint32_t n2 = hi0 ^ c3 ^ k1;
        const uint32_t n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// Particle g = offset + i uses counter (lo32(g), hi32(g), 0, 0) and key (lo32(seed), hi32(seed))
// (reading R6).
void particle_words(uint64_t seed, uint64_t g, uint32_t w[4]) {
    const uint32_t ctr[4] = {(uint32_t)(g & 0xffffffffu), (uint32_t)(g >> 32), 0u, 0u};
    const uint32_t key[2] = {(uint32_t)(seed & 0xffffffffu), (uint32_t)(seed >> 32)};
    philox4x32_10(ctr, key, w);
}

// ---------------------------------------------------------------- S0: parameters
struct Params {
    ld kappa, kstar, a, b, c;
};

// Table I lines 1-4.  B(3/2,kappa*) through the gamma function as PAPER.md:250
// allows: B(p,q) = Gamma(p) Gamma(q) / Gamma(p+q).
Params params_of(ld kappa) {
    Params P;
    P.kappa = kappa;
    P.kstar = kappa - 0.5L;                                              // Eq. (16)
    const ld B = expl(lgammal(1.5L) + lgammal(P.kstar) - lgammal(P.kstar + 1.5L));
    P.a = (1.0L / kappa) * powl(2.0L / (3.0L * B), 2.0L / 3.0L);         // Eq. (13)
    P.c = (0.123L * kappa * kappa - 1.12L * kappa + 2.56L) /
          (kappa * kappa - 7.89L * kappa + 15.6L);                       // Eq. (20)
    P.b = powl(P.kstar * 1.5L * B, 1.0L / P.kstar) * (P.kstar / kappa) * P.c;  // Eq. (17) times c
    return P;
}

const ld TWO32 = 4294967296.0L;
const ld TWO31 = 2147483648.0L;
const ld TWO30 = 1073741824.0L;
const ld PI_L = 3.14159265358979323846264338327950288L;
const ld LN2_L = 0.693147180559945309417232121458176568L;

// ---------------------------------------------------------------- S2-S4: speed, literal
// Table I lines 6-7 exactly as printed; returns x = (V/theta)^2.
ld x_literal(uint32_t w0, const Params& P) {
    const ld U1 = ((ld)w0 + 0.5L) / TWO32;
    const ld L = -P.kstar * (powl(1.0L - powl(U1, 2.0L / 3.0L), -1.0L / P.kstar) - 1.0L);
    const ld A = P.a + P.c * L;
    return -2.0L * L / (A + sqrtl(A * A - 4.0L * P.b * L));
}

// ---------------------------------------------------------------- S2-S4: speed, cancellation-free
// Same steps; each written so that nothing cancels (readings R3, R7).
ld L_of_uniform(ld U1, ld t1, bool upper_half, const Params& P) {
    const ld lnU1 = upper_half ? log1pl(-t1) : logl(U1);
    const ld E = (2.0L / 3.0L) * lnU1;                                    // ln U1^{2/3} <= 0
    const ld lnS = (E > -LN2_L) ? logl(-expm1l(E)) : log1pl(-expl(E));   // ln(1 - U1^{2/3})
    const ld M = -lnS / P.kstar;                                          // >= 0
    return -P.kstar * expm1l(M);                                          // Eq. (25); L < 0
}

ld L_stable(uint32_t w0, const Params& P) {
    const ld U1 = ((ld)w0 + 0.5L) / TWO32;
    const ld t1 = ((ld)(uint32_t)(~w0) + 0.5L) / TWO32;                  // 1 - U1, exact
    return L_of_uniform(U1, t1, w0 >= 0x80000000u, P);
}

ld x_of_L(ld L, const Params& P) {
    const ld A = P.a + P.c * L;
    const ld D = sqrtl(A * A - 4.0L * P.b * L);                           // -4bL > 0 so D > |A|
    // Eq. (24) prints both forms of the positive root; use the one that adds.
    return (A >= 0.0L) ? (-2.0L * L / (A + D)) : ((D - A) / (2.0L * P.b));
}

ld x_stable(uint32_t w0, const Params& P) { return x_of_L(L_stable(w0, P), P); }

// 64-bit U1 (reading R20): U1 = (W + 1/2)/2^64 with W = w0 2^32 + w3,
// the word the 32-bit generator discards.  1 - U1 = (~W + 1/2)/2^64 from the integer complement again.
// W + 1/2 needs 65 bits when W >= 2^63; there the branch uses t1 (exact for the small ~W that matter), and
// the other way round, so each branch sees its own argument to 2^-64 relative.
ld L_stable64(uint32_t w0, uint32_t w3, const Params& P) {
    const uint64_t W = ((uint64_t)w0 << 32) | (uint64_t)w3;
    const ld TWO64 = TWO32 * TWO32;
    const ld U1 = ((ld)W + 0.5L) / TWO64;
    const ld t1 = ((ld)(~W) + 0.5L) / TWO64;
    return L_of_uniform(U1, t1, (W >> 63) != 0, P);
}
ld x_stable64(uint32_t w0, uint32_t w3, const Params& P) { return x_of_L(L_stable64(w0, w3, P), P); }

// ---------------------------------------------------------------- S5: direction
struct Dir {
    ld mu, sth, cphi, sphi;
};

// Table I lines 8-10 as printed.
Dir dir_literal(uint32_t w1, uint32_t w2) {
    const ld U2 = ((ld)w1 + 0.5L) / TWO32;
    const ld U3 = ((ld)w2 + 0.5L) / TWO32;
    Dir d;
    d.mu = 2.0L * U2 - 1.0L;
    d.sth = 2.0L * sqrtl(U2 * (1.0L - U2));
    d.cphi = cosl(2.0L * PI_L * U3);
    d.sphi = sinl(2.0L * PI_L * U3);
    return d;
}

// Same quantities with 1-U2 and 2U2-1 taken from the integer and the azimuth reduced by
// quarter turns on the integer, so cos/sin are evaluated only on |angle| <= pi/4.
Dir dir_stable(uint32_t w1, uint32_t w2) {
    Dir d;
    const ld U2 = ((ld)w1 + 0.5L) / TWO32;
    const ld t2 = ((ld)(uint32_t)(~w1) + 0.5L) / TWO32;
    d.mu = ((ld)(int32_t)(w1 ^ 0x80000000u) + 0.5L) / TWO31;
    d.sth = 2.0L * sqrtl(U2 * t2);
    // 2 pi U3 = (pi/2) * (w2 + 1/2) / 2^30 quarter turns.  k = nearest quarter turn, rem in (-1/2, 1/2).
    const uint64_t k = ((uint64_t)w2 + 0x20000000ull) >> 30;              // 0..4
    const ld rem = ((ld)((int64_t)w2 - (int64_t)(k << 30)) + 0.5L) / TWO30;
    const ld ang = 0.5L * PI_L * rem;
    const ld cr = cosl(ang), sr = sinl(ang);
    switch (k & 3u) {
        case 0: d.cphi = cr;  d.sphi = sr;  break;
        case 1: d.cphi = -sr; d.sphi = cr;  break;
        case 2: d.cphi = -cr; d.sphi = -sr; break;
        default: d.cphi = sr; d.sphi = -cr; break;
    }
    return d;
}

bool params_ok(double kappa, double theta) {
    return std::isfinite(kappa) && std::isfinite(theta) && kappa > 1.5 && theta >= 0.0;
}

}  // namespace

extern "C" {

// Philox4x32-10 of one (counter, key); pinned by the published known-answer vectors.
void oracle_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
    philox4x32_10(ctr, key, out);
}

// Words the generator uses for particles offset .. offset+n-1 (w3 is drawn and discarded).
void oracle_words(int64_t n, uint64_t seed, uint64_t offset, uint32_t* w0, uint32_t* w1, uint32_t* w2) {
    for (int64_t i = 0; i < n; ++i) {
        uint32_t w[4];
        particle_words(seed, offset + (uint64_t)i, w);
        w0[i] = w[0]; w1[i] = w[1]; w2[i] = w[2];
    }
}

// S0, rounded once to double.  Returns 0, or -1 if kappa is outside the domain kappa > 3/2.
int oracle_params(double kappa, double* kstar, double* a, double* b, double* c) {
    if (!params_ok(kappa, 1.0)) return -1;
    const Params P = params_of((ld)kappa);
    *kstar = (double)P.kstar; *a = (double)P.a; *b = (double)P.b; *c = (double)P.c;
    return 0;
}

// x = (V/theta)^2 as a function of the first word only (S2-S4), stable and literal forms,
// and L of Eq. (25) (stable form).
int oracle_x_of_w0(int64_t n, const uint32_t* w0, double kappa, double* x) {
    if (!params_ok(kappa, 1.0)) return -1;
    const Params P = params_of((ld)kappa);
    for (int64_t i = 0; i < n; ++i) x[i] = (double)x_stable(w0[i], P);
    return 0;
}
int oracle_x_of_w0_literal(int64_t n, const uint32_t* w0, double kappa, double* x) {
    if (!params_ok(kappa, 1.0)) return -1;
    const Params P = params_of((ld)kappa);
    for (int64_t i = 0; i < n; ++i) x[i] = (double)x_literal(w0[i], P);
    return 0;
}
int oracle_L_of_w0(int64_t n, const uint32_t* w0, double kappa, double* L) {
    if (!params_ok(kappa, 1.0)) return -1;
    const Params P = params_of((ld)kappa);
    for (int64_t i = 0; i < n; ++i) L[i] = (double)L_stable(w0[i], P);
    return 0;
}

// The same with the 64-bit U1 built from (w0, w3).
int oracle_x_of_w0w3(int64_t n, const uint32_t* w0, const uint32_t* w3, double kappa, double* x) {
    if (!params_ok(kappa, 1.0)) return -1;
    const Params P = params_of((ld)kappa);
    for (int64_t i = 0; i < n; ++i) x[i] = (double)x_stable64(w0[i], w3[i], P);
    return 0;
}

// Direction cosines (mu, sth*cos phi, sth*sin phi) from words (w1, w2), stable form (S5).
void oracle_direction(int64_t n, const uint32_t* w1, const uint32_t* w2, double* nx, double* ny, double* nz) {
    for (int64_t i = 0; i < n; ++i) {
        const Dir d = dir_stable(w1[i], w2[i]);
        nx[i] = (double)d.mu; ny[i] = (double)(d.sth * d.cphi); nz[i] = (double)(d.sth * d.sphi);
    }
}

// Velocities from given words (so tests can drive chosen words through S2-S6).
int oracle_velocity_of_words(int64_t n, const uint32_t* w0, const uint32_t* w1, const uint32_t* w2,
                             double kappa, double theta, double* vx, double* vy, double* vz) {
    if (!params_ok(kappa, theta)) return -1;
    const Params P = params_of((ld)kappa);
    for (int64_t i = 0; i < n; ++i) {
        const ld V = (ld)theta * sqrtl(x_stable(w0[i], P));
        const Dir d = dir_stable(w1[i], w2[i]);
        vx[i] = (double)(V * d.mu);
        vy[i] = (double)(V * d.sth * d.cphi);
        vz[i] = (double)(V * d.sth * d.sphi);
    }
    return 0;
}

// The generator: particle i (0 <= i < n) is a pure function of (seed, offset+i, kappa, theta).
int oracle_sample(int64_t n, double kappa, double theta, uint64_t seed, uint64_t offset,
                  double* vx, double* vy, double* vz) {
    if (n < 0 || !params_ok(kappa, theta)) return -1;
    const Params P = params_of((ld)kappa);
    for (int64_t i = 0; i < n; ++i) {
        uint32_t w[4];
        particle_words(seed, offset + (uint64_t)i, w);
        const ld V = (ld)theta * sqrtl(x_stable(w[0], P));
        const Dir d = dir_stable(w[1], w[2]);
        vx[i] = (double)(V * d.mu);
        vy[i] = (double)(V * d.sth * d.cphi);
        vz[i] = (double)(V * d.sth * d.sphi);
    }
    return 0;
}

// The generator with the 64-bit U1 (flag KAPPAGEN_U1_64 of the library); w3[] (optional) receives the fourth word.
int oracle_sample_u64(int64_t n, double kappa, double theta, uint64_t seed, uint64_t offset,
                      double* vx, double* vy, double* vz, uint32_t* w3_out) {
    if (n < 0 || !params_ok(kappa, theta)) return -1;
    const Params P = params_of((ld)kappa);
    for (int64_t i = 0; i < n; ++i) {
        uint32_t w[4];
        particle_words(seed, offset + (uint64_t)i, w);
        const ld V = (ld)theta * sqrtl(x_stable64(w[0], w[3], P));
        const Dir d = dir_stable(w[1], w[2]);
        vx[i] = (double)(V * d.mu);
        vy[i] = (double)(V * d.sth * d.cphi);
        vz[i] = (double)(V * d.sth * d.sphi);
        if (w3_out) w3_out[i] = w[3];
    }
    return 0;
}
int oracle_velocity_of_words_u64(int64_t n, const uint32_t* w0, const uint32_t* w1, const uint32_t* w2, const uint32_t* w3,
                                 double kappa, double theta, double* vx, double* vy, double* vz) {
    if (!params_ok(kappa, theta)) return -1;
    const Params P = params_of((ld)kappa);
    for (int64_t i = 0; i < n; ++i) {
        const ld V = (ld)theta * sqrtl(x_stable64(w0[i], w3[i], P));
        const Dir d = dir_stable(w1[i], w2[i]);
        vx[i] = (double)(V * d.mu);
        vy[i] = (double)(V * d.sth * d.cphi);
        vz[i] = (double)(V * d.sth * d.sphi);
    }
    return 0;
}

// Speed over theta, sqrt(x), of each particle (S1-S4 only): the quantity paper test 2 histograms with bins
// of width Delta v = 1/5.  u64 != 0: the 64-bit U1 of reading R20.
int oracle_speed_over_theta(int64_t n, double kappa, uint64_t seed, uint64_t offset, int u64, double* s) {
    if (n < 0 || !params_ok(kappa, 1.0)) return -1;
    const Params P = params_of((ld)kappa);
    for (int64_t i = 0; i < n; ++i) {
        uint32_t w[4];
        particle_words(seed, offset + (uint64_t)i, w);
        s[i] = (double)sqrtl(u64 ? x_stable64(w[0], w[3], P) : x_stable(w[0], P));
    }
    return 0;
}

// Table I typed in verbatim (see header).  Same interface as oracle_sample.
int oracle_sample_literal(int64_t n, double kappa, double theta, uint64_t seed, uint64_t offset,
                          double* vx, double* vy, double* vz) {
    if (n < 0 || !params_ok(kappa, theta)) return -1;
    const Params P = params_of((ld)kappa);
    for (int64_t i = 0; i < n; ++i) {
        uint32_t w[4];
        particle_words(seed, offset + (uint64_t)i, w);
        const ld V = (ld)theta * sqrtl(x_literal(w[0], P));
        const Dir d = dir_literal(w[1], w[2]);
        vx[i] = (double)(V * d.mu);
        vy[i] = (double)(V * d.sth * d.cphi);
        vz[i] = (double)(V * d.sth * d.sphi);
    }
    return 0;
}

// Positions of the PIC particle record (kappagen_load_cells; reading R22 -- they are not in the paper):
// the offset of particle g inside its cell, in units of the cell size, from a SECOND Philox block of the same
// particle, counter (lo32 g, hi32 g, 0, 2), same key; words 0,1,2 -> x,y,z as midpoint uniforms of `bits` bits,
// ((w >> (32 - bits)) + 1/2) / 2^bits: bits = 23 is what a float holds exactly, bits = 32 a double.
int oracle_positions(int64_t n, uint64_t seed, uint64_t offset, int bits, double* fx, double* fy, double* fz) {
    if (n < 0 || bits < 1 || bits > 32) return -1;
    const uint32_t key[2] = {(uint32_t)(seed & 0xffffffffu), (uint32_t)(seed >> 32)};
    double* f[3] = {fx, fy, fz};
    for (int64_t i = 0; i < n; ++i) {
        const uint64_t g = offset + (uint64_t)i;
        const uint32_t ctr[4] = {(uint32_t)(g & 0xffffffffu), (uint32_t)(g >> 32), 0u, 2u};
        uint32_t w[4];
        philox4x32_10(ctr, key, w);
        for (int q = 0; q < 3; ++q)
            f[q][i] = (double)(((ld)(w[q] >> (32 - bits)) + 0.5L) / ldexpl(1.0L, bits));
    }
    return 0;
}

// PIC-style, cell-major: particle g = cell*ppc + j uses counter offset+g and its cell's
// (kappa, theta); the cell's drift is added last (reading R11).  drift == NULL: none;
// drift_stride == 0: one shared (dx,dy,dz); drift_stride == 1: [ncell][3].  A cell whose kappa
// or theta is outside the domain yields NaN for all its particles.  tx,ty,tz (optional, may be
// NULL) receive the thermal part without drift.
int oracle_sample_cells(int64_t ncell, int32_t ppc, const double* kappa, const double* theta,
                        const double* drift, int64_t drift_stride, uint64_t seed, uint64_t offset,
                        double* vx, double* vy, double* vz, double* tx, double* ty, double* tz) {
    if (ncell < 0 || ppc < 0) return -1;
    for (int64_t cell = 0; cell < ncell; ++cell) {
        const bool ok = params_ok(kappa[cell], theta[cell]);
        Params P = {};
        if (ok) P = params_of((ld)kappa[cell]);
        ld d3[3] = {0.0L, 0.0L, 0.0L};
        if (drift) for (int q = 0; q < 3; ++q) d3[q] = (ld)drift[3 * cell * drift_stride + q];
        for (int32_t j = 0; j < ppc; ++j) {
            const int64_t i = cell * (int64_t)ppc + j;
            ld t3[3];
            if (ok) {
                uint32_t w[4];
                particle_words(seed, offset + (uint64_t)i, w);
                const ld V = (ld)theta[cell] * sqrtl(x_stable(w[0], P));
                const Dir d = dir_stable(w[1], w[2]);
                t3[0] = V * d.mu; t3[1] = V * d.sth * d.cphi; t3[2] = V * d.sth * d.sphi;
            } else {
                t3[0] = t3[1] = t3[2] = (ld)NAN;
            }
            vx[i] = (double)(t3[0] + d3[0]); vy[i] = (double)(t3[1] + d3[1]); vz[i] = (double)(t3[2] + d3[2]);
            if (tx) { tx[i] = (double)t3[0]; ty[i] = (double)t3[1]; tz[i] = (double)t3[2]; }
        }
    }
    return 0;
}

// Per-cell velocity moments of the same particles (the fused loader of SURVEY.md section 8(f) f1: what a
// PIC code computes right after loading -- momentum and the energy density of Eq. (5)):
//   mom[4*cell + 0..2] = sum_j (vx, vy, vz),   mom[4*cell + 3] = sum_j (vx^2 + vy^2 + vz^2)
// over the cell's ppc particles, drift included, accumulated in long double and rounded once.  abs1
// (optional) receives sum_j (|vx| + |vy| + |vz|) per cell, the scale of the admissible rounding error.
int oracle_cells_moments(int64_t ncell, int32_t ppc, const double* kappa, const double* theta,
                         const double* drift, int64_t drift_stride, uint64_t seed, uint64_t offset,
                         double* mom, double* abs1) {
    if (ncell < 0 || ppc < 0) return -1;
    for (int64_t cell = 0; cell < ncell; ++cell) {
        const bool ok = params_ok(kappa[cell], theta[cell]);
        Params P = {};
        if (ok) P = params_of((ld)kappa[cell]);
        ld d3[3] = {0.0L, 0.0L, 0.0L};
        if (drift) for (int q = 0; q < 3; ++q) d3[q] = (ld)drift[3 * cell * drift_stride + q];
        ld s[4] = {0.0L, 0.0L, 0.0L, 0.0L}, a1 = 0.0L;
        for (int32_t j = 0; j < ppc; ++j) {
            const int64_t i = cell * (int64_t)ppc + j;
            if (!ok) { s[0] = s[1] = s[2] = s[3] = a1 = (ld)NAN; break; }
            uint32_t w[4];
            particle_words(seed, offset + (uint64_t)i, w);
            const ld V = (ld)theta[cell] * sqrtl(x_stable(w[0], P));
            const Dir d = dir_stable(w[1], w[2]);
            const ld v3[3] = {V * d.mu + d3[0], V * d.sth * d.cphi + d3[1], V * d.sth * d.sphi + d3[2]};
            for (int q = 0; q < 3; ++q) { s[q] += v3[q]; s[3] += v3[q] * v3[q]; a1 += fabsl(v3[q]); }
        }
        for (int q = 0; q < 4; ++q) mom[4 * cell + q] = (double)s[q];
        if (abs1) abs1[cell] = (double)a1;
    }
    return 0;
}

int oracle_version(void) { return 1; }

}  // extern "C"
