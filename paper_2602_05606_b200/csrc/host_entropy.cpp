// host_entropy.cpp -- the host half of paper test 2: from a histogram of |v|/theta
// (kappagen_speed_histogram) the discrete relative entropy of Eqs. (26)-(27),
//     D(P||Q) = sum_i (P(i) + eps) ln((P(i) + eps) / (Q(i) + eps)),   Q(i) = hist[i] / N,
// against the baseline probabilities P(i) = the Kappa distribution (Eq. 2) integrated over bin i, "with
// Delta v = 1/5", taken from its CDF, Eq. (3): F(x) = I_{x/(x+kappa)}(3/2, kappa - 1/2), x = v^2/theta^2
// -- or, for comparison, against the generator's own CDF G(x), Eq. (7)/(A11).
// Bins: [i dv, (i+1) dv) for i < nbins-1; the last bin is open-ended, so that both P and Q sum to one
// (reading R21).  Plain host arithmetic in long double; compiled by g++.
#include <cmath>
#include <cstdint>

#include "../../include/kappagen.h"
#include "host_params.hpp"

namespace {

typedef long double ld;

// The continued fraction of the incomplete beta function, DLMF 8.17.22:
//     I_x(a,b) = x^a (1-x)^b / (a B(a,b)) * 1 / (1 + d_1 / (1 + d_2 / (1 + ...))),
//     d_{2m}   =  m (b - m) x / ((a + 2m - 1)(a + 2m)),
//     d_{2m+1} = -(a + m)(a + b + m) x / ((a + 2m)(a + 2m + 1)).
ld beta_cf_term(int j, ld a, ld b, ld x) {
    const ld m = (ld)(j / 2);
    if (j % 2 == 0) return m * (b - m) * x / ((a + 2.0L * m - 1.0L) * (a + 2.0L * m));
    return -(a + m) * (a + b + m) * x / ((a + 2.0L * m) * (a + 2.0L * m + 1.0L));
}

// 1 / (1 + d_1 / (1 + d_2 / ...)) by the modified Lentz recurrence for f = b_0 + a_1/(b_1 + a_2/(b_2 + ...)) with every
// b_j = 1 and a_j = d_j (DLMF 3.10(iii) names the method): C_j = 1 + d_j / C_{j-1}, D_j = 1 / (1 + d_j D_{j-1}),
// f_j = f_{j-1} C_j D_j, from f_0 = C_0 = 1, D_0 = 0; a vanishing denominator is replaced by the smallest long double
// that still inverts.  Converges fast for x < (a + 1) / (a + b + 2), which is how betainc_both() calls it.
ld beta_cf(ld a, ld b, ld x) {
    const ld floor_ld = 1e-4000L;
    ld f = 1.0L, C = 1.0L, D = 0.0L;
    for (int j = 1; j <= 4000; ++j) {
        const ld dj = beta_cf_term(j, a, b, x);
        ld den = 1.0L + dj * D;
        if (fabsl(den) < floor_ld) den = floor_ld;
        D = 1.0L / den;
        C = 1.0L + dj / C;
        if (fabsl(C) < floor_ld) C = floor_ld;
        const ld step = C * D;
        f *= step;
        if (fabsl(step - 1.0L) < 1e-19L) break;
    }
    return 1.0L / f;
}

// Regularized incomplete beta I_x(a,b) and its complement, each computed without cancellation.
void betainc_both(ld a, ld b, ld x, ld* I, ld* Ic) {
    if (x <= 0.0L) { *I = 0.0L; *Ic = 1.0L; return; }
    if (x >= 1.0L) { *I = 1.0L; *Ic = 0.0L; return; }
    const ld lnfront = lgammal(a + b) - lgammal(a) - lgammal(b) + a * logl(x) + b * log1pl(-x);
    const ld front = expl(lnfront);
    if (x < (a + 1.0L) / (a + b + 2.0L)) {
        *I = front * beta_cf(a, b, x) / a;
        *Ic = 1.0L - *I;
    } else {
        *Ic = front * beta_cf(b, a, 1.0L - x) / b;
        *I = 1.0L - *Ic;
    }
}

// Survival function 1 - CDF of x = v^2/theta^2 at speed v (in units of theta).
ld survival(ld v, double kappa, int which, const kappagen::TableIParams<double>& T) {
    const ld x = v * v;
    if (which == KAPPAGEN_ENTROPY_VS_EXACT) {
        ld I, Ic;
        betainc_both(1.5L, (ld)kappa - 0.5L, x / (x + (ld)kappa), &I, &Ic);          // Eq. (3)
        return Ic;
    }
    const ld ks = T.kstar, h = ((ld)T.a * x + (ld)T.b * x * x) / (1.0L + (ld)T.c * x);
    if (!(x > 0.0L)) return 1.0L;
    const ld q = expl(-ks * log1pl(h / ks));                                            // exp_{q*}(-h), Eq. (8)
    return -expm1l(1.5L * log1pl(-q));                                                  // 1 - (1-q)^{3/2}, Eq. (7)/(A11)
}

}  // namespace

extern "C" int kappagen_relative_entropy(const unsigned long long* hist, int32_t nbins, double dv, double kappa,
                                         double eps, int which, double* D_out) {
    const char* fn = "kappagen_relative_entropy";
    if (!hist || !D_out) {
        kappagen::set_error("%s: NULL histogram or output", fn);
        return KAPPAGEN_ENULL;
    }
    if (nbins < 2 || !(dv > 0.0) || !std::isfinite(dv) || !(eps >= 0.0) || !kappagen::domain_ok(kappa, 0.0) ||
        (which != KAPPAGEN_ENTROPY_VS_EXACT && which != KAPPAGEN_ENTROPY_VS_APPROX)) {
        kappagen::set_error("%s: need nbins >= 2, dv > 0, eps >= 0, kappa > 3/2, which in {0,1}", fn);
        return KAPPAGEN_EINVAL;
    }
    ld total = 0.0L;
    for (int32_t i = 0; i < nbins; ++i) total += (ld)hist[i];
    if (!(total > 0.0L)) {
        kappagen::set_error("%s: empty histogram", fn);
        return KAPPAGEN_EINVAL;
    }
    const kappagen::TableIParams<double> T = kappagen::host_table1(kappa);
    ld D = 0.0L, s_lo = 1.0L;                                   // survival at the bin's lower edge (v = 0)
    for (int32_t i = 0; i < nbins; ++i) {
        const ld s_hi = (i == nbins - 1) ? 0.0L : survival((ld)(i + 1) * (ld)dv, kappa, which, T);
        const ld P = s_lo - s_hi;                               // both tails small: no cancellation where it matters
        const ld Q = (ld)hist[i] / total;
        D += (P + (ld)eps) * logl((P + (ld)eps) / (Q + (ld)eps));
        s_lo = s_hi;
    }
    *D_out = (double)D;
    return KAPPAGEN_OK;
}
