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

// Continued fraction of the incomplete beta function (modified Lentz iteration, the classical
// evaluation of I_x(a,b): DLMF 8.17.22).
ld betacf(ld a, ld b, ld x) {
    const ld tiny = 1e-4000L;
    const ld qab = a + b, qap = a + 1.0L, qam = a - 1.0L;
    ld c = 1.0L, d = 1.0L - qab * x / qap;
    if (fabsl(d) < tiny) d = tiny;
    d = 1.0L / d;
    ld h = d;
    for (int m = 1; m <= 2000; ++m) {
        const ld m2 = 2.0L * m;
        ld aa = m * (b - m) * x / ((qam + m2) * (a + m2));
        d = 1.0L + aa * d; if (fabsl(d) < tiny) d = tiny;
        c = 1.0L + aa / c; if (fabsl(c) < tiny) c = tiny;
        d = 1.0L / d;
        h *= d * c;
        aa = -(a + m) * (qab + m) * x / ((a + m2) * (qap + m2));
        d = 1.0L + aa * d; if (fabsl(d) < tiny) d = tiny;
        c = 1.0L + aa / c; if (fabsl(c) < tiny) c = tiny;
        d = 1.0L / d;
        const ld del = d * c;
        h *= del;
        if (fabsl(del - 1.0L) < 1e-19L) break;
    }
    return h;
}

// Regularized incomplete beta I_x(a,b) and its complement, each computed without cancellation.
void betainc_both(ld a, ld b, ld x, ld* I, ld* Ic) {
    if (x <= 0.0L) { *I = 0.0L; *Ic = 1.0L; return; }
    if (x >= 1.0L) { *I = 1.0L; *Ic = 0.0L; return; }
    const ld lnfront = lgammal(a + b) - lgammal(a) - lgammal(b) + a * logl(x) + b * log1pl(-x);
    const ld front = expl(lnfront);
    if (x < (a + 1.0L) / (a + b + 2.0L)) {
        *I = front * betacf(a, b, x) / a;
        *Ic = 1.0L - *I;
    } else {
        *Ic = front * betacf(b, a, 1.0L - x) / b;
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
