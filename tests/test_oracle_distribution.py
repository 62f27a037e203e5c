"""Pins for the oracle end to end against the EXACT Kappa distribution (Eqs. (1)-(6)) and against the
accuracy statements the paper prints: the generator samples G (Eq. 7), which is
close to, not equal to, F (Eq. 3) -- so every gate is "exact result within the approximation error"."""
import math

import numpy as np
import pytest
from scipy import integrate, special

import oracle

KAPPAS = (1.6, 2.0, 3.0, 4.0, 6.0, 10.0)


def F_exact(x, kappa):
    """Eq. (3): regularized incomplete beta I_{x/(x+kappa)}(3/2, kappa-1/2)."""
    return special.betainc(1.5, kappa - 0.5, x / (x + kappa))


def f_exact(x, kappa):
    """Eq. (2) PAPER.md:37."""
    return (x / kappa) ** 0.5 * (1 + x / kappa) ** (-(kappa + 1)) / (kappa * special.beta(1.5, kappa - 0.5))


def sup_G_minus_F_via_oracle(kappa, npts=400_001):
    """sup_x |G(x) - F(x)| = sup_u |u - F(G^{-1}(u))| with G^{-1} taken from the oracle itself."""
    w = np.linspace(0, 2**32 - 1, npts).astype(np.uint64).astype(np.uint32)
    u = (w.astype(np.float64) + 0.5) / 2**32
    return float(np.max(np.abs(F_exact(oracle.x_of_w0(w, kappa), kappa) - u)))


def ks_distance(sorted_cdf_values):
    n = sorted_cdf_values.size
    i = np.arange(1, n + 1, dtype=np.float64)
    return float(max(np.max(i / n - sorted_cdf_values), np.max(sorted_cdf_values - (i - 1) / n)))


def test_approximation_error_sizes_match_the_paper():
    sup = {k: sup_G_minus_F_via_oracle(k) for k in KAPPAS + (2.6, 4.2, 7.5)}
    # "remarkably accurate for kappa <~ 3", "remarkably low for kappa < 4"
    for k in (1.6, 2.0, 2.6, 3.0):
        assert sup[k] < 1.5e-4
    # Pinsker: sup|G-F| <= sqrt(D/2) with the printed D ~ 1e-6 for kappa >~ 5
    for k in (6.0, 7.5, 10.0):
        assert sup[k] < 1.0e-3
    # worst around the transition kappa ~ 4.1-4.2, still tiny
    assert sup[4.2] == max(sup.values()) and 5e-4 < sup[4.2] < 2.5e-3


@pytest.mark.parametrize("kappa,n", [(k, 10_000_000) for k in (1.6, 2.0, 3.0, 4.0, 6.0, 10.0)])   # north_star: 1e7 samples
def test_ks_against_exact_kappa_cdf(kappa, n):
    theta = 0.7
    vx, vy, vz = oracle.sample(n, kappa, theta, seed=1, offset=0)
    x = np.sort((vx * vx + vy * vy + vz * vz) / theta**2)
    band = 1.95 / math.sqrt(n)                                  # 99.9 % Kolmogorov quantile
    ks = ks_distance(F_exact(x, kappa))
    assert ks <= sup_G_minus_F_via_oracle(kappa, 100_001) + band, ks
    if kappa == 4.0 and n >= 10_000_000:
        # at N_p >~ 1e7 the approximation becomes detectable near kappa ~ 4.1
        assert ks > band


def test_energy_closed_form_eq5_by_quadrature():
    # <x> = 3 kappa / (2 kappa - 3)  (Eq. 5 with m theta^2 / 2 per unit x)
    for kappa in (2.0, 3.0, 4.1, 10.0):
        val, _ = integrate.quad(lambda t: math.exp(t) * math.exp(t) * f_exact(math.exp(t), kappa), -40, 60, limit=400)
        assert val == pytest.approx(3 * kappa / (2 * kappa - 3), rel=1e-8)


def mean_x_under_G(kappa, xcut=None):
    """<min(x, xcut)> under the generator's own distribution, by quadrature over u of the oracle's
    inverse: int_0^1 min(x(u), xcut) du on the 32-bit word grid collapses to a mean over words; here a
    fine stratified subsample of words (every 2^12-th, tails dense) is enough for 1e-6."""
    w_mid = np.arange(1 << 20, (1 << 32) - (1 << 20), 1 << 12, dtype=np.uint64)
    w_lo = np.arange(0, 1 << 20, dtype=np.uint64)
    w_hi = np.arange((1 << 32) - (1 << 20), 1 << 32, dtype=np.uint64)

    def part(w, weight):
        x = oracle.x_of_w0(w.astype(np.uint32), kappa)
        if xcut is not None:
            x = np.minimum(x, xcut)
        return float(np.sum(x)) * weight

    return (part(w_lo, 1.0) + part(w_hi, 1.0) + part(w_mid + (1 << 11), float(1 << 12))) / 2.0**32


def test_energy_error_of_the_approximation_as_printed(facts):
    err = {}
    for kappa in (2.0, 2.5, 3.0, 4.1, 6.0, 10.0):
        exact = 3 * kappa / (2 * kappa - 3)
        err[kappa] = (mean_x_under_G(kappa) - exact) / exact
    # "within an error of 1e-3, except for the largest error at kappa ~ 4.1"
    for kappa in (2.0, 2.5, 3.0, 6.0, 10.0):
        assert abs(err[kappa]) < facts["energy_error_bound"]
    # "It becomes zero at kappa ~ 2.5"
    assert abs(err[2.5]) < 5e-5
    # "O(10^-2.5) near kappa ~ 4.1", and energy is LOST there ("0.19% of the energy density is erroneously lost")
    assert err[4.1] < 0 and abs(math.log10(abs(err[4.1])) - facts["energy_error_peak_log10"]) < 0.3


def test_tail_population_deficit_at_kappa_4p1(facts):
    # density underestimated by ~1 % in v > 3 theta at kappa = 4.1; Eq. (6): that tail
    # carries ~19 % of the energy.
    kappa, x3 = 4.1, 9.0
    lo, hi = 0, 2**32 - 1
    while hi - lo > 1:                     # invert the oracle's monotone map at x = 9 by bisection on the word
        mid = (lo + hi) // 2
        if oracle.x_of_w0([mid], kappa)[0] < x3:
            lo = mid
        else:
            hi = mid
    tail_G = 1.0 - (hi + 0.5) / 2**32
    tail_F = 1.0 - F_exact(x3, kappa)
    assert 1 - tail_G / tail_F == pytest.approx(facts["tail_density_deficit_kappa4p1"], abs=0.005)
    FE = special.betainc(2.5, kappa - 1.5, x3 / (x3 + kappa))     # Eq. (6)
    assert 1 - FE == pytest.approx(facts["tail_energy_fraction_kappa4p1_v3"], abs=0.005)


@pytest.mark.parametrize("kappa", KAPPAS)
def test_censored_second_moment_of_samples(kappa):
    # heavy tails: Var(x) is infinite for kappa <= 5/2, so gate the censored moment <min(x, x_c)>,
    # x_c = G^{-1}(1 - 1e-4) (SURVEY 8(c)-E gate M2), at 5 standard errors.
    n = 2_000_000
    theta = 1.0
    wc = int((1 - 1e-4) * 2**32)
    xc = oracle.x_of_w0([wc], kappa)[0]
    vx, vy, vz = oracle.sample(n, kappa, theta, seed=1, offset=0)
    xs = np.minimum(vx * vx + vy * vy + vz * vz, xc)
    want = mean_x_under_G(kappa, xc)
    assert abs(xs.mean() - want) < 5 * xs.std() / math.sqrt(n)


def test_second_moment_closed_form_kappa3(facts):
    # north_star: <v^2> = 3 kappa theta^2 / (2 kappa - 3) for kappa > 3/2; kappa = 3 has finite variance.
    n, kappa, theta = 4_000_000, 3.0, 0.5
    vx, vy, vz = oracle.sample(n, kappa, theta, seed=2, offset=10**9)
    v2 = vx * vx + vy * vy + vz * vz
    exact = 3 * kappa * theta**2 / (2 * kappa - 3)
    var_x = kappa**2 * (15 / 4) / ((kappa - 1.5) * (kappa - 2.5)) - (3 * kappa / (2 * kappa - 3)) ** 2
    sigma = theta**2 * math.sqrt(var_x / n)
    assert abs(v2.mean() - exact) < 5 * sigma + facts["energy_error_bound"] * exact
    # isotropy of the velocities themselves: zero mean, equal variances (each <v^2>/3)
    for c in (vx, vy, vz):
        assert abs(c.mean()) < 5 * math.sqrt(exact / 3 / n)
    third = [float((c * c).mean()) for c in (vx, vy, vz)]
    assert max(third) - min(third) < 5 * theta**2 * math.sqrt(var_x / n) * 1.5


def test_most_probable_speed_is_theta():
    # "the Kappa distributions have their maximum at the most probable speed |v| = theta"
    n, theta = 4_000_000, 2.0
    for kappa in (3.0, 7.5):
        vx, vy, vz = oracle.sample(n, kappa, theta, seed=3, offset=0)
        v = np.sqrt(vx * vx + vy * vy + vz * vz)
        hist, edges = np.histogram(v, bins=np.arange(0.0, 3.0 * theta, 0.1 * theta))
        centre = 0.5 * (edges[:-1] + edges[1:])
        assert abs(centre[np.argmax(hist)] - theta) <= 0.1 * theta
