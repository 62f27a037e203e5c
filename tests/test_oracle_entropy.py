"""Pins for the oracle side of paper test 2 (Eqs. (26)-(27)):
speeds, histogram with Delta v = 1/5, bin probabilities and the discrete relative entropy -- and the product's
host function kappagen_relative_entropy against them (host arithmetic only, no GPU involved).

What the paper fixes: the large-N plateau of D for the proposed method is the continuous KL divergence of
the approximation, 'remarkably low for kappa < 4', peaking near kappa ~ 4.2 and ~1e-6 for kappa >~ 5
(SURVEY.md section 4 [probe]: 5.3e-8 at 3, 7.7e-6 at 4.1); below N ~ 1e7 the particle noise hides it
and D falls like 1/N."""
import ctypes

import numpy as np
import pytest
from scipy import integrate, special

import oracle
from paper_2602_05606_b200 import kappagen as kg

DV = 0.2                      # "Delta v = 1/5"


def kappa_speed_pdf(v, kappa):
    """4 pi v^2 f(v), Eq. (1) with theta = 1: the omni-directional speed density."""
    norm = special.gamma(kappa + 1) / ((np.pi * kappa) ** 1.5 * special.gamma(kappa - 0.5))
    return 4 * np.pi * v * v * norm * (1 + v * v / kappa) ** (-(kappa + 1))


@pytest.mark.parametrize("kappa", (2.0, 3.0, 4.1, 7.5))
def test_exact_bin_probabilities_are_the_integral_of_eq1(kappa):
    """'we numerically integrate the Kappa distribution in each histogram bin': quadrature of the
    density Eq. (1) against the CDF route Eq. (3) that bin_probabilities takes."""
    P = oracle.bin_probabilities(kappa, DV, 64, "exact")
    assert abs(P.sum() - 1) < 1e-14 and np.all(P > 0)
    for i in (0, 1, 4, 5, 17, 40):
        q, _ = integrate.quad(kappa_speed_pdf, i * DV, (i + 1) * DV, args=(kappa,), epsabs=0, epsrel=1e-12)
        assert P[i] == pytest.approx(q, rel=1e-10)
    tail, _ = integrate.quad(kappa_speed_pdf, 63 * DV, np.inf, args=(kappa,), epsabs=0, epsrel=1e-12)
    assert P[63] == pytest.approx(tail, rel=1e-9)             # the open-ended last bin (reading R21)
    assert np.argmax(P) in (4, 5)                             # the speed density peaks at |v| = theta


def test_plateau_of_the_relative_entropy_has_the_shape_the_paper_describes():
    """N -> infinity: Q -> the generator's own bin probabilities, so D -> sum P_F ln(P_F/P_G), which the paper
    says is 'essentially similar' to the continuous D of Fig. 4(a).  What the PAPER fixes is the
    shape (remarkably low for kappa < 4, a peak near kappa ~ 4.2, ~1e-6 beyond kappa ~ 5) -- the last
    two assertions.  The two numbers 5.3e-8 and 7.7e-6 are NOT printed in the paper (Fig. 4(a) shows them only as
    circles): they are the SURVEY.md section 4 [probe] values, an independent 400 001-point quadrature of Eqs. (2),
    (7), kept here as a regression pin of the bin-probability code, not as a paper fact."""
    def plateau(kappa):
        PF = oracle.bin_probabilities(kappa, DV, 2048, "exact")
        PG = oracle.bin_probabilities(kappa, DV, 2048, "approx")
        return float(np.sum(PF * np.log(PF / PG)))
    assert plateau(3.0) == pytest.approx(5.3e-8, rel=0.15)
    assert plateau(4.1) == pytest.approx(7.7e-6, rel=0.15)
    assert 3e-7 < plateau(7.5) < 3e-6                          # "~1e-6 for kappa >~ 5"
    assert plateau(4.2) > plateau(3.0) * 50 and plateau(4.2) > plateau(7.5)      # the peak near 4.2


def test_noise_floor_scales_like_one_over_n():
    """Well-populated bins: 2 N D is asymptotically chi-square with (bins - 1) degrees of freedom, so
    D ~ (bins-1)/(2N), 'antiproportional to the number of particles'."""
    kappa, nb = 3.0, 20
    d = []
    for n in (100_000, 400_000):
        h = oracle.speed_histogram(oracle.speed_over_theta(n, kappa, 5), DV, nb)
        assert h.sum() == n
        d.append(2 * n * oracle.relative_entropy(h, kappa, DV))
    assert all(5 < x < 45 for x in d), d                       # chi-square(19): P(<5) ~ P(>45) < 1e-3


def test_speeds_are_the_norm_of_the_sampled_velocities():
    n, kappa = 5000, 4.1
    s = oracle.speed_over_theta(n, kappa, 9, 123)
    vx, vy, vz = oracle.sample(n, kappa, 2.5, 9, 123)
    assert np.allclose(s, np.sqrt(vx * vx + vy * vy + vz * vz) / 2.5, rtol=4e-16, atol=0)
    s64 = oracle.speed_over_theta(n, kappa, 9, 123, u64=True)
    ux, uy, uz = oracle.sample_u64(n, kappa, 2.5, 9, 123)
    assert np.allclose(s64, np.sqrt(ux * ux + uy * uy + uz * uz) / 2.5, rtol=4e-16, atol=0)


@pytest.mark.parametrize("kappa", (1.6, 3.0, 4.1, 7.5, 15.0))
@pytest.mark.parametrize("which", (0, 1))
def test_product_host_entropy_equals_the_oracle_reference(kappa, which):
    """kappagen_relative_entropy (long double, own continued-fraction incomplete beta) against the scipy-based
    reference above, on a real histogram and on degenerate ones."""
    h = oracle.speed_histogram(oracle.speed_over_theta(200_000, kappa, 1), DV, 512)
    want = oracle.relative_entropy(h, kappa, DV, 1e-10, "exact" if which == 0 else "approx")
    got = kg.relative_entropy(h, kappa, DV, 1e-10, which)
    assert got == pytest.approx(want, rel=1e-9, abs=1e-15)
    one = np.zeros(8, dtype=np.uint64)
    one[3] = 7
    assert kg.relative_entropy(one, kappa, DV, 1e-10, which) == pytest.approx(
        oracle.relative_entropy(one, kappa, DV, 1e-10, "exact" if which == 0 else "approx"), rel=1e-9)


def test_product_host_entropy_status_codes():
    L = kg.lib()
    h = (ctypes.c_uint64 * 4)(1, 2, 3, 4)
    out = ctypes.c_double()
    assert L.kappagen_relative_entropy(None, 4, DV, 3.0, 1e-10, 0, ctypes.byref(out)) == kg.ENULL
    assert L.kappagen_relative_entropy(h, 1, DV, 3.0, 1e-10, 0, ctypes.byref(out)) == kg.EINVAL
    assert L.kappagen_relative_entropy(h, 4, 0.0, 3.0, 1e-10, 0, ctypes.byref(out)) == kg.EINVAL
    assert L.kappagen_relative_entropy(h, 4, DV, 1.5, 1e-10, 0, ctypes.byref(out)) == kg.EINVAL
    assert L.kappagen_relative_entropy(h, 4, DV, 3.0, 1e-10, 2, ctypes.byref(out)) == kg.EINVAL
    z = (ctypes.c_uint64 * 4)(0, 0, 0, 0)
    assert L.kappagen_relative_entropy(z, 4, DV, 3.0, 1e-10, 0, ctypes.byref(out)) == kg.EINVAL
    assert L.kappagen_relative_entropy(h, 4, DV, 3.0, 1e-10, 0, ctypes.byref(out)) == kg.OK and out.value > 0
