"""Pins for oracle S0 (Table I lines 1-4; Eqs. (13),(16),(17),(20)) against what the paper prints
and against an evaluation in 40-digit arithmetic with mpmath's own beta function (the oracle goes
through lgammal instead)."""
import math

import mpmath as mp
import numpy as np
import pytest

import oracle

KAPPAS = (1.6, 2.0, 2.5, 3.0, 4.0, 4.1, 6.0, 7.5, 10.0, 15.0, 100.0)


def mp_params(kappa):
    mp.mp.dps = 40
    k = mp.mpf(kappa)
    ks = k - mp.mpf(1) / 2
    B = mp.beta(mp.mpf(3) / 2, ks)
    a = (1 / k) * (2 / (3 * B)) ** (mp.mpf(2) / 3)
    c = (mp.mpf("0.123") * k**2 - mp.mpf("1.12") * k + mp.mpf("2.56")) / (k**2 - mp.mpf("7.89") * k + mp.mpf("15.6"))
    b = (ks * mp.mpf(3) / 2 * B) ** (1 / ks) * (ks / k) * c
    return ks, a, b, c


@pytest.mark.parametrize("kappa", KAPPAS)
def test_params_match_40_digit_evaluation(kappa):
    got = oracle.params(kappa)
    want = mp_params(kappa)
    for g, w in zip(got, want):
        assert abs(g - float(w)) <= 2.3e-16 * abs(float(w))


def test_printed_start_values_two_thirds(facts):
    # PAPER.md:106 "Starting from 2/3 at kappa = 3/2"
    ks, a, b, c = oracle.params(1.5 + 1e-9)
    assert a == pytest.approx(facts["a_at_kappa_1p5"], rel=1e-7)
    assert b / c == pytest.approx(facts["b_over_c_at_kappa_1p5"], rel=1e-7)


def test_printed_limits_large_kappa(facts):
    # Eq. (18)
    lim = (4.0 / (3.0 * math.sqrt(math.pi))) ** (2.0 / 3.0)
    assert round(lim, 3) == facts["a_limit"]
    ks, a, b, c = oracle.params(1e6)
    assert a == pytest.approx(lim, rel=1e-5)
    assert b / c == pytest.approx(facts["b_over_c_limit"], rel=1e-4)


def test_a_and_b_over_c_increase_and_cross_near_4p1(facts):
    ks_grid = np.linspace(1.51, 20.0, 1850)
    a = np.array([oracle.params(k)[1] for k in ks_grid])
    bc = np.array([oracle.params(k)[2] / oracle.params(k)[3] for k in ks_grid])
    assert np.all(np.diff(a) > 0) and np.all(np.diff(bc) > 0)      # "increase monotonically" PAPER.md:106
    sign = np.sign(a - bc)
    cross = np.nonzero(np.diff(sign))[0]
    assert len(cross) == 1
    assert abs(ks_grid[cross[0]] - facts["a_bc_intersection_kappa"]) < 0.1


def test_c_approx_extrema_as_printed(facts):
    # maximum ~1.6 at kappa ~3.9, minimum ~0.02 at kappa ~4.7
    grid = np.linspace(1.51, 10.0, 8491)
    c = np.array([oracle.params(k)[3] for k in grid])
    imax, imin = int(np.argmax(c)), int(np.argmin(c))
    assert abs(c[imax] - facts["c_max"]) < 0.05 and abs(grid[imax] - facts["c_max_kappa"]) < 0.05
    assert abs(c[imin] - facts["c_min"]) < 0.005 and abs(grid[imin] - facts["c_min_kappa"]) < 0.05
    assert np.all(c > 0)  # b, c > 0 is what keeps the discriminant of Eq. (24) positive


def test_c_at_4_is_exactly_6_fifths():
    # (0.123*16 - 1.12*4 + 2.56) / (16 - 7.89*4 + 15.6) = 0.048 / 0.04
    assert oracle.params(4.0)[3] == pytest.approx(1.2, rel=1e-15)


def test_kappa_star_is_kappa_minus_half():
    for k in KAPPAS:
        assert oracle.params(k)[0] == k - 0.5  # Eq. (16)


def test_domain():
    for bad in (1.5, 1.0, -2.0, float("nan"), float("inf")):
        with pytest.raises(ValueError):
            oracle.params(bad)
