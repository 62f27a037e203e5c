"""Pins for oracle S2-S4 (U1 -> L -> x = V^2/theta^2; Eqs. (22)-(25), Table I lines 6-7).

The inverse is pinned against the FORWARD definition G(x) of Eq. (7)/(A11) evaluated in 40-digit
arithmetic (round trip), against Table I typed literally in 50-digit arithmetic, against the
Appendix asymptotics Eqs. (12) and (15), and by monotonicity."""
import mpmath as mp
import numpy as np
import pytest

import oracle
from paper_2602_05606_b200.workloads import edge_words
from test_oracle_params import mp_params

KAPPAS = (1.6, 2.0, 3.0, 4.0, 6.0, 10.0)
WORDS = edge_words(n_random=600)


def G_mp(x, kappa):
    """Eq. (A11); returns (G, 1-G) so both ends can be compared relatively."""
    ks, a, b, c = mp_params(kappa)
    x = mp.mpf(x)
    h = (a * x + b * x * x) / (1 + c * x)
    q = (1 + h / ks) ** (-ks)            # exp_{q*}(-h), Eq. (8) with q* = 1 + 1/kappa*
    G = (1 - q) ** (mp.mpf(3) / 2)
    return G, 1 - G


@pytest.mark.parametrize("kappa", KAPPAS)
def test_round_trip_through_forward_cdf(kappa):
    mp.mp.dps = 40
    x = oracle.x_of_w0(WORDS, kappa)
    ks = kappa - 0.5
    tol = (1.5 + ks) * 1.2e-16 * 2      # x is rounded once to double; d ln G/d ln x <= 3/2, d ln(1-G)/d ln x >= -kappa*
    worst = 0.0
    for w, xi in zip(WORDS.tolist(), x.tolist()):
        u = (mp.mpf(w) + mp.mpf(1) / 2) / 2**32
        G, Gc = G_mp(xi, kappa)
        err = max(abs(G - u) / u, abs(Gc - (1 - u)) / (1 - u))
        worst = max(worst, float(err))
    assert worst <= tol, worst


def table1_x_mp(w0, kappa):
    """Table I lines 6-7 typed verbatim in 50-digit arithmetic."""
    ks, a, b, c = mp_params(kappa)
    U1 = (mp.mpf(w0) + mp.mpf(1) / 2) / 2**32
    L = -ks * ((1 - U1 ** (mp.mpf(2) / 3)) ** (-1 / ks) - 1)
    return -2 * L / ((a + c * L) + mp.sqrt((a + c * L) ** 2 - 4 * b * L)), L


@pytest.mark.parametrize("kappa", KAPPAS)
def test_stable_form_equals_table1_in_50_digits(kappa):
    mp.mp.dps = 50
    x = oracle.x_of_w0(WORDS, kappa)
    L = oracle.L_of_w0(WORDS, kappa)
    worst = 0.0
    for w, xi, Li in zip(WORDS.tolist(), x.tolist(), L.tolist()):
        xm, Lm = table1_x_mp(w, kappa)
        assert Li < 0                                   # "Note that L is negative" PAPER.md:176
        worst = max(worst, float(abs(xi - xm) / xm), float(abs(Li - Lm) / abs(Lm)))
    assert worst <= 1.3e-16, worst                      # one rounding to double (2^-53 = 1.11e-16) + long-double noise


@pytest.mark.parametrize("kappa", KAPPAS)
def test_literal_table1_agrees_where_it_does_not_cancel(kappa):
    # long double literal evaluation: fine in the bulk, loses digits toward both ends (R7)
    bulk = WORDS[(WORDS > 2**26) & (WORDS < 2**32 - 2**26)]
    xs, xl = oracle.x_of_w0(bulk, kappa), oracle.x_of_w0_literal(bulk, kappa)
    assert np.max(np.abs(xs - xl) / xs) < 1e-14
    # and at the extremes the literal form is visibly worse than the stable one (what R7 is about)
    ends = np.array([0, 1, 2, 2**32 - 3, 2**32 - 2, 2**32 - 1], dtype=np.uint32)
    xs, xl = oracle.x_of_w0(ends, kappa), oracle.x_of_w0_literal(ends, kappa)
    assert np.all(np.isfinite(xl)) and np.max(np.abs(xs - xl) / xs) < 1e-8


@pytest.mark.parametrize("kappa", KAPPAS)
def test_monotone_in_the_word(kappa):
    x = oracle.x_of_w0(WORDS, kappa)
    assert np.all(np.diff(x) > 0)
    lo = np.arange(0, 1 << 16, dtype=np.uint32)
    hi = np.arange((1 << 32) - (1 << 16), 1 << 32, dtype=np.uint64).astype(np.uint32)
    mid = np.arange((1 << 31) - (1 << 15), (1 << 31) + (1 << 15), dtype=np.uint64).astype(np.uint32)
    for win in (lo, mid, hi):
        assert np.all(np.diff(oracle.x_of_w0(win, kappa)) > 0)


@pytest.mark.parametrize("kappa", KAPPAS)
def test_small_x_asymptote_eq12(kappa):
    # Eq. (12): G = a^{3/2} x^{3/2} {1 + (3/2) q x + O(x^2)}, q = (b-ac)/a - (kappa*+1)a/(2 kappa*)
    # => U1^{2/3} / (a x) = 1 + q x + O(x^2)
    ks, a, b, c = oracle.params(kappa)
    q = (b - a * c) / a - (ks + 1) * a / (2 * ks)
    w = np.array([0, 1, 5, 100, 4000, 70000], dtype=np.uint32)
    x = oracle.x_of_w0(w, kappa)
    u = (w.astype(np.float64) + 0.5) / 2**32
    ratio = u ** (2.0 / 3.0) / (a * x)
    assert np.all(np.abs(ratio - 1 - q * x) <= 20 * x * x + 1e-14)
    assert np.all(np.abs(ratio - 1) >= 0.5 * abs(q) * x - 1e-14)   # the first-order term is really there


@pytest.mark.parametrize("kappa", (1.6, 2.0, 3.0))
def test_large_x_asymptote_eq15(kappa):
    # Eq. (15): 1 - G = (3/2) (c kappa*/b)^{kappa*} x^{-kappa*} (1 + O(1/x))
    ks, a, b, c = oracle.params(kappa)
    w = np.array([2**32 - 1, 2**32 - 2, 2**32 - 7], dtype=np.uint32)
    x = oracle.x_of_w0(w, kappa)
    t = ((2**32 - 1 - w.astype(np.float64)) + 0.5) / 2**32
    lead = 1.5 * (c * ks / b) ** ks * x ** (-ks)
    K = (c * ks / b) * abs(ks + (a * c - b) / c**2)                  # size of the x^{-1} term in (A14)
    assert np.all(np.abs(t / lead - 1) <= 3 * K / x + t)


@pytest.mark.parametrize("kappa", KAPPAS)
def test_quadratic_residual(kappa):
    # x solves b x^2 + (a + cL) x + L = 0 (Eq. (22) -> (24))
    ks, a, b, c = oracle.params(kappa)
    x, L = oracle.x_of_w0(WORDS, kappa), oracle.L_of_w0(WORDS, kappa)
    res = b * x * x + (a + c * L) * x + L
    scale = b * x * x + np.abs(a + c * L) * x + np.abs(L)
    assert np.max(np.abs(res) / scale) < 1e-15


def test_extreme_speeds_at_32_bits():
    # the largest representable speed^2, from the asymptote Eq. (15) inverted at 1-U = 2^-33
    for kappa in (1.6, 2.0, 3.0):
        ks, a, b, c = oracle.params(kappa)
        xmax = oracle.x_of_w0([2**32 - 1], kappa)[0]
        approx = (c * ks / b) * (1.5 / 2.0**-33) ** (1 / ks)
        assert xmax == pytest.approx(approx, rel=3e-3 if kappa > 2.5 else 1e-5)
