"""Pins for the 64-bit-U1 variant of the oracle (reading R20):
U1 = (w0 2^32 + w3 + 1/2)/2^64, the discarded fourth Philox word deepening both ends of the uniform.
Same kinds of pins as test_oracle_inverse.py: the forward CDF of Eq. (A11) in 40 digits, Table I typed
literally in 50 digits, monotonicity across the word boundary, the asymptote Eq. (15), and the relation
to the 32-bit generator (its midpoint lies between the two central 64-bit points)."""
import mpmath as mp
import numpy as np
import pytest

import oracle
from test_oracle_inverse import G_mp
from test_oracle_params import mp_params

KAPPAS = (1.6, 2.0, 3.0, 4.0, 6.0, 10.0)


def edge_pairs():
    hi = [0, 1, 2, 3, 7, 2**16, 2**31 - 1, 2**31, 2**31 + 1, 2**32 - 2**16, 2**32 - 8, 2**32 - 3, 2**32 - 2, 2**32 - 1]
    lo = [0, 1, 2, 5, 2**15, 2**31 - 1, 2**31, 2**32 - 6, 2**32 - 2, 2**32 - 1]
    rng = np.random.Generator(np.random.PCG64(64))
    pairs = [(h, l) for h in hi for l in lo] + [tuple(int(v) for v in rng.integers(0, 2**32, 2)) for _ in range(300)]
    pairs = sorted(set(pairs), key=lambda p: (p[0] << 32) | p[1])
    return np.array([p[0] for p in pairs], dtype=np.uint32), np.array([p[1] for p in pairs], dtype=np.uint32)


W0, W3 = edge_pairs()


@pytest.mark.parametrize("kappa", KAPPAS)
def test_round_trip_through_forward_cdf_at_64_bits(kappa):
    mp.mp.dps = 45
    x = oracle.x_of_w0w3(W0, W3, kappa)
    ks = kappa - 0.5
    tol = (1.5 + ks) * 1.2e-16 * 2
    worst = 0.0
    for h, l, xi in zip(W0.tolist(), W3.tolist(), x.tolist()):
        u = (mp.mpf((h << 32) | l) + mp.mpf(1) / 2) / mp.mpf(2) ** 64
        G, Gc = G_mp(xi, kappa)
        worst = max(worst, float(max(abs(G - u) / u, abs(Gc - (1 - u)) / (1 - u))))
    assert worst <= tol, worst


@pytest.mark.parametrize("kappa", KAPPAS)
def test_equals_table1_in_50_digits_with_the_64_bit_uniform(kappa):
    mp.mp.dps = 60
    ks, a, b, c = mp_params(kappa)
    x = oracle.x_of_w0w3(W0, W3, kappa)
    worst = 0.0
    for h, l, xi in zip(W0.tolist(), W3.tolist(), x.tolist()):
        U1 = (mp.mpf((h << 32) | l) + mp.mpf(1) / 2) / mp.mpf(2) ** 64
        L = -ks * ((1 - U1 ** (mp.mpf(2) / 3)) ** (-1 / ks) - 1)             # Eq. (25), Table I line 6
        xm = -2 * L / ((a + c * L) + mp.sqrt((a + c * L) ** 2 - 4 * b * L))  # Eq. (24), Table I line 7
        worst = max(worst, float(abs(xi - xm) / xm))
    assert worst <= 1.3e-16, worst


@pytest.mark.parametrize("kappa", KAPPAS)
def test_monotone_across_the_word_boundary_and_brackets_the_32_bit_point(kappa):
    x = oracle.x_of_w0w3(W0, W3, kappa)
    d = np.diff(x)                                                 # pairs are sorted by the 64-bit integer
    assert np.all(d >= 0) and np.mean(d > 0) > 0.9                 # neighbours 2^-64 apart can round to one double
    w0 = np.array([0, 1, 77, 2**31 - 1, 2**31, 2**32 - 2], dtype=np.uint32)
    top = oracle.x_of_w0w3(w0, np.full(w0.size, 2**32 - 1, dtype=np.uint32), kappa)
    nxt = oracle.x_of_w0w3(w0 + 1, np.zeros(w0.size, dtype=np.uint32), kappa)
    assert np.all(top <= nxt) and np.all(top[:3] < nxt[:3])        # 2^-64 apart: resolved in double only for small U1
    # the 32-bit midpoint (w0 + 1/2)/2^32 = (w0 2^32 + 2^31)/2^64 lies between the 64-bit points w3 = 2^31 -+ 2^24
    # (a 2^-64 step is below the resolution of a double unless U1 is tiny, hence the wider bracket)
    w0 = np.concatenate([w0, [2**32 - 1]]).astype(np.uint32)
    below = oracle.x_of_w0w3(w0, np.full(w0.size, 2**31 - 2**24, dtype=np.uint32), kappa)
    above = oracle.x_of_w0w3(w0, np.full(w0.size, 2**31 + 2**24, dtype=np.uint32), kappa)
    mid = oracle.x_of_w0(w0, kappa)
    assert np.all(below < mid) and np.all(mid < above)
    assert np.all(((above - below) / mid)[3:5] < 1e-8)             # 2^-39 wide in U1: tight away from the ends


@pytest.mark.parametrize("kappa", (1.6, 2.0, 3.0))
def test_extreme_speed_follows_eq15_at_2_to_minus_65(kappa):
    # Eq. (15) PAPER.md:97 inverted at 1 - U1 = 2^-65: x_max = (c kappa*/b) (1.5 / 2^-65)^(1/kappa*)
    ks, a, b, c = oracle.params(kappa)
    xmax = oracle.x_of_w0w3([2**32 - 1], [2**32 - 1], kappa)[0]
    approx = (c * ks / b) * (1.5 / 2.0 ** -65) ** (1 / ks)
    assert xmax == pytest.approx(approx, rel=1e-6)
    x32 = oracle.x_of_w0([2**32 - 1], kappa)[0]
    assert xmax / x32 == pytest.approx(2.0 ** (32 / ks), rel=1e-4)   # the tail reaches 2^(32/kappa*) further in v^2


def test_sample_u64_changes_the_speed_only_and_uses_the_fourth_word():
    n, kappa, theta, seed, off = 5000, 2.0, 0.7, 99, 2**32 - 2500
    (vx, vy, vz), w3 = oracle.sample_u64(n, kappa, theta, seed, off, return_w3=True)
    sx, sy, sz = oracle.sample(n, kappa, theta, seed, off)
    w0, w1, w2 = oracle.words(n, seed, off)
    # the fourth word is the block's fourth output (pinned by the known-answer vectors for seed 0 below)
    want = oracle.velocity_of_words_u64(w0, w1, w2, w3, kappa, theta)
    assert all(np.array_equal(a, b) for a, b in zip((vx, vy, vz), want))
    # same direction, speed within the 2^-32 bracket of the 32-bit point
    v64 = np.sqrt(vx**2 + vy**2 + vz**2)
    v32 = np.sqrt(sx**2 + sy**2 + sz**2)
    assert np.allclose(vx / v64, sx / v32, rtol=0, atol=1e-14) and np.allclose(vz / v64, sz / v32, rtol=0, atol=1e-14)
    u = (w0.astype(np.float64) + 0.5) / 2**32
    assert np.all(np.abs(v64 / v32 - 1) < 2.0**-31 / np.minimum(u, 1 - u))
    assert np.max(np.abs(v64 / v32 - 1)) > 1e-12                  # and it is not the same generator
    _, w3z = oracle.sample_u64(3, 2.0, 1.0, 0, 0, return_w3=True)
    assert [int(v) for v in w3z] == [0x9b00dbd8, 0x097eff67, 0x459135e4]    # SURVEY.md 8(c)-D1, particles 0,1,2 of seed 0
