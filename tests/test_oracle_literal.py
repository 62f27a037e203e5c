"""Pins for the LITERAL evaluator of the oracle (oracle_sample_literal -> x_literal, dir_literal): Table I
typed in verbatim, lines 5-10, in the paper's order and notation.

It is not the function GPU parity is measured against (that is oracle.sample, the cancellation-free form of
the same real numbers, reading R7); it exists so that a reader can check the oracle against the
paper by eye, and these tests tie the two together: the literal form against a 50-digit mpmath evaluation of
Table I typed here once more from the paper, and against oracle.sample wherever the literal form is sound."""
import mpmath as mp
import numpy as np
import pytest

import oracle
from test_oracle_params import mp_params


def table1_mp(w0, w1, w2, kappa, theta):
    """Table I lines 5-10 in 50-digit arithmetic; U_j = (w + 1/2)/2^32 (reading R3)."""
    ks, a, b, c = mp_params(kappa)
    U1, U2, U3 = ((mp.mpf(w) + mp.mpf(1) / 2) / 2**32 for w in (w0, w1, w2))
    L = -ks * ((1 - U1 ** (mp.mpf(2) / 3)) ** (-1 / ks) - 1)                       # line 6, Eq. (25)
    V = theta * mp.sqrt(-2 * L / ((a + c * L) + mp.sqrt((a + c * L) ** 2 - 4 * b * L)))   # line 7, Eq. (24)
    vx = V * (2 * U2 - 1)                                                          # line 8
    vy = 2 * V * mp.sqrt(U2 * (1 - U2)) * mp.cos(2 * mp.pi * U3)                   # line 9
    vz = 2 * V * mp.sqrt(U2 * (1 - U2)) * mp.sin(2 * mp.pi * U3)                   # line 10
    return vx, vy, vz


@pytest.mark.parametrize("kappa,theta,seed,offset", [(3.0, 1.0, 0, 0), (1.6, 0.1, 42, 2**32 - 700), (7.5, 2.5, 9, 12345)])
def test_literal_sampler_equals_table1_in_50_digits(kappa, theta, seed, offset):
    mp.mp.dps = 50
    n = 1500
    w0, w1, w2 = oracle.words(n, seed, offset)
    got = oracle.sample(n, kappa, theta, seed, offset, literal=True)
    # the literal long-double form is sound away from the ends of U1 (reading R7) and away from the zeros of the
    # three components (2U2-1, cos, sin are formed by subtraction / from a rounded 2 pi U3 there)
    U2 = (w1.astype(np.float64) + 0.5) / 2**32
    U3 = (w2.astype(np.float64) + 0.5) / 2**32
    sound = (w0 > 2**26) & (w0 < 2**32 - 2**26) & (np.abs(2 * U2 - 1) > 1e-3) \
        & (np.abs(np.cos(2 * np.pi * U3)) > 1e-3) & (np.abs(np.sin(2 * np.pi * U3)) > 1e-3)
    assert sound.sum() > 0.9 * n
    worst = 0.0
    for i in np.nonzero(sound)[0][:600]:
        want = table1_mp(int(w0[i]), int(w1[i]), int(w2[i]), kappa, mp.mpf(theta))
        for q in range(3):
            worst = max(worst, float(abs(got[q][i] - want[q]) / abs(want[q])))
    # long double eps 5.4e-20; conditioning <= 2^6 (U1 window) x 1e3 (component window); one rounding to double
    assert worst <= 2e-16, worst


@pytest.mark.parametrize("kappa", [2.0, 4.0, 10.0])
def test_literal_and_stable_samplers_agree_in_the_bulk(kappa):
    n, theta, seed = 200_000, 0.7, 5
    w0, w1, w2 = oracle.words(n, seed, 0)
    lit = oracle.sample(n, kappa, theta, seed, 0, literal=True)
    stab = oracle.sample(n, kappa, theta, seed, 0)
    bulk = (w0 > 2**26) & (w0 < 2**32 - 2**26)
    for q in range(3):
        # absolute comparison on the scale of the speed: the literal cos/sin carry an ABSOLUTE error of
        # 2 pi eps_ld, the literal 2U2-1 an absolute error of eps_ld -- relative only away from their zeros
        speed = np.sqrt(stab[0] ** 2 + stab[1] ** 2 + stab[2] ** 2)
        assert np.max(np.abs(lit[q] - stab[q])[bulk] / speed[bulk]) < 1e-15
    # the polar axis is x (reading R8): vx carries 2U2-1, whose sign is the top bit of w1
    assert np.array_equal(lit[0] > 0, w1 >= 2**31)
    # and (vy, vz) = (cos, sin): vz > 0 on the first half turn of U3 (w2 < 2^31), vy > 0 on the outer quarters
    assert np.array_equal(lit[2] > 0, w2 < 2**31)
    assert np.array_equal(lit[1] > 0, (w2 < 2**30) | (w2 >= 3 * 2**30))
