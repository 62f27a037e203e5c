"""Pins for oracle S5-S6 (Table I lines 8-10): isotropic direction from (U2, U3)."""
import math

import mpmath as mp
import numpy as np

import oracle
from paper_2602_05606_b200.workloads import edge_words

W = edge_words(n_random=1500)
RNG = np.random.Generator(np.random.PCG64(11))
W1 = W
W2 = RNG.permutation(W)


def test_unit_norm_and_v2_equals_V2():
    nx, ny, nz = oracle.direction(W1, W2)
    assert np.max(np.abs(nx * nx + ny * ny + nz * nz - 1.0)) < 5e-16
    w0 = RNG.permutation(W)
    for kappa, theta in ((2.0, 0.1), (6.0, 3.0)):
        vx, vy, vz = oracle.velocity_of_words(w0, W1, W2, kappa, theta)
        V2 = theta * theta * oracle.x_of_w0(w0, kappa)
        assert np.max(np.abs(vx * vx + vy * vy + vz * vz - V2) / V2) < 1e-15


def test_table1_lines_8_to_10_in_50_digits():
    # vx = V(2U2-1), vy = 2V sqrt(U2(1-U2)) cos(2 pi U3), vz = ... sin(2 pi U3); x is the polar axis (R8)
    mp.mp.dps = 50
    nx, ny, nz = oracle.direction(W1, W2)
    worst = 0.0
    for a, b, gx, gy, gz in zip(W1.tolist(), W2.tolist(), nx.tolist(), ny.tolist(), nz.tolist()):
        U2 = (mp.mpf(a) + mp.mpf(1) / 2) / 2**32
        U3 = (mp.mpf(b) + mp.mpf(1) / 2) / 2**32
        wx = 2 * U2 - 1
        s = 2 * mp.sqrt(U2 * (1 - U2))
        wy, wz = s * mp.cos(2 * mp.pi * U3), s * mp.sin(2 * mp.pi * U3)
        for g, w in ((gx, wx), (gy, wy), (gz, wz)):
            worst = max(worst, float(abs(g - w) / abs(w)))
    assert worst <= 1.2e-16, worst      # strict per-component relative error, zeros of cos/sin included


def test_closed_form_next_to_the_zeros():
    # words adjacent to each quarter turn: |cos| or |sin| = sin(pi * 2^-32) exactly
    tiny = float(mp.sin(mp.pi * mp.mpf(2) ** -32))
    assert abs(tiny - 7.3146e-10) < 1e-14
    w1 = np.full(8, 0x80000000, dtype=np.uint32)          # mu = 2^-32, sth ~ 1
    w2 = np.array([0, 2**30 - 1, 2**30, 2**31 - 1, 2**31, 3 * 2**30 - 1, 3 * 2**30, 2**32 - 1], dtype=np.uint64).astype(np.uint32)
    nx, ny, nz = oracle.direction(w1, w2)
    sth = math.sqrt(1 - 2.0**-64)
    want_y = [1, tiny, -tiny, -1, -1, -tiny, tiny, 1]
    want_z = [tiny, 1, 1, tiny, -tiny, -1, -1, -tiny]
    for i in range(8):
        for got, want in ((ny[i], want_y[i]), (nz[i], want_z[i])):
            if abs(want) == 1:
                assert abs(got - want * sth) < 1e-15
            else:
                assert abs(got - want * sth) <= 1.2e-16 * tiny
    assert np.all(nx == 2.0**-32)


def test_exact_symmetries_under_complement():
    nx, ny, nz = oracle.direction(W1, W2)
    mx, my, mz = oracle.direction(~W1, W2)     # U2 -> 1-U2: mu -> -mu, sin(theta) unchanged
    assert np.array_equal(mx, -nx) and np.array_equal(my, ny) and np.array_equal(mz, nz)
    px, py, pz = oracle.direction(W1, ~W2)     # U3 -> 1-U3: phi -> -phi
    assert np.array_equal(px, nx) and np.array_equal(py, ny) and np.array_equal(pz, -nz)


def test_isotropy_of_direction_cosines():
    # means 0 and variances 1/3 for every component, whatever kappa
    n = 2_000_000
    _, w1, w2 = oracle.words(n, 31337, 0)
    comps = oracle.direction(w1, w2)
    for c in comps:
        assert abs(c.mean()) < 5 * math.sqrt(1 / 3 / n)
        assert abs((c * c).mean() - 1 / 3) < 5 * math.sqrt((1 / 5 - 1 / 9) / n)
    for i in range(3):
        for j in range(i + 1, 3):
            assert abs((comps[i] * comps[j]).mean()) < 5 * math.sqrt(1 / 15 / n) * 1.5
    # azimuth is uniform: quadrant counts of (ny, nz)
    quad = (comps[1] > 0).astype(int) * 2 + (comps[2] > 0).astype(int)
    cnt = np.bincount(quad, minlength=4)
    assert np.max(np.abs(cnt - n / 4)) < 5 * math.sqrt(n * 3 / 16)
