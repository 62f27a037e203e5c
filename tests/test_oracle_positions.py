"""Pins for oracle.positions (the position half of the PIC particle record, kappagen_load_cells; DESIGN.md
reading R22: positions are not in the paper, they come from a second Philox4x32-10 block of the same particle,
counter (lo32 g, hi32 g, 0, 2)).

The pin is an INDEPENDENT Philox4x32-10 written here in pure Python integers from the SC'11 description and
itself checked against the published known-answer vectors (tests/golden/philox4x32_10_kat.txt); on top of it the
definition ((w >> (32-bits)) + 1/2)/2^bits is evaluated in exact rational arithmetic.  Plus what any mistake in
the counter layout, the word order or the bit selection would break: exact representability in the record's
element type, distinctness from the velocity block, uniformity, independence from the velocity uniforms, and
invariance under chunking.
"""
from fractions import Fraction

import numpy as np

import oracle
from test_oracle_philox import _kats

M0, M1, W0, W1 = 0xD2511F53, 0xCD9E8D57, 0x9E3779B9, 0xBB67AE85
MASK = 0xFFFFFFFF


def philox_py(ctr, key):
    c0, c1, c2, c3 = ctr
    k0, k1 = key
    for r in range(10):
        p0, p1 = M0 * c0, M1 * c2
        c0, c1, c2, c3 = (p1 >> 32) ^ c1 ^ k0, p1 & MASK, (p0 >> 32) ^ c3 ^ k1, p0 & MASK
        k0, k1 = (k0 + W0) & MASK, (k1 + W1) & MASK
    return [c0, c1, c2, c3]


def test_the_python_philox_reproduces_the_published_vectors():
    for ctr, key, want in _kats():
        assert philox_py(ctr, key) == want


def test_positions_are_the_second_block_counter_word3_equals_2():
    seed = (0x1234ABCD << 32) | 0x0BADF00D
    for offset in (0, 2**32 - 3, 2**40 + 17, 2**64 - 2):
        n = 6
        for bits in (23, 32):
            fx, fy, fz = oracle.positions(n, seed, offset, bits)
            for i in range(n):
                g = (offset + i) % 2**64
                w = philox_py([g & MASK, g >> 32, 0, 2], [seed & MASK, seed >> 32])
                for q, f in enumerate((fx, fy, fz)):
                    want = Fraction(2 * (w[q] >> (32 - bits)) + 1, 2 ** (bits + 1))
                    assert Fraction(float(f[i])) == want          # exact: the double holds the midpoint exactly


def test_exactly_representable_in_the_record_type_and_inside_the_open_interval():
    f = np.concatenate(oracle.positions(200_000, 5, 0, 23))
    assert np.array_equal(f.astype(np.float32).astype(np.float64), f)   # 23-bit midpoints fit a float exactly
    assert f.min() > 0.0 and f.max() < 1.0
    k = f * 2**24                                                        # odd integers below 2^24
    assert np.array_equal(k, np.round(k)) and np.all(k.astype(np.int64) % 2 == 1)
    g = np.concatenate(oracle.positions(1000, 5, 0, 32))
    assert np.array_equal(g * 2**33, np.round(g * 2**33)) and g.min() > 0.0 and g.max() < 1.0


def test_distinct_from_the_velocity_block_and_chunk_invariant():
    n, seed = 5000, 9
    fx, fy, fz = oracle.positions(n, seed, 0, 32)
    w0, w1, w2 = oracle.words(n, seed, 0)
    u = [(w.astype(np.float64) + 0.5) / 2**32 for w in (w0, w1, w2)]
    for a in (fx, fy, fz):
        for b in u:
            assert np.mean(a == b) < 1e-3                                 # another block, not the velocity words again
    a = oracle.positions(3000, seed, 100, 23)
    b = oracle.positions(1000, seed, 1100, 23)
    for q in range(3):
        assert np.array_equal(a[q][1000:2000], b[q])


def test_uniform_and_independent_of_the_velocity_uniforms():
    n, seed = 400_000, 21
    f = oracle.positions(n, seed, 0, 23)
    band = 1.95 / np.sqrt(n)                                              # 99.9 % Kolmogorov quantile
    grid = (np.arange(1, n + 1) - 0.5) / n
    for a in f:
        ks = np.max(np.abs(np.sort(a) - grid)) + 0.5 / n
        assert ks <= band, ks
        assert abs(a.mean() - 0.5) < 5 * np.sqrt(1 / 12 / n)
        assert abs(a.var() - 1 / 12) < 5 * np.sqrt(1 / 180 / n)
    w = oracle.words(n, seed, 0)
    u = [(x.astype(np.float64) + 0.5) / 2**32 for x in w]
    lim = 5 / np.sqrt(n)
    for i, a in enumerate(f):
        for j, b in enumerate(f):
            if i < j:
                assert abs(np.corrcoef(a, b)[0, 1]) < lim
        for b in u:
            assert abs(np.corrcoef(a, b)[0, 1]) < lim
