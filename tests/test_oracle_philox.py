"""Pins for oracle S1 (Philox4x32-10) and the particle -> (counter, key) layout (R6)."""
import os

import numpy as np

import oracle

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "philox4x32_10_kat.txt")


def _kats():
    out = []
    with open(GOLDEN) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            lhs, rhs = line.split("->")
            ctr, key = lhs.split(";")
            out.append(([int(x, 16) for x in ctr.split()], [int(x, 16) for x in key.split()],
                        [int(x, 16) for x in rhs.split()]))
    return out


def test_known_answer_vectors():
    kats = _kats()
    assert len(kats) == 3
    for ctr, key, want in kats:
        got = oracle.philox4x32_10(ctr, key)
        assert [int(x) for x in got] == want


def test_particle_zero_is_first_kat():
    # seed 0, particle 0 -> counter (0,0,0,0), key (0,0): the first published vector; w3 is dropped.
    w0, w1, w2 = oracle.words(1, 0, 0)
    assert (int(w0[0]), int(w1[0]), int(w2[0])) == (0x6627E8D5, 0xE169C58D, 0xBC57AC4C)


def test_layout_counter_is_particle_index_key_is_seed():
    # words(seed, offset+i) must equal Philox(ctr=(lo(g),hi(g),0,0), key=(lo(seed),hi(seed))).
    seed = 0xA4093822_299F31D0
    for g in (0, 1, 2, 0xFFFFFFFF, 0x1_0000_0000, 0x1234_5678_9ABC_DEF0, 2**64 - 1):
        want = oracle.philox4x32_10([g & 0xFFFFFFFF, g >> 32, 0, 0], [seed & 0xFFFFFFFF, seed >> 32])
        w0, w1, w2 = oracle.words(1, seed, g)
        assert (w0[0], w1[0], w2[0]) == (want[0], want[1], want[2])


def test_offset_counts_particles_and_carries_into_high_word():
    seed = 5
    base = 2**32 - 1000
    a = oracle.words(2000, seed, base)
    b1 = oracle.words(1000, seed, base)
    b2 = oracle.words(1000, seed, base + 1000)  # crosses g = 2^32
    for k in range(3):
        assert np.array_equal(a[k], np.concatenate([b1[k], b2[k]]))
    # g = 2^32 differs from g = 0 (the carry reaches ctr[1])
    assert oracle.words(1, seed, 2**32)[0][0] != oracle.words(1, seed, 0)[0][0]
    # high half of the seed reaches key[1]
    assert oracle.words(1, 1, 0)[0][0] != oracle.words(1, 1 + 2**32, 0)[0][0]


def test_words_look_uniform():
    # not a pin of the constants (the KATs are), just a guard against a truncated round loop
    w0, w1, w2 = oracle.words(200_000, 99, 0)
    for w in (w0, w1, w2):
        u = (w.astype(np.float64) + 0.5) / 2**32
        assert abs(u.mean() - 0.5) < 5 * (1 / 12**0.5) / 200_000**0.5
        bits = np.unpackbits(w.view(np.uint8)).mean()
        assert abs(bits - 0.5) < 5 * 0.5 / (32 * 200_000) ** 0.5
    assert abs(np.corrcoef(w0.astype(np.float64), w1.astype(np.float64))[0, 1]) < 0.02
