"""The method's edge cases through the code path that SHIPS.

kappagen_sample runs whole tiles through a path of its own -- one Philox head per tile, round 1's product by
constant additions (float), packed pairs (float) / eight interleaved chains (double).  The hooks
kappagen_words_tile and kappagen_velocity_of_words_tile go through exactly those device functions:
  * words: bit-exact against the oracle across 2^32 boundaries of the counter, where the tile path must hand over
    to the per-group and per-particle paths and back;
  * velocities: bit-identical to the scalar hook (kappagen_velocity_of_words) AND within the north_star tolerance
    of the oracle on workloads.edge_words(20000) -- w = 0, 2^32-1, the quarter-turn neighbours, both sides of every
    select -- for all kappa of C2 and the two ends of the accepted range."""
import numpy as np
import pytest
import torch

import oracle
from gpu_util import TAIL_BITS, TOL, rel_err, report, u32
from paper_2602_05606_b200 import kappagen as kg
from paper_2602_05606_b200 import workloads as wl

pytestmark = pytest.mark.gpu

TILE = 2048          # particles per tile of both sample kernels (256 threads x 8 particles)


@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("seed,offset,n", [
    (42, 0, 5 * TILE + 77),                          # whole tiles + ragged tail
    (42, 2**32 - 3 * TILE - 5, 7 * TILE + 3),        # a tile that straddles 2^32: before, across, after
    (7, 2**32 - TILE, 3 * TILE),                     # the boundary exactly at a tile edge
    (7, 2**32 - TILE - 1, 3 * TILE),                 # ... and one particle off it
    (123, 2**33 - 4 * TILE + 1, 8 * TILE),           # high counter word = 1 -> 2
    (5, 2**64 - 3 * TILE - 9, 6 * TILE),             # 64-bit wrap of the counter
    (0xA4093822_299F31D0, 2**40 + 12345, 4 * TILE + 1),
])
def test_words_through_the_tile_path_are_bit_exact(dtype, seed, offset, n):
    got = kg.words_tile(n, seed, offset, dtype)
    want = oracle.words(n, seed, offset % 2**64)
    for g, w in zip(got[:3], want):
        assert np.array_equal(u32(g), w)
    _, w3 = oracle.sample_u64(n, 2.0, 1.0, seed, offset % 2**64, return_w3=True)
    assert np.array_equal(u32(got[3]), w3)
    # and the group path (kappagen_words) agrees with it word for word
    for g, h in zip(got, kg.words4(n, seed, offset)):
        assert torch.equal(g, h)


def edge_triplets(n_random=20000):
    w = wl.edge_words(n_random=n_random)
    rng = np.random.Generator(np.random.PCG64(5))
    w0 = np.concatenate([w, rng.permutation(w), w])
    w1 = np.concatenate([rng.permutation(w), w, w])
    w2 = np.concatenate([rng.permutation(w), rng.permutation(w), w])
    return w0, w1, w2


@pytest.mark.parametrize("kappa", wl.C2_KAPPAS + (1.5001, 1e6))
@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_edge_words_through_the_shipped_tile_body(kappa, dtype):
    w0, w1, w2 = edge_triplets()
    dev = [torch.from_numpy(a.view(np.int32)).cuda() for a in (w0, w1, w2)]
    for theta in (0.37, 3e11):                       # folded and unfolded coefficient forms (float)
        tile = kg.velocity_of_words_tile(*dev, kappa, theta, dtype)
        scalar = kg.velocity_of_words(*dev, kappa, theta, dtype)
        for a, b in zip(tile, scalar):
            assert torch.equal(a, b)                 # packed / interleaved body == scalar chain, bit for bit
        want = oracle.velocity_of_words(w0, w1, w2, kappa, theta)
        errs = np.maximum.reduce([rel_err(g.cpu().numpy(), r) for g, r in zip(tile, want)])
        head, tail = w0 < 2**TAIL_BITS, w0 >= 2**32 - 2**TAIL_BITS
        rep = dict(head=float(errs[head].max()), tail=float(errs[tail].max()), bulk=float(errs[~(head | tail)].max()))
        report(test="edge_words_tile", kappa=kappa, dtype=dtype, theta=theta, **rep)
        assert max(rep.values()) <= TOL[dtype], rep
        assert all(bool(torch.isfinite(g).all()) for g in tile)


@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_edge_words_through_the_tile_body_with_64_bit_u1(dtype):
    w0, w1, w2 = edge_triplets(n_random=4000)
    rng = np.random.Generator(np.random.PCG64(6))
    w3 = rng.permutation(w0)
    dev = [torch.from_numpy(a.view(np.int32)).cuda() for a in (w0, w1, w2, w3)]
    for kappa in (1.6, 4.0):
        tile = kg.velocity_of_words_tile(dev[0], dev[1], dev[2], kappa, 0.5, dtype, w3=dev[3], flags=kg.U1_64)
        scalar = kg.velocity_of_words_u64(*dev, kappa, 0.5, dtype)
        for a, b in zip(tile, scalar):
            assert torch.equal(a, b)
        want = oracle.velocity_of_words_u64(w0, w1, w2, w3, kappa, 0.5)
        err = max(float(rel_err(g.cpu().numpy(), r).max()) for g, r in zip(tile, want))
        assert err <= TOL[dtype], err


@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_sample_is_the_tile_body_on_the_tile_words(dtype):
    """Closes the loop: kappagen_sample == tile body applied to tile words, bit for bit, across a 2^32 boundary."""
    n, seed, off, kappa, theta = 9 * TILE + 5, 42, 2**32 - 4 * TILE - 3, 2.0, 0.1
    w = kg.words_tile(n, seed, off, dtype)
    a = kg.velocity_of_words_tile(w[0], w[1], w[2], kappa, theta, dtype)
    b = kg.sample(n, kappa, theta, seed, off, dtype)
    for x, y in zip(a, b):
        assert torch.equal(x, y)
