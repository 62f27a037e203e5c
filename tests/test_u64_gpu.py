"""GPU parity of the 64-bit-U1 variant (kappagen_sample_flags with KAPPAGEN_U1_64; SURVEY.md section 8(f) f2,
DESIGN.md reading R20): all four Philox words bit-exact, velocities within the north_star tolerances
against the oracle's sample_u64 over random streams and over (w0, w3) pairs that stress both ends of the
64-bit uniform (where 1 - U1 is as small as 2^-65 and the speed reaches v/theta ~ 1e9 at kappa = 1.6)."""
import numpy as np
import pytest
import torch

import oracle
from gpu_util import TOL, max_rel_err, report, u32
from paper_2602_05606_b200 import kappagen as kg
from test_oracle_u64 import edge_pairs

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("seed,offset,n", [(0, 0, 100_000), (99, 2**32 - 1001, 2003), (7, 2**64 - 500, 1000)])
def test_four_words_bit_exact(seed, offset, n):
    got = kg.words4(n, seed, offset)
    (_, _, _), w3 = oracle.sample_u64(n, 2.0, 1.0, seed, offset % 2**64, return_w3=True)
    want = oracle.words(n, seed, offset % 2**64) + (w3,)
    for g, w in zip(got, want):
        assert np.array_equal(u32(g), w)


@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("kappa", [1.6, 2.0, 3.0, 10.0])
def test_sample_u64_parity(kappa, dtype):
    n, theta, seed, offset = 300_007, 0.7, 5, 2**33 - 1234
    got = kg.sample_flags(n, kappa, theta, seed, offset, dtype, kg.U1_64)
    want = oracle.sample_u64(n, kappa, theta, seed, offset)
    err = max_rel_err(got, want)
    report(test="sample_u64", kappa=kappa, dtype=dtype, max_rel_err=err)
    assert err <= TOL[dtype], err
    # flags = 0 is kappagen_sample, bit for bit; the flag changes the speed only slightly in the bulk
    plain = kg.sample_flags(n, kappa, theta, seed, offset, dtype, 0)
    ref = kg.sample(n, kappa, theta, seed, offset, dtype)
    assert all(torch.equal(a, b) for a, b in zip(plain, ref))
    assert not torch.equal(plain[0], got[0])


@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("kappa", [1.6, 2.0, 4.0, 10.0])
def test_edge_pairs_of_the_64_bit_uniform(kappa, dtype):
    w0, w3 = edge_pairs()
    rng = np.random.Generator(np.random.PCG64(3))
    w1 = rng.integers(0, 2**32, w0.size, dtype=np.uint64).astype(np.uint32)
    w2 = rng.integers(0, 2**32, w0.size, dtype=np.uint64).astype(np.uint32)
    t = [torch.from_numpy(w.view(np.int32)).cuda() for w in (w0, w1, w2, w3)]
    got = kg.velocity_of_words_u64(t[0], t[1], t[2], t[3], kappa, 1.0, dtype)
    want = oracle.velocity_of_words_u64(w0, w1, w2, w3, kappa, 1.0)
    err = max_rel_err(got, want)
    report(test="edge_pairs_u64", kappa=kappa, dtype=dtype, max_rel_err=err,
           vmax_over_theta=float(np.sqrt(sum(w**2 for w in want)).max()))
    assert err <= TOL[dtype], err
    assert all(bool(torch.isfinite(g).all()) for g in got)


def test_unknown_flag_is_rejected_and_chunks_continue():
    L = kg.lib()
    x = torch.empty(16, device="cuda")
    assert L.kappagen_sample_flags(16, 2.0, 1.0, 0, 0, kg.F32, 2, x.data_ptr(), x.data_ptr(), x.data_ptr(), None) == kg.EINVAL
    n = 10_001
    one = kg.sample_flags(n, 1.6, 1.0, 123, 10, "f32", kg.U1_64)
    a = kg.sample_flags(4000, 1.6, 1.0, 123, 10, "f32", kg.U1_64)
    b = kg.sample_flags(n - 4000, 1.6, 1.0, 123, 4010, "f32", kg.U1_64)
    for o, p, q in zip(one, a, b):
        assert torch.equal(o, torch.cat([p, q]))
