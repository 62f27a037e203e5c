"""kappagen_math_planes, the tracked "math + stores without Philox" ceiling: it must run the sampler's own S2-S6 on the
affine words its header states, so its output is compared bit for bit with kappagen_velocity_of_words_tile (the
sampler's straight-line tile body fed from memory) on those words, and with the oracle within tolerance."""
import numpy as np
import pytest
import torch

import oracle
from gpu_util import TOL, max_rel_err
from paper_2602_05606_b200 import kappagen as kg

pytestmark = pytest.mark.gpu


def affine_words(n, offset):
    g = (np.arange(n, dtype=np.uint64) + np.uint64(offset)) & np.uint64(0xFFFFFFFF)
    return [((g * np.uint64(m) + np.uint64(a)) & np.uint64(0xFFFFFFFF)).astype(np.uint32)
            for m, a in zip(kg.MATH_PLANES_MUL, kg.MATH_PLANES_ADD)]


@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("n,offset", [(3 * 3072 * 5 + 17, 0), (40_000, 2**32 - 9000), (5, 123)])
@pytest.mark.parametrize("kappa,theta", [(2.0, 0.1), (4.1, 1e-12)])
def test_math_planes_is_the_sampler_math_on_affine_words(dtype, n, offset, kappa, theta):
    w = affine_words(n, offset)
    dw = [torch.from_numpy(x.view(np.int32)).cuda() for x in w]
    got = kg.math_planes(n, kappa, theta, offset, dtype)
    ref = kg.velocity_of_words_tile(dw[0], dw[1], dw[2], kappa, theta, dtype)
    for q in range(3):
        assert torch.equal(got[q], ref[q])
    want = oracle.velocity_of_words(w[0], w[1], w[2], kappa, theta)
    assert max_rel_err(got, want) <= TOL[dtype]


def test_math_planes_rejects_misaligned_planes_and_bad_parameters():
    buf = [torch.empty(129, dtype=torch.float32, device="cuda") for _ in range(3)]
    with pytest.raises(kg.KappagenError) as e:
        kg.math_planes(128, 2.0, 1.0, 0, "f32", out=tuple(b[1:] for b in buf))
    assert e.value.status == kg.EALIGN
    with pytest.raises(kg.KappagenError) as e:
        kg.math_planes(128, 1.5, 1.0, 0, "f32")
    assert e.value.status == kg.EINVAL
