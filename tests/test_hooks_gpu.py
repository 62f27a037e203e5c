"""The measurement hooks and the workspace variant of the end-to-end call (include/kappagen.h):
kappagen_philox_planes (bit-exact against oracle.words, every path), kappagen_sample_host_ws (same bits as
kappagen_sample, nothing allocated inside), kappagen_pipe_probe (sane, reproducible pipe rates)."""
import numpy as np
import pytest
import torch

import oracle
from paper_2602_05606_b200 import kappagen as kg
from gpu_util import u32

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("seed,offset,n", [(0, 0, 100_003), (42, 2**32 - 70_001, 140_002), (7, 2**64 - 9, 4100),
                                           ((5 << 32) | 9, 2**33 - 2048 * 3 - 5, 2048 * 7 + 3), (1, 0, 1), (1, 5, 3)])
def test_philox_planes_bit_exact(seed, offset, n):
    got = kg.philox_planes(n, seed, offset)
    want = oracle.words(n, seed, offset)
    for g, w in zip(got, want):
        assert np.array_equal(u32(g), w)
    # element-aligned planes: the scalar-store instantiation writes the same words and nothing else
    buf = [torch.full((n + 9,), -1, dtype=torch.int32, device="cuda") for _ in range(3)]
    kg.philox_planes(n, seed, offset, out=tuple(b[1:1 + n] for b in buf))
    for b, w in zip(buf, want):
        assert np.array_equal(u32(b[1:1 + n]), w)
        assert int(b[0]) == -1 and bool((b[1 + n:] == -1).all())


@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_sample_host_ws_equals_sample(dtype):
    n = (1 << 22) * 2 + 12345                                    # three chunks, the last one ragged
    tdt = torch.float32 if dtype == "f32" else torch.float64
    ws = torch.empty(kg.sample_host_workspace_bytes(n, dtype), dtype=torch.uint8, device="cuda")
    sa, sb = torch.cuda.Stream(), torch.cuda.Stream()
    host = tuple(torch.empty(n, dtype=tdt, pin_memory=True) for _ in range(3))
    kg.sample_host_ws(n, 1.6, 0.5, 77, 2**32 - n // 2, dtype, host, ws, sa, sb)
    dev = kg.sample(n, 1.6, 0.5, 77, 2**32 - n // 2, dtype)
    for h, d in zip(host, dev):
        assert torch.equal(h, d.cpu())
    again = kg.sample_host(n, 1.6, 0.5, 77, 2**32 - n // 2, dtype)
    for h, a in zip(host, again):
        assert torch.equal(h, a)
    with pytest.raises(kg.KappagenError) as e:
        kg.sample_host_ws(n, 1.6, 0.5, 77, 0, dtype, host, ws, sa, sa)
    assert e.value.status == kg.EINVAL
    with pytest.raises(kg.KappagenError) as e:
        kg.sample_host_ws(n, 1.6, 0.5, 77, 0, dtype, host, ws[:1024], sa, sb)
    assert e.value.status == kg.EWORKSPACE


def test_pipe_probe_rates():
    assert kg.pipe_probe_count() >= 16
    rates = {}
    for mix in range(6):                                          # the six single-kind mixes
        cyc, counts = kg.pipe_probe(mix, 8, 1024)
        (kind, cnt), = counts.items()
        rates[kind] = (cyc - 0.4) / cnt                           # ~3 loop instructions per iteration
    # one warp instruction per scheduler: quarter-rate wide multiply, half-rate ALU / FP64 / IMAD, 8-cycle MUFU
    assert 3.8 <= rates["IMAD.WIDE.U32"] <= 5.5, rates
    assert 1.8 <= rates["LOP3"] <= 2.4 and 1.8 <= rates["FFMA2"] <= 2.4 and 1.8 <= rates["DFMA"] <= 2.6, rates
    assert 7.5 <= rates["MUFU.EX2"] <= 8.6 and 1.8 <= rates["IMAD"] <= 2.5, rates
    with pytest.raises(kg.KappagenError):
        kg.pipe_probe(kg.pipe_probe_count(), 8, 10)


@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_prepared_workspace_gives_the_bits_of_sample_cells(dtype):
    """Table I lines 1-4 "are required only once": kappagen_cells_prepare once, then
    kappagen_sample_cells_prepared for several (ppc, seed, offset) -- each bit-identical to kappagen_sample_cells."""
    npd = np.float32 if dtype == "f32" else np.float64
    rng = np.random.Generator(np.random.PCG64(8))
    ncell = 777
    kap = torch.from_numpy((1.6 + 6 * rng.random(ncell)).astype(npd)).cuda()
    th = torch.from_numpy((0.1 + rng.random(ncell)).astype(npd)).cuda()
    drift = torch.from_numpy((0.05 * rng.standard_normal(3 * ncell)).astype(npd)).cuda()
    ws = kg.cells_prepare(kap, th, drift, 1)
    for ppc, seed, offset in ((64, 1, 0), (37, 2, 2**32 - 1000), (256, 3, 12345)):
        got = kg.sample_cells_prepared(ncell, ppc, ws, seed, offset, dtype)
        want = kg.sample_cells(ppc, kap, th, drift, 1, seed, offset)
        for g, w in zip(got, want):
            assert torch.equal(g, w)
    with pytest.raises(kg.KappagenError) as e:
        kg.sample_cells_prepared(ncell, 64, ws[:100], 1, 0, dtype)
    assert e.value.status == kg.EWORKSPACE
