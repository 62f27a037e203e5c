"""Very many particles per cell (ppc above ~6.4e4, where (tile + ppc) * ppc >= 2^32 and the 32-bit multiply-high that
finds a group's cell inside a tile is no longer exact).  Such calls used to leave the straight-line tile path; they now
stay on it and find the cell by one compare (a tile then touches at most two cells: cells_ahead() in kernels.cuh).
Checked: the tile path (16-byte aligned planes) against the guarded per-group path (planes shifted by one element, which
the header promises "writes the same values") bit for bit, the particle records against the planes, the cell ids, the
fused moments, and one case against the oracle."""
import numpy as np
import pytest
import torch

import oracle
from gpu_util import TOL, rel_err
from paper_2602_05606_b200 import kappagen as kg

pytestmark = pytest.mark.gpu

TD = {"f32": torch.float32, "f64": torch.float64}
PPCS = [1 << 17, 70000, 65540, 1 << 16, 262148]          # 2^16 still has its multiply-high constant in double (tile 1024)


def _cells(dtype, ncell):
    rng = np.random.Generator(np.random.PCG64(31))
    kap = torch.tensor(rng.uniform(1.7, 6.0, ncell), dtype=TD[dtype], device="cuda")
    th = torch.tensor(rng.uniform(0.2, 1.5, ncell), dtype=TD[dtype], device="cuda")
    drift = torch.tensor(rng.normal(0, 0.1, (ncell, 3)), dtype=TD[dtype], device="cuda")
    return kap, th, drift


@pytest.mark.parametrize("ppc", PPCS)
@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_tile_path_equals_guarded_path_for_large_ppc(dtype, ppc):
    ncell = 5
    n = ncell * ppc
    kap, th, drift = _cells(dtype, ncell)
    seed, offset = 77, 2**32 - 3 * ppc - 1000                         # crosses a 2^32 counter boundary inside a cell
    tile = kg.sample_cells(ppc, kap, th, drift, 1, seed, offset)
    buf = [torch.empty(n + 1, dtype=TD[dtype], device="cuda") for _ in range(3)]
    guarded = kg.sample_cells(ppc, kap, th, drift, 1, seed, offset, out=tuple(b[1:] for b in buf))
    for q in range(3):
        assert torch.equal(tile[q], guarded[q])
    rec = kg.load_cells(ppc, kap, th, drift, 1, None, 100, seed, offset)
    for q in range(3):
        assert torch.equal(rec[:, 4 + q], tile[q])
    ids = rec[:, 3].contiguous().view(torch.int32 if dtype == "f32" else torch.int64)
    assert torch.equal(ids.to(torch.int64), 100 + torch.arange(n, device="cuda") // ppc)
    planes, mom = kg.sample_cells_moments(ppc, kap, th, drift, 1, seed, offset)
    for q in range(3):
        assert torch.equal(planes[q], tile[q])
        want = tile[q].view(ncell, ppc).double().sum(1)
        assert torch.allclose(mom[:, q].double(), want, rtol=2e-3 if dtype == "f32" else 1e-10, atol=ppc * (1e-4 if dtype == "f32" else 1e-12))


def test_large_ppc_against_the_oracle():
    ppc, ncell, dtype = 70000, 3, "f64"
    kap, th, drift = _cells(dtype, ncell)
    got = kg.sample_cells(ppc, kap, th, drift, 1, 9, 12345)
    want, therm = oracle.sample_cells(ppc, kap.cpu().numpy(), th.cpu().numpy(), drift.cpu().numpy().ravel(), 1, 9, 12345, thermal=True)
    d = drift.cpu().numpy()
    for q in range(3):
        scale = np.abs(therm[q]) + np.repeat(np.abs(d[:, q]), ppc)
        assert np.all(np.abs(got[q].cpu().numpy() - want[q]) <= TOL[dtype] * scale)
