"""The only error channel of per-cell inputs (include/kappagen.h, kappagen_sample_cells): a cell with kappa <= 3/2
(PAPER.md:35), theta < 0 or a non-finite value gets NaN in ALL its particles -- in both element types and through every
entry point that reads per-cell parameters (planes, prepared workspace, fused moments, particle records); its
neighbours are untouched.  The NaN pattern is also compared with the oracle's."""
import numpy as np
import pytest
import torch

import oracle
from paper_2602_05606_b200 import kappagen as kg

pytestmark = pytest.mark.gpu

NPDT = {"f32": np.float32, "f64": np.float64}
BAD = {1: ("kappa", 1.5), 4: ("kappa", float("nan")), 6: ("theta", -0.25), 9: ("theta", float("inf")),
       12: ("kappa", float("-inf")), 13: ("kappa", 0.0)}
COLD = 15                                                   # theta == 0 is valid: the cell sits at its drift


def _cells(dtype, ncell=24):
    rng = np.random.Generator(np.random.PCG64(99))
    kap = rng.uniform(1.6, 8.0, ncell).astype(NPDT[dtype])
    th = rng.uniform(0.1, 2.0, ncell).astype(NPDT[dtype])
    good_k, good_t = kap.copy(), th.copy()
    for c, (which, v) in BAD.items():
        (kap if which == "kappa" else th)[c] = v
    th[COLD] = 0.0
    good_t[COLD] = 0.0
    drift = rng.normal(0, 0.1, (ncell, 3)).astype(NPDT[dtype])
    return kap, th, good_k, good_t, drift


def _dev(*arrays):
    return tuple(torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in arrays)


@pytest.mark.parametrize("ppc", [8, 5, 64])
@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_invalid_cells_are_nan_everywhere_and_only_there(dtype, ppc):
    kap, th, good_k, good_t, drift = _cells(dtype)
    ncell = kap.size
    dk, dt, dgk, dgt, dd = _dev(kap, th, good_k, good_t, drift)
    got = kg.sample_cells(ppc, dk, dt, dd, 1, 5, 1000)
    ref = kg.sample_cells(ppc, dgk, dgt, dd, 1, 5, 1000)                 # same cells, all made valid
    want = oracle.sample_cells(ppc, kap.astype(np.float64), th.astype(np.float64), drift.astype(np.float64).ravel(), 1, 5, 1000)
    bad = np.zeros(ncell, dtype=bool)
    bad[list(BAD)] = True
    mask = torch.from_numpy(np.repeat(bad, ppc)).cuda()
    for q in range(3):
        assert torch.isnan(got[q][mask]).all(), "component %d of an invalid cell is not NaN" % q
        assert torch.equal(got[q][~mask], ref[q][~mask])
        assert not torch.isnan(ref[q]).any()
        assert np.array_equal(np.isnan(want[q]), np.repeat(bad, ppc))
    cold = slice(COLD * ppc, (COLD + 1) * ppc)
    for q in range(3):
        assert torch.equal(got[q][cold], dd[COLD, q].expand(ppc))

    # the prepared workspace carries the same NaNs
    ws = kg.cells_prepare(dk, dt, dd, 1)
    prep = kg.sample_cells_prepared(ncell, ppc, ws, 5, 1000, dtype)
    for q in range(3):
        assert torch.equal(torch.isnan(prep[q]), mask) and torch.equal(prep[q][~mask], got[q][~mask])

    # fused moments: NaN sums for invalid cells, in the stored planes too
    planes, mom = kg.sample_cells_moments(ppc, dk, dt, dd, 1, 5, 1000)
    mbad = torch.from_numpy(bad).cuda()
    assert torch.isnan(mom[mbad]).all() and not torch.isnan(mom[~mbad]).any()
    for q in range(3):
        assert torch.equal(torch.isnan(planes[q]), mask)
    _, mom_only = kg.sample_cells_moments(ppc, dk, dt, dd, 1, 5, 1000, store=False)
    assert torch.isnan(mom_only[mbad]).all() and not torch.isnan(mom_only[~mbad]).any()

    # particle records: velocity columns NaN, positions / cell id / weight still written
    rec = kg.load_cells(ppc, dk, dt, dd, 1, None, 0, 5, 1000)
    assert torch.isnan(rec[mask][:, 4:7]).all() and not torch.isnan(rec[~mask][:, 4:7]).any()
    assert not torch.isnan(rec[:, 0:3]).any() and torch.equal(rec[:, 7], torch.ones_like(rec[:, 7]))
