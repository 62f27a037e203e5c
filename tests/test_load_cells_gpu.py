"""kappagen_load_cells (second half): the PIC particle record
{fx, fy, fz, cell_id, vx, vy, vz, weight} against the oracle -- positions and cell ids bit-exact, velocities
within the north_star tolerance relative to |v_thermal| + |drift| (reading R11), and bit-identical to what
kappagen_sample_cells writes; every code path (bulk-copy whole tiles, ragged tail, ppc not a multiple of the
group, tile across a 2^32 counter boundary), both dtypes, guard bands around the record array."""
import numpy as np
import pytest
import torch

import oracle
from paper_2602_05606_b200 import kappagen as kg
from paper_2602_05606_b200 import workloads as wl
from gpu_util import TOL, report

pytestmark = pytest.mark.gpu

NP = {"f32": np.float32, "f64": np.float64}
TD = {"f32": torch.float32, "f64": torch.float64}
IT = {"f32": torch.int32, "f64": torch.int64}
BITS = {"f32": 23, "f64": 32}


def _inputs(ncell, dtype, seed=3, per_cell_drift=False):
    rng = np.random.Generator(np.random.PCG64(seed))
    kap = (1.6 + 8.4 * rng.random(ncell)).astype(NP[dtype])
    th = (0.05 + rng.random(ncell)).astype(NP[dtype])
    drift = (rng.standard_normal(3 * ncell if per_cell_drift else 3) * 0.1).astype(NP[dtype])
    wgt = (0.5 + rng.random(ncell)).astype(NP[dtype])
    return kap, th, drift, wgt


def _check(ncell, ppc, dtype, offset=0, cell_base=0, per_cell_drift=False, weight=True, seed=11):
    kap, th, drift, wgt = _inputs(ncell, dtype, per_cell_drift=per_cell_drift)
    n = ncell * ppc
    stride = 1 if per_cell_drift else 0
    dk, dt, dd, dw = (torch.from_numpy(a).cuda() for a in (kap, th, drift, wgt))
    pad = 64
    buf = torch.full((n + 2 * pad, 8), float("nan"), dtype=TD[dtype], device="cuda")
    rec = kg.load_cells(ppc, dk, dt, dd, stride, dw if weight else None, cell_base, seed, offset, out=buf[pad:pad + n])
    torch.cuda.synchronize()
    assert torch.isnan(buf[:pad]).all() and torch.isnan(buf[pad + n:]).all()          # nothing written outside
    got = rec.cpu()
    # positions and ids: bit-exact
    f = oracle.positions(n, seed, offset, BITS[dtype])
    for q in range(3):
        assert np.array_equal(got[:, q].numpy().astype(np.float64), f[q]), "position %d" % q
    ids = got[:, 3].contiguous().view(IT[dtype]).numpy()
    assert np.array_equal(ids, cell_base + np.repeat(np.arange(ncell, dtype=np.int64), ppc))
    want_w = np.repeat(wgt, ppc) if weight else np.ones(n, dtype=NP[dtype])
    assert np.array_equal(got[:, 7].numpy(), want_w)
    # velocities: tolerance against the oracle, bit-identical to kappagen_sample_cells
    want, therm = oracle.sample_cells(ppc, kap, th, drift, stride, seed, offset, thermal=True)
    d3 = drift.astype(np.float64).reshape(-1, 3)
    worst = 0.0
    for q in range(3):
        dq = np.repeat(d3[:, q], ppc) if per_cell_drift else np.full(n, d3[0, q])
        err = np.abs(got[:, 4 + q].numpy().astype(np.float64) - want[q]) / (np.abs(therm[q]) + np.abs(dq))
        worst = max(worst, float(err.max(initial=0.0)))
    assert worst <= TOL[dtype], worst
    planes = kg.sample_cells(ppc, dk, dt, dd, stride, seed, offset)
    for q in range(3):
        assert torch.equal(rec[:, 4 + q], planes[q]), "velocity column %d differs from kappagen_sample_cells" % q
    return worst


@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("ncell,ppc", [(700, 64), (64, 256), (1031, 8), (300, 37), (5000, 4), (9, 1), (3, 5000)])
def test_records_against_the_oracle(ncell, ppc, dtype):
    worst = _check(ncell, ppc, dtype, weight=(ncell % 2 == 1))
    report(test="load_cells", ncell=ncell, ppc=ppc, dtype=dtype, max_rel_err=worst)


@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_per_cell_drift_cell_base_and_counter_carry(dtype):
    _check(200, 64, dtype, offset=2**32 - 5000, cell_base=123456, per_cell_drift=True)
    _check(130, 16, dtype, offset=2**40 + 3, cell_base=2**31 - 130 if dtype == "f32" else 2**40, per_cell_drift=False)


def test_status_codes():
    k = torch.full((4,), 3.0, device="cuda")
    with pytest.raises(kg.KappagenError) as e:
        kg.load_cells(8, k, k, None, 0, None, 2**31 - 3, 0, 0)               # id does not fit int32
    assert e.value.status == kg.EINVAL
    with pytest.raises(kg.KappagenError) as e:
        kg.load_cells(8, k, k, None, 0, None, 0, 0, 0, workspace=torch.empty(16, dtype=torch.uint8, device="cuda"))
    assert e.value.status == kg.EWORKSPACE
    out = kg.load_cells(0, k, k)                                             # ppc = 0: nothing to do
    assert out.shape == (0, 8)


def test_config4_shape_slab_full_parity():
    """BASELINE.json configs[3] shape (x-y planes of 256 x 256 cells x 64 particles, Harris-like theta, drift
    (0, 0, 0.02)): two z planes of the grid as one call with the offsets a rank owning them would use."""
    cfg = wl.C4
    z0, z1 = 30, 32
    kap, th = wl.cell_arrays(cfg, z_planes=(z0, z1))
    ncell = kap.size
    cell_begin = z0 * cfg.nx * cfg.ny
    drift = np.array(cfg.drift, dtype=np.float32)
    n = ncell * cfg.ppc
    rec = kg.load_cells(cfg.ppc, torch.from_numpy(kap).cuda(), torch.from_numpy(th).cuda(), torch.from_numpy(drift).cuda(), 0,
                        None, cell_begin, cfg.seed, cell_begin * cfg.ppc)
    got = rec.cpu()
    f = oracle.positions(n, cfg.seed, cell_begin * cfg.ppc, 23)
    for q in range(3):
        assert np.array_equal(got[:, q].numpy().astype(np.float64), f[q])
    want, therm = oracle.sample_cells(cfg.ppc, kap, th, drift, 0, cfg.seed, cell_begin * cfg.ppc, thermal=True)
    for q in range(3):
        err = np.abs(got[:, 4 + q].numpy().astype(np.float64) - want[q]) / (np.abs(therm[q]) + abs(float(drift[q])))
        assert err.max() <= TOL["f32"]
    ids = got[:, 3].contiguous().view(torch.int32).numpy()
    assert ids[0] == cell_begin and ids[-1] == cell_begin + ncell - 1
