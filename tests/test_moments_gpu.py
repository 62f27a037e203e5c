"""GPU parity of the fused loader kappagen_sample_cells_moments: per-cell
(sum vx, sum vy, sum vz, sum |v|^2) reduced inside the generating kernel, against the oracle's extended
precision sums of the same particles.

Tolerance (derived from the arithmetic): each summand carries the per-component
tolerance tol of the sampler, and a sum of ppc terms formed in the output type adds at most ppc*eps of the
sum of magnitudes, so  |sum_gpu - sum_ref| <= (tol + ppc*eps) * sum_j (|thermal_j| + |drift|)  per component
(the sampler's own error scale, reading R11), and  |s2_gpu - s2_ref| <= sum_j 2 |v_j| tol (|thermal_j| + |drift|)
+ (ppc+3)*eps * s2_ref  for the sum of squares."""
import numpy as np
import pytest
import torch

import oracle
from gpu_util import TOL, report
from paper_2602_05606_b200 import kappagen as kg
from paper_2602_05606_b200 import workloads as wl

pytestmark = pytest.mark.gpu
EPS = {"f32": 2.0 ** -24, "f64": 2.0 ** -53}


def check_moments(got, ppc, kap, th, drift, stride, seed, offset, dtype):
    dr = None if drift is None else np.asarray(drift, dtype=np.float64)
    k64, t64 = kap.astype(np.float64), th.astype(np.float64)
    want, _ = oracle.cells_moments(ppc, k64, t64, dr, stride, seed, offset)
    v, therm = oracle.sample_cells(ppc, k64, t64, dr, stride, seed, offset, thermal=True)
    g = got.cpu().numpy().astype(np.float64)
    assert g.shape == want.shape
    assert np.array_equal(np.isnan(g), np.isnan(want))
    ok = ~np.isnan(want[:, 0])
    worst = 0.0
    b2 = np.zeros(want.shape[0])
    for q in range(3):
        if dr is None:
            d = 0.0
        elif stride == 0:
            d = abs(dr[q])
        else:
            d = np.repeat(np.abs(dr.reshape(-1, 3)[:, q]), ppc)
        each = np.abs(therm[q]) + d                       # the sampler's error scale per particle (reading R11)
        scale = each.reshape(-1, ppc).sum(axis=1)
        bound = (TOL[dtype] + ppc * EPS[dtype]) * scale + 1e-300
        r = np.abs(g[:, q] - want[:, q])[ok] / bound[ok]
        worst = max(worst, float(r.max(initial=0.0)))
        b2 += (2 * np.abs(v[q]) * TOL[dtype] * each).reshape(-1, ppc).sum(axis=1)
    bound = b2 + (ppc + 3) * EPS[dtype] * want[:, 3] + 1e-300
    worst = max(worst, float((np.abs(g[:, 3] - want[:, 3])[ok] / bound[ok]).max(initial=0.0)))
    return worst


# ppc: 64 -> shuffle tree, direct store (float L=16, double L=32); 8 -> direct with short segments; 256 and 1024
# -> one warp (or more) per cell, shuffle then atomics; 5 and 37 -> groups straddle cells, atomics; 1 -> degenerate
@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("ppc", [64, 8, 4, 2, 256, 1024, 5, 37, 1])
def test_moments_match_oracle_sums(dtype, ppc):
    cfg = wl.CellsConfig(nx=16, ny=8, nz=6 if ppc <= 64 else 2, ppc=ppc)
    npdt = np.float32 if dtype == "f32" else np.float64
    kap, th = wl.cell_arrays(cfg, dtype=npdt)
    drift = np.array(cfg.drift, dtype=npdt)
    planes, mom = kg.sample_cells_moments(ppc, torch.from_numpy(kap).cuda(), torch.from_numpy(th).cuda(),
                                          torch.from_numpy(drift).cuda(), 0, cfg.seed, 1000)
    worst = check_moments(mom, ppc, kap, th, drift, 0, cfg.seed, 1000, dtype)
    report(test="cells_moments", dtype=dtype, ppc=ppc, worst_over_bound=worst)
    assert worst <= 1.0, worst
    # the planes written by the fused call are those of kappagen_sample_cells, bit for bit
    ref = kg.sample_cells(ppc, torch.from_numpy(kap).cuda(), torch.from_numpy(th).cuda(), torch.from_numpy(drift).cuda(),
                          0, cfg.seed, 1000)
    for a, b in zip(planes, ref):
        assert torch.equal(a, b)
    # moments only (NULL planes): same sums; bit-identical where the summation order is fixed (shuffle tree)
    none, mom2 = kg.sample_cells_moments(ppc, torch.from_numpy(kap).cuda(), torch.from_numpy(th).cuda(),
                                         torch.from_numpy(drift).cuda(), 0, cfg.seed, 1000, store=False)
    assert none is None
    g = 4 if dtype == "f32" else 2
    lanes = ppc // g
    if ppc % g == 0 and lanes <= 32 and lanes & (lanes - 1) == 0:
        assert torch.equal(mom, mom2)
    else:
        assert check_moments(mom2, ppc, kap, th, drift, 0, cfg.seed, 1000, dtype) <= 1.0


def test_moments_per_cell_drift_invalid_cells_and_status_codes():
    ppc = 64
    kap = np.array([2.0, 1.5, 3.0, 4.0, 2.5], dtype=np.float32)      # 1.5 invalid
    th = np.array([1.0, 1.0, -1.0, 0.0, 0.3], dtype=np.float32)       # negative theta invalid; 0 = cold cell
    drift = (np.arange(15, dtype=np.float32) * 0.01).reshape(5, 3)
    _, mom = kg.sample_cells_moments(ppc, torch.from_numpy(kap).cuda(), torch.from_numpy(th).cuda(),
                                     torch.from_numpy(drift).cuda(), 1, 3, 0)
    assert check_moments(mom, ppc, kap, th, drift, 1, 3, 0, "f32") <= 1.0
    m = mom.cpu().numpy()
    assert np.all(np.isnan(m[1])) and np.all(np.isnan(m[2]))
    assert np.allclose(m[3, :3], ppc * drift[3], rtol=1e-5)            # cold cell: only the drift
    L = kg.lib()
    k = torch.from_numpy(kap).cuda()
    t = torch.from_numpy(th).cuda()
    ws = torch.empty(5 * 32, dtype=torch.uint8, device="cuda")
    args = (5, ppc, k.data_ptr(), t.data_ptr(), None, 0, 0, 0, kg.F32, None, None, None)
    assert L.kappagen_sample_cells_moments(*args, None, ws.data_ptr(), ws.numel(), None) == kg.ENULL
    assert L.kappagen_sample_cells_moments(*args, mom.data_ptr() + 4, ws.data_ptr(), ws.numel(), None) == kg.EALIGN
    assert L.kappagen_sample_cells_moments(*args, mom.data_ptr(), ws.data_ptr(), 16, None) == kg.EWORKSPACE
    assert L.kappagen_sample_cells_moments(0, ppc, None, None, None, 0, 0, 0, kg.F32, None, None, None, None, None, 0, None) == kg.OK


def test_config4_moments_full_size_sampled_cells_and_energy():
    """configs[3] at full size (256x256x64 cells x 64): moments-only call; oracle sums on sampled z planes;
    the mean drift <vz> = 0.02 and the summed energy against Eq. (5) per cell (kappa in [2,5): heavy tails, so
    the energy check is on the median over cells of s2/(ppc theta^2) / (3 kappa/(2 kappa - 3)), a robust statistic)."""
    cfg = wl.C4
    kap, th = wl.cell_arrays(cfg)
    drift = np.array(cfg.drift, dtype=np.float32)
    kd, td, dd = torch.from_numpy(kap).cuda(), torch.from_numpy(th).cuda(), torch.from_numpy(drift).cuda()
    _, mom = kg.sample_cells_moments(cfg.ppc, kd, td, dd, 0, cfg.seed, 0, store=False)
    per = cfg.nx * cfg.ny
    for iz in (0, 31, 63):
        c0, c1 = iz * per, iz * per + 2048
        worst = check_moments(mom[c0:c1], cfg.ppc, kap[c0:c1], th[c0:c1], drift, 0, cfg.seed, c0 * cfg.ppc, "f32")
        report(test="config4_moments", iz=iz, worst_over_bound=worst)
        assert worst <= 1.0, worst
    m = mom.double()
    n = cfg.ncell * cfg.ppc
    mean_vz = float(m[:, 2].sum()) / n
    assert abs(mean_vz - 0.02) < 2e-5, mean_vz
    k64 = torch.from_numpy(kap.astype(np.float64)).cuda()
    t64 = torch.from_numpy(th.astype(np.float64)).cuda()
    thermal2 = (m[:, 3] - 2 * 0.02 * m[:, 2] + cfg.ppc * 0.02 ** 2) / (cfg.ppc * t64 ** 2)
    ratio = thermal2 / (3 * k64 / (2 * k64 - 3))
    med = float(ratio.median())
    assert 0.8 < med < 1.0, med          # medians of heavy-tailed sample means sit below the mean
