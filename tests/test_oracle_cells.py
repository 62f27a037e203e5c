"""oracle_sample_cells (PIC-style, BASELINE.json configs[3]) reduces to oracle_sample cell by cell;
input recipe of workloads.cell_arrays."""
import numpy as np

import oracle
from paper_2602_05606_b200 import workloads as wl


def test_cells_reduce_to_uniform_sample_plus_drift():
    ppc, seed, offset = 5, 7, 1000
    kappa = np.array([2.0, 3.5, 4.75, 2.0])
    theta = np.array([0.05, 0.06, 0.0, 0.07])
    drift = np.array([0.0, 0.0, 0.02])
    (vx, vy, vz), (tx, ty, tz) = oracle.sample_cells(ppc, kappa, theta, drift, 0, seed, offset, thermal=True)
    for cell in range(4):
        sx, sy, sz = oracle.sample(ppc, kappa[cell], theta[cell], seed, offset + cell * ppc)
        sl = slice(cell * ppc, (cell + 1) * ppc)
        assert np.array_equal(tx[sl], sx) and np.array_equal(ty[sl], sy) and np.array_equal(tz[sl], sz)
        assert np.array_equal(vx[sl], sx) and np.array_equal(vy[sl], sy)
        assert np.allclose(vz[sl], sz + 0.02, rtol=0, atol=2.3e-16 * 0.25)   # one rounding vs two
    assert np.all(tx[10:15] == 0) and np.all(vz[10:15] == 0.02)        # theta = 0 -> cold cell


def test_per_cell_drift_stride_and_invalid_cells_are_nan():
    ppc = 3
    kappa = np.array([2.0, 1.5, 3.0])        # 1.5 is outside kappa > 3/2
    theta = np.array([1.0, 1.0, -1.0])       # negative theta is invalid too
    drift = np.arange(9, dtype=np.float64).reshape(3, 3)
    vx, vy, vz = oracle.sample_cells(ppc, kappa, theta, drift, 1, 3, 0)
    sx, sy, sz = oracle.sample(ppc, 2.0, 1.0, 3, 0)
    assert np.allclose(vx[:3], sx + 0.0) and np.allclose(vy[:3], sy + 1.0) and np.allclose(vz[:3], sz + 2.0)
    assert np.all(np.isnan(vx[3:])) and np.all(np.isnan(vy[3:])) and np.all(np.isnan(vz[3:]))
    nx, ny, nz = oracle.sample_cells(ppc, kappa[:1], theta[:1], None, 0, 3, 0)
    assert np.array_equal(nx, sx) and np.array_equal(nz, sz)


def test_cell_arrays_recipe():
    cfg = wl.CellsConfig(nx=8, ny=4, nz=6, ppc=2)
    kap, th = wl.cell_arrays(cfg)
    assert kap.dtype == np.float32 and kap.size == cfg.ncell == th.size
    assert kap.min() >= 2.0 and kap.max() <= 5.0 and kap.std() > 0.5
    th3 = th.reshape(cfg.nz, cfg.ny, cfg.nx)
    assert np.all(th3 == th3[:, :1, :1])                     # theta depends on z only
    assert np.all(np.diff(th3[:, 0, 0]) > 0)                 # tanh profile
    assert np.allclose(th3[cfg.nz // 2 - 1, 0, 0] + th3[cfg.nz // 2, 0, 0], 2 * cfg.theta0, rtol=1e-6)
    # a sub-range of planes sees the same values as the full grid
    k2, t2 = wl.cell_arrays(cfg, z_planes=(2, 4))
    per = cfg.nx * cfg.ny
    assert np.array_equal(k2, kap[2 * per:4 * per]) and np.array_equal(t2, th[2 * per:4 * per])


def test_shard_range_partitions():
    for n in (0, 1, 10, 1 << 28, 1000003):
        for world in (1, 2, 3, 8):
            edges = [wl.shard_range(n, r, world) for r in range(world)]
            assert edges[0][0] == 0 and edges[-1][1] == n
            assert all(edges[r][1] == edges[r + 1][0] for r in range(world - 1))
            sizes = [e - b for b, e in edges]
            assert max(sizes) - min(sizes) <= 1
