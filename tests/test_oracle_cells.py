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


# ------------------------------------------------------------------ fused loader moments
def test_moments_of_one_particle_cells_are_the_pinned_velocities():
    """ppc = 1: the 'sums' are the single particle's (vx, vy, vz, |v|^2), which test_oracle_inverse /
    test_oracle_direction pin independently (50-digit Table I, round trip, closed forms)."""
    n = 257
    kappa = np.linspace(1.6, 10.0, n)
    theta = np.linspace(0.01, 2.0, n)
    drift = np.array([0.1, -0.2, 0.02])
    mom, abs1 = oracle.cells_moments(1, kappa, theta, drift, 0, 11, 5)
    (vx, vy, vz) = oracle.sample_cells(1, kappa, theta, drift, 0, 11, 5)
    assert np.allclose(mom[:, 0], vx, rtol=2e-16, atol=0) and np.allclose(mom[:, 1], vy, rtol=2e-16, atol=0)
    assert np.allclose(mom[:, 2], vz, rtol=2e-16, atol=0)
    assert np.allclose(mom[:, 3], vx * vx + vy * vy + vz * vz, rtol=1e-15, atol=0)
    assert np.allclose(abs1, np.abs(vx) + np.abs(vy) + np.abs(vz), rtol=1e-15, atol=0)


def test_moments_are_the_cellwise_sums_in_extended_precision():
    """Brute force: numpy longdouble sums of sample_cells' output, cell by cell, a second route to the same
    numbers (per-cell drift with stride 1, ppc not a multiple of anything, one cold and one invalid cell)."""
    ppc = 37
    kappa = np.array([2.0, 3.5, 4.75, 1.2, 6.0])
    theta = np.array([0.05, 0.06, 0.0, 0.07, 1.0])
    drift = np.arange(15, dtype=np.float64).reshape(5, 3) * 0.01
    mom, abs1 = oracle.cells_moments(ppc, kappa, theta, drift, 1, 7, 123456789)
    vx, vy, vz = oracle.sample_cells(ppc, kappa, theta, drift, 1, 7, 123456789)
    for cell in range(5):
        sl = slice(cell * ppc, (cell + 1) * ppc)
        if cell == 3:
            assert np.all(np.isnan(mom[cell])) and np.isnan(abs1[cell])
            continue
        x, y, z = (a[sl].astype(np.longdouble) for a in (vx, vy, vz))
        want = np.array([x.sum(), y.sum(), z.sum(), (x * x + y * y + z * z).sum()], dtype=np.float64)
        scale = np.array([np.abs(x).sum(), np.abs(y).sum(), np.abs(z).sum(), want[3]], dtype=np.float64)
        assert np.all(np.abs(mom[cell] - want) <= 4e-16 * scale + 1e-300)
    assert np.allclose(mom[2, :3], ppc * drift[2]) and np.isclose(mom[2, 3], ppc * np.sum(drift[2] ** 2))   # cold cell


def test_energy_density_of_many_cells_matches_eq5_with_the_papers_energy_error():
    """Eq. (5): <v^2> = 3 kappa theta^2 / (2 kappa - 3); the approximate generator's own
    value differs by the paper's energy error, 'within 1e-3' away from kappa ~ 4.1: at
    kappa = 6 the mean of the per-cell sum of v^2, drift removed, must sit within 5 sigma + 1e-3 of Eq. (5).
    Var(x) = kappa^2 (15/4)/((kappa-3/2)(kappa-5/2)) - <x>^2 for the beta-prime variable."""
    kappa0, theta0, ppc, ncell = 6.0, 0.3, 64, 4096
    drift = np.array([0.0, 0.0, 0.02])
    mom, _ = oracle.cells_moments(ppc, np.full(ncell, kappa0), np.full(ncell, theta0), drift, 0, 3, 0)
    n = ppc * ncell
    # sum (v + d)^2 = sum v^2 + 2 d . sum v + n d^2  ->  thermal <v^2>
    sum_v = mom[:, :3].sum(axis=0) - n * drift
    v2 = (mom[:, 3].sum() - 2.0 * drift @ sum_v - n * drift @ drift) / n / theta0 ** 2
    exact = 3 * kappa0 / (2 * kappa0 - 3)
    var = kappa0 ** 2 * 3.75 / ((kappa0 - 1.5) * (kappa0 - 2.5)) - exact ** 2
    assert abs(v2 - exact) <= 5 * np.sqrt(var / n) + 1e-3 * exact
    # momentum: <v> = drift within 5 sigma, sigma^2 = <v^2>/3 per component
    assert np.all(np.abs(sum_v / n) <= 5 * theta0 * np.sqrt(exact / 3 / n))
