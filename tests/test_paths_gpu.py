"""GPU parity of the other entry points: kappagen_sample_cells (BASELINE.json configs[3]),
kappagen_sample_host (the end-to-end path), the packed-pair kernel against the scalar test hook, and
the statistical validation of the rejection baseline (exact Kappa distribution, Eq. (3), Eq. (5))."""
import numpy as np
import pytest
import torch
from scipy import special, stats

import oracle
from gpu_util import TOL, max_rel_err, report, u32
from paper_2602_05606_b200 import kappagen as kg
from paper_2602_05606_b200 import workloads as wl

pytestmark = pytest.mark.gpu


def cells_check(cfg, kap, th, drift, stride, got, cell0=0, dtype="f32"):
    """|got - want| <= tol (|thermal| + |drift|) per component (SURVEY.md 8(c)-F drift rule)."""
    dr = None if drift is None else np.asarray(drift, dtype=np.float64)
    want, therm = oracle.sample_cells(cfg.ppc, kap.astype(np.float64), th.astype(np.float64), dr, stride, cfg.seed,
                                      cell0 * cfg.ppc, thermal=True)
    worst = 0.0
    for q in range(3):
        g = got[q].cpu().numpy().astype(np.float64)
        if dr is None:
            d = 0.0
        elif stride == 0:
            d = abs(dr[q])
        else:
            d = np.repeat(np.abs(dr.reshape(-1, 3)[:, q]), cfg.ppc)
        scale = np.abs(therm[q]) + d
        ok = scale > 0
        worst = max(worst, float(np.max(np.abs(g - want[q])[ok] / scale[ok], initial=0.0)))
        assert np.array_equal(np.isnan(g), np.isnan(want[q]))
    return worst


@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("ppc", [64, 5, 1])
def test_cells_small_grid_full_parity(dtype, ppc):
    cfg = wl.CellsConfig(nx=32, ny=16, nz=12, ppc=ppc)
    npdt = np.float32 if dtype == "f32" else np.float64
    kap, th = wl.cell_arrays(cfg, dtype=npdt)
    drift = np.array(cfg.drift, dtype=npdt)
    got = kg.sample_cells(ppc, torch.from_numpy(kap).cuda(), torch.from_numpy(th).cuda(), torch.from_numpy(drift).cuda(),
                          0, cfg.seed, 0)
    err = cells_check(cfg, kap, th, drift, 0, got, dtype=dtype)
    report(test="cells_small", dtype=dtype, ppc=ppc, max_err_rel_to_thermal_plus_drift=err)
    assert err <= TOL[dtype], err


def test_cells_per_cell_drift_invalid_cells_and_no_drift():
    cfg = wl.CellsConfig(nx=8, ny=8, nz=4, ppc=7)
    kap, th = wl.cell_arrays(cfg)
    kap = kap.copy(); th = th.copy()
    kap[3] = 1.5; th[10] = -1.0; kap[17] = np.nan; th[20] = 0.0          # invalid, invalid, invalid, cold
    rng = np.random.Generator(np.random.PCG64(4))
    drift = rng.normal(0, 0.05, size=(cfg.ncell, 3)).astype(np.float32)
    dk, dt = torch.from_numpy(kap).cuda(), torch.from_numpy(th).cuda()
    got = kg.sample_cells(cfg.ppc, dk, dt, torch.from_numpy(drift).cuda(), 1, cfg.seed, 123)
    want, therm = oracle.sample_cells(cfg.ppc, kap.astype(np.float64), th.astype(np.float64), drift.astype(np.float64).ravel(),
                                      1, cfg.seed, 123, thermal=True)
    for q in range(3):
        g = got[q].cpu().numpy().astype(np.float64)
        assert np.array_equal(np.isnan(g), np.isnan(want[q]))
        ok = ~np.isnan(g)
        scale = np.abs(therm[q]) + np.repeat(np.abs(drift[:, q].astype(np.float64)), cfg.ppc)
        assert np.all(np.abs(g - want[q])[ok] <= TOL["f32"] * scale[ok] + 1e-30)
    for cell in (3, 10, 17):
        assert torch.isnan(got[0][cell * cfg.ppc:(cell + 1) * cfg.ppc]).all()
    cold = slice(20 * cfg.ppc, 21 * cfg.ppc)
    assert torch.equal(got[2][cold], torch.full((cfg.ppc,), float(drift[20, 2]), device="cuda"))
    nod = kg.sample_cells(cfg.ppc, dk, dt, None, 0, cfg.seed, 123)
    for q in range(3):
        g = nod[q].cpu().numpy().astype(np.float64)
        ok = ~np.isnan(g) & (therm[q] != 0)
        assert np.all(np.abs(g - therm[q])[ok] <= TOL["f32"] * np.abs(therm[q])[ok])


def test_cells_equal_uniform_sample_when_parameters_are_uniform():
    ncell, ppc = 1000, 64
    kap = torch.full((ncell,), 2.0, dtype=torch.float32, device="cuda")
    th = torch.full((ncell,), 0.1, dtype=torch.float32, device="cuda")
    a = kg.sample_cells(ppc, kap, th, None, 0, 42, 77)
    b = kg.sample(ncell * ppc, 2.0, float(np.float32(0.1)), 42, 77, "f32")
    for x, y in zip(a, b):          # folded and unfolded coefficient forms differ by roundings only
        assert torch.allclose(x, y, rtol=2e-6, atol=0)


def test_config4_full_size_sampled_parity_and_mean_drift():
    cfg = wl.C4
    kap, th = wl.cell_arrays(cfg)
    drift = np.array(cfg.drift, dtype=np.float32)
    got = kg.sample_cells(cfg.ppc, torch.from_numpy(kap).cuda(), torch.from_numpy(th).cuda(), torch.from_numpy(drift).cuda(),
                          0, cfg.seed, 0)
    torch.cuda.synchronize()
    assert got[0].numel() == 1 << 28
    rng = np.random.Generator(np.random.PCG64(8))
    worst = 0.0
    starts = [0, cfg.ncell - 64] + [int(c) for c in rng.integers(0, cfg.ncell - 64, size=40)]
    for c0 in starts:
        sl = slice(c0 * cfg.ppc, (c0 + 64) * cfg.ppc)
        worst = max(worst, cells_check(cfg, kap[c0:c0 + 64], th[c0:c0 + 64], drift, 0, [g[sl] for g in got], cell0=c0))
    report(test="config4_sampled", max_err_rel_to_thermal_plus_drift=worst)
    assert worst <= TOL["f32"], worst
    assert torch.isfinite(got[0]).all() and torch.isfinite(got[1]).all() and torch.isfinite(got[2]).all()
    mz = got[2].double().mean().item()                           # <vz> = drift (cfg.drift[2] = 0.02)
    sig = float(np.sqrt(np.mean(th.astype(np.float64) ** 2) * 2.0 / (1 << 28)))     # generous: <x>/3 < 2 for kappa >= 2
    assert abs(mz - 0.02) < 6 * sig, (mz, sig)


@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_pair_kernel_is_bit_identical_to_scalar_hook(dtype):
    n, kappa, theta, seed, off = 70_001, 2.0, 0.1, 42, 2**32 - 30_000
    w = kg.words(n, seed, off)
    a = kg.velocity_of_words(*w, kappa, theta, dtype)
    b = kg.sample(n, kappa, theta, seed, off, dtype)
    for x, y in zip(a, b):
        assert torch.equal(x, y)


@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_extreme_theta_takes_the_unfolded_path(dtype):
    n, kappa, seed = 50_000, 3.0, 5
    for theta in (1e-12, 3e11, 2.0**-30, 2.0**30):
        got = kg.sample(n, kappa, theta, seed, 0, dtype)
        want = oracle.sample(n, kappa, theta, seed, 0)
        assert max_rel_err(got, want) <= TOL[dtype]


@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_sample_host_equals_device_sample(dtype):
    n = (1 << 22) * 2 + 12345                              # three chunks, ragged tail
    dev = kg.sample(n, 2.0, 0.1, 42, 999, dtype)
    host = kg.sample_host(n, 2.0, 0.1, 42, 999, dtype)
    pageable = kg.sample_host(1000, 2.0, 0.1, 42, 999, dtype, pin=False)
    for d, h, p in zip(dev, host, pageable):
        assert torch.equal(d.cpu(), h)
        assert torch.equal(d[:1000].cpu(), p)


def kappa_cdf(x, kappa):
    """Exact CDF of x = v^2/theta^2, Eq. (3)."""
    return special.betainc(1.5, kappa - 0.5, x / (x + kappa))


@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("kappa", [1.6, 2.0, 3.0, 10.0])
def test_baseline_mt_samples_the_exact_kappa_distribution(kappa, dtype):
    n, theta = 4_000_000, 0.5
    trips = torch.zeros(2, dtype=torch.int64, device="cuda")
    v = kg.baseline_mt(n, kappa, theta, 11, 0, dtype, trip_counters=trips)
    x = ((v[0].double() ** 2 + v[1].double() ** 2 + v[2].double() ** 2) / theta**2).cpu().numpy()
    ks = stats.kstest(x, lambda t: kappa_cdf(t, kappa)).statistic
    band = 1.95 / np.sqrt(n)                                 # 99.9 % Kolmogorov quantile
    lane, warp = (float(t) / n for t in trips.cpu().numpy())
    report(test="baseline_mt", kappa=kappa, dtype=dtype, ks=float(ks), band=band, trips_per_lane=lane, trips_per_warp=warp)
    assert ks <= band, (ks, band)
    for q in range(3):                                       # direction cosines: mean 0, variance 1/3
        c = (v[q].double() / torch.sqrt(torch.tensor(x, device="cuda")) / theta).cpu().numpy()
        assert abs(c.mean()) < 5 * np.sqrt(1 / 3 / n) and abs((c**2).mean() - 1 / 3) < 5 * np.sqrt(4 / 45 / n)
    # Marsaglia-Tsang acceptance rate, Eq. (28), k = kappa - 1/2: a lane makes 1/p1 trips on average
    # ("3 + 2/p1 variates per particle on CPUs"); a warp waits for its slowest lane and
    # makes mu_1(1 - p1, 32) trips, Eq. (30): 1.80, 1.60, 1.37, 1.10 at these four kappa.
    k = kappa - 0.5
    p1 = np.exp(k - 1.0 / 3.0) * special.gamma(k) / (np.sqrt(2 * np.pi) * (k - 1.0 / 3.0) ** (k - 0.5))
    rho = 1.0 - p1
    mu1 = 3.0 - (1.0 - rho) ** 32 - (1.0 - rho**2) ** 32
    assert abs(mu1 - {1.6: 1.80, 2.0: 1.60, 3.0: 1.37, 10.0: 1.10}[kappa]) < 0.006
    report(test="baseline_mt_trips", kappa=kappa, dtype=dtype, lane=lane, one_over_p1=1 / p1, warp=warp, mu1_eq30=mu1)
    assert abs(lane - 1.0 / p1) <= 0.001, (lane, 1.0 / p1)
    assert abs(warp - mu1) <= 0.01, (warp, mu1)
