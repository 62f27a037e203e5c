"""Multi-GPU readiness on one GPU (index-range sharding, no collective): R ranks run one after
the other, each on its own shard with the offsets a rank would pass (`offset + begin`, cells: `offset +
cell_begin * ppc`), and the concatenation must be BIT-IDENTICAL to the single call -- for the uniform sampler,
the per-cell sampler, the fused moments, the particle records and the summed speed histograms.  No rank waits on
another (nothing here emulates a collective); the scaling curve itself is unmeasured (one GPU per round)."""
import numpy as np
import pytest
import torch

from paper_2602_05606_b200 import kappagen as kg
from paper_2602_05606_b200 import workloads as wl

pytestmark = pytest.mark.gpu

RANKS = (2, 3, 8)


@pytest.mark.parametrize("world", RANKS)
@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_sample_shards_concatenate_to_the_single_call(world, dtype):
    n, offset = 1_000_003, 2**32 - 400_000                      # the shards straddle a 2^32 counter boundary
    one = kg.sample(n, 2.5, 0.3, 17, offset, dtype)
    parts = tuple(torch.empty_like(o) for o in one)
    for r in range(world):
        b, e = wl.shard_range(n, r, world)
        kg.sample(e - b, 2.5, 0.3, 17, offset + b, dtype, out=tuple(p[b:e] for p in parts))
    for p, o in zip(parts, one):
        assert torch.equal(p, o)


@pytest.mark.parametrize("world", RANKS)
@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_cells_shards_by_z_planes(world, dtype):
    """configs[3] shape, smaller grid: ranks own contiguous z-plane ranges; per-cell arrays are cut with
    workloads.cell_arrays(z_planes=...) exactly as a rank would build them."""
    cfg = wl.CellsConfig(nx=32, ny=16, nz=24, ppc=64)
    npd = np.float32 if dtype == "f32" else np.float64
    offset = 12345
    kap, th = wl.cell_arrays(cfg, dtype=npd)
    drift = torch.tensor(cfg.drift, dtype=torch.float32 if dtype == "f32" else torch.float64, device="cuda")
    dk, dt = torch.from_numpy(kap).cuda(), torch.from_numpy(th).cuda()
    one = kg.sample_cells(cfg.ppc, dk, dt, drift, 0, cfg.seed, offset)
    _, mom_one = kg.sample_cells_moments(cfg.ppc, dk, dt, drift, 0, cfg.seed, offset)
    rec_one = kg.load_cells(cfg.ppc, dk, dt, drift, 0, None, 0, cfg.seed, offset)
    per_plane = cfg.nx * cfg.ny
    planes, moms, recs = [], [], []
    for r in range(world):
        z0, z1 = wl.shard_range(cfg.nz, r, world)
        k_r, t_r = wl.cell_arrays(cfg, z_planes=(z0, z1), dtype=npd)
        cell_begin = z0 * per_plane
        assert np.array_equal(k_r, kap[cell_begin:cell_begin + k_r.size])
        a, b = torch.from_numpy(k_r).cuda(), torch.from_numpy(t_r).cuda()
        off_r = offset + cell_begin * cfg.ppc
        planes.append(kg.sample_cells(cfg.ppc, a, b, drift, 0, cfg.seed, off_r))
        moms.append(kg.sample_cells_moments(cfg.ppc, a, b, drift, 0, cfg.seed, off_r)[1])
        recs.append(kg.load_cells(cfg.ppc, a, b, drift, 0, None, cell_begin, cfg.seed, off_r))
    for q in range(3):
        assert torch.equal(torch.cat([p[q] for p in planes]), one[q])
    assert torch.equal(torch.cat(moms), mom_one)                 # ppc = 64: the fixed-order shuffle mode
    assert torch.equal(torch.cat(recs).view(torch.uint8), rec_one.view(torch.uint8))


@pytest.mark.parametrize("world", RANKS)
def test_cells_shards_with_ragged_ppc(world):
    """ppc = 37: groups straddle cells, shard boundaries fall inside tiles -- the packed, the per-group and the
    per-particle paths must give the same bits for the same particle."""
    ncell, ppc = 3001, 37
    rng = np.random.Generator(np.random.PCG64(5))
    kap = (1.7 + 5 * rng.random(ncell)).astype(np.float32)
    th = (0.1 + rng.random(ncell)).astype(np.float32)
    drift = torch.tensor([0.01, -0.02, 0.03], dtype=torch.float32, device="cuda")
    dk, dt = torch.from_numpy(kap).cuda(), torch.from_numpy(th).cuda()
    one = kg.sample_cells(ppc, dk, dt, drift, 0, 3, 99)
    parts = []
    for r in range(world):
        b, e = wl.shard_range(ncell, r, world)
        parts.append(kg.sample_cells(ppc, dk[b:e].contiguous(), dt[b:e].contiguous(), drift, 0, 3, 99 + b * ppc))
    for q in range(3):
        assert torch.equal(torch.cat([p[q] for p in parts]), one[q])


@pytest.mark.parametrize("world", RANKS)
@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_histograms_of_the_shards_sum_to_the_single_call(world, dtype):
    n, nbins = 3_000_001, 256
    one = kg.speed_histogram(n, 3.0, 4, 7, dtype, 0, 0.2, nbins)
    total = torch.zeros_like(one)
    for r in range(world):
        b, e = wl.shard_range(n, r, world)
        total += kg.speed_histogram(e - b, 3.0, 4, 7 + b, dtype, 0, 0.2, nbins)     # the reduction a caller would all-reduce
    assert torch.equal(total, one) and int(one.sum()) == n
