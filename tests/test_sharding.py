"""The N>1 path on CPU: index-range sharding with no data-path collective (SURVEY.md
section 8(e)).  Two `gloo` ranks each take workloads.shard_range(n, rank, 2), generate their range with the
oracle at offset + begin, and rank 0 checks that the concatenation is bit-identical to the one-shot stream --
the property that lets bench.py / a PIC code give every GPU its own range and never exchange anything.
The collective used here (all_gather of the results) is test plumbing, exactly like bench.py's barrier."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import oracle
from paper_2602_05606_b200 import workloads as wl


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, n, offset, ok):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        b, e = wl.shard_range(n, rank, world)
        v = oracle.sample(e - b, 1.6, 1.0, 123, offset + b)
        w = oracle.words(e - b, 123, offset + b)
        # pad to the largest shard so that all_gather sees equal shapes
        m = max(wl.shard_range(n, r, world)[1] - wl.shard_range(n, r, world)[0] for r in range(world))
        mine = torch.zeros(6, m, dtype=torch.float64)
        for j in range(3):
            mine[j, :e - b] = torch.from_numpy(v[j])
            mine[3 + j, :e - b] = torch.from_numpy(w[j].astype(np.float64))      # uint32 is exact in double
        parts = [torch.zeros_like(mine) for _ in range(world)]
        dist.all_gather(parts, mine)
        if rank == 0:
            want_v = oracle.sample(n, 1.6, 1.0, 123, offset)
            want_w = oracle.words(n, 123, offset)
            good = True
            for j in range(3):
                got_v = np.concatenate([parts[r][j, :wl.shard_range(n, r, world)[1] - wl.shard_range(n, r, world)[0]].numpy()
                                        for r in range(world)])
                got_w = np.concatenate([parts[r][3 + j, :wl.shard_range(n, r, world)[1] - wl.shard_range(n, r, world)[0]].numpy()
                                        for r in range(world)])
                good = good and np.array_equal(got_v, want_v[j]) and np.array_equal(got_w, want_w[j].astype(np.float64))
            ok.value = 1 if good else 0
        dist.barrier()
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("n,offset", [(20001, 0), (4097, 2**32 - 2000)])
def test_two_gloo_ranks_reproduce_the_one_shot_stream(n, offset):
    oracle.lib()                                   # build once in the parent
    ctx = mp.get_context("spawn")
    ok = ctx.Value("i", -1)
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, n, offset, ok)) for r in range(2)]
    for p in procs:
        p.start()
    for p in procs:
        p.join(120)
        assert p.exitcode == 0
    assert ok.value == 1


@pytest.mark.parametrize("n,world", [(0, 2), (1, 2), (7, 3), (2**28, 8), (10**8 + 1, 4)])
def test_shard_ranges_tile_the_index_range(n, world):
    edges = [wl.shard_range(n, r, world) for r in range(world)]
    assert edges[0][0] == 0 and edges[-1][1] == n
    for (b0, e0), (b1, e1) in zip(edges, edges[1:]):
        assert e0 == b1 and b0 <= e0
    sizes = [e - b for b, e in edges]
    assert max(sizes) - min(sizes) <= 1


def test_cell_shards_see_the_same_inputs_as_the_full_grid():
    """configs[3] sharded by z planes: a rank's kappa[]/theta[] slice equals the full grid's slice."""
    cfg = wl.CellsConfig(nx=8, ny=4, nz=6)
    full_k, full_t = wl.cell_arrays(cfg)
    per_plane = cfg.nx * cfg.ny
    for rank in range(2):
        z0, z1 = wl.shard_range(cfg.nz, rank, 2)
        k, t = wl.cell_arrays(cfg, z_planes=(z0, z1))
        assert np.array_equal(k, full_k[z0 * per_plane:z1 * per_plane])
        assert np.array_equal(t, full_t[z0 * per_plane:z1 * per_plane])
