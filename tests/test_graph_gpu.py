"""The device entry points only enqueue kernels on the caller's stream (no allocation, no synchronisation), so
they can be recorded into a CUDA graph: small launch-bound calls (1e6 particles take 16 us, mostly launch) are
replayed without the per-call host cost.  Replay must reproduce the direct calls bit for bit."""
import pytest
import torch

from paper_2602_05606_b200 import kappagen as kg
from paper_2602_05606_b200 import workloads as wl

pytestmark = pytest.mark.gpu


def test_sample_calls_replay_from_a_cuda_graph():
    n, chunks = 1_000_000, 8
    planes = tuple(torch.empty(n * chunks, dtype=torch.float32, device="cuda") for _ in range(3))
    hist = torch.zeros(64, dtype=torch.int64, device="cuda")
    cfg = wl.CellsConfig(nx=16, ny=8, nz=4, ppc=64)
    kap, th = wl.cell_arrays(cfg)
    k, t = torch.from_numpy(kap).cuda(), torch.from_numpy(th).cuda()
    d = torch.tensor(cfg.drift, dtype=torch.float32, device="cuda")
    cells = tuple(torch.empty(cfg.ncell * cfg.ppc, dtype=torch.float32, device="cuda") for _ in range(3))
    mom = torch.empty((cfg.ncell, 4), dtype=torch.float32, device="cuda")
    ws = torch.empty(kg.cells_workspace_bytes(cfg.ncell, "f32"), dtype=torch.uint8, device="cuda")
    recs = torch.empty((cfg.ncell * cfg.ppc, 8), dtype=torch.float32, device="cuda")
    words = tuple(torch.empty(n, dtype=torch.int32, device="cuda") for _ in range(3))

    def enqueue(stream):
        for c in range(chunks):
            kg.sample(n, 3.0, 1.0, 0, c * n, "f32", out=tuple(p[c * n:(c + 1) * n] for p in planes), stream=stream)
        kg.speed_histogram(n, 3.0, 0, 0, "f32", 0, 0.2, 64, hist=hist, stream=stream)
        kg.sample_cells_moments(cfg.ppc, k, t, d, 0, cfg.seed, 0, out=cells, moments=mom, workspace=ws, stream=stream)
        kg.load_cells(cfg.ppc, k, t, d, 0, None, 7, cfg.seed, 0, out=recs, workspace=ws, stream=stream)   # bulk-copy stores
        kg.philox_planes(n, 5, 11, out=words, stream=stream)

    enqueue(torch.cuda.current_stream())
    torch.cuda.synchronize()
    want = [p.clone() for p in planes] + [c.clone() for c in cells] + [mom.clone(), recs.clone()] + [w.clone() for w in words]
    want_hist = hist.clone()

    for p in planes + cells:
        p.zero_()
    mom.zero_()
    recs.zero_()
    for w in words:
        w.zero_()
    g = torch.cuda.CUDAGraph()
    side = torch.cuda.Stream()
    with torch.cuda.stream(side):
        with torch.cuda.graph(g, stream=side):
            enqueue(side)
    hist.zero_()
    g.replay()
    torch.cuda.synchronize()
    got = list(planes) + list(cells) + [mom, recs] + list(words)
    assert all(torch.equal(a, b) for a, b in zip(got, want))
    assert torch.equal(hist, want_hist)
    one = kg.sample(n * chunks, 3.0, 1.0, 0, 0, "f32")
    assert all(torch.equal(a, b) for a, b in zip(planes, one))        # and the chunks continue the stream
