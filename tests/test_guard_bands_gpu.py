"""Out-of-bounds writes, checked without a sanitizer: every output buffer is carved out of a larger
allocation filled with a sentinel, with guard bands on both sides; after the call the guards must be intact.
Ragged sizes, misaligned planes (scalar-store path), the cells / moments / histogram / words entry points."""
import numpy as np
import pytest
import torch

from paper_2602_05606_b200 import kappagen as kg
from paper_2602_05606_b200 import workloads as wl

pytestmark = pytest.mark.gpu
GUARD = 64


def carve(n, dtype, shift=0, fill=-777.0):
    """A length-n view starting GUARD + shift elements into a sentinel-filled buffer."""
    buf = torch.full((n + 2 * GUARD + 8,), fill, dtype=dtype, device="cuda")
    return buf, buf[GUARD + shift:GUARD + shift + n]


def intact(buf, n, shift, fill=-777.0):
    lo, hi = buf[:GUARD + shift], buf[GUARD + shift + n:]
    return bool((lo == fill).all()) and bool((hi == fill).all())


@pytest.mark.parametrize("dtype,tdt", [("f32", torch.float32), ("f64", torch.float64)])
@pytest.mark.parametrize("n", [1, 3, 5, 127, 2047, 2049, 4097, 100_003])
@pytest.mark.parametrize("shift", [0, 1])
def test_sample_writes_only_its_planes(dtype, tdt, n, shift):
    bufs, views = zip(*(carve(n, tdt, shift) for _ in range(3)))
    for flags in (0, kg.U1_64):
        kg.sample_flags(n, 2.0, 0.5, 3, 2**32 - 50, dtype, flags, out=views)
        torch.cuda.synchronize()
        assert all(intact(b, n, shift) for b in bufs)
        assert all(bool(torch.isfinite(v).all()) and bool((v != -777.0).all()) for v in views)
    kg.baseline_mt(n, 2.0, 0.5, 3, 0, dtype, out=views)
    torch.cuda.synchronize()
    assert all(intact(b, n, shift) for b in bufs)


@pytest.mark.parametrize("dtype,tdt", [("f32", torch.float32), ("f64", torch.float64)])
@pytest.mark.parametrize("ppc", [1, 5, 64, 100])
def test_cells_and_moments_write_only_their_outputs(dtype, tdt, ppc):
    cfg = wl.CellsConfig(nx=7, ny=3, nz=5, ppc=ppc)
    kap, th = wl.cell_arrays(cfg, dtype=np.float32 if dtype == "f32" else np.float64)
    k, t = torch.from_numpy(kap).cuda(), torch.from_numpy(th).cuda()
    d = torch.tensor(cfg.drift, dtype=tdt, device="cuda")
    n = cfg.ncell * ppc
    bufs, views = zip(*(carve(n, tdt, 0) for _ in range(3)))
    mbuf, mview = carve(4 * cfg.ncell, tdt, 0)
    need = kg.cells_workspace_bytes(cfg.ncell, dtype)
    wbuf = torch.full((need + 2 * GUARD,), 0x5A, dtype=torch.uint8, device="cuda")
    ws = wbuf[GUARD:GUARD + need]
    kg.sample_cells_moments(ppc, k, t, d, 0, 7, 0, out=views, moments=mview.view(cfg.ncell, 4), workspace=ws)
    torch.cuda.synchronize()
    assert all(intact(b, n, 0) for b in bufs) and intact(mbuf, 4 * cfg.ncell, 0)
    assert bool((wbuf[:GUARD] == 0x5A).all()) and bool((wbuf[GUARD + need:] == 0x5A).all())
    assert bool((mview != -777.0).all())


def test_words_and_histogram_write_only_their_outputs():
    n = 4099
    bufs, views = zip(*(carve(n, torch.int32, 0, fill=-777) for _ in range(4)))
    L = kg.lib()
    assert L.kappagen_words4(n, 1, 2**32 - 9, *(v.data_ptr() for v in views), None) == kg.OK
    torch.cuda.synchronize()
    assert all(intact(b, n, 0, fill=-777) for b in bufs)
    for nbins in (2, 33, 4096):
        hbuf = torch.full((nbins + 2 * GUARD,), -777, dtype=torch.int64, device="cuda")
        h = hbuf[GUARD:GUARD + nbins]
        h.zero_()
        kg.speed_histogram(50_001, 1.6, 2, 0, "f32", 0, 0.2, nbins, hist=h)
        torch.cuda.synchronize()
        assert bool((hbuf[:GUARD] == -777).all()) and bool((hbuf[GUARD + nbins:] == -777).all())
        assert int(h.sum()) == 50_001
