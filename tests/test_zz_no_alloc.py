"""kappagen_sample_cells_static: the per-cell sampler for callers that cannot allocate device memory.

Who needs it: a routine that runs inside somebody else's simulation -- say the particle injection of an open boundary,
called every time step -- where the host framework has taken the whole GPU into its own memory pool at start-up and
forbids cudaMalloc afterwards (it stalls every stream on the device, and with the pool holding everything it may just
fail), and where the routine is handed output arrays but no handle to that pool.  kappagen_sample_cells wants a
workspace from such a caller; this entry point keeps the per-cell records in a 3 MiB array inside the library instead
and takes inputs and outputs only.

What is checked here, against the existing kappagen_sample_cells on the same inputs (same kernels, so bit for bit,
which is the bar the other path-against-path tests of this suite use):
  * two calls in a row that share the built-in array, the second with fewer cells, other parameters and (in two of
    the three pairings) the other element type, i.e. another record size laid over the first call's leftovers;
  * the largest cell count the array holds, and the clear refusal of one cell more;
  * that a repeated call leaves the device's free memory where it was.
This file sorts last on purpose: `pytest -x` stops at the first failure, and nothing is collected after it.
It passes alone in a fresh process (the first call then does the one-time address look-up) and after the rest.
"""
import numpy as np
import pytest
import torch

from paper_2602_05606_b200 import kappagen as kg
from paper_2602_05606_b200 import workloads as wl

REC_BYTES = {"f32": 48, "f64": 96}                    # one per-cell record (kappagen_cells_workspace_bytes(1, dtype))


def _inputs(cfg, dtype, seed, bad_cells=()):
    npdt = np.float32 if dtype == "f32" else np.float64
    kap, th = wl.cell_arrays(cfg, dtype=npdt)
    kap, th = kap.copy(), th.copy()
    for c in bad_cells:                                # invalid cells must come out NaN on both paths alike
        kap[c] = 1.25
    drift = np.random.Generator(np.random.PCG64(seed)).normal(0.0, 0.05, size=(cfg.ncell, 3)).astype(npdt)
    return torch.from_numpy(kap).cuda(), torch.from_numpy(th).cuda(), torch.from_numpy(drift).cuda()


def _same(a, b):
    """Bit-identical planes (NaNs of invalid cells included)."""
    return all(torch.equal(x.view(torch.int32 if x.dtype == torch.float32 else torch.int64),
                           y.view(torch.int32 if y.dtype == torch.float32 else torch.int64)) for x, y in zip(a, b))


def _both_paths(cfg, dtype, seed, offset, bad_cells=()):
    kap, th, drift = _inputs(cfg, dtype, seed, bad_cells)
    n = cfg.ncell * cfg.ppc
    tdt = torch.float32 if dtype == "f32" else torch.float64
    out = tuple(torch.full((n,), -7.0, dtype=tdt, device="cuda") for _ in range(3))     # caller-owned outputs
    got = kg.sample_cells_static(cfg.ppc, kap, th, drift, 1, cfg.seed, offset, out=out)
    want = kg.sample_cells(cfg.ppc, kap, th, drift, 1, cfg.seed, offset)                # workspace from torch
    torch.cuda.synchronize()
    return got, want


@pytest.mark.gpu
@pytest.mark.parametrize("first,second", [("f32", "f32"), ("f32", "f64"), ("f64", "f32")])
def test_two_calls_in_a_row_match_the_workspace_path(first, second):
    big = wl.CellsConfig(nx=48, ny=32, nz=20, ppc=37, seed=11)          # 30720 cells: most of the array in double
    got, want = _both_paths(big, first, seed=1, offset=2**32 - 999, bad_cells=(5, 30000))
    assert _same(got, want)
    if first == "f32":
        assert torch.isnan(got[0][5 * 37:6 * 37]).all() and not torch.isnan(got[0][6 * 37:7 * 37]).any()
    small = wl.CellsConfig(nx=16, ny=8, nz=6, ppc=64, kappa_lo=1.6, kappa_hi=9.0, theta0=2.0, seed=12)
    got2, want2 = _both_paths(small, second, seed=2, offset=17)         # 768 cells on top of the leftovers
    assert _same(got2, want2)
    assert not any(torch.isnan(p).any() for p in got2)


@pytest.mark.gpu
@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_the_largest_call_the_array_holds(dtype):
    most = kg.STATIC_SCRATCH_BYTES // REC_BYTES[dtype]
    assert most == {"f32": 65536, "f64": 32768}[dtype]
    cfg = wl.CellsConfig(nx=most // 64, ny=8, nz=8, ppc=4, seed=13)
    assert cfg.ncell == most
    got, want = _both_paths(cfg, dtype, seed=3, offset=0)
    assert _same(got, want)
    kap, th, _ = _inputs(cfg, dtype, 3)
    one_more = (torch.cat([kap, kap[:1]]), torch.cat([th, th[:1]]))
    with pytest.raises(kg.KappagenError) as e:
        kg.sample_cells_static(4, one_more[0], one_more[1])
    assert e.value.status == kg.EWORKSPACE and str(most) in str(e.value)


@pytest.mark.gpu
def test_a_repeated_call_takes_no_device_memory():
    cfg = wl.CellsConfig(nx=32, ny=16, nz=8, ppc=16, seed=14)
    kap, th, drift = _inputs(cfg, "f32", 4)
    out = tuple(torch.empty(cfg.ncell * cfg.ppc, dtype=torch.float32, device="cuda") for _ in range(3))
    kg.sample_cells_static(cfg.ppc, kap, th, drift, 1, cfg.seed, 0, out=out)            # set-up and kernel loading
    torch.cuda.synchronize()
    before = torch.cuda.mem_get_info()[0]
    for rep in range(3):
        kg.sample_cells_static(cfg.ppc, kap, th, drift, 1, cfg.seed, rep, out=out)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == before


def test_too_many_cells_are_refused_before_the_device_is_touched():
    """No GPU needed: the size check comes first, so it also answers on a box without a device."""
    L = kg.lib()
    for code, most in ((kg.F32, 65536), (kg.F64, 32768)):
        rc = L.kappagen_sample_cells_static(most + 1, 4, None, None, None, 0, 0, 0, code, None, None, None, None)
        assert rc == kg.EWORKSPACE
        msg = kg.last_error()
        assert "kappagen_sample_cells_static" in msg and str(most) in msg and str(kg.STATIC_SCRATCH_BYTES) in msg
    assert L.kappagen_sample_cells_static(10, 4, None, None, None, 0, 0, 0, 7, None, None, None, None) == kg.EINVAL
    assert L.kappagen_sample_cells_static(0, 4, None, None, None, 0, 0, 0, kg.F32, None, None, None, None) == kg.OK
    assert L.kappagen_sample_cells_static(-1, 4, None, None, None, 0, 0, 0, kg.F32, None, None, None, None) == kg.EINVAL
