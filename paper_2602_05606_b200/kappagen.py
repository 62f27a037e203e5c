"""Thin ctypes binding over libkappagen (include/kappagen.h).  Argument marshalling only: every step
of the hot path runs in the CUDA kernels behind the C ABI.  PyTorch is used to allocate device
memory and to name the current stream; tensors are passed as raw pointers.

There is no CPU fallback.  If libkappagen.so has not been built, the first call raises
KappagenNotBuilt with the build command; on a machine without a CUDA device the library returns
KAPPAGEN_ECUDA and the binding raises KappagenError.
"""
from __future__ import annotations

import ctypes
import os

import torch

F32, F64 = 0, 1
U1_64 = 1                      # kappagen_sample_flags: 64-bit U1 from (w0, w3)
OK, EINVAL, ENULL, EALIGN, EWORKSPACE, ECUDA = 0, -1, -2, -3, -4, -5
_STATUS = {EINVAL: "KAPPAGEN_EINVAL", ENULL: "KAPPAGEN_ENULL", EALIGN: "KAPPAGEN_EALIGN",
           EWORKSPACE: "KAPPAGEN_EWORKSPACE", ECUDA: "KAPPAGEN_ECUDA"}
_SO = os.path.join(os.path.dirname(os.path.abspath(__file__)), "libkappagen.so")
_lib = None


class KappagenNotBuilt(RuntimeError):
    pass


class KappagenError(RuntimeError):
    def __init__(self, status: int, text: str):
        super().__init__("%s (%d): %s" % (_STATUS.get(status, "?"), status, text))
        self.status = status


def lib() -> ctypes.CDLL:
    """Load libkappagen.so (in-tree).  Fails loudly when it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(_SO):
            raise KappagenNotBuilt("%s is missing: build it with `python -m paper_2602_05606_b200.build` "
                                   "(or __graft_entry__.build()); there is no CPU fallback" % _SO)
        L = ctypes.CDLL(_SO)
        i64, u64, f64, i32, vp, sz = (ctypes.c_int64, ctypes.c_uint64, ctypes.c_double, ctypes.c_int32,
                                      ctypes.c_void_p, ctypes.c_size_t)
        ci = ctypes.c_int
        L.kappagen_sample.argtypes = [i64, f64, f64, u64, u64, ci, vp, vp, vp, vp]
        L.kappagen_sample_flags.argtypes = [i64, f64, f64, u64, u64, ci, ctypes.c_uint32, vp, vp, vp, vp]
        L.kappagen_words4.argtypes = [i64, u64, u64, vp, vp, vp, vp, vp]
        L.kappagen_velocity_of_words_u64.argtypes = [i64, vp, vp, vp, vp, f64, f64, ci, vp, vp, vp, vp]
        L.kappagen_speed_histogram.argtypes = [i64, f64, u64, u64, ci, ctypes.c_uint32, f64, i32, vp, vp]
        L.kappagen_relative_entropy.argtypes = [vp, i32, f64, f64, f64, ci, ctypes.POINTER(ctypes.c_double)]
        L.kappagen_sample_cells.argtypes = [i64, i32, vp, vp, vp, i64, u64, u64, ci, vp, vp, vp, vp, sz, vp]
        L.kappagen_sample_cells_static.argtypes = [i64, i32, vp, vp, vp, i64, u64, u64, ci, vp, vp, vp, vp]
        L.kappagen_sample_cells_moments.argtypes = [i64, i32, vp, vp, vp, i64, u64, u64, ci, vp, vp, vp, vp, vp, sz, vp]
        L.kappagen_cells_prepare.argtypes = [i64, vp, vp, vp, i64, ci, vp, sz, vp]
        L.kappagen_sample_cells_prepared.argtypes = [i64, i32, u64, u64, ci, vp, vp, vp, vp, sz, vp]
        L.kappagen_cells_workspace_bytes.argtypes = [i64, ci]
        L.kappagen_cells_workspace_bytes.restype = sz
        L.kappagen_sample_host.argtypes = [i64, f64, f64, u64, u64, ci, vp, vp, vp]
        L.kappagen_sample_host_ws.argtypes = [i64, f64, f64, u64, u64, ci, vp, vp, vp, vp, sz, vp, vp]
        L.kappagen_sample_host_workspace_bytes.argtypes = [i64, ci]
        L.kappagen_sample_host_workspace_bytes.restype = sz
        L.kappagen_load_cells.argtypes = [i64, i32, vp, vp, vp, i64, vp, i64, u64, u64, ci, vp, vp, sz, vp]
        L.kappagen_philox_planes.argtypes = [i64, u64, u64, vp, vp, vp, vp]
        L.kappagen_math_planes.argtypes = [i64, f64, f64, u64, ci, vp, vp, vp, vp]
        L.kappagen_pipe_probe.argtypes = [ci, ci, ci, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ci)]
        L.kappagen_baseline_mt.argtypes = [i64, f64, f64, u64, u64, ci, vp, vp, vp, vp, vp]
        L.kappagen_words.argtypes = [i64, u64, u64, vp, vp, vp, vp]
        L.kappagen_words_tile.argtypes = [i64, u64, u64, ci, vp, vp, vp, vp, vp]
        L.kappagen_velocity_of_words_tile.argtypes = [i64, vp, vp, vp, vp, f64, f64, ci, ctypes.c_uint32, vp, vp, vp, vp]
        L.kappagen_velocity_of_words.argtypes = [i64, vp, vp, vp, f64, f64, ci, vp, vp, vp, vp]
        dp = ctypes.POINTER(ctypes.c_double)
        L.kappagen_params.argtypes = [f64, dp, dp, dp, dp]
        L.kappagen_last_error.restype = ctypes.c_char_p
        for name in ("kappagen_speed_histogram", "kappagen_relative_entropy", "kappagen_sample", "kappagen_sample_flags", "kappagen_words4", "kappagen_velocity_of_words_u64",
                     "kappagen_sample_cells", "kappagen_sample_cells_static", "kappagen_sample_cells_moments", "kappagen_sample_host", "kappagen_baseline_mt",
                     "kappagen_words", "kappagen_velocity_of_words", "kappagen_params", "kappagen_version",
                     "kappagen_words_tile", "kappagen_velocity_of_words_tile", "kappagen_sample_host_ws",
                     "kappagen_load_cells", "kappagen_cells_prepare", "kappagen_sample_cells_prepared", "kappagen_philox_planes", "kappagen_math_planes", "kappagen_pipe_probe", "kappagen_pipe_probe_count"):
            getattr(L, name).restype = ci
        _lib = L
    return _lib


def last_error() -> str:
    return lib().kappagen_last_error().decode()


def version() -> int:
    return lib().kappagen_version()


def _check(rc: int) -> None:
    if rc != OK:
        raise KappagenError(rc, last_error())


def _dtype_code(dtype) -> int:
    if dtype in (torch.float32, "f32", F32):
        return F32
    if dtype in (torch.float64, "f64", F64):
        return F64
    raise ValueError("dtype must be float32/'f32' or float64/'f64'")


def _torch_dtype(code: int):
    return torch.float32 if code == F32 else torch.float64


def _stream(stream) -> int:
    if stream is None:
        if not torch.cuda.is_available():
            return 0        # host-side argument checks still work; anything that launches returns KAPPAGEN_ECUDA
        stream = torch.cuda.current_stream()
    return stream.cuda_stream if hasattr(stream, "cuda_stream") else int(stream)


def _dev(t, dtype, min_numel: int, what: str):
    """A device tensor whose data_ptr() the library may use: CUDA, contiguous, of `dtype`, >= min_numel elements."""
    if not isinstance(t, torch.Tensor) or not t.is_cuda:
        raise ValueError("%s must be a CUDA tensor" % what)
    if dtype is not None and t.dtype not in (dtype if isinstance(dtype, tuple) else (dtype,)):
        raise ValueError("%s must have dtype %s, got %s" % (what, dtype, t.dtype))
    if not t.is_contiguous() or t.numel() < min_numel:
        raise ValueError("%s must be contiguous with >= %d elements (has %d)" % (what, min_numel, t.numel()))
    return t


def _same_device(*ts):
    devs = {t.device for t in ts if t is not None}
    if len(devs) > 1:
        raise ValueError("all tensors of one call must live on the same device, got %s" % sorted(map(str, devs)))


def _planes(n: int, code: int, out, device):
    if out is None:
        return tuple(torch.empty(n, dtype=_torch_dtype(code), device=device) for _ in range(3))
    vx, vy, vz = out
    for t in (vx, vy, vz):
        _dev(t, _torch_dtype(code), n, "output plane")
    _same_device(vx, vy, vz)
    return vx, vy, vz


def _cell_inputs(ppc: int, kappa, theta, drift, drift_stride: int):
    """Checks shared by sample_cells / sample_cells_moments / load_cells_record; returns (code, ncell)."""
    code = _dtype_code(kappa.dtype)
    ncell = kappa.numel()
    _dev(kappa, None, ncell, "kappa")
    _dev(theta, kappa.dtype, ncell, "theta")
    if theta.numel() != ncell:
        raise ValueError("kappa and theta must have the same length")
    if drift_stride not in (0, 1):
        raise ValueError("drift_stride must be 0 (one shared vector) or 1 (per cell)")
    if drift is not None:
        _dev(drift, kappa.dtype, 3 if drift_stride == 0 else 3 * ncell, "drift")
    _same_device(kappa, theta, drift)
    if ppc < 0:
        raise ValueError("ppc must be >= 0")
    return code, ncell


def params(kappa: float):
    """Table I lines 1-4 on the host: (kappa*, a, b, c)."""
    v = [ctypes.c_double() for _ in range(4)]
    _check(lib().kappagen_params(kappa, *[ctypes.byref(x) for x in v]))
    return tuple(x.value for x in v)


def sample(n: int, kappa: float, theta: float, seed: int, offset: int = 0, dtype="f32", out=None,
           stream=None, device="cuda"):
    """kappagen_sample: returns (vx, vy, vz) device tensors (or fills `out`)."""
    code = _dtype_code(dtype)
    vx, vy, vz = _planes(n, code, out, device)
    _check(lib().kappagen_sample(n, kappa, theta, seed, offset, code, vx.data_ptr(), vy.data_ptr(), vz.data_ptr(),
                                 _stream(stream)))
    return vx, vy, vz


def sample_flags(n: int, kappa: float, theta: float, seed: int, offset: int = 0, dtype="f32", flags: int = 0, out=None,
                 stream=None, device="cuda"):
    """kappagen_sample_flags: kappagen_sample with options (flags = U1_64: 64-bit U1 from (w0, w3))."""
    code = _dtype_code(dtype)
    vx, vy, vz = _planes(n, code, out, device)
    _check(lib().kappagen_sample_flags(n, kappa, theta, seed, offset, code, flags, vx.data_ptr(), vy.data_ptr(),
                                       vz.data_ptr(), _stream(stream)))
    return vx, vy, vz


def cells_workspace_bytes(ncell: int, dtype="f32") -> int:
    return lib().kappagen_cells_workspace_bytes(ncell, _dtype_code(dtype))


def sample_cells(ppc: int, kappa: torch.Tensor, theta: torch.Tensor, drift=None, drift_stride: int = 0,
                 seed: int = 0, offset: int = 0, out=None, workspace=None, stream=None):
    """kappagen_sample_cells: kappa, theta (and drift) are device tensors of the output dtype."""
    code, ncell = _cell_inputs(ppc, kappa, theta, drift, drift_stride)
    vx, vy, vz = _planes(ncell * ppc, code, out, kappa.device)
    _same_device(kappa, vx)
    need = cells_workspace_bytes(ncell, code)
    if workspace is None:
        workspace = torch.empty(max(need, 16), dtype=torch.uint8, device=kappa.device)
    _dev(workspace, None, 0, "workspace")
    _check(lib().kappagen_sample_cells(ncell, ppc, kappa.data_ptr(), theta.data_ptr(),
                                       drift.data_ptr() if drift is not None else None, drift_stride, seed, offset,
                                       code, vx.data_ptr(), vy.data_ptr(), vz.data_ptr(), workspace.data_ptr(),
                                       workspace.numel() * workspace.element_size(), _stream(stream)))
    return vx, vy, vz


STATIC_SCRATCH_BYTES = 3 << 20      # KAPPAGEN_STATIC_SCRATCH_BYTES of include/kappagen.h


def sample_cells_static(ppc: int, kappa: torch.Tensor, theta: torch.Tensor, drift=None, drift_stride: int = 0,
                        seed: int = 0, offset: int = 0, out=None, stream=None):
    """kappagen_sample_cells_static: sample_cells for code that may not allocate device memory (a routine inside a
    simulation whose framework owns the whole GPU through its own pool and bans cudaMalloc after start-up).  No
    workspace argument: the per-cell records go to a 3 MiB array built into the library, so one call takes at most
    65536 float / 32768 double cells (more raises KappagenError with EWORKSPACE), calls that overlap on the GPU
    corrupt each other, and the first call on a device should be made outside stream capture.  Pass `out` (three
    preallocated planes) to keep this wrapper from allocating them with torch.  Same values as sample_cells."""
    code, ncell = _cell_inputs(ppc, kappa, theta, drift, drift_stride)
    vx, vy, vz = _planes(ncell * ppc, code, out, kappa.device)
    _same_device(kappa, vx)
    _check(lib().kappagen_sample_cells_static(ncell, ppc, kappa.data_ptr(), theta.data_ptr(),
                                              drift.data_ptr() if drift is not None else None, drift_stride, seed,
                                              offset, code, vx.data_ptr(), vy.data_ptr(), vz.data_ptr(), _stream(stream)))
    return vx, vy, vz


def cells_prepare(kappa: torch.Tensor, theta: torch.Tensor, drift=None, drift_stride: int = 0, workspace=None, stream=None):
    """kappagen_cells_prepare: Table I lines 1-4 per cell (+ drift) into the workspace, once; returns the workspace."""
    code, ncell = _cell_inputs(1, kappa, theta, drift, drift_stride)
    need = cells_workspace_bytes(ncell, code)
    if workspace is None:
        workspace = torch.empty(max(need, 16), dtype=torch.uint8, device=kappa.device)
    _dev(workspace, None, 0, "workspace")
    _same_device(kappa, workspace)
    _check(lib().kappagen_cells_prepare(ncell, kappa.data_ptr(), theta.data_ptr(), drift.data_ptr() if drift is not None else None,
                                        drift_stride, code, workspace.data_ptr(), workspace.numel() * workspace.element_size(),
                                        _stream(stream)))
    return workspace


def sample_cells_prepared(ncell: int, ppc: int, workspace: torch.Tensor, seed: int = 0, offset: int = 0, dtype="f32", out=None,
                          stream=None):
    """kappagen_sample_cells_prepared: velocities from a workspace filled by cells_prepare."""
    code = _dtype_code(dtype)
    _dev(workspace, None, 0, "workspace")
    vx, vy, vz = _planes(ncell * ppc, code, out, workspace.device)
    _same_device(workspace, vx)
    _check(lib().kappagen_sample_cells_prepared(ncell, ppc, seed, offset, code, vx.data_ptr(), vy.data_ptr(), vz.data_ptr(),
                                                workspace.data_ptr(), workspace.numel() * workspace.element_size(), _stream(stream)))
    return vx, vy, vz


def sample_cells_moments(ppc: int, kappa: torch.Tensor, theta: torch.Tensor, drift=None, drift_stride: int = 0,
                         seed: int = 0, offset: int = 0, out=None, moments=None, workspace=None, stream=None,
                         store: bool = True):
    """kappagen_sample_cells_moments: returns ((vx, vy, vz) or None, moments[ncell, 4]).  store=False passes
    NULL planes: moments only, no velocity reaches HBM."""
    code, ncell = _cell_inputs(ppc, kappa, theta, drift, drift_stride)
    planes = _planes(ncell * ppc, code, out, kappa.device) if store else None
    if moments is None:
        moments = torch.empty((ncell, 4), dtype=kappa.dtype, device=kappa.device)
    _dev(moments, kappa.dtype, 4 * ncell, "moments")
    need = cells_workspace_bytes(ncell, code)
    if workspace is None:
        workspace = torch.empty(max(need, 16), dtype=torch.uint8, device=kappa.device)
    _dev(workspace, None, 0, "workspace")
    _same_device(kappa, moments, workspace, *(planes or ()))
    ptrs = [p.data_ptr() for p in planes] if store else [None, None, None]
    _check(lib().kappagen_sample_cells_moments(ncell, ppc, kappa.data_ptr(), theta.data_ptr(),
                                               drift.data_ptr() if drift is not None else None, drift_stride, seed,
                                               offset, code, ptrs[0], ptrs[1], ptrs[2], moments.data_ptr(),
                                               workspace.data_ptr(), workspace.numel() * workspace.element_size(),
                                               _stream(stream)))
    return planes, moments


def sample_host(n: int, kappa: float, theta: float, seed: int, offset: int = 0, dtype="f32", out=None,
                pin: bool = True):
    """kappagen_sample_host: host (CPU) tensors in, filled synchronously; the end-to-end path."""
    code = _dtype_code(dtype)
    if out is None:
        out = tuple(torch.empty(n, dtype=_torch_dtype(code), pin_memory=pin) for _ in range(3))
    vx, vy, vz = out
    for t in (vx, vy, vz):
        if t.is_cuda or t.dtype != _torch_dtype(code) or t.numel() < n or not t.is_contiguous():
            raise ValueError("sample_host needs contiguous CPU tensors of the requested dtype")
    _check(lib().kappagen_sample_host(n, kappa, theta, seed, offset, code, vx.data_ptr(), vy.data_ptr(), vz.data_ptr()))
    return vx, vy, vz


def sample_host_workspace_bytes(n: int, dtype="f32") -> int:
    return int(lib().kappagen_sample_host_workspace_bytes(n, _dtype_code(dtype)))


def sample_host_ws(n: int, kappa: float, theta: float, seed: int, offset: int, dtype, out, workspace, stream_a, stream_b):
    """kappagen_sample_host_ws: as sample_host, with the caller's device staging workspace (uint8 CUDA tensor) and two
    streams; nothing is allocated or created inside the call."""
    code = _dtype_code(dtype)
    vx, vy, vz = out
    for t in (vx, vy, vz):
        if t.is_cuda or t.dtype != _torch_dtype(code) or t.numel() < n or not t.is_contiguous():
            raise ValueError("sample_host_ws needs contiguous CPU tensors of the requested dtype")
    _dev(workspace, None, 0, "workspace")
    _check(lib().kappagen_sample_host_ws(n, kappa, theta, seed, offset, code, vx.data_ptr(), vy.data_ptr(), vz.data_ptr(),
                                         workspace.data_ptr(), workspace.numel() * workspace.element_size(),
                                         _stream(stream_a), _stream(stream_b)))
    return vx, vy, vz


def load_cells(ppc: int, kappa: torch.Tensor, theta: torch.Tensor, drift=None, drift_stride: int = 0, weight=None,
               cell_base: int = 0, seed: int = 0, offset: int = 0, out=None, workspace=None, stream=None):
    """kappagen_load_cells: one record {fx, fy, fz, cell_id, vx, vy, vz, weight} per particle; returns records[n, 8]
    (the cell id sits in column 3 as integer BITS: view it with .view(torch.int32 / torch.int64))."""
    code, ncell = _cell_inputs(ppc, kappa, theta, drift, drift_stride)
    n = ncell * ppc
    if weight is not None:
        _dev(weight, kappa.dtype, ncell, "weight")
    if out is None:
        out = torch.empty((n, 8), dtype=kappa.dtype, device=kappa.device)
    _dev(out, kappa.dtype, 8 * n, "records")
    need = cells_workspace_bytes(ncell, code)
    if workspace is None:
        workspace = torch.empty(max(need, 16), dtype=torch.uint8, device=kappa.device)
    _dev(workspace, None, 0, "workspace")
    _same_device(kappa, weight, out, workspace)
    _check(lib().kappagen_load_cells(ncell, ppc, kappa.data_ptr(), theta.data_ptr(),
                                     drift.data_ptr() if drift is not None else None, drift_stride,
                                     weight.data_ptr() if weight is not None else None, cell_base, seed, offset, code,
                                     out.data_ptr(), workspace.data_ptr(), workspace.numel() * workspace.element_size(),
                                     _stream(stream)))
    return out


def philox_planes(n: int, seed: int, offset: int = 0, out=None, stream=None, device="cuda"):
    """kappagen_philox_planes: S1 + S6 only (the float sampler's measured ceiling); three int32 tensors of uint32 bits."""
    if out is None:
        out = tuple(torch.empty(n, dtype=torch.int32, device=device) for _ in range(3))
    for t in out:
        _dev(t, (torch.int32, torch.uint32, torch.float32), n, "word plane")
    _same_device(*out)
    _check(lib().kappagen_philox_planes(n, seed, offset, out[0].data_ptr(), out[1].data_ptr(), out[2].data_ptr(), _stream(stream)))
    return out


MATH_PLANES_MUL = (0x9E3779B1, 0x85EBCA77, 0xC2B2AE3D)       # kappagen_math_planes: w_k = lo32(g) * MUL[k] + ADD[k] mod 2^32
MATH_PLANES_ADD = (0x7F4A7C15, 0x165667B1, 0x27D4EB2F)


def math_planes(n: int, kappa: float, theta: float, offset: int = 0, dtype="f32", out=None, stream=None, device="cuda"):
    """kappagen_math_planes: S2-S6 + stores on affine words of the index (the sampler's ceiling from the math side)."""
    code = _dtype_code(dtype)
    vx, vy, vz = _planes(n, code, out, device)
    _check(lib().kappagen_math_planes(n, kappa, theta, offset, code, vx.data_ptr(), vy.data_ptr(), vz.data_ptr(), _stream(stream)))
    return vx, vy, vz


PIPE_KINDS = ("IMAD.WIDE.U32", "LOP3", "FFMA2", "MUFU.EX2", "DFMA", "IMAD")


def pipe_probe_count() -> int:
    return int(lib().kappagen_pipe_probe_count())


def pipe_probe(mix: int, warps_per_scheduler: int = 8, iters: int = 2048):
    """kappagen_pipe_probe: (cycles per loop iteration per warp, {kind: instructions per iteration})."""
    cyc = ctypes.c_double()
    counts = (ctypes.c_int * 6)()
    _check(lib().kappagen_pipe_probe(mix, warps_per_scheduler, iters, ctypes.byref(cyc), counts))
    return cyc.value, {k: int(c) for k, c in zip(PIPE_KINDS, counts) if c}


def baseline_mt(n: int, kappa: float, theta: float, seed: int, offset: int = 0, dtype="f32", out=None,
                trip_counters=None, stream=None, device="cuda"):
    """kappagen_baseline_mt: the rejection-based comparison generator (exact Kappa distribution)."""
    code = _dtype_code(dtype)
    vx, vy, vz = _planes(n, code, out, device)
    if trip_counters is not None:
        _dev(trip_counters, (torch.int64, torch.uint64), 2, "trip_counters")
    _check(lib().kappagen_baseline_mt(n, kappa, theta, seed, offset, code, vx.data_ptr(), vy.data_ptr(), vz.data_ptr(),
                                      _stream(stream), trip_counters.data_ptr() if trip_counters is not None else None))
    return vx, vy, vz


def words(n: int, seed: int, offset: int = 0, stream=None, device="cuda"):
    """kappagen_words: the Philox words particle i consumes, as three int32 tensors holding uint32 bits."""
    w = tuple(torch.empty(n, dtype=torch.int32, device=device) for _ in range(3))
    _check(lib().kappagen_words(n, seed, offset, w[0].data_ptr(), w[1].data_ptr(), w[2].data_ptr(), _stream(stream)))
    return w


def words4(n: int, seed: int, offset: int = 0, stream=None, device="cuda"):
    """kappagen_words4: all four words of each particle's Philox block (int32 tensors holding uint32 bits)."""
    w = tuple(torch.empty(n, dtype=torch.int32, device=device) for _ in range(4))
    _check(lib().kappagen_words4(n, seed, offset, w[0].data_ptr(), w[1].data_ptr(), w[2].data_ptr(), w[3].data_ptr(),
                                 _stream(stream)))
    return w


def velocity_of_words_u64(w0, w1, w2, w3, kappa: float, theta: float, dtype="f32", stream=None):
    """kappagen_velocity_of_words_u64: S2-S6 with the 64-bit U1 from (w0, w3)."""
    code = _dtype_code(dtype)
    n = w0.numel()
    for w in (w0, w1, w2, w3):
        _dev(w, torch.int32, n, "words")
        if w.numel() != n:
            raise ValueError("words must have equal length")
    vx, vy, vz = _planes(n, code, None, w0.device)
    _check(lib().kappagen_velocity_of_words_u64(n, w0.data_ptr(), w1.data_ptr(), w2.data_ptr(), w3.data_ptr(), kappa,
                                                theta, code, vx.data_ptr(), vy.data_ptr(), vz.data_ptr(), _stream(stream)))
    return vx, vy, vz


def velocity_of_words(w0, w1, w2, kappa: float, theta: float, dtype="f32", stream=None):
    """kappagen_velocity_of_words: S2-S6 on caller-chosen words (int32 device tensors holding uint32 bits)."""
    code = _dtype_code(dtype)
    n = w0.numel()
    for w in (w0, w1, w2):
        _dev(w, torch.int32, n, "words")
        if w.numel() != n:
            raise ValueError("words must have equal length")
    vx, vy, vz = _planes(n, code, None, w0.device)
    _check(lib().kappagen_velocity_of_words(n, w0.data_ptr(), w1.data_ptr(), w2.data_ptr(), kappa, theta, code,
                                            vx.data_ptr(), vy.data_ptr(), vz.data_ptr(), _stream(stream)))
    return vx, vy, vz

def words_tile(n: int, seed: int, offset: int = 0, dtype="f32", stream=None, device="cuda"):
    """kappagen_words_tile: all four words, drawn through the tile path of kappagen_sample's kernel for `dtype`."""
    w = tuple(torch.empty(n, dtype=torch.int32, device=device) for _ in range(4))
    _check(lib().kappagen_words_tile(n, seed, offset, _dtype_code(dtype), w[0].data_ptr(), w[1].data_ptr(), w[2].data_ptr(),
                                     w[3].data_ptr(), _stream(stream)))
    return w


def velocity_of_words_tile(w0, w1, w2, kappa: float, theta: float, dtype="f32", w3=None, flags: int = 0, stream=None):
    """kappagen_velocity_of_words_tile: S2-S6 on caller-chosen words through the shipped straight-line tile body."""
    code = _dtype_code(dtype)
    n = w0.numel()
    for w in (w0, w1, w2) + ((w3,) if w3 is not None else ()):
        _dev(w, torch.int32, n, "words")
        if w.numel() != n:
            raise ValueError("words must have equal length")
    vx, vy, vz = _planes(n, code, None, w0.device)
    _check(lib().kappagen_velocity_of_words_tile(n, w0.data_ptr(), w1.data_ptr(), w2.data_ptr(),
                                                 w3.data_ptr() if w3 is not None else None, kappa, theta, code, flags,
                                                 vx.data_ptr(), vy.data_ptr(), vz.data_ptr(), _stream(stream)))
    return vx, vy, vz


def speed_histogram(n: int, kappa: float, seed: int, offset: int = 0, dtype="f32", flags: int = 0, dv: float = 0.2,
                    nbins: int = 512, hist=None, stream=None, device="cuda"):
    """kappagen_speed_histogram: accumulates the counts of |v|/theta into `hist` (int64 device tensor holding
    unsigned 64-bit counters, zeroed here when not given)."""
    if hist is None:
        hist = torch.zeros(nbins, dtype=torch.int64, device=device)
    _dev(hist, (torch.int64, torch.uint64), nbins, "hist")
    _check(lib().kappagen_speed_histogram(n, kappa, seed, offset, _dtype_code(dtype), flags, dv, nbins, hist.data_ptr(),
                                          _stream(stream)))
    return hist


def relative_entropy(hist, kappa: float, dv: float = 0.2, eps: float = 1e-10, which: int = 0) -> float:
    """kappagen_relative_entropy (Eq. 27) of a histogram (any integer tensor/array; copied to the host)."""
    import numpy as np
    h = np.ascontiguousarray(hist.cpu().numpy() if hasattr(hist, "cpu") else hist).astype(np.uint64)
    out = ctypes.c_double(0.0)
    _check(lib().kappagen_relative_entropy(h.ctypes.data, h.size, dv, kappa, eps, which, ctypes.byref(out)))
    return out.value
