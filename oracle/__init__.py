"""ctypes loader for the CPU oracle (oracle/kappagen_oracle.cpp).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this package.  It imports nothing from
paper_2602_05606_b200 and the CUDA path imports nothing from here.

`build()` compiles the C++ source with g++ into oracle/libkappagen_oracle.so (git-ignored);
`lib()` builds on demand and returns the loaded library with argument types set.  The thin
numpy wrappers below only marshal arguments.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "kappagen_oracle.cpp")
_SO = os.path.join(_HERE, "libkappagen_oracle.so")
_lock = threading.Lock()
_lib = None

_u32p = ctypes.POINTER(ctypes.c_uint32)
_f64p = ctypes.POINTER(ctypes.c_double)


def build(force: bool = False) -> str:
    """Compile the oracle if the .so is missing or older than its source."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        tmp = _SO + ".tmp.%d" % os.getpid()
        # -O2 without -ffast-math: the oracle's arithmetic is exactly what the source says.
        cmd = ["g++", "-std=c++17", "-O2", "-fPIC", "-shared", "-Wall", "-Wextra", "-o", tmp, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
        os.replace(tmp, _SO)
    return _SO


def lib() -> ctypes.CDLL:
    global _lib
    with _lock:
        if _lib is None:
            L = ctypes.CDLL(build())
            i64, u64, f64, i32 = ctypes.c_int64, ctypes.c_uint64, ctypes.c_double, ctypes.c_int32
            L.oracle_philox4x32_10.argtypes = [_u32p, _u32p, _u32p]
            L.oracle_philox4x32_10.restype = None
            L.oracle_words.argtypes = [i64, u64, u64, _u32p, _u32p, _u32p]
            L.oracle_words.restype = None
            L.oracle_params.argtypes = [f64, _f64p, _f64p, _f64p, _f64p]
            L.oracle_params.restype = ctypes.c_int
            for name in ("oracle_x_of_w0", "oracle_x_of_w0_literal", "oracle_L_of_w0"):
                f = getattr(L, name)
                f.argtypes = [i64, _u32p, f64, _f64p]
                f.restype = ctypes.c_int
            L.oracle_direction.argtypes = [i64, _u32p, _u32p, _f64p, _f64p, _f64p]
            L.oracle_direction.restype = None
            L.oracle_velocity_of_words.argtypes = [i64, _u32p, _u32p, _u32p, f64, f64, _f64p, _f64p, _f64p]
            L.oracle_velocity_of_words.restype = ctypes.c_int
            for name in ("oracle_sample", "oracle_sample_literal"):
                f = getattr(L, name)
                f.argtypes = [i64, f64, f64, u64, u64, _f64p, _f64p, _f64p]
                f.restype = ctypes.c_int
            L.oracle_sample_cells.argtypes = [i64, i32, _f64p, _f64p, _f64p, i64, u64, u64,
                                              _f64p, _f64p, _f64p, _f64p, _f64p, _f64p]
            L.oracle_sample_cells.restype = ctypes.c_int
            L.oracle_positions.argtypes = [i64, u64, u64, ctypes.c_int, _f64p, _f64p, _f64p]
            L.oracle_positions.restype = ctypes.c_int
            L.oracle_cells_moments.argtypes = [i64, i32, _f64p, _f64p, _f64p, i64, u64, u64, _f64p, _f64p]
            L.oracle_cells_moments.restype = ctypes.c_int
            L.oracle_x_of_w0w3.argtypes = [i64, _u32p, _u32p, f64, _f64p]
            L.oracle_x_of_w0w3.restype = ctypes.c_int
            L.oracle_sample_u64.argtypes = [i64, f64, f64, u64, u64, _f64p, _f64p, _f64p, _u32p]
            L.oracle_sample_u64.restype = ctypes.c_int
            L.oracle_velocity_of_words_u64.argtypes = [i64, _u32p, _u32p, _u32p, _u32p, f64, f64, _f64p, _f64p, _f64p]
            L.oracle_velocity_of_words_u64.restype = ctypes.c_int
            L.oracle_speed_over_theta.argtypes = [i64, f64, u64, u64, ctypes.c_int, _f64p]
            L.oracle_speed_over_theta.restype = ctypes.c_int
            L.oracle_version.restype = ctypes.c_int
            _lib = L
    return _lib


def _u32(a):
    return np.ascontiguousarray(a, dtype=np.uint32)


def _p32(a):
    return a.ctypes.data_as(_u32p)


def _p64(a):
    return a.ctypes.data_as(_f64p)


def philox4x32_10(ctr, key) -> np.ndarray:
    c, k, out = _u32(ctr), _u32(key), np.zeros(4, dtype=np.uint32)
    assert c.shape == (4,) and k.shape == (2,)
    lib().oracle_philox4x32_10(_p32(c), _p32(k), _p32(out))
    return out


def words(n: int, seed: int, offset: int):
    w = [np.empty(n, dtype=np.uint32) for _ in range(3)]
    lib().oracle_words(n, seed, offset, _p32(w[0]), _p32(w[1]), _p32(w[2]))
    return tuple(w)


def params(kappa: float):
    v = [ctypes.c_double() for _ in range(4)]
    rc = lib().oracle_params(kappa, *[ctypes.byref(x) for x in v])
    if rc != 0:
        raise ValueError("kappa must be finite and > 3/2")
    return tuple(x.value for x in v)  # (kappa*, a, b, c)


def _of_w0(name, w0, kappa):
    w0 = _u32(w0)
    out = np.empty(w0.size, dtype=np.float64)
    if getattr(lib(), name)(w0.size, _p32(w0), kappa, _p64(out)) != 0:
        raise ValueError("bad kappa")
    return out


def x_of_w0(w0, kappa: float) -> np.ndarray:
    return _of_w0("oracle_x_of_w0", w0, kappa)


def x_of_w0_literal(w0, kappa: float) -> np.ndarray:
    return _of_w0("oracle_x_of_w0_literal", w0, kappa)


def L_of_w0(w0, kappa: float) -> np.ndarray:
    return _of_w0("oracle_L_of_w0", w0, kappa)


def direction(w1, w2):
    w1, w2 = _u32(w1), _u32(w2)
    n = [np.empty(w1.size, dtype=np.float64) for _ in range(3)]
    lib().oracle_direction(w1.size, _p32(w1), _p32(w2), _p64(n[0]), _p64(n[1]), _p64(n[2]))
    return tuple(n)


def velocity_of_words(w0, w1, w2, kappa: float, theta: float):
    w0, w1, w2 = _u32(w0), _u32(w1), _u32(w2)
    v = [np.empty(w0.size, dtype=np.float64) for _ in range(3)]
    rc = lib().oracle_velocity_of_words(w0.size, _p32(w0), _p32(w1), _p32(w2), kappa, theta,
                                        _p64(v[0]), _p64(v[1]), _p64(v[2]))
    if rc != 0:
        raise ValueError("bad kappa/theta")
    return tuple(v)


def sample(n: int, kappa: float, theta: float, seed: int, offset: int = 0, literal: bool = False):
    v = [np.empty(n, dtype=np.float64) for _ in range(3)]
    f = lib().oracle_sample_literal if literal else lib().oracle_sample
    if f(n, kappa, theta, seed, offset, _p64(v[0]), _p64(v[1]), _p64(v[2])) != 0:
        raise ValueError("bad arguments")
    return tuple(v)


def sample_cells(ppc: int, kappa, theta, drift, drift_stride: int, seed: int, offset: int = 0,
                 thermal: bool = False):
    kappa = np.ascontiguousarray(kappa, dtype=np.float64)
    theta = np.ascontiguousarray(theta, dtype=np.float64)
    ncell = kappa.size
    n = ncell * ppc
    v = [np.empty(n, dtype=np.float64) for _ in range(3)]
    t = [np.empty(n, dtype=np.float64) for _ in range(3)] if thermal else None
    dptr = None
    if drift is not None:
        drift = np.ascontiguousarray(drift, dtype=np.float64)
        dptr = _p64(drift)
    null = ctypes.cast(None, _f64p)
    rc = lib().oracle_sample_cells(ncell, ppc, _p64(kappa), _p64(theta), dptr if dptr is not None else null,
                                   drift_stride, seed, offset, _p64(v[0]), _p64(v[1]), _p64(v[2]),
                                   _p64(t[0]) if t else null, _p64(t[1]) if t else null,
                                   _p64(t[2]) if t else null)
    if rc != 0:
        raise ValueError("bad arguments")
    return (tuple(v), tuple(t)) if thermal else tuple(v)


def positions(n: int, seed: int, offset: int = 0, bits: int = 23):
    """Offsets (fx, fy, fz) in (0,1) of the particles inside their cells: the second Philox block of each particle
    (counter word 3 = 2), midpoint uniforms of `bits` bits (23: exact in float, 32: exact in double); reading R22."""
    f = [np.empty(n, dtype=np.float64) for _ in range(3)]
    if lib().oracle_positions(n, seed, offset, bits, _p64(f[0]), _p64(f[1]), _p64(f[2])) != 0:
        raise ValueError("bad arguments")
    return tuple(f)


def cells_moments(ppc: int, kappa, theta, drift, drift_stride: int, seed: int, offset: int = 0):
    """Per-cell (sum vx, sum vy, sum vz, sum |v|^2) of sample_cells' particles, drift included, and the
    per-cell sum of |vx|+|vy|+|vz| (the scale of the admissible rounding error).  Returns (mom[ncell,4], abs1)."""
    kappa = np.ascontiguousarray(kappa, dtype=np.float64)
    theta = np.ascontiguousarray(theta, dtype=np.float64)
    ncell = kappa.size
    mom = np.empty((ncell, 4), dtype=np.float64)
    abs1 = np.empty(ncell, dtype=np.float64)
    null = ctypes.cast(None, _f64p)
    dptr = null
    if drift is not None:
        drift = np.ascontiguousarray(drift, dtype=np.float64)
        dptr = _p64(drift)
    rc = lib().oracle_cells_moments(ncell, ppc, _p64(kappa), _p64(theta), dptr, drift_stride, seed, offset,
                                    _p64(mom), _p64(abs1))
    if rc != 0:
        raise ValueError("bad arguments")
    return mom, abs1


# ---- 64-bit U1 from (w0, w3): SURVEY.md section 8(f) f2, reading R20
def x_of_w0w3(w0, w3, kappa: float) -> np.ndarray:
    w0, w3 = _u32(w0), _u32(w3)
    x = np.empty(w0.size, dtype=np.float64)
    if lib().oracle_x_of_w0w3(w0.size, _p32(w0), _p32(w3), kappa, _p64(x)) != 0:
        raise ValueError("bad kappa")
    return x


def sample_u64(n: int, kappa: float, theta: float, seed: int, offset: int = 0, return_w3: bool = False):
    v = [np.empty(n, dtype=np.float64) for _ in range(3)]
    w3 = np.empty(n, dtype=np.uint32)
    if lib().oracle_sample_u64(n, kappa, theta, seed, offset, _p64(v[0]), _p64(v[1]), _p64(v[2]), _p32(w3)) != 0:
        raise ValueError("bad arguments")
    return (tuple(v), w3) if return_w3 else tuple(v)


def velocity_of_words_u64(w0, w1, w2, w3, kappa: float, theta: float):
    w0, w1, w2, w3 = _u32(w0), _u32(w1), _u32(w2), _u32(w3)
    v = [np.empty(w0.size, dtype=np.float64) for _ in range(3)]
    if lib().oracle_velocity_of_words_u64(w0.size, _p32(w0), _p32(w1), _p32(w2), _p32(w3), kappa, theta,
                                          _p64(v[0]), _p64(v[1]), _p64(v[2])) != 0:
        raise ValueError("bad arguments")
    return tuple(v)


# ---- paper test 2: speed histogram and discrete relative entropy, SURVEY.md section 8(f) f3
def speed_over_theta(n: int, kappa: float, seed: int, offset: int = 0, u64: bool = False) -> np.ndarray:
    """|v|/theta = sqrt(x) per particle (S1-S4), long double rounded to double."""
    s = np.empty(n, dtype=np.float64)
    if lib().oracle_speed_over_theta(n, kappa, seed, offset, 1 if u64 else 0, _p64(s)) != 0:
        raise ValueError("bad arguments")
    return s


def speed_histogram(s, dv: float, nbins: int) -> np.ndarray:
    """Counts of s = |v|/theta in bins [i dv, (i+1) dv), i < nbins-1; the last bin is open-ended (reading R21)."""
    idx = np.minimum(np.floor(np.asarray(s, dtype=np.float64) / dv).astype(np.int64), nbins - 1)
    return np.bincount(idx, minlength=nbins).astype(np.uint64)


def bin_probabilities(kappa: float, dv: float, nbins: int, which: str = "exact") -> np.ndarray:
    """P(i): the distribution of |v|/theta integrated over each bin.  "exact": the Kappa distribution, Eq. (2)
    integrated through its CDF Eq. (3), F(x) = I_{x/(x+kappa)}(3/2, kappa-1/2), x = v^2/theta^2.
    "approx": the generator's own CDF G(x), Eq. (7)/(A11)."""
    from scipy import special
    v = np.arange(nbins, dtype=np.float64) * dv
    x = v * v
    # survival functions 1 - CDF at the lower bin edges, each formed without cancellation so that the far
    # tail bins keep their relative accuracy: 1 - I_y(a,b) = I_{1-y}(b,a);  1 - (1-q)^{3/2} = -expm1(1.5 log1p(-q))
    if which == "exact":
        surv = special.betainc(kappa - 0.5, 1.5, kappa / (x + kappa))
    else:
        ks, a, b, c = params(kappa)
        h = (a * x + b * x * x) / (1.0 + c * x)
        q = np.exp(-ks * np.log1p(h / ks))                    # exp_{q*}(-h), Eq. (8)
        with np.errstate(divide="ignore"):
            surv = -np.expm1(1.5 * np.log1p(-q))             # q = 1 at v = 0: survival 1
        surv[0] = 1.0
    return -np.diff(np.concatenate([surv, [0.0]]))            # last bin open-ended


def relative_entropy(hist, kappa: float, dv: float, eps: float = 1e-10, which: str = "exact") -> float:
    """Eq. (27): D(P||Q) = sum_i (P(i)+eps) ln((P(i)+eps)/(Q(i)+eps)), P the baseline
    (analytic) bin probabilities, Q(i) = hist[i]/N the Monte Carlo ones, eps = 1e-10."""
    hist = np.asarray(hist, dtype=np.float64)
    P = bin_probabilities(kappa, dv, hist.size, which)
    Q = hist / hist.sum()
    return float(np.sum((P + eps) * np.log((P + eps) / (Q + eps))))
