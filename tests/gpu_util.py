"""Helpers for the -m gpu parity tests: compare CUDA output (through the C ABI binding) with the oracle."""
from __future__ import annotations

import json
import os

import numpy as np

TOL = {"f32": 4e-6, "f64": 1e-12}      # BASELINE.json north_star: max relative error per component
TAIL_BITS = 12                          # "documented tail region": w0 >= 2^32 - 2^12, and the head w0 < 2^12

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
REPORT = os.path.join(ROOT, "gpurun_out", "parity_report.jsonl")


def u32(t):
    """int32 device tensor holding uint32 bits -> numpy uint32."""
    return t.cpu().numpy().view(np.uint32)


def rel_err(got, want):
    """Strict per-component relative error |got - want| / |want| in double (0/0 = 0)."""
    got = np.asarray(got, dtype=np.float64)
    want = np.asarray(want, dtype=np.float64)
    diff = np.abs(got - want)
    with np.errstate(divide="ignore", invalid="ignore"):
        r = np.where(want != 0, diff / np.abs(want), np.where(diff == 0, 0.0, np.inf))
    return r


def max_rel_err(gpu_planes, ref_planes):
    return max(float(np.max(rel_err(g.cpu().numpy() if hasattr(g, "cpu") else g, r), initial=0.0))
               for g, r in zip(gpu_planes, ref_planes))


def report(**kw):
    """Append one JSON line to gpurun_out/parity_report.jsonl (scratch; summarised into profiles/ by hand)."""
    try:
        os.makedirs(os.path.dirname(REPORT), exist_ok=True)
        with open(REPORT, "a") as f:
            f.write(json.dumps(kw) + "\n")
    except OSError:
        pass
