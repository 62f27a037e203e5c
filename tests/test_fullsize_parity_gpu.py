"""Full element-wise parity at FULL size for BASELINE.json configs[1], [2], [3], [4] (C2's six kappa, C3 fp32 and fp64,
C4, C5):
every particle of the GPU output against the oracle, the oracle run over disjoint index ranges on all host
cores (SURVEY.md section 8(c)-F "Coverage at scale": counter-based => trivially splittable).

The north_star asks for the error "excluding the documented tail region u -> 1, where the error is reported
separately": the maxima are taken separately over the head `w0 < 2^12`, the tail `w0 >= 2^32 - 2^12` and the
bulk (reading R19), all three are gated by the tolerance (the stable evaluation excludes nothing),
and one JSON line per configuration goes to gpurun_out/parity_report.jsonl; profiles/r02_parity.md is that
table, transcribed.
"""
from __future__ import annotations

import os
from concurrent.futures import ThreadPoolExecutor

import numpy as np
import pytest
import torch

import oracle
from paper_2602_05606_b200 import kappagen as kg
from paper_2602_05606_b200 import workloads as wl
from gpu_util import TAIL_BITS, TOL, report

pytestmark = pytest.mark.gpu

CHUNK = 1 << 22                       # particles per oracle call (one worker, ~0.1 GB of doubles)
HEAD = np.uint32(1 << TAIL_BITS)
TAIL = np.uint32((1 << 32) - (1 << TAIL_BITS))


class Worst:
    """Running maxima of the relative error over head / tail / bulk, and where the overall maximum sits."""

    def __init__(self):
        self.err = {"head": 0.0, "tail": 0.0, "bulk": 0.0}
        self.count = {"head": 0, "tail": 0, "bulk": 0}
        self.at = (-1, -1)

    def merge(self, other):
        top = max(self.err.values())
        for k in self.err:
            self.err[k] = max(self.err[k], other.err[k])
            self.count[k] += other.count[k]
        if max(other.err.values()) > top:
            self.at = other.at


def _classify(rel, w0, begin):
    """rel[3][m] relative errors of one chunk -> Worst."""
    w = Worst()
    r = np.maximum(np.maximum(rel[0], rel[1]), rel[2])
    head, tail = w0 < HEAD, w0 >= TAIL
    for name, mask in (("head", head), ("tail", tail)):
        w.count[name] = int(mask.sum())
        if w.count[name]:
            w.err[name] = float(r[mask].max())
    bulk = ~(head | tail)
    w.count["bulk"] = int(bulk.sum())
    w.err["bulk"] = float(r[bulk].max())
    i = int(np.argmax(r))
    w.at = (begin + i, int(np.argmax([rel[q][i] for q in range(3)])))
    return w


def _run_chunks(n, job):
    """job(begin, m) -> Worst for particles [begin, begin+m); all host cores; returns the merged Worst."""
    total = Worst()
    begins = list(range(0, n, CHUNK))
    with ThreadPoolExecutor(max_workers=os.cpu_count() or 1) as pool:
        for w in pool.map(lambda b: job(b, min(CHUNK, n - b)), begins):
            total.merge(w)
    assert sum(total.count.values()) == n
    return total


def _check_sample(got, n, kappa, theta, seed, offset, dtype, name):
    """Every particle of `got` (three device planes) against oracle.sample."""
    host = [g.cpu().numpy() for g in got]          # pageable copies, outside any timing

    def job(begin, m):
        want = oracle.sample(m, kappa, theta, seed, offset + begin)
        w0 = oracle.words(m, seed, offset + begin)[0]
        rel = [np.abs(host[q][begin:begin + m].astype(np.float64) - want[q]) / np.abs(want[q]) for q in range(3)]
        return _classify(rel, w0, begin)

    w = _run_chunks(n, job)
    report(test="fullsize_parity", config=name, dtype=dtype, n=n, kappa=kappa, theta=theta, seed=seed, offset=offset,
           max_rel_err=w.err, particles=w.count, worst_particle=w.at[0], worst_component="xyz"[w.at[1]],
           tol=TOL[dtype], host_threads=os.cpu_count())
    assert max(w.err.values()) <= TOL[dtype], (name, w.err, w.at)
    # 2^28 uniform words put about 2^8 particles into each 2^-20 end region: the report is not vacuous
    assert w.count["head"] > 0 and w.count["tail"] > 0, w.count
    return w


@pytest.mark.parametrize("cfg", [wl.C3_F32, wl.C3_F64], ids=lambda c: c.name)
def test_config3_every_particle(cfg):
    got = kg.sample(cfg.n, cfg.kappa, cfg.theta, cfg.seed, cfg.offset, cfg.dtype)
    torch.cuda.synchronize()
    _check_sample(got, cfg.n, cfg.kappa, cfg.theta, cfg.seed, cfg.offset, cfg.dtype, cfg.name)


@pytest.mark.parametrize("cfg", wl.C2, ids=lambda c: c.name)
def test_config2_every_particle(cfg):
    """configs[1]: 10^8 particles at each kappa of the paper's scan (1.6 ... 10), every particle (SURVEY.md section
    8(c)-F: "Full element-wise parity for C1, C2"); the statistical side of this configuration is test_config2_gpu's."""
    got = kg.sample(cfg.n, cfg.kappa, cfg.theta, cfg.seed, cfg.offset, cfg.dtype)
    torch.cuda.synchronize()
    _check_sample(got, cfg.n, cfg.kappa, cfg.theta, cfg.seed, cfg.offset, cfg.dtype, cfg.name)


def test_config5_every_particle_of_the_chunked_run():
    """The four 2^28 chunks of configs[4] (consecutive Philox offsets), each written by its own call, against
    the oracle stream; bit-identity of chunked and one-shot output is test_parity_gpu's."""
    c = wl.C5
    chunk = c.n // wl.C5_CHUNKS
    total = Worst()
    for j in range(wl.C5_CHUNKS):
        got = kg.sample(chunk, c.kappa, c.theta, c.seed, j * chunk, c.dtype)
        torch.cuda.synchronize()
        total.merge(_check_sample(got, chunk, c.kappa, c.theta, c.seed, j * chunk, c.dtype, "C5 chunk %d" % j))
        del got
    report(test="fullsize_parity", config="C5 (4 chunks of 2^28)", dtype=c.dtype, n=c.n, max_rel_err=total.err,
           particles=total.count, tol=TOL[c.dtype])


def test_config4_every_particle():
    """configs[3]: 256 x 256 x 64 cells x 64 particles, per-cell kappa and theta, drift (0, 0, 0.02).  The bound is
    relative to |v_thermal| + |drift| (reading R11: a correctly rounded add can do no better)."""
    cfg = wl.C4
    kap, th = wl.cell_arrays(cfg)
    drift = np.array(cfg.drift, dtype=np.float32)
    got = kg.sample_cells(cfg.ppc, torch.from_numpy(kap).cuda(), torch.from_numpy(th).cuda(),
                          torch.from_numpy(drift).cuda(), 0, cfg.seed, 0)
    torch.cuda.synchronize()
    host = [g.cpu().numpy() for g in got]
    n = cfg.ncell * cfg.ppc
    cells_per_job = CHUNK // cfg.ppc

    def job(begin, m):
        c0, c1 = begin // cfg.ppc, (begin + m) // cfg.ppc
        assert (c1 - c0) * cfg.ppc == m and c1 - c0 <= cells_per_job
        want, therm = oracle.sample_cells(cfg.ppc, kap[c0:c1], th[c0:c1], drift, 0, cfg.seed, begin, thermal=True)
        w0 = oracle.words(m, cfg.seed, begin)[0]
        rel = [np.abs(host[q][begin:begin + m].astype(np.float64) - want[q]) /
               (np.abs(therm[q]) + abs(float(drift[q]))) for q in range(3)]
        return _classify(rel, w0, begin)

    w = _run_chunks(n, job)
    report(test="fullsize_parity", config=cfg.name, dtype=cfg.dtype, n=n, max_rel_err=w.err, particles=w.count,
           worst_particle=w.at[0], worst_component="xyz"[w.at[1]], tol=TOL[cfg.dtype], host_threads=os.cpu_count(),
           note="error relative to |v_thermal| + |drift|")
    assert max(w.err.values()) <= TOL[cfg.dtype], (w.err, w.at)
