"""Seeded, synthetic input generators shared by the tests (oracle side and CUDA side) and bench.py.

This module holds NONE of the method's arithmetic: no Philox, no CDF, no parameters a/b/c.  It only
names the BASELINE.json configurations and builds the input arrays (per-cell kappa/theta/drift, and
lists of 32-bit test words) with numpy.  The paper's workloads are themselves synthetic ("generate
10^8 particles, as a function of kappa"; 10^6 particles; 10^2-10^3
particles per cell), so these inputs ARE the paper's benchmark shapes.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np


@dataclass(frozen=True)
class SampleConfig:
    """One kappagen_sample call shape from BASELINE.json `configs`."""
    name: str
    n: int
    kappa: float
    theta: float
    seed: int
    dtype: str  # "f32" | "f64"
    offset: int = 0


# BASELINE.json configs[0]: the small case the oracle finishes in ~1 s (paper test 1).
C1 = SampleConfig("C1", 1_000_000, 3.0, 1.0, 0, "f64")
# configs[1]: kappa sweep, 1e8 particles each, fp32 (paper test 3's shape).
C2_KAPPAS = (1.6, 2.0, 3.0, 4.0, 6.0, 10.0)
C2 = tuple(SampleConfig("C2_k%g" % k, 100_000_000, k, 1.0, 1, "f32") for k in C2_KAPPAS)
# configs[2]: the bandwidth / roofline run.
C3_F32 = SampleConfig("C3_f32", 1 << 28, 2.0, 0.1, 42, "f32")
C3_F64 = SampleConfig("C3_f64", 1 << 28, 2.0, 0.1, 42, "f64")
# configs[4]: 2^30 particles in 4 chunks of 2^28, heavy tail.
C5 = SampleConfig("C5", 1 << 30, 1.6, 1.0, 123, "f32")
C5_CHUNKS = 4


@dataclass(frozen=True)
class CellsConfig:
    """BASELINE.json configs[3]: PIC-style initialisation."""
    name: str = "C4"
    nx: int = 256
    ny: int = 256
    nz: int = 64
    ppc: int = 64
    kappa_lo: float = 2.0
    kappa_hi: float = 5.0
    theta0: float = 0.05
    theta_amp: float = 0.5
    layer_halfwidth: float = 8.0
    drift: tuple = (0.0, 0.0, 0.02)
    seed: int = 7
    dtype: str = "f32"

    @property
    def ncell(self) -> int:
        return self.nx * self.ny * self.nz


C4 = CellsConfig()


def cell_arrays(cfg: CellsConfig, z_planes=None, dtype=np.float32):
    """Per-cell kappa[] and theta[] of config 4, cell = (iz*ny + iy)*nx + ix (x fastest).

    kappa[cell] ~ Uniform[kappa_lo, kappa_hi) from numpy's PCG64 seeded with cfg.seed, drawn for the
    whole grid in cell order (so a sub-range of z planes sees the same values as the full grid);
    theta[cell] = theta0 * (1 + theta_amp * tanh(z / layer_halfwidth)), z = iz + 1/2 - nz/2 (cell
    centre height about the mid-plane, in cells): a Harris-like layer.  Values are rounded to `dtype`
    (the element type the library reads) and returned as that dtype; both the oracle and the CUDA
    path read these same arrays.  `z_planes=(z0, z1)` returns only cells of planes z0 <= iz < z1.
    """
    z0, z1 = (0, cfg.nz) if z_planes is None else z_planes
    assert 0 <= z0 <= z1 <= cfg.nz
    per_plane = cfg.nx * cfg.ny
    rng = np.random.Generator(np.random.PCG64(cfg.seed))
    # PCG64 can jump, but drawing plane by plane keeps this obviously right; planes are 65536 cells.
    kap = np.empty((z1 - z0) * per_plane, dtype=np.float64)
    for iz in range(cfg.nz):
        u = rng.random(per_plane)
        if z0 <= iz < z1:
            kap[(iz - z0) * per_plane:(iz - z0 + 1) * per_plane] = cfg.kappa_lo + (cfg.kappa_hi - cfg.kappa_lo) * u
        if iz >= z1:
            break
    z = np.arange(z0, z1, dtype=np.float64) + 0.5 - 0.5 * cfg.nz
    th_plane = cfg.theta0 * (1.0 + cfg.theta_amp * np.tanh(z / cfg.layer_halfwidth))
    th = np.repeat(th_plane, per_plane)
    return kap.astype(dtype), th.astype(dtype)


def edge_words(n_random: int = 3000, seed: int = 2602) -> np.ndarray:
    """32-bit test words that stress both ends of the uniform: every m*2^e and its complement for
    m in {0,1,2,3,5,7}, the words around each quarter and half of the range, plus random words.
    Sorted, unique, dtype uint32."""
    ws = set()
    for m in (0, 1, 2, 3, 5, 7):
        for e in range(33):
            v = m << e
            if v < (1 << 32):
                ws.add(v)
                ws.add((~v) & 0xFFFFFFFF)
    for q in range(0, 5):
        base = q << 30
        for d in (-2, -1, 0, 1, 2):
            v = base + d
            if 0 <= v < (1 << 32):
                ws.add(v)
    for e in range(1, 8):  # eighth turns: |angle| = pi/4 boundaries of the azimuth reduction
        base = e << 29
        for d in (-1, 0, 1):
            ws.add(base + d)
    rng = np.random.Generator(np.random.PCG64(seed))
    ws.update(int(v) for v in rng.integers(0, 1 << 32, size=n_random, dtype=np.uint64))
    return np.array(sorted(ws), dtype=np.uint32)


def shard_range(n: int, rank: int, world: int):
    """Contiguous index range [begin, end) of rank `rank` out of `world` for n particles (or cells):
    the data-parallel partition of SURVEY.md section 8(e).  No collective is needed: a rank calls the
    library with offset + begin."""
    base, rem = divmod(n, world)
    begin = rank * base + min(rank, rem)
    return begin, begin + base + (1 if rank < rem else 0)
