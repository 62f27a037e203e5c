"""Host logic of bench.py (no GPU): the roofline objects follow from the kernel time by the arithmetic DESIGN.md
section 5 states, for both dtypes, and carry the keys the bench contract asks for."""
import json
import math

import bench


def test_roofline_objects_follow_from_the_kernel_time():
    n = 1 << 28
    peak, _, mhz = bench.measured_peaks()
    r32 = bench.roofline_of("f32", n, 1.15, 1.14, 1.20, ceiling_ms=0.60)
    assert r32["bound"] == "hbm" and r32["unit"] == "GB/s" and r32["peak"] == peak
    assert math.isclose(r32["achieved"], 12 * n / 1.15e-3 / 1e9, rel_tol=1e-12)
    assert math.isclose(r32["frac"], r32["achieved"] / peak, rel_tol=1e-12) and r32["frac"] == r32["frac_hbm"]
    assert math.isclose(r32["frac_pipe"], 19 * n / 1.15e-3 / (148 * 32 * mhz * 1e6), rel_tol=1e-12)
    assert math.isclose(r32["frac_of_ceiling"], 0.60 / 1.15, rel_tol=1e-12)
    assert r32["target"] == {"kind": "hbm", "frac": 0.80, "met": r32["frac"] >= 0.80}
    r64 = bench.roofline_of("f64", n, 2.07, 2.06, 2.10)
    assert r64["bound"] == "alu" and r64["frac"] == r64["frac_pipe"]
    assert math.isclose(r64["frac_pipe"], 85 * n / 2.07e-3 / (148 * 64 * mhz * 1e6), rel_tol=1e-12)
    assert math.isclose(r64["frac_hbm"], 24 * n / 2.07e-3 / 1e9 / peak, rel_tol=1e-12)
    assert 0.5 < r64["shared_port"]["frac"] < 1.2 and "ceiling" not in r64
    for r in (r32, r64):
        for key in ("bound", "achieved", "peak", "unit", "frac", "traffic", "kernel_ms", "ncu"):
            assert key in r
        assert r["ncu"]["source"]["from"].startswith("profiles/")        # copied figures name their source
        json.dumps(r)                                                   # the object is JSON-serialisable


def test_workload_is_configs_2():
    with open(bench.os.path.join(bench.ROOT, "BASELINE.json")) as f:
        base = json.load(f)
    assert "2^28 particles, kappa=2.0, theta=0.1" in base["configs"][2] and "seed=42" in base["configs"][2]
    assert (bench.N_STEP, bench.KAPPA, bench.THETA, bench.SEED) == (1 << 28, 2.0, 0.1, 42)
    c = bench.config_dict("f32", 4)
    assert "configs[2]" in c["workload"] and c["particles_per_step_per_gpu"] == 1 << 28 and "x4" in c["parallelism"]
