"""Host logic of bench.py (no GPU): the roofline objects follow from the kernel time by the arithmetic DESIGN.md
section 5 states, for both dtypes, and carry the keys the bench contract asks for."""
import json
import math

import bench


def test_roofline_objects_follow_from_the_kernel_time():
    n = 1 << 28
    peak, _, mhz = bench.measured_peaks()
    r32 = bench.roofline_of("f32", n, 1.15, 1.14, 1.20, ceiling_ms=0.60)
    # the headline names the measured limiter (the multiply pipe), the north_star's HBM figure stays beside it as the target
    assert r32["bound"] == "alu" and r32["unit"] == "G mul.wide.u32/s" and r32["frac"] == r32["frac_pipe"]
    assert math.isclose(r32["hbm"]["achieved"], 12 * n / 1.15e-3 / 1e9, rel_tol=1e-12) and r32["hbm"]["peak"] == peak
    assert math.isclose(r32["frac_hbm"], r32["hbm"]["achieved"] / peak, rel_tol=1e-12)
    assert math.isclose(r32["frac_pipe"], 19 * n / 1.15e-3 / (148 * 32 * mhz * 1e6), rel_tol=1e-12)
    assert r32["pipe"]["algorithmic_ops_per_particle"] == 19 and r32["pipe"]["executed_ops_per_particle"] == 18.1
    assert math.isclose(r32["pipe"]["frac_executed"], r32["frac_pipe"] * 18.1 / 19, rel_tol=1e-12)
    assert math.isclose(r32["frac_of_ceiling"], 0.60 / 1.15, rel_tol=1e-12)
    assert r32["target"] == {"kind": "hbm", "frac": 0.80, "achieved_frac": r32["frac_hbm"], "met": r32["frac_hbm"] >= 0.80}
    r64 = bench.roofline_of("f64", n, 2.07, 2.06, 2.10)
    assert r64["bound"] == "alu" and r64["frac"] == r64["frac_pipe"]
    assert math.isclose(r64["frac_pipe"], 85 * n / 2.07e-3 / (148 * 64 * mhz * 1e6), rel_tol=1e-12)
    assert math.isclose(r64["frac_hbm"], 24 * n / 2.07e-3 / 1e9 / peak, rel_tol=1e-12)
    cyc = 2.07e-3 * mhz * 1e6 * 148 * 4 * 32 / n
    assert math.isclose(r64["mix_bound"]["frac"], 259.3 / cyc, rel_tol=1e-12) and "ceiling" not in r64
    assert math.isclose(r64["mix_bound"]["fp64_pipe_frac_at_bound"], 85 * 2 / 259.3, rel_tol=1e-12)   # 2 cycles per FP64 warp instruction
    r64m = bench.roofline_of("f64", n, 2.07, 2.06, 2.10, None, 1.64)
    assert math.isclose(r64m["math_only"]["fp64_pipe_frac"], r64["frac_pipe"] * 2.07 / 1.64, rel_tol=1e-12)
    assert math.isclose(r64m["math_only"]["philox_share_of_sampler_time"], 1 - 1.64 / 2.07, rel_tol=1e-12)
    for r in (r32, r64):
        for key in ("bound", "achieved", "peak", "unit", "frac", "traffic", "kernel_ms", "ncu"):
            assert key in r
        assert r["ncu"]["source"]["from"].startswith("profiles/")        # copied figures name their source
        assert r["traffic"] == r["ncu"]["dram_bytes_per_launch"]
        json.dumps(r)                                                   # the object is JSON-serialisable


def test_workload_is_configs_2():
    with open(bench.os.path.join(bench.ROOT, "BASELINE.json")) as f:
        base = json.load(f)
    assert "2^28 particles, kappa=2.0, theta=0.1" in base["configs"][2] and "seed=42" in base["configs"][2]
    assert (bench.N_STEP, bench.KAPPA, bench.THETA, bench.SEED) == (1 << 28, 2.0, 0.1, 42)
    c = bench.config_dict("f32", 4)
    assert "configs[2]" in c["workload"] and c["particles_per_step_per_gpu"] == 1 << 28 and "x4" in c["parallelism"]


def test_ncu_constants_come_from_the_tracked_profile():
    with open(bench.os.path.join(bench.ROOT, "profiles", "r03_ncu.json")) as f:
        j = json.load(f)
    for d in ("f32", "f64"):
        assert bench.NCU_TRAFFIC_BYTES[d] == j["sample_kernel"][d]["dram_bytes_per_launch"]
        assert bench.NCU_PIPE_PCT[d] == j["sample_kernel"][d]["pipe_busy_pct"]
        # a capture with wasted traffic would show here: ncu's DRAM bytes stay within 5 % of the algorithmic bytes
        assert abs(bench.NCU_TRAFFIC_BYTES[d] / (3 * (4 if d == "f32" else 8) * (1 << 28)) - 1) < 0.05
    assert "command" in j["source"] and "kernels_as_of_commit" in j["source"]
    assert "_work" not in j["source"]["command"]


def test_reference_arm_says_what_it_ran(capsys):
    class A:
        gpus, steps, warmup, dtype = 1, 1, 0, "f32"
    old, bench.REF_SAMPLE = bench.REF_SAMPLE, 1 << 12
    try:
        bench.run_reference(A)
    finally:
        bench.REF_SAMPLE = old
    line = json.loads(capsys.readouterr().out.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["dtype"] == "f64" and line["gpu_launches"] == 0
    assert line["config"]["particles_per_step_per_gpu"] == 1 << 12            # the sample it ran, not the GPU arm's 2^28
    assert "long double" in line["config"]["workload"] and line["config"]["full_workload_particles_per_step"] == 1 << 28
    assert line["e2e"]["value"] == line["value"] == line["cpu_baseline"]["value"]
