"""bench.py -- throughput of the kappagen hot path on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--dtype f32|f64] [--impl ours|reference]

A "step" is one pass of the whole hot path (S1-S6: Philox -> q-exponential inverse -> direction ->
SoA stores) over one batch: kappagen_sample(2^28, kappa=2.0, theta=0.1, seed=42, offset=step*2^28)
= BASELINE.json configs[2], the configuration its metric ("particles/s ... at 2^28 particles") is
quoted on.  Under torchrun every rank does the same amount of work on its own index range (weak
scaling, no collective: SURVEY.md section 8(e)).  Prints ONE JSON line on rank 0.

`--impl reference` times the CPU oracle (oracle/, as it stands, one thread) on a bounded sample of
the same workload; it is a deliberately slow checker, not a competitor.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "kappa_particles_per_second"
UNIT = "particles/s"
N_STEP = 1 << 28                       # particles per step per GPU (configs[2])
KAPPA, THETA, SEED = 2.0, 0.1, 42
REF_SAMPLE = 1 << 20                   # particles per step of the --impl reference arm
CPU_BASELINE_SAMPLE = 1 << 24          # particles of the cpu_baseline leg (~10-20 s of one core)
FALLBACK_HBM_GBS = 6650.0              # B200_PROFILING.md fallback when MEASURED_PEAKS.json is absent
FALLBACK_SM_MHZ = 1965.0               # B200 maximum SM clock (MEASURED_PEAKS.json sm_max_mhz when present)
N_SM = 148
# ncu figures of one sample_kernel launch at 2^28 particles (dram__bytes_read.sum + dram__bytes_write.sum, busy
# fraction of the pipes) come from the tracked profiles/r03_ncu.json, which names the capture command, the commit the
# kernels were at and the markdown summary that holds the same numbers.  They are NOT measured by this run: the line
# prints them under "ncu" with that source so that nobody takes them for it.
def load_ncu():
    with open(os.path.join(ROOT, "profiles", "r03_ncu.json")) as f:
        j = json.load(f)
    src = dict(j["source"], note="copied from an ncu --set full capture, not measured by this run")
    return src, {d: j["sample_kernel"][d]["dram_bytes_per_launch"] for d in ("f32", "f64")}, \
        {d: j["sample_kernel"][d]["pipe_busy_pct"] for d in ("f32", "f64")}


NCU_CAPTURE, NCU_TRAFFIC_BYTES, NCU_PIPE_PCT = load_ncu()


def probe_mix_cycles():
    """Cycles per 32 particles of a dependency-free, memory-free loop with the double sampler's exact instruction mix at
    its 3 warps per scheduler (kappagen_pipe_probe mix 21, profiles/r03_pipe_rates.md via r03_ncu.json)."""
    with open(os.path.join(ROOT, "profiles", "r03_ncu.json")) as f:
        return float(json.load(f)["pipe_probe"]["double_sampler_mix"]["cycles_per_iteration"]["w3"])
# Algorithmic work per particle on the arithmetic pipes (instruction counts from cuobjdump -sass,
# rates from kappagen_pipe_probe = profiles/r03_pipe_rates.md), in thread-operations per clock per SM:
#   f32: Philox4x32-10 with counter words 2,3 = 0 needs 19 32x32->64-bit multiplies; IMAD.WIDE issues at a quarter of
#        the 128-lane FMA rate (probe: 4.1 cycles per warp instruction per scheduler) -> 32 /clk/SM.
#   f64: the double chain is 85 FP64 instructions (DFMA/DMUL/DADD/DSETP) per particle; 64 /clk/SM.  On sm_100 the FP64
#        pipe and the FMA-heavy pipe (Philox's IMAD.WIDE) overlap only in part: a loop of the kernel's exact mix, free of
#        dependencies and memory, takes 259.3 cycles per 32 particles (profiles/r03_fp64_limit.md), the kernel 288.
ALU_WORK = {"f32": (19, 32, "G mul.wide.u32/s", "fmaheavy (IMAD.WIDE.U32, quarter rate)"),
            "f64": (85, 64, "G FP64 instr/s", "fp64 (DFMA/DMUL/DADD)")}
# What the SASS executes per particle on that pipe: the shared Philox head per tile leaves 18.1 of the 19 algorithmic
# multiplies (17.1 IMAD.WIDE + 1 IMAD.HI, profiles/r02_fp32_limit.md); the double chain executes its 85.
ALU_EXECUTED = {"f32": 18.1, "f64": 85.0}
TARGETS = {"f32": ("hbm", 0.80), "f64": ("alu", 0.70)}         # BASELINE.json north_star, last sentence
BOUND = {"f32": "alu", "f64": "alu"}                           # the measured limiter of each kernel (ncu pipe figures)


def measured_peaks():
    """(HBM GB/s, its source, SM MHz) from the driver-written MEASURED_PEAKS.json, else the profiling guide's fallback."""
    peak, which, mhz = FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)", FALLBACK_SM_MHZ
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            j = json.load(f)
        peak, which = float(j["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, copy read+write)"
        mhz = float(j.get("sm_max_mhz", mhz))
    except Exception:
        pass
    return peak, which, mhz


def roofline_of(dtype, n, kern_ms, kern_min, kern_max, ceiling_ms=None, math_ms=None):
    """The roofline object of sample_kernel<dtype> from this run's CUDA-event time per launch.
    `bound`/`achieved`/`peak`/`frac` name the pipe that actually limits the kernel (both dtypes: an arithmetic pipe,
    "alu"): algorithmic pipe operations per second against the pipe's issue rate.  The north_star's own figures stay
    beside it: `frac_hbm` (HBM write fraction against the measured copy peak) and `target` (f32: 0.80 of HBM, judged on
    frac_hbm; f64: 0.70 of the FP64 pipe, judged on frac_pipe)."""
    es = 4 if dtype == "f32" else 8
    peak, which, mhz = measured_peaks()
    ops, per_clk, alu_unit, pipe = ALU_WORK[dtype]
    rate = n / (kern_ms * 1e-3)
    hbm = {"achieved": 3 * es * rate / 1e9, "peak": peak, "unit": "GB/s", "algorithmic_bytes_per_launch": 3 * es * n,
           "peak_source": which}
    hbm["frac"] = hbm["achieved"] / peak
    alu_peak = N_SM * per_clk * mhz * 1e6 / 1e9
    alu = {"achieved": ops * rate / 1e9, "peak": alu_peak, "unit": alu_unit, "pipe": pipe,
           "algorithmic_ops_per_particle": ops,
           "peak_source": "%d SMs x %d thread-ops/clk/SM x %.0f MHz (DESIGN.md section 5, profiles/r03_pipe_rates.md)" % (N_SM, per_clk, mhz)}
    alu["frac"] = alu["achieved"] / alu_peak
    alu["executed_ops_per_particle"] = ALU_EXECUTED[dtype]
    alu["frac_executed"] = alu["frac"] * ALU_EXECUTED[dtype] / ops
    kind, goal = TARGETS[dtype]
    judged = hbm["frac"] if kind == "hbm" else alu["frac"]
    head = dict(hbm) if BOUND[dtype] == "hbm" else dict(alu)
    r = {"bound": BOUND[dtype], "achieved": head["achieved"], "peak": head["peak"], "unit": head["unit"], "frac": head["frac"],
         "traffic": NCU_TRAFFIC_BYTES[dtype], "kernel": "sample_kernel<%s>" % dtype, "kernel_ms": kern_ms,
         "kernel_ms_min": kern_min, "kernel_ms_max": kern_max, "frac_hbm": hbm["frac"], "frac_pipe": alu["frac"],
         "hbm": hbm, "pipe": alu, "target": {"kind": kind, "frac": goal, "achieved_frac": judged, "met": judged >= goal},
         "ncu": {"source": NCU_CAPTURE, "dram_bytes_per_launch": NCU_TRAFFIC_BYTES[dtype], "pipe_busy_pct": NCU_PIPE_PCT[dtype]}}
    if dtype == "f32":
        r["bound_note"] = ("compute-bound: the FMA-heavy pipe (Philox's IMAD.WIDE + packed FMA) limits the kernel, not HBM; "
                           "frac = frac_pipe is the multiply pipe (19 algorithmic multiplies per particle; frac_executed "
                           "counts the 18.1 the SASS issues), frac_hbm the HBM write fraction the north_star asks for "
                           "(target), frac_of_ceiling the same kernel with steps S2-S5 stripped (kappagen_philox_planes)")
    else:
        cyc = kern_ms * 1e-3 * mhz * 1e6 * N_SM * 4 * 32 / n           # scheduler cycles per 32 particles
        bound = probe_mix_cycles()
        r["mix_bound"] = {"cycles_per_32_particles": cyc, "probe_mix_cycles": bound, "frac": bound / cyc,
                          "fp64_pipe_frac_at_bound": ops * 32 / (per_clk / 4) / bound,
                          "note": "kappagen_pipe_probe mix 21 = this kernel's instruction mix per particle (85 FP64, 18 wide "
                                  "multiplies, 56 ALU, 6 MUFU, 9 IMAD) without dependencies or memory, at the kernel's 3 warps per "
                                  "scheduler: the bound of ANY schedule of this mix (profiles/r03_fp64_limit.md); frac = how close "
                                  "the kernel is to it"}
    if ceiling_ms is not None:
        r["ceiling"] = {"kernel": "philox_planes_kernel (S1 + S6 only, 12 B/particle)", "kernel_ms": ceiling_ms,
                        "particles_per_s": n / (ceiling_ms * 1e-3)}
        r["frac_of_ceiling"] = ceiling_ms / kern_ms
    if math_ms is not None:
        cyc = lambda ms: ms * 1e-3 * mhz * 1e6 * N_SM * 4 * 32 / n
        r["math_only"] = {"kernel": "math_planes_kernel (S2-S6 + stores, words from one IMAD each)", "kernel_ms": math_ms,
                          "particles_per_s": n / (math_ms * 1e-3), "cycles_per_32_particles": cyc(math_ms),
                          "sampler_cycles_per_32_particles": cyc(kern_ms), "philox_share_of_sampler_time": 1.0 - math_ms / kern_ms}
        if dtype == "f64":
            r["math_only"]["fp64_pipe_frac"] = ops * n / (math_ms * 1e-3) / 1e9 / alu_peak
    return r


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--dtype", choices=["f32", "f64"], default="f32")
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--e2e-steps", type=int, default=5)
    ap.add_argument("--no-extras", action="store_true", help="skip the fp64 / baseline / cells extra timings")
    ap.add_argument("--dist-backend", choices=["nccl", "gloo"], default="nccl",
                    help="process group of the N>1 run; the data path has no collective, the group only carries the barrier, "
                         "the max over ranks and the shard check (gloo: ranks may share one GPU, see --device-index)")
    ap.add_argument("--device-index", type=int, default=None,
                    help="CUDA device of this rank instead of LOCAL_RANK (to exercise the N>1 branch on a one-GPU box)")
    ap.add_argument("--pipe-rates", action="store_true",
                    help="print the kappagen_pipe_probe table (markdown) that profiles/r03_pipe_rates.md holds, and exit")
    ap.add_argument("--sweep", action="store_true",
                    help="also time kappagen_sample over 1e6 ... 2^30 particles and kappa 1.6 ... 10 (extras.sweep)")
    return ap.parse_args()


def reference_config_dict():
    """What the --impl reference arm runs: a bounded sample of the same workload on the host, in the oracle's arithmetic."""
    return {"workload": "bounded sample of BASELINE.json configs[2]: %d particles per step (not 2^28), kappa=2.0, theta=0.1, "
                        "seed=42, oracle.sample on one host thread, long double arithmetic returned as f64 planes, "
                        "Philox offset advances by %d per step" % (REF_SAMPLE, REF_SAMPLE),
            "particles_per_step_per_gpu": REF_SAMPLE, "kappa": KAPPA, "theta": THETA, "seed": SEED,
            "parallelism": "none: rank 0's host cores only, no GPU", "arithmetic": "long double -> f64",
            "full_workload_particles_per_step": N_STEP}


def config_dict(dtype, world):
    return {"workload": "BASELINE.json configs[2]: 2^28 particles per step per GPU, kappa=2.0, theta=0.1, seed=42, "
                        "%s SoA vx/vy/vz, Philox offset advances by 2^28 per step" % dtype,
            "particles_per_step_per_gpu": N_STEP, "kappa": KAPPA, "theta": THETA, "seed": SEED,
            "parallelism": "index-range sharding x%d, no collective" % world,
            "l2": "write-only path; each step writes %.2f GB of output (> 126 MB L2), no L2 flush needed"
                  % (N_STEP * 3 * (4 if dtype == "f32" else 8) / 1e9)}


# --------------------------------------------------------------------------- reference arm (CPU oracle)
def oracle_rate(n, offset=0):
    """Time oracle.sample on n particles of the workload, one thread.  Returns particles/s."""
    import oracle
    t0 = time.perf_counter()
    oracle.sample(n, KAPPA, THETA, SEED, offset)
    return n / (time.perf_counter() - t0)


def oracle_rate_all_cores(n):
    """The same oracle function over disjoint index ranges on every host core (counter-based, so the split is
    trivial; ctypes releases the GIL).  Returns (particles/s, threads)."""
    import concurrent.futures as cf
    import oracle
    cores = os.cpu_count() or 1
    per = (n + cores - 1) // cores
    oracle.lib()
    t0 = time.perf_counter()
    with cf.ThreadPoolExecutor(cores) as ex:
        list(ex.map(lambda r: oracle.sample(min(per, n - r * per), KAPPA, THETA, SEED, r * per) if r * per < n else None,
                    range(cores)))
    return n / (time.perf_counter() - t0), cores


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    oracle.lib()
    for w in range(max(args.warmup, 0)):
        oracle.sample(REF_SAMPLE, KAPPA, THETA, SEED, w * REF_SAMPLE)
    t0 = time.perf_counter()
    for s in range(args.steps):
        oracle.sample(REF_SAMPLE, KAPPA, THETA, SEED, s * REF_SAMPLE)
    dt = time.perf_counter() - t0
    value = args.steps * REF_SAMPLE / dt
    sample = "%d particles per step of configs[2] (kappa=2.0, theta=0.1, seed=42), long double, 1 thread" % REF_SAMPLE
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * dt / max(args.steps, 1), "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": reference_config_dict(),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


# --------------------------------------------------------------------------- clocks
class ClockSampler(threading.Thread):
    """Samples SM clock and clock-event reasons through NVML while the timed region runs."""

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.samples, self.reasons, self.max_mhz = index, [], set(), None
        self._stop_evt = threading.Event()
        self.ok = False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
            self.ok = True
        except Exception:
            self.nv = None

    def run(self):
        if not self.ok:
            return
        nv = self.nv
        names = {nv.nvmlClocksEventReasonHwSlowdown: "hw_slowdown",
                 nv.nvmlClocksEventReasonHwThermalSlowdown: "hw_thermal_slowdown",
                 nv.nvmlClocksEventReasonSwThermalSlowdown: "sw_thermal_slowdown",
                 nv.nvmlClocksEventReasonSwPowerCap: "sw_power_cap",
                 nv.nvmlClocksEventReasonHwPowerBrakeSlowdown: "hw_power_brake_slowdown"}
        while not self._stop_evt.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                for bit, name in names.items():
                    if r & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            time.sleep(0.005)

    def mark(self):
        self.first_timed = len(self.samples)

    def stop(self):
        self._stop_evt.set()
        if self.is_alive():
            self.join()
        timed = sorted(self.samples[getattr(self, "first_timed", 0):])
        s = timed if timed else sorted(self.samples)
        return {"sm_mhz": s[len(s) // 2] if s else None, "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(timed), "samples_incl_warmup": len(self.samples)}


# --------------------------------------------------------------------------- our arm
def time_launches(fn, steps, warmup, torch):
    """Run fn(step) warmup+steps times on the current stream; returns (total_ms, [per-launch ms])."""
    for s in range(warmup):
        fn(s)
    torch.cuda.synchronize()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    t_begin, t_end = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t_begin.record()
    for s in range(steps):
        ev[s][0].record()
        fn(warmup + s)
        ev[s][1].record()
    t_end.record()
    torch.cuda.synchronize()
    return t_begin.elapsed_time(t_end), [a.elapsed_time(b) for a, b in ev]


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2602_05606_b200 import kappagen as kg

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback for the product path")
    if args.device_index is not None:
        local = args.device_index
    torch.cuda.set_device(local)
    nccl = args.dist_backend == "nccl"
    if world > 1:
        if nccl:
            dist.init_process_group("nccl", device_id=torch.device("cuda", local))
        else:
            dist.init_process_group("gloo")

    def max_over_ranks(x):
        t = torch.tensor([x], dtype=torch.float64, device="cuda" if nccl else "cpu")
        if world > 1:
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item())
    from paper_2602_05606_b200 import build as kbuild
    if rank == 0:
        kbuild.build()                                  # no-op when the in-tree library is up to date
    if world > 1:
        dist.barrier()
    kg.lib()                                            # fail loudly now if libkappagen.so is missing
    dtype, n = args.dtype, N_STEP
    tdt = torch.float32 if dtype == "f32" else torch.float64
    es = 4 if dtype == "f32" else 8
    planes = tuple(torch.empty(n, dtype=tdt, device="cuda") for _ in range(3))
    stream = torch.cuda.current_stream()

    def step(s):
        # rank r owns the index range [ (s*world + r) * n, +n ): contiguous shards, no exchange
        kg.sample(n, KAPPA, THETA, SEED, (s * world + rank) * n, dtype, out=planes, stream=stream)

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    sampler = ClockSampler(local)
    sampler.start()                                     # polls every 5 ms from the warm-up on; the device stays loaded
    for s in range(max(args.warmup, 3)):
        step(s)
    barrier()
    sampler.mark()                                      # samples from here on belong to the timed region
    total_ms, per_launch = time_launches(step, args.steps, 0, torch)
    barrier()
    clocks = sampler.stop()
    total_ms = max_over_ranks(total_ms)
    value = world * n * args.steps / (total_ms * 1e-3)
    shards = None
    if world > 1:                                       # what each rank's last timed step wrote, and from which offset
        mine = {"rank": rank, "offset": ((args.steps - 1) * world + rank) * n, "device": local,
                "vx_head": [float(v) for v in planes[0][:4].double().cpu()]}
        shards = [None] * world
        dist.all_gather_object(shards, mine)
    kern_ms = sum(per_launch) / len(per_launch)

    # ---- end to end through the C ABI with HOST buffers (device->host copies inside the timed region)
    host = tuple(torch.empty(n, dtype=tdt, pin_memory=True) for _ in range(3))
    ws = torch.empty(kg.sample_host_workspace_bytes(n, dtype), dtype=torch.uint8, device="cuda")
    sa, sb = torch.cuda.Stream(), torch.cuda.Stream()   # the caller's: the call allocates and creates nothing
    kg.sample_host_ws(n, KAPPA, THETA, SEED, rank * n, dtype, host, ws, sa, sb)  # warm-up (also faults the pages in)
    barrier()
    t0 = time.perf_counter()
    e2e_each = []
    for s in range(args.e2e_steps):
        t1 = time.perf_counter()
        kg.sample_host_ws(n, KAPPA, THETA, SEED, (s * world + rank) * n, dtype, host, ws, sa, sb)   # synchronous
        e2e_each.append(time.perf_counter() - t1)
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0
    e2e_value = world * n * args.e2e_steps / max_over_ranks(e2e_s)
    checksum = float(host[0][:1024].double().abs().sum())                         # the host result is read
    del host, ws

    line = None
    if rank == 0:
        ceiling_ms = None
        if dtype == "f32":                               # the same launch shape with S2-S5 stripped: Philox + stores
            wp = tuple(p.view(torch.int32) for p in planes)
            _, cms = time_launches(lambda s: kg.philox_planes(n, SEED, s * n, out=wp, stream=stream), 10, 3, torch)
            ceiling_ms = sum(cms) / len(cms)
        # ... and with S1 stripped instead: the math and the stores on affine words (kappagen_math_planes)
        _, mms = time_launches(lambda s: kg.math_planes(n, KAPPA, THETA, s * n, dtype, out=planes, stream=stream), 10, 3, torch)
        math_ms = sum(mms) / len(mms)
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
            "ms_per_step": total_ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": dtype, "data": "synthetic", "config": config_dict(dtype, world),
            "clocks": clocks, "gpu_launches": args.steps,
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 3 * es * n * world,
                    "steps": args.e2e_steps, "api": "kappagen_sample_host_ws (pinned host planes, caller's staging workspace and streams)",
                    "checksum": checksum, "ms_per_step": [round(1e3 * t, 3) for t in e2e_each],
                    "value_at_median_step": world * n / sorted(e2e_each)[len(e2e_each) // 2]},
            "roofline": roofline_of(dtype, n, kern_ms, min(per_launch), max(per_launch), ceiling_ms, math_ms),
        }
        if shards is not None:
            line["shards"] = shards
            line["config"]["dist_backend"] = args.dist_backend
        if world == 1:                                   # the other dtype of the metric ("fp32/fp64"), same workload, this run
            other = "f64" if dtype == "f32" else "f32"
            op = tuple(torch.empty(n, dtype=torch.float64 if other == "f64" else torch.float32, device="cuda") for _ in range(3))
            _, oms = time_launches(lambda s: kg.sample(n, KAPPA, THETA, SEED, s * n, other, out=op, stream=stream), 20, 3, torch)
            k = sum(oms) / len(oms)
            _, mms = time_launches(lambda s: kg.math_planes(n, KAPPA, THETA, s * n, other, out=op, stream=stream), 10, 3, torch)
            line["roofline_" + other] = roofline_of(other, n, k, min(oms), max(oms), None, sum(mms) / len(mms))
            line["value_" + other] = n / (k * 1e-3)
            del op
        if world == 1 and not args.no_extras:
            line["extras"] = extras(kg, torch, dtype)
        if world == 1 and args.sweep:
            line.setdefault("extras", {})["sweep"] = sweep(kg, torch)
        if world == 1:
            rate = oracle_rate(CPU_BASELINE_SAMPLE)
            line["cpu_baseline"] = {"value": rate, "unit": UNIT, "cores": 1, "kind": "oracle",
                                    "sample": "first %d particles of configs[2] (kappa=2.0, theta=0.1, seed=42), "
                                              "oracle.sample in long double on one host thread" % CPU_BASELINE_SAMPLE}
            rate_all, cores = oracle_rate_all_cores(4 * CPU_BASELINE_SAMPLE)
            line["cpu_baseline"]["all_cores"] = {"value": rate_all, "unit": UNIT, "cores": cores,
                                                 "sample": "first %d particles, split into %d index ranges" % (4 * CPU_BASELINE_SAMPLE, cores)}
        print(json.dumps(line))
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


def extras(kg, torch, dtype):
    """Reported beside the headline (N=1 only): the other dtype and the rejection baseline at the same size."""
    out = {}
    n = N_STEP
    st = torch.cuda.current_stream()
    p64 = tuple(torch.empty(n, dtype=torch.float64, device="cuda") for _ in range(3))
    p32 = tuple(x.view(torch.float32)[:n] for x in p64)
    planes = {"f32": p32, "f64": p64}
    other = "f64" if dtype == "f32" else "f32"
    es = {"f32": 4, "f64": 8}
    _, ms = time_launches(lambda s: kg.sample(n, KAPPA, THETA, SEED, s * n, other, out=planes[other], stream=st), 10, 3, torch)
    k = sum(ms) / len(ms)
    out["sample_" + other] = {"particles_per_s": n / (k * 1e-3), "kernel_ms": k, "write_GBps": 3 * es[other] * n / (k * 1e-3) / 1e9}
    for dt in ("f32", "f64"):
        _, ms = time_launches(lambda s: kg.baseline_mt(n, KAPPA, THETA, SEED, s * n, dt, out=planes[dt], stream=st), 5, 2, torch)
        k = sum(ms) / len(ms)
        out["baseline_mt_" + dt] = {"particles_per_s": n / (k * 1e-3), "kernel_ms": k, "write_GBps": 3 * es[dt] * n / (k * 1e-3) / 1e9}
    # configs[3]: PIC-style per-cell parameters, 256x256x64 cells x 64 particles (pre-kernel + sampling kernel)
    from paper_2602_05606_b200 import workloads as wl
    cfg = wl.C4
    kap, th = wl.cell_arrays(cfg)
    kd, td = torch.from_numpy(kap).cuda(), torch.from_numpy(th).cuda()
    dd = torch.tensor(cfg.drift, dtype=torch.float32, device="cuda")
    ws = torch.empty(kg.cells_workspace_bytes(cfg.ncell, "f32"), dtype=torch.uint8, device="cuda")
    nc = cfg.ncell * cfg.ppc
    _, ms = time_launches(lambda s: kg.sample_cells(cfg.ppc, kd, td, dd, 0, cfg.seed, s * nc, out=p32, workspace=ws, stream=st),
                          5, 2, torch)
    k = sum(ms) / len(ms)
    out["sample_cells_f32_config4"] = {"particles_per_s": nc / (k * 1e-3), "ms": k, "write_GBps": 12 * nc / (k * 1e-3) / 1e9}
    # Table I lines 1-4 "are required only once": the per-cell records prepared outside, sampling only
    kg.cells_prepare(kd, td, dd, 0, workspace=ws, stream=st)
    _, ms = time_launches(lambda s: kg.sample_cells_prepared(cfg.ncell, cfg.ppc, ws, cfg.seed, s * nc, "f32", out=p32, stream=st),
                          5, 2, torch)
    k = sum(ms) / len(ms)
    out["sample_cells_prepared_f32_config4"] = {"particles_per_s": nc / (k * 1e-3), "ms": k, "write_GBps": 12 * nc / (k * 1e-3) / 1e9,
                                                "note": "kappagen_cells_prepare (0.1 ms) outside the timed call"}
    # the fused loader: planes + per-cell moments in one kernel, and moments only
    mom = torch.empty((cfg.ncell, 4), dtype=torch.float32, device="cuda")
    _, ms = time_launches(lambda s: kg.sample_cells_moments(cfg.ppc, kd, td, dd, 0, cfg.seed, s * nc, out=p32, moments=mom,
                                                            workspace=ws, stream=st), 5, 2, torch)
    k = sum(ms) / len(ms)
    out["sample_cells_moments_f32_config4"] = {"particles_per_s": nc / (k * 1e-3), "ms": k}
    _, ms = time_launches(lambda s: kg.sample_cells_moments(cfg.ppc, kd, td, dd, 0, cfg.seed, s * nc, moments=mom, workspace=ws,
                                                            stream=st, store=False), 5, 2, torch)
    k = sum(ms) / len(ms)
    out["cells_moments_only_f32_config4"] = {"particles_per_s": nc / (k * 1e-3), "ms": k}
    # the particle loader (second half): 32-byte AoS records {fx,fy,fz,cell,vx,vy,vz,w}, one kernel,
    # against the SoA sampler followed by three strided copies into the record array (which still lacks the positions)
    rec = torch.empty((nc, 8), dtype=torch.float32, device="cuda")
    _, ms = time_launches(lambda s: kg.load_cells(cfg.ppc, kd, td, dd, 0, None, 0, cfg.seed, s * nc, out=rec, workspace=ws, stream=st),
                          5, 2, torch)
    k = sum(ms) / len(ms)
    out["load_cells_f32_config4"] = {"particles_per_s": nc / (k * 1e-3), "ms": k, "write_GBps": 32 * nc / (k * 1e-3) / 1e9,
                                     "record_bytes": 32}

    def soa_then_interleave(s):
        kg.sample_cells(cfg.ppc, kd, td, dd, 0, cfg.seed, s * nc, out=p32, workspace=ws, stream=st)
        for q in range(3):
            rec[:, 4 + q].copy_(p32[q][:nc])
    _, ms = time_launches(soa_then_interleave, 5, 2, torch)
    k = sum(ms) / len(ms)
    out["sample_cells_then_interleave_f32_config4"] = {"particles_per_s": nc / (k * 1e-3), "ms": k,
                                                       "note": "velocities only: positions, ids and weights not written"}
    del rec
    # paper test 2 on the device: generate and bin 2^28 speeds, no velocity written
    hist = torch.zeros(512, dtype=torch.int64, device="cuda")
    for dt in ("f32", "f64"):
        _, ms = time_launches(lambda s: kg.speed_histogram(n, 4.1, 1, s * n, dt, 0, 0.2, 512, hist=hist, stream=st), 5, 2, torch)
        k = sum(ms) / len(ms)
        out["speed_histogram_" + dt] = {"particles_per_s": n / (k * 1e-3), "ms": k}
    return out


def sweep(kg, torch):
    """The paper's benchmark shape (particles generated as a function of kappa) over the sizes the
    north_star names: 1e6 ... 2^30 particles, kappa 1.6 ... 10, both dtypes (2^30 in fp32 only: 12.9 GB)."""
    out = []
    st = torch.cuda.current_stream()
    for dt, tdt, sizes in (("f32", torch.float32, (10**6, 10**7, 10**8, 1 << 28, 1 << 30)),
                           ("f64", torch.float64, (10**6, 10**7, 10**8, 1 << 28))):
        planes = tuple(torch.empty(max(sizes), dtype=tdt, device="cuda") for _ in range(3))
        for n in sizes:
            view = tuple(p[:n] for p in planes)
            for kappa in (1.6, 3.0, 10.0):
                _, ms = time_launches(lambda s: kg.sample(n, kappa, 1.0, 1, s * n, dt, out=view, stream=st), 4, 2, torch)
                k = min(ms)
                out.append({"dtype": dt, "n": n, "kappa": kappa, "ms": k, "particles_per_s": n / (k * 1e-3)})
        del planes
    return out


def pipe_rates():
    """The issue-rate probe of every mix at 1, 2, 4, 8 warps per scheduler: cycles per loop iteration per warp."""
    import torch
    from paper_2602_05606_b200 import kappagen as kg
    if not torch.cuda.is_available():
        raise SystemExit("--pipe-rates needs a CUDA device")
    ws = (1, 2, 3, 4, 8)                                  # 3 = the double sampler's warps per scheduler (one block of 384)
    print("| mix | instructions per iteration | " + " | ".join("w=%d" % w for w in ws) + " | sum of single-kind costs at w=8 |")
    print("|---|---|" + "---|" * (len(ws) + 1))
    single = {}
    rows = []
    for mix in range(kg.pipe_probe_count()):
        cyc = [kg.pipe_probe(mix, w, 2048) for w in ws]
        counts = cyc[0][1]
        if len(counts) == 1:
            (kind, cnt), = counts.items()
            single[kind] = cyc[-1][0] / cnt
        rows.append((mix, counts, [c[0] for c in cyc]))
    for mix, counts, c in rows:
        add = sum(single.get(k, float("nan")) * v for k, v in counts.items())
        print("| %d | %s | %s | %.1f |" % (mix, " + ".join("%d %s" % (v, k) for k, v in counts.items()),
                                          " | ".join("%.1f" % x for x in c), add))
    print()
    print("cycles per warp instruction per scheduler at w=8 (loop overhead of ~3 instructions per iteration included): " +
          ", ".join("%s %.2f" % (k, v) for k, v in single.items()))


def main():
    args = parse_args()
    if args.pipe_rates:
        pipe_rates()
        return
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
