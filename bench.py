#!/usr/bin/env python
"""bench.py -- throughput of the first-passage-time hot path (BASELINE.json metric: trajectory-steps/s and escapes/s on
one B200, fraction of the FP64 pipe peak).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload c2] [--impl ours|reference] [--no-extra]

A "step" is one pass of the whole hot path (claim ids -> Philox -> Box-Muller -> integrate -> escape test -> refill ->
results by id) over one batch: BASELINE.json configs[1] (C2: RCSJ constant bias, stochastic Heun, fp64, 10^5
trajectories, seed 2), i.e. ONE fpt_simulate call.  Inputs are generated inside the kernel from (seed, trajectory id), so
there are no input arrays; outputs (20 B per trajectory) stay in HBM for `value` and are copied to pinned host memory for
`e2e` (fpt_simulate_host).  L2 is flushed between timed steps.  With N > 1 (torchrun) every rank integrates its own
10^5-trajectory id range (first_id = rank * n_traj; no data-path collective): weak scaling.

`--impl reference` times the ORACLE (oracle/fpt_oracle.cpp, OpenMP over trajectories) on the host cores, each step a
bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "trajectory-steps/s"
UNIT = "steps/s"

PROFILES = os.path.join(ROOT, "profiles")


def kernel_source_sha() -> str:
    """sha256 over the CUDA sources the kernels are built from, comments and blank lines stripped: ties a stored measurement to
    the CODE it was taken on (rewording a comment does not invalidate a capture, changing a statement does)."""
    import hashlib
    import re
    h = hashlib.sha256()
    csrc = os.path.join(ROOT, "paper_1802_05065_b200", "csrc")
    for name in sorted(os.listdir(csrc)):
        if name.endswith((".cu", ".cuh")):
            text = open(os.path.join(csrc, name), encoding="utf-8").read()
            text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
            text = re.sub(r"//[^\n]*", "", text)
            code = "\n".join(line.rstrip() for line in text.splitlines() if line.strip())
            h.update(name.encode())
            h.update(code.encode())
    return h.hexdigest()[:16]


def ncu_traffic(workload: str, n_traj: int):
    """dram__bytes_read.sum + dram__bytes_write.sum of ONE integrator launch of this workload, from the `ncu --set full`
    capture recorded in profiles/ncu_traffic.json -- or None when there is no capture of this workload, or the kernel
    sources have changed since it was taken (the record carries their hash)."""
    try:
        rec = json.load(open(os.path.join(PROFILES, "ncu_traffic.json")))
    except (OSError, ValueError):
        return None, "no profiles/ncu_traffic.json"
    e = rec.get("captures", {}).get(f"{workload}@{n_traj}")
    if e is None:
        return None, "no capture of this workload"
    if e.get("kernel_source_sha") != kernel_source_sha():
        return None, f"capture {e.get('file')} was taken on other kernel sources ({e.get('kernel_source_sha')})"
    return int(e["dram_bytes_read"]) + int(e["dram_bytes_write"]), e.get("file")


def sass_counts():
    """profiles/sass_counts.json (written by build(): python -m paper_1802_05065_b200.sasscount --write)."""
    try:
        return json.load(open(os.path.join(PROFILES, "sass_counts.json")))["per_step"]
    except (OSError, ValueError, KeyError):
        return {}


def sass_key(kind: str, params: dict) -> str:
    return (f"{kind}_f{'32' if params['precision'] == 'fp32' else '64'}_{'ud' if params['model'] == 'underdamped' else 'od'}_"
            f"{params['scheme']}_{'sin' if params['amp'] != 0.0 else 'nosin'}_{'ramp' if params['nu'] != 0.0 else 'const'}")


def executed_per_step(counts: dict, params: dict, kernel: int):
    """FP64 (FP32) pipe instructions the kernel that ran executes per trajectory step, from its SASS: the persistent
    kernel's step loop, or consumer loop + producer loop of the specialised kernel."""
    cls = "fp32" if params["precision"] == "fp32" else "fp64"
    if kernel == 2:
        e = counts.get(sass_key("specialised", params))
        return None if not e else round(e["consumer_loop"][cls] + e["producer_loop"][cls], 2)
    e = counts.get(sass_key("persistent", params))
    return None if not e else e["step_loop"][cls]


# ------------------------------------------------------------------------------------------------------------------
class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    BAD = {"hw_slowdown": 0x8, "hw_thermal_slowdown": 0x40, "sw_thermal_slowdown": 0x20}
    NOTE = {"sw_power_cap": 0x4}

    def __init__(self, index: int, period_s: float = 0.01):
        super().__init__(daemon=True)
        self.index, self.period, self.samples, self.reasons = index, period_s, [], set()
        self.max_mhz = None
        self._stop_evt = threading.Event()
        self.ok = False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self.ok = True
        except Exception:
            self.nv = None

    def run(self):
        while self.ok and not self._stop_evt.is_set():
            try:
                self.samples.append(float(self.nv.nvmlDeviceGetClockInfo(self.h, self.nv.NVML_CLOCK_SM)))
                r = int(self.nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
                for name, bit in {**self.BAD, **self.NOTE}.items():
                    if r & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            time.sleep(self.period)

    def stop(self) -> dict:
        self._stop_evt.set()
        if self.is_alive():
            self.join()
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": 0}
        return {"sm_mhz": statistics.median(self.samples), "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(self.samples)}


def host_cores() -> int:
    try:
        return len(os.sched_getaffinity(0))
    except Exception:
        return os.cpu_count() or 1


# ------------------------------------------------------------------------------------------------------------------
def oracle_rate(w: dict, budget_s: float, n_max: int, first_id: int = 0):
    """Time the oracle (all host cores) on the first ids of workload `w`; returns (steps/s, escapes/s, ids, seconds, cores)."""
    import numpy as np
    import oracle
    p = oracle.make_params(**dict(w["params"], first_id=first_id))
    cores = oracle.omp_threads()
    n0 = min(n_max, 64 * cores)
    t0 = time.perf_counter()
    r = oracle.simulate(p, n0, w["seed"], w["t_max"])
    dt0 = time.perf_counter() - t0
    n = int(min(n_max, max(n0, n0 * budget_s / max(dt0, 1e-3))))
    if n > n0 * 1.5:
        t0 = time.perf_counter()
        r = oracle.simulate(p, n, w["seed"], w["t_max"])
        dt0 = time.perf_counter() - t0
    else:
        n = n0
    steps = float(np.sum(r["k"]))
    return steps / dt0, float(np.sum(r["status"] == 0)) / dt0, n, dt0, cores


TWINS = {"c3_fast": ("c3", dict(nu=1e-3, t_max=1050.0), 1 << 19),
         "c5_T0.1": ("c5", dict(temperature=0.1, t_max=2000.0), 1 << 20),
         "c4_fast": ("c4", dict(nu=1e-4, t_max=5500.0), 1 << 18)}


def resolve_workload(fpt, name: str):
    """(workload dict, trajectory count of a throughput-shaped twin or None)."""
    if name in TWINS:
        base, ov, n = TWINS[name]
        return fpt.workload(base, **ov), n
    return fpt.workload(name), None


def config_dict(args, w, n_traj: int) -> dict:
    """The `config` object of the JSON line: the same in both arms (ours / reference), world size excluded."""
    return {"workload": f"{args.workload}: BASELINE.json configs[{int(args.workload[1]) - 1}]"
                        + (" parameters, scaled twin" if args.workload in TWINS else ""), "n_traj_per_gpu": n_traj,
            "seed": w["seed"], "t_max": w["t_max"], "params": {k2: v for k2, v in w["params"].items()},
            "l2": "no input arrays (inputs are generated in-kernel from seed and id); 256 MiB written between timed steps",
            "parallelism": "independent id ranges, one per GPU, no collective"}


def bench_n_traj(args, w, n_twin):
    n_traj = n_twin or w["n_traj"]
    if args.workload in ("c3", "c4", "c5"):       # full configs take minutes: bench them on a fixed id range
        n_traj = min(n_traj, 1 << 16)
    if args.n_traj > 0:
        n_traj = args.n_traj
    return n_traj


def run_reference(args, rank: int):
    """--impl reference: the oracle on the host cores (rank 0 only)."""
    if rank != 0:
        return
    import paper_1802_05065_b200 as fpt
    w, n_twin = resolve_workload(fpt, args.workload)
    n_traj = bench_n_traj(args, w, n_twin)
    per_step_budget = max(1.0, min(15.0, 90.0 / max(1, args.steps + args.warmup)))
    rates, esc, ids, secs = [], [], 0, 0.0
    cores = host_cores()
    for i in range(args.warmup + args.steps):
        r, e, n, dt, cores = oracle_rate(w, per_step_budget, n_traj, first_id=0)
        if i >= args.warmup:
            rates.append(r); esc.append(e); ids = n; secs += dt
    value = statistics.mean(rates)
    sample = f"ids [0,{ids}) of the {n_traj} of the config per step, OpenMP over trajectories, {cores} threads"
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * secs / max(1, args.steps), "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64" if w["params"]["precision"] == "fp64" else "f32", "data": "synthetic",
            "config": config_dict(args, w, n_traj), "oracle_ids_per_step": ids,
            "escapes_per_s": statistics.mean(esc),
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------------------------------------
def time_workload(fpt, torch, w, n_traj, steps, warmup, flush, first_id=0, hist=False, opts=None):
    """Device-timed steps of one workload through fpt_simulate_ex; returns dict(ms list, this call's statistics, outputs)."""
    p = fpt.make_params(**dict(w["params"], first_id=first_id))
    out = fpt.binding._alloc_outputs(n_traj)
    d_stats = fpt.alloc_stats()
    h = None
    if hist and w.get("hist"):
        of, lo, hi, nb = w["hist"]
        h = (of, lo, hi, nb, torch.zeros(nb + 2, dtype=torch.int64, device="cuda"))

    def one():
        fpt.simulate_ex(p, n_traj, w["seed"], w["t_max"], hist=h, opts=opts, stats=d_stats, out=out)

    for _ in range(warmup):
        one()
    torch.cuda.synchronize()
    ms = []
    for _ in range(steps):
        if flush is not None:
            flush.add_(1)                       # write a buffer larger than L2 between timed steps
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        one()
        e1.record()
        e1.synchronize()
        ms.append(e0.elapsed_time(e1))
    return {"ms": ms, "stats": fpt.read_stats(d_stats), "out": out}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="c2", choices=["c1", "c2", "c3", "c4", "c5", "c3_fast", "c4_fast", "c5_T0.1"],
                    help="c2 = BASELINE.json configs[1] (the metric's workload).  c3/c4/c5 are the FULL configs' parameters on 65536 "
                         "ids (minutes to hours per step); the *_fast / c5_T0.1 twins keep every parameter but the ramp rate / "
                         "temperature, so a step lasts ~0.1-0.3 s (what the extra_workloads block and the ncu captures use)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--n-traj", type=int, default=0, help="override the trajectories per step (0 = the config's own count)")
    ap.add_argument("--no-extra", action="store_true", help="skip the throughput-shaped extra workloads and the CPU baseline")
    ap.add_argument("--no-time-slice", action="store_true", help="main workload: forbid time slicing (profiling the unsliced geometry)")
    ap.add_argument("--no-stated", action="store_true", help="skip the two stated-parameter legs (c3, c5: ~45 s together)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))

    if args.impl == "reference":
        run_reference(args, rank)
        return

    import numpy as np
    import torch
    import paper_1802_05065_b200 as fpt
    fpt.lib()                                    # fails loudly if the CUDA extension is missing
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    w, n_twin = resolve_workload(fpt, args.workload)
    n_traj = bench_n_traj(args, w, n_twin)
    n64 = w["n64_ref"]
    fp32 = w["params"]["precision"] == "fp32"
    flush = torch.zeros(256 << 20, dtype=torch.uint8, device="cuda")     # 256 MiB > 126 MB L2

    # roofline denominator, measured live under ~1 s of load: FP64 (FP32 for the fp32 variant) thread-instructions / s
    peak, clk_hz = (fpt.fp32_peak if fp32 else fpt.fp64_peak)(1.0)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-timed region: exactly K steps
    first_id = fpt.sharding.shard_range(n_traj * world, rank, world)[0]      # rank r integrates ids [r*n, (r+1)*n)
    main_opts = fpt.launch_opts(time_slice=False) if args.no_time_slice else None
    time_workload(fpt, torch, w, n_traj, 0, args.warmup, flush, first_id, opts=main_opts)          # warm-up
    sampler = ClockSampler(local_rank)
    barrier()
    sampler.start()
    t_wall0 = time.perf_counter()
    res = time_workload(fpt, torch, w, n_traj, args.steps, 0, flush, first_id, opts=main_opts)
    barrier()
    t_wall = time.perf_counter() - t_wall0
    clocks = sampler.stop()
    st = res["stats"]
    dev_s = sum(res["ms"]) * 1e-3
    f, g, s = res["out"]
    k = torch.where(s == 0, torch.round(f / w["params"]["dt"]), torch.full_like(f, float(st["n_cap"]))).to(torch.int64)
    useful = int(k.sum().item())
    assert useful == st["useful_steps"], (useful, st["useful_steps"])               # counters agree with the outputs
    escaped = int((s == 0).sum().item())

    # ---- end to end through the public host-buffer call (pinned host outputs, D2H inside the timed region)
    hf = torch.empty(n_traj, dtype=torch.float64).pin_memory()
    hg = torch.empty(n_traj, dtype=torch.float64).pin_memory()
    hs = torch.empty(n_traj, dtype=torch.int32).pin_memory()
    p_host = fpt.make_params(**dict(w["params"], first_id=first_id))
    for _ in range(2):
        fpt.simulate_host(p_host, n_traj, w["seed"], w["t_max"], hf, hg, hs)
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        fpt.simulate_host(p_host, n_traj, w["seed"], w["t_max"], hf, hg, hs)
    barrier()
    e2e_s = time.perf_counter() - t0
    assert torch.equal(hf, f.cpu()) and torch.equal(hs, s.cpu())

    # ---- max over ranks
    tv = torch.tensor([dev_s, e2e_s], dtype=torch.float64, device="cuda")
    tot = torch.tensor([float(useful), float(escaped)], dtype=torch.float64, device="cuda")
    if dist is not None:
        dist.all_reduce(tv, op=dist.ReduceOp.MAX)
        dist.all_reduce(tot, op=dist.ReduceOp.SUM)
    dev_s, e2e_s = float(tv[0]), float(tv[1])
    useful_all, escaped_all = float(tot[0]), float(tot[1])
    value = useful_all * args.steps / dev_s
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": 1e3 * dev_s / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32" if fp32 else "f64", "data": "synthetic",
        "config": config_dict(args, w, n_traj),
        "escapes_per_s": escaped_all * args.steps / dev_s,
        "censored": int(st["n_censored"]), "lane_efficiency": st["lane_efficiency"],
        "launch": {"grid": st["grid"], "block": st["block"], "check_every": st["check_every"],
                   "kernel": fpt.binding.KERNEL[st["kernel"]], "time_slices": st["time_slices"]},
        "wall_s_timed_region": t_wall, "ms_each_step": [round(x, 3) for x in res["ms"]],
        "e2e": {"value": useful_all * args.steps / e2e_s, "unit": UNIT, "h2d_bytes_per_step": 96,
                "d2h_bytes_per_step": n_traj * 20, "api": "fpt_simulate_host (pinned host outputs; inputs = 96-byte fpt_params)"},
        "gpu_launches": 2 * args.steps,         # per step: the integrator kernel + the 1-thread statistics export (and a 128-byte memset)
        "clocks": clocks,
    }
    per_gpu_rate = (useful * args.steps / (sum(res["ms"]) * 1e-3))
    counts = sass_counts()
    n_exec = executed_per_step(counts, w["params"], st["kernel"])
    traffic, traffic_src = ncu_traffic(args.workload, n_traj)
    cls = "FP32" if fp32 else "FP64"
    line["roofline"] = {
        "bound": "alu", "achieved": per_gpu_rate * n64 / 1e9, "peak": peak / 1e9,
        "unit": f"G {cls} thread-instr/s",
        "frac": per_gpu_rate * n64 / peak,
        "traffic": traffic, "traffic_source": traffic_src,
        "note": f"achieved = steps/s x {n64} reference {cls}-pipe instructions per step (SURVEY 8(a)); peak = "
                f"{'FFMA' if fp32 else 'DFMA'} chains measured live by fpt_fp{'32' if fp32 else '64'}_peak after 1 s of load "
                f"(SM clock seen {clk_hz / 1e6:.0f} MHz); MEASURED_PEAKS.json has no {cls} figure",
        "hbm_bytes_per_step_algorithmic": n_traj * 20,
        # what the kernel that ran really executes per step (profiles/sass_counts.json, from cuobjdump -sass at build time)
        "instr_per_step_executed": n_exec,
        "frac_executed": None if n_exec is None else per_gpu_rate * n_exec / peak,
        "kernel_source_sha": kernel_source_sha(),
    }

    if rank == 0 and world == 1 and not args.no_extra:
        # ---- throughput-shaped workloads: (i) the configs' parameters with the ramp rate / temperature changed so that a
        # step lasts ~0.1-0.3 s (twins), (ii) configs 3 and 5 at their STATED parameters on a bounded id range (one timed
        # step each, ~15-30 s): the numbers behind the 60 % target, timed by whoever runs this file
        extra = {}
        shapes = [("c2_x42", "c2", dict(), 1 << 22, False, 3, None),
                  ("c3_fast_ramp",) + TWINS["c3_fast"] + (True, 3, None),
                  ("c5_T0.1",) + TWINS["c5_T0.1"] + (False, 3, None),
                  ("c4_fast_ramp",) + TWINS["c4_fast"] + (False, 3, None),
                  # config 4's own launch geometry (65 536 trajectories: 3.46 blocks of 128 per SM -> 3 per SM, time-sliced)
                  ("c4_fast_ramp_stated_geometry",) + TWINS["c4_fast"][:2] + (1 << 16, False, 3, None)]
        if not args.no_stated:
            # the full configs keep every SM full (10^6 and 4 x 10^6 trajectories); their samples here are launched the same
            # way: one whole wave of config 3 (ramped: every trajectory lasts about as long, so a ragged last wave would idle
            # the GPU for a whole trajectory), 2^17 ids of config 5 on the full config's 3 blocks of 128 threads per SM
            full = fpt.launch_opts(block=128, blocks_per_sm=3, specialise=False)
            wave = time_workload(fpt, torch, fpt.workload("c3", t_max=10.0), 1 << 20, 0, 1, None, 0)["stats"]
            shapes += [("c3_stated_one_wave", "c3", dict(), wave["grid"] * wave["block"], True, 1, None),
                       ("c5_stated_ids_0_131072", "c5", dict(), 1 << 17, False, 1, full)]
        for name, base, ov, n, hist, reps, opts in shapes:
            ww = fpt.workload(base, **ov)
            if reps > 1:
                r = time_workload(fpt, torch, ww, n, reps, 1, flush, 0, hist=hist, opts=opts)
            else:                                   # long step: warm the kernel up on the same ids with the cap cut to 1e-4 of it
                time_workload(fpt, torch, fpt.workload(base, t_max=ww["t_max"] * 1e-4), n, 0, 1, None, 0, hist=hist, opts=opts)
                r = time_workload(fpt, torch, ww, n, 1, 0, flush, 0, hist=hist, opts=opts)
            sec = statistics.median(r["ms"]) * 1e-3
            stx = r["stats"]
            is32 = ww["params"]["precision"] == "fp32"
            pk = peak if is32 == fp32 else (fpt.fp32_peak if is32 else fpt.fp64_peak)(0.5)[0]
            nx = executed_per_step(counts, ww["params"], stx["kernel"])
            rate = stx["useful_steps"] / sec
            extra[name] = {"n_traj": n, "overrides": ov, "steps_per_s": rate, "escapes_per_s": stx["n_escaped"] / sec,
                           "ms": sec * 1e3, "censored": stx["n_censored"], "lane_efficiency": stx["lane_efficiency"],
                           "roofline_frac": rate * ww["n64_ref"] / pk, "n_ref_per_step": ww["n64_ref"],
                           "instr_per_step_executed": nx, "frac_executed": None if nx is None else rate * nx / pk,
                           "launch": {"grid": stx["grid"], "block": stx["block"], "check_every": stx["check_every"],
                                      "kernel": fpt.binding.KERNEL[stx["kernel"]], "time_slices": stx["time_slices"]},
                           "dtype": "f32" if is32 else "f64"}
        line["extra_workloads"] = extra
        # ---- the oracle as it stands on the host cores, bounded sample of the same workload
        r_cpu, e_cpu, ids, secs, cores = oracle_rate(w, 15.0, n_traj)
        line["cpu_baseline"] = {"value": r_cpu, "unit": UNIT, "cores": cores, "kind": "oracle",
                                "sample": f"ids [0,{ids}) of the bench workload, {secs:.1f} s, OpenMP over trajectories",
                                "escapes_per_s": e_cpu}
    if rank == 0:
        print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
