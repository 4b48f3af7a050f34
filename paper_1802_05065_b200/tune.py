"""Launch-geometry / poll-interval sweep (what the `profiles/*_geometry_sweep.txt` tables were made with).

    python -m paper_1802_05065_b200.tune [workload ...] [--k 16,64] [--geoms 128x1,128x2,256x2]

Times fpt_simulate for every (K, block x blocks-per-SM) combination on the throughput-shaped twins of the configs and
prints steps/s, the fraction of the measured FP64 / FP32 peak, the lane efficiency and a hash of the outputs (which must
not depend on the geometry).  0x0 = the library's default geometry, K = 0 its default poll interval.
"""
from __future__ import annotations

import argparse
import hashlib
import statistics

WORKLOADS = {
    "c2": ("c2", {}, 100000),
    "c2_1M": ("c2", {}, 1 << 20),
    "c3_fast": ("c3", dict(nu=1e-3, t_max=1050.0), 1 << 19),
    "c5_T0.1": ("c5", dict(temperature=0.1, t_max=2000.0), 1 << 20),
    "c1": ("c1", {}, 10000),
    "c1_big": ("c1", {}, 1 << 21),
    "c4_fast": ("c4", dict(nu=1e-4, t_max=5500.0), 1 << 18),
    "c4_under": ("c4", dict(nu=1e-4, t_max=5500.0), 65536),
}


def main():
    import torch
    from . import binding as fpt
    from .workloads import workload
    ap = argparse.ArgumentParser()
    ap.add_argument("workloads", nargs="*", default=list(WORKLOADS))
    ap.add_argument("--k", default="0")
    ap.add_argument("--geoms", default="0x0,128x1,128x2,128x3,128x4,256x1,256x2")
    ap.add_argument("--schedule", default="dynamic", choices=["dynamic", "static"],
                    help="static = the split of the paper's Appendix A (lane j owns runs j, j+L, ...), for the scheduler A/B")
    args = ap.parse_args()
    ks = [int(x) for x in args.k.split(",")]
    geoms = [tuple(int(y) for y in g.split("x")) for g in args.geoms.split(",")]
    peak64, peak32 = fpt.fp64_peak(0.5)[0], fpt.fp32_peak(0.5)[0]
    for name in args.workloads:
        base, ov, n = WORKLOADS[name]
        w = workload(base, **ov)
        ref = None
        for k in ks:
            for block, per_sm in geoms:
                fpt.set_launch(block, per_sm, 0)
                fpt.set_schedule(args.schedule)
                try:
                    prm = fpt.make_params(**dict(w["params"], check_every=k))
                    out = fpt._alloc_outputs(n)
                    ms = []
                    for i in range(4):
                        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                        e0.record()
                        fpt.simulate(prm, n, w["seed"], w["t_max"], out=out)
                        e1.record()
                        e1.synchronize()
                        if i:
                            ms.append(e0.elapsed_time(e1))
                    st = fpt.last_stats()
                finally:
                    fpt.set_launch(0, 0, 0)
                    fpt.set_schedule("dynamic")
                h = hashlib.md5(out[0].cpu().numpy().tobytes() + out[2].cpu().numpy().tobytes()).hexdigest()[:8]
                ref = ref or h
                sec = statistics.median(ms) * 1e-3
                peak = peak32 if w["params"]["precision"] == "fp32" else peak64
                print(f"{name:9s} K={st['check_every']:3d} block={st['block']:3d} per_sm={per_sm} grid={st['grid']:5d} ms={sec * 1e3:9.3f} "
                      f"steps/s={st['useful_steps'] / sec:.3e} frac={st['useful_steps'] / sec * w['n64_ref'] / peak:.3f} "
                      f"lane_eff={st['lane_efficiency']:.3f} runs_per_lane={n / (st['grid'] * st['block']):.1f} {h}{'' if h == ref else ' MISMATCH'}", flush=True)


if __name__ == "__main__":
    main()
