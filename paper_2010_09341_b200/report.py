"""Per-configuration timing report: python -m paper_2010_09341_b200.report [--configs cfg1,cfg2,...] [--json out]

Runs the BASELINE.json configurations through the C ABI on cuda:0 (full sizes, refine after every iteration,
seed 0) and prints one line per configuration: device time per iteration from the library's own CUDA events
(vegas_last_sums: memset + all launches + finalize), events/s, the batch-size sweep of configs[2]
(events/s against events_per_launch; PAPER.md:L57-L65 is the paper's version of that study), the launch
shape, the pass fraction, and the measured pipe rates.  GPU only: there is no CPU fallback.  This is the
script behind the results table in BASELINE.md; bench.py is the single-line benchmark the driver runs.
"""
from __future__ import annotations

import argparse
import json
import statistics
import time

from . import vegas as V
from . import workloads as W


def run_config(name, w, n_iter=None, epl=0, tune=False):
    g = V.from_workload(w)
    if w.integrand_id == W.LO_2TO2_TAB:
        g.set_table(W.pdf_table())
    n_iter = n_iter or w.n_iter
    g.iterate(w.n_events, epl, w.seed)          # untimed warm-up on the uniform grid
    tuned = None
    if tune and w.n_events >= 10**6:
        cands = [c for c in (10**4, 10**5, 10**6, 10**7, 10**8) if c <= w.n_events]
        tuned = g.tune_events_per_launch(w.n_events, cands, seed=w.seed)
    g.reset()
    import torch
    ms, wall, res, passf, rms = [], [], [], [], []
    for _ in range(n_iter):
        t0 = time.perf_counter()
        I, s, _ = g.iterate(w.n_events, epl, w.seed, want_hist=False)
        wall.append((time.perf_counter() - t0) * 1e3)
        ms.append(g.last_sums()[2])
        passf.append(g.last_npass() / w.n_events)
        res.append((I, s))
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        g.refine_enqueue(w.alpha)
        e1.record()
        g.refine_collect()
        rms.append(e0.elapsed_time(e1))     # refine_kernel on the current stream
    out = {"config": name, "workload": w.name, "n_events": w.n_events, "events_per_launch": epl or w.n_events,
           "iterations": n_iter, "kernel_ms_median": statistics.median(ms), "kernel_ms_best": min(ms),
           "events_per_s_median": w.n_events / (statistics.median(ms) * 1e-3),
           "events_per_s_best": w.n_events / (min(ms) * 1e-3),
           "wall_ms_median": statistics.median(wall), "refine_ms_median": statistics.median(rms), "launch_shape": g.launch_shape(),
           "launch_plan": dict(zip(("launches", "stream_lanes", "ctas_per_launch", "extra_cta_every"),
                                   V.plan_launches(w.n_events, epl or w.n_events, g.launch_shape()["threads_per_cta"],
                                                   g.device_info()["sm_count"] * g.launch_shape()["ctas_per_sm"]))),
           "pass_fraction_first_last": [passf[0], passf[-1]], "last_result": res[-1],
           "tuned_events_per_launch": tuned[0] if tuned else None, "tune_ms": tuned[1] if tuned else None}
    g.close()
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--configs", default="cfg1,cfg2,cfg3,cfg4,cfg5")
    ap.add_argument("--json", default="")
    args = ap.parse_args()
    rows = []
    pipes = {n: V.pipe_rate(k) for n, k in (("dfma", V.PIPE_DFMA), ("ffma", V.PIPE_FFMA), ("imad_wide", V.PIPE_IMAD_WIDE),
                                           ("lop3", V.PIPE_LOP3), ("shared_f64_add", V.PIPE_SHARED_F64_ADD),
                                           ("shared_f64_add_r8", V.PIPE_SHARED_F64_ADD_R8),
                                           ("shared_f64_rmw_plain", V.PIPE_SHARED_F64_RMW_PLAIN),
                                           ("shared_u32_add", V.PIPE_SHARED_U32_ADD), ("dfma_3reg", V.PIPE_DFMA_3REG),
                                           ("mix_event_loop", V.PIPE_MIX_EVENT_LOOP))}
    print(json.dumps({"pipe_rates_thread_instr_per_s": pipes}))
    for name in args.configs.split(","):
        w = W.ALL[name]()
        if name == "cfg3":
            for epl in w.batch_sizes:
                rows.append(run_config("cfg3/epl=%d" % epl, w, epl=epl))
                print(json.dumps(rows[-1]))
        else:
            rows.append(run_config(name, w, epl=w.events_per_launch, tune=True))
            print(json.dumps(rows[-1]))
    if args.json:
        with open(args.json, "w") as f:
            json.dump({"pipes": pipes, "rows": rows}, f, indent=1)


if __name__ == "__main__":
    main()
