#!/usr/bin/env python
"""bench.py -- events/s per Vegas iteration (BASELINE.json metric) on the headline workload.

A step = one pass of the whole hot path: one Vegas iteration over n_events (S1-S6: Philox draw, grid map,
integrand, compensated sums, histograms, finalize) followed by the grid refinement (S7), on
BASELINE.json configs[1] (d=8 double Gaussian, 50 bins, 1e8 events per iteration, FP64, seed 0).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg2|cfg4|cfg5|cfg1] [--epl E]
  python bench.py --impl reference ...      # the CPU oracle, as it stands, on the host cores

Prints ONE JSON line (rank 0).  `value` = events of all ranks / device time (CUDA events, max over ranks);
`e2e` = the same through vegas_iterate/vegas_refine with host result buffers (D2H of I, sigma, histogram
inside the timed region; the path has no host inputs: events are generated in registers from
(seed, iteration, event index)); `roofline` and `cpu_baseline` as described in DESIGN.md "Measurement".
Multi-GPU: the path does not shard in this build ("replicas only"): --gpus N runs N
independent replicas, one process per GPU, no data-path collective.
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

from paper_2010_09341_b200 import workloads as W  # noqa: E402

METRIC = "events/sec per Vegas iteration"
UNIT = "events/s"

# Algorithmic FP work per event (FMA = 2 FLOPs, exp/cos/div
# expanded to the sequences nvcc emits).  fp64 FLOPs for the fp64 configs, fp32 FLOPs for cfg4.
# cfg5: 130 per event that passes the cuts, 14 per rejected one (mean taken with the measured pass fraction).
ALGO_FLOPS = {"cfg1": 67.0, "cfg2": 154.0, "cfg2_u32": 154.0, "cfg4": 232.0, "cfg5": (130.0, 14.0)}
# FP pipe lanes per SM (B200): 64 fp64, 128 fp32.  Peak = SMs * lanes * 2 FLOP * max SM clock.
FP_LANES = {"f64": 64, "f32": 128}
# dram__bytes_read.sum + dram__bytes_write.sum of one 1e8-event iterate_kernel launch, from the ncu --set full
# captures summarised in profiles/r01[c-e]_ncu_full_<cfg>_iterate.md (the algorithmic HBM traffic is ~0: one table
# read and one d*N flush per CTA)
NCU_TRAFFIC_BYTES = {"cfg2": 36352, "cfg4": 73216, "cfg5": 44032}   # r01c-r01e captures: 35-44 KB (cfg2, cfg5), 70-73 KB (cfg4)


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--workload", default="cfg2", choices=["cfg1", "cfg2", "cfg4", "cfg5", "cfg2_u32"])
    ap.add_argument("--n-events", type=int, default=0, help="override events per iteration (parity/debug only)")
    ap.add_argument("--epl", type=int, default=0, help="events per launch (0 = whole iteration in one launch)")
    ap.add_argument("--ctas-per-sm", type=int, default=0)
    ap.add_argument("--threads", type=int, default=0)
    ap.add_argument("--replicas", type=int, default=0)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-sample", type=int, default=10**8, help="events of the cpu_baseline oracle step")
    ap.add_argument("--ref-sample", type=int, default=10**7, help="events per step of --impl reference")
    return ap.parse_args()


def workload(args):
    w = W.ALL[args.workload]()
    n = args.n_events or w.n_events
    return w, n


def dtype_of(w):
    return "f32" if w.precision == W.FP32_EVAL else "f64"


def config_of(args, w, n, shape=None):
    cfg = {"workload": "%s: %s, d=%d, %d bins, %d events/iteration, alpha=%.1f, seed=%d (%s)" % (
        args.workload, w.name, w.dim, w.nbins, n, w.alpha, w.seed, w.note),
        "events_per_launch": args.epl or n,
        "l2": "n/a: no HBM-resident inputs (events are generated in registers from (seed, iteration, event index)); "
              "the table/histogram live in shared memory"}
    if shape:
        cfg["launch_shape"] = shape
    return cfg


# ---------------------------------------------------------------------------------------------------
# clocks during the timed region (NVML polling thread)
# ---------------------------------------------------------------------------------------------------
class ClockSampler:
    def __init__(self, index):
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop = threading.Event()
        self._thr = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self._nv = pynvml
            self._h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self._h, pynvml.NVML_CLOCK_SM)
        except Exception as e:  # no NVML: report that instead of numbers
            self._nv = None
            self.error = repr(e)

    def _run(self):
        nv = self._nv
        names = {"hw_slowdown": 0x8, "sw_power_cap": 0x4, "sw_thermal_slowdown": 0x20, "hw_thermal_slowdown": 0x40,
                 "hw_power_brake_slowdown": 0x80, "sync_boost": 0x10, "display_clock_setting": 0x100,
                 "applications_clocks_setting": 0x2}
        while not self._stop.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self._h, nv.NVML_CLOCK_SM))
                r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self._h)
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            time.sleep(0.002)

    def start(self):
        if self._nv:
            self._thr = threading.Thread(target=self._run, daemon=True)
            self._thr.start()

    def stop(self):
        self._stop.set()
        if self._thr:
            self._thr.join()
        if not self._nv:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "error": self.error}
        s = sorted(self.samples)
        return {"sm_mhz": s[len(s) // 2] if s else None, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(s)}


# ---------------------------------------------------------------------------------------------------
# the CPU oracle legs (cpu_baseline of the b200 arm; the whole of --impl reference)
# ---------------------------------------------------------------------------------------------------
def oracle_steps(w, n_sample, steps, warmup):
    """Times `steps` oracle steps (iterate over n_sample events + refine) on all host cores."""
    from oracle import oracle as O
    cores = max(1, len(os.sched_getaffinity(0)))
    o = O.Oracle(w.dim, w.nbins, w.integrand_id, w.params, w.precision)
    for _ in range(warmup):
        o.iterate(n_sample, w.seed, threads=cores)
        o.refine(w.alpha)
    t0 = time.perf_counter()
    for _ in range(steps):
        o.iterate(n_sample, w.seed, threads=cores)
        o.refine(w.alpha)
    dt = time.perf_counter() - t0
    return dt, cores


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    w, n = workload(args)
    n_sample = min(n, args.ref_sample)
    dt, cores = oracle_steps(w, n_sample, args.steps, args.warmup)
    value = n_sample * args.steps / dt
    out = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": dtype_of(w), "data": "synthetic",
        "config": config_of(args, w, n),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle",
                         "sample": "%d of %d events per step (iterate + refine), %d steps, oracle/vegas_oracle.c on %d threads"
                                   % (n_sample, n, args.steps, cores)},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(out))


# ---------------------------------------------------------------------------------------------------
# the B200 arm
# ---------------------------------------------------------------------------------------------------
def max_over_ranks(values, device="cpu"):
    """Element-wise maximum of a list of floats over all ranks (identity without a process group): the
    replicas-only multi-GPU timing rule -- every rank reports the slowest rank's time."""
    import torch
    import torch.distributed as dist
    t = torch.tensor(values, dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(v) for v in t.tolist()]


def aggregate_value(events_per_rank_step, steps, world, ms):
    """Whole-job throughput of `world` independent replicas: all ranks' events over the slowest rank's time."""
    return float(events_per_rank_step) * steps * world / (ms * 1e-3)


def run_b200(args):
    import torch
    import torch.distributed as dist
    from paper_2010_09341_b200 import vegas as V

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    w, n = workload(args)
    epl = args.epl or n
    g = V.from_workload(w, device="cuda:%d" % local)
    if args.ctas_per_sm or args.threads:
        g.set_launch_shape(args.ctas_per_sm, args.threads)
    if args.replicas:
        g.set_hist_replicas(args.replicas)
    shape = g.launch_shape()
    info = g.device_info()
    # measured pipe rates (thread-instructions/s), same process, right before the timed region
    pipes = {name: V.pipe_rate(kind) for name, kind in (("dfma", V.PIPE_DFMA), ("ffma", V.PIPE_FFMA),
             ("imad_wide", V.PIPE_IMAD_WIDE), ("lop3", V.PIPE_LOP3), ("shared_f64_add", V.PIPE_SHARED_F64_ADD))} if rank == 0 else {}

    def step_async():
        nl = g.iterate_enqueue(n, epl, w.seed)
        g.refine_enqueue(w.alpha)           # S7, no host round trip; outcome collected after the timed region
        return nl + 1                       # iterate launches (S6 runs in their last CTA) + the refine kernel

    # ---- device-timed region ----
    g.reset()
    for _ in range(args.warmup):
        step_async()
    g.refine_collect()
    sampler = ClockSampler(local)
    barrier()
    sampler.start()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    launches, iter_ms = 0, 0.0
    ev0.record()
    for _ in range(args.steps):
        launches += step_async()
    ev1.record()
    barrier()
    clocks = sampler.stop()
    dev_ms = ev0.elapsed_time(ev1)
    g.refine_collect()                      # VegasError(EGRID) if a refinement of the timed region was rejected
    # the library's own CUDA events around each iteration's memset + launches + finalize (last 64 kept)
    kept = min(args.steps, 64)
    iter_ms = sum(g.iteration_kernel_ms(b) for b in range(kept)) * (args.steps / kept)
    I, s, _ = g.iterate_collect(want_hist=False)
    pass_fraction = g.last_npass() / float(n)

    # ---- end-to-end region: the public blocking calls with host result buffers ----
    g.reset()
    for _ in range(args.warmup):
        g.iterate(n, epl, w.seed)
        g.refine(w.alpha)
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        g.iterate(n, epl, w.seed)           # D2H: I, sigma, histogram
        g.refine(w.alpha)
    torch.cuda.synchronize(dev)
    e2e_ms = (time.perf_counter() - t0) * 1e3

    dev_ms, e2e_ms, iter_ms = max_over_ranks([dev_ms, e2e_ms, iter_ms], dev)

    if rank == 0:
        total_events = float(n) * args.steps * world
        value = aggregate_value(n, args.steps, world, dev_ms)
        dt = dtype_of(w)
        kern_s = iter_ms * 1e-3 / args.steps          # average duration of one iteration's kernels
        fpe = ALGO_FLOPS[args.workload]
        if isinstance(fpe, tuple):
            fpe = fpe[0] * pass_fraction + fpe[1] * (1.0 - pass_fraction)
        flops = fpe * n
        peak = info["sm_count"] * FP_LANES[dt] * 2 * (clocks.get("sm_max_mhz") or info["sm_clock_khz"] / 1e3) * 1e6 / 1e12
        achieved = flops / kern_s / 1e12
        peak_measured = 2.0 * pipes["dfma" if dt == "f64" else "ffma"] / 1e12
        out = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": dev_ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": dt, "data": "synthetic", "config": config_of(args, w, n, shape),
            "clocks": clocks,
            "e2e": {"value": total_events / (e2e_ms * 1e-3), "unit": UNIT, "h2d_bytes_per_step": 0,
                    "d2h_bytes_per_step": 16 + w.dim * w.nbins * 8 + 4,
                    "note": "vegas_iterate + vegas_refine with host result buffers, host wall clock"},
            "gpu_launches": launches,
            "roofline": {"bound": "alu", "achieved": achieved, "peak": peak, "unit": "TFLOP/s", "frac": achieved / peak,
                         "traffic": NCU_TRAFFIC_BYTES.get(args.workload) if n == w.n_events and epl == n else None,
                         "traffic_unit": "bytes per launch (ncu, profiles/r01c_*)", "kernel": "iterate_kernel", "kernel_ms": kern_s * 1e3,
                         "flops_per_event": fpe,
                         "peak_source": "SMs x %d %s lanes x 2 x max SM clock (B200 unit counts; DESIGN.md section 7)" % (FP_LANES[dt], dt),
                         "peak_measured": peak_measured, "frac_of_measured": achieved / peak_measured,
                         "peak_measured_source": "2 x vegas_pipe_rate(%s) in this process before the timed region" % ("DFMA" if dt == "f64" else "FFMA"),
                         "pipe_rates_thread_instr_per_s": pipes,
                         "note": "issue-slot and IMAD.WIDE co-bounds: DESIGN.md section 7"},
            "result": {"integral": I, "error": s, "pass_fraction": pass_fraction},
        }
        if not args.no_cpu_baseline and world == 1:
            ns = min(n, args.cpu_sample)
            cdt, cores = oracle_steps(w, ns, 1, 0)
            n1 = min(ns, 5 * 10**6)
            from oracle import oracle as _O
            o1 = _O.Oracle(w.dim, w.nbins, w.integrand_id, w.params, w.precision)
            t1 = time.perf_counter()
            o1.iterate(n1, w.seed, threads=1)
            o1.refine(w.alpha)
            t1 = time.perf_counter() - t1
            out["cpu_baseline"] = {"value": ns / cdt, "unit": UNIT, "cores": cores, "kind": "oracle",
                                   "single_thread": {"value": n1 / t1, "unit": UNIT, "cores": 1,
                                                     "sample": "one step over the first %d events, plain single-threaded C loop" % n1},
                                   "sample": "one step (iterate + refine) over the first %d of %d events of the same "
                                             "workload, oracle/vegas_oracle.c on %d threads" % (ns, n, cores)}
        print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


def main():
    args = parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_b200(args)


if __name__ == "__main__":
    main()
