#!/usr/bin/env python
"""bench.py -- events/s per Vegas iteration (BASELINE.json metric) on the headline workload.

A step = one pass of the whole hot path: one Vegas iteration over n_events (S1-S6: Philox draw, grid map,
integrand, compensated sums, histograms, finalize) followed by the grid refinement (S7) -- vegas_step_enqueue, on
BASELINE.json configs[1] (d=8 double Gaussian, 50 bins, 1e8 events per iteration, FP64, seed 0).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg2|cfg4|cfg5|cfg1] [--epl E]
  python bench.py --impl reference ...      # the CPU oracle, as it stands, on the host cores

Prints ONE JSON line (rank 0).  `value` = events of the whole job / device time (CUDA events, max over ranks);
`e2e` = the same through vegas_iterate/vegas_refine with host result buffers (D2H of I, sigma, histogram
inside the timed region; the path has no host inputs: events are generated in registers from
(seed, iteration, event index)); `roofline` and `cpu_baseline` as described in DESIGN.md "Measurement".
Multi-GPU (--gpus N under torchrun): the iteration is SHARDED: rank g runs the events
[g n/N, (g+1) n/N) of the same n-event iteration, ONE all-reduce (NCCL) of the 8 + d*N partial sums per iteration,
then S6 and the identical refinement on every rank -- total work fixed, "scaling": "strong".
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
# What one launch of the committed iterate kernel executed per event and moved through DRAM, from the round-3 ncu
# captures (profiles/r03_kernel_counts.md names the commands; written by `python -m paper_2010_09341_b200.ncu_counts`).
# The algorithmic HBM traffic is ~0: one table read and one d*N flush per CTA.
KERNEL_COUNTS_CSV = os.path.join(ROOT, "profiles", "r03_kernel_counts.csv")


def kernel_counts(workload, w=None, shape=None):
    """(row, note): the row of profiles/r03_kernel_counts.csv for this workload (dict of floats) -- or (None, why) when
    there is none, when the kernel sources changed since the capture (the row's src_sha is not this tree's), or when the
    instance the row was captured from, iterate_kernel<F, D, NB, RS, TREP, HB, MAXT, MINB>, is not the shape running
    now (dim, bins, 2^RS histogram replicas, threads per CTA): stale counts must not pass for co-bounds."""
    import csv
    import re
    from paper_2010_09341_b200 import build as B
    try:
        with open(KERNEL_COUNTS_CSV) as fh:
            rows = [r for r in csv.DictReader(fh) if r["workload"] == workload]
    except OSError:
        return None, "no %s" % os.path.relpath(KERNEL_COUNTS_CSV, ROOT)
    if not rows:
        return None, "no row for %s in %s" % (workload, os.path.relpath(KERNEL_COUNTS_CSV, ROOT))
    row = rows[0]
    text = ("workload", "kernel", "src_sha")
    kc = {k: (v if k in text else float(v)) for k, v in row.items()}
    if kc.get("src_sha") != B.kernel_source_sha():
        return None, "the kernel sources changed since the capture (csv %s, tree %s): recapture" % (kc.get("src_sha"), B.kernel_source_sha())
    m = re.search(r"<\s*\w+\s*,\s*(\d+),\s*(\d+),\s*(-?\d+),\s*(\d+),\s*(\d+),\s*(\d+),\s*(\d+)\s*>", kc["kernel"])
    if m and w is not None and shape is not None:
        D, NB, RS, _, _, MAXT, _ = (int(v) for v in m.groups())
        if (D, NB) != (w.dim, w.nbins) or (RS >= 0 and (1 << RS) != shape["hist_replicas"]) or MAXT < shape["threads_per_cta"]:
            return None, "captured instance %s is not the running shape %s" % (kc["kernel"], shape)
    return kc, None


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
    ap.add_argument("--no-other-configs", action="store_true", help="skip the other_configs block (cfg1, cfg3, cfg4, cfg5)")
    ap.add_argument("--cpu-sample", type=int, default=10**8, help="events of the cpu_baseline oracle step")
    ap.add_argument("--ref-sample", type=int, default=10**7, help="events per step of --impl reference")
    ap.add_argument("--dist-backend", default="nccl", choices=["nccl", "gloo"],
                    help="gloo lets two ranks share one GPU (a check of the sharded path on a 1-GPU box; not a measurement)")
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


def aggregate_value(events_per_step, steps, ms):
    """Whole-job throughput of the sharded run: the n events of every step (all ranks' shards together) over the slowest
    rank's time."""
    return float(events_per_step) * steps / (ms * 1e-3)


def nccl_lines(path, limit=12):
    """The communicator lines NCCL wrote to its debug file (topology / algorithm evidence for the N > 1 run)."""
    keep = []
    try:
        with open(path) as fh:
            for ln in fh:
                if any(k in ln for k in ("comm 0x", "NVLS", "Connected all", "nRanks", "Init COMPLETE", "Channel 00/")):
                    keep.append(ln.strip()[:200])
    except OSError:
        pass
    return keep[:limit]


def other_configs(V, torch, info, clock_hz, steps=5):
    """The BASELINE.json configurations besides the headline one, so that the driver's record carries them too: device
    time (CUDA events on the stream the kernels are launched on, which is torch's current stream) of `steps` whole
    steps after 2 untimed ones.  cfg1: fused steps replayed by vegas_run_integration's CUDA graphs (the latency-bound
    case: microseconds per step); cfg3: one iteration + refinement per events_per_launch of the batch-size study;
    cfg4, cfg5: fused steps as in the headline measurement.  roofline_frac = algorithmic FLOPs (ALGO_FLOPS) per second
    over SMs x lanes x 2 x max SM clock of the dtype's pipe."""
    def frac(w, name, events_per_s, pass_fraction=1.0):
        fpe = ALGO_FLOPS[name]
        if isinstance(fpe, tuple):
            fpe = fpe[0] * pass_fraction + fpe[1] * (1.0 - pass_fraction)
        peak = info["sm_count"] * FP_LANES[dtype_of(w)] * 2 * clock_hz
        return fpe * events_per_s / peak

    def timed(fn, n_steps):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record()
        for _ in range(n_steps):
            fn()
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / n_steps

    out = {}
    # cfg1: 1e5 events per step; 160 graph-replayed steps after a 16-step warm-up run
    w = W.cfg1()
    g = V.from_workload(w)
    g.run_integration(16, w.n_events, 0, w.seed, w.alpha)
    g.run_integration(160, w.n_events, 0, w.seed, w.alpha)
    ms = g.last_sums()[2]                                 # the run's average device time per step
    out["cfg1"] = {"us_per_step": ms * 1e3, "events_per_s": w.n_events / (ms * 1e-3), "steps": 160,
                   "roofline_frac": frac(w, "cfg1", w.n_events / (ms * 1e-3)), "dtype": dtype_of(w),
                   "path": "vegas_run_integration (CUDA graphs of 16 fused steps)"}
    g.close()
    # cfg3: the batch-size study
    w = W.cfg3()
    g = V.from_workload(w)
    rows = []
    for epl in w.batch_sizes:
        g.reset()

        def step():
            g.iterate_enqueue(w.n_events, epl, w.seed)
            g.refine_enqueue(w.alpha)
        for _ in range(2):
            step()
        ms = timed(step, steps)
        g.refine_collect()
        rows.append({"events_per_launch": epl, "ms_per_iter": ms, "events_per_s": w.n_events / (ms * 1e-3),
                     "roofline_frac": frac(w, "cfg2", w.n_events / (ms * 1e-3))})
    out["cfg3"] = {"rows": rows, "dtype": dtype_of(w), "steps": steps, "path": "vegas_iterate_enqueue + vegas_refine_enqueue"}
    g.close()
    for name in ("cfg4", "cfg5"):
        w = W.ALL[name]()
        g = V.from_workload(w)
        g.reset()

        def step():
            g.step_enqueue(w.n_events, w.n_events, w.seed, w.alpha)
        for _ in range(2):
            step()
        ms = timed(step, steps)
        g.refine_collect()
        g.iterate_collect(want_hist=False)
        pf = g.last_npass() / float(w.n_events)
        out[name] = {"ms_per_iter": ms, "events_per_s": w.n_events / (ms * 1e-3), "steps": steps, "dtype": dtype_of(w),
                     "roofline_frac": frac(w, name, w.n_events / (ms * 1e-3), pf), "pass_fraction": pf,
                     "path": "vegas_step_enqueue (fused step)"}
        g.close()
    return out


def run_b200(args):
    import torch
    import torch.distributed as dist
    from paper_2010_09341_b200 import sharded as S
    from paper_2010_09341_b200 import vegas as V

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    local = local % torch.cuda.device_count()            # (--dist-backend gloo: several ranks may share one GPU)
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    nccl_log = None
    if world > 1:
        if args.dist_backend == "nccl":
            nccl_log = "/tmp/vegas_bench_nccl_%d.log" % os.getpid()
            os.environ.setdefault("NCCL_DEBUG", "INFO")
            os.environ.setdefault("NCCL_DEBUG_SUBSYS", "INIT,GRAPH")
            os.environ.setdefault("NCCL_DEBUG_FILE", nccl_log)
            dist.init_process_group("nccl", device_id=dev)
        else:
            dist.init_process_group("gloo")

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    w, n = workload(args)
    first, count = S.shard_range(n, rank, world)         # this rank's share of every iteration (all of it at N = 1)
    epl = args.epl or max(count, 1)
    g = V.from_workload(w, device="cuda:%d" % local)
    if args.ctas_per_sm or args.threads:
        g.set_launch_shape(args.ctas_per_sm, args.threads)
    if args.replicas:
        g.set_hist_replicas(args.replicas)
    shape = g.launch_shape()
    info = g.device_info()
    # measured pipe rates (thread-instructions/s), same process, right before the timed region
    pipes = {name: V.pipe_rate(kind) for name, kind in (("dfma", V.PIPE_DFMA), ("ffma", V.PIPE_FFMA),
             ("imad_wide", V.PIPE_IMAD_WIDE), ("lop3", V.PIPE_LOP3), ("shared_f64_add", V.PIPE_SHARED_F64_ADD),
             ("dfma_3reg", V.PIPE_DFMA_3REG), ("mix_event_loop", V.PIPE_MIX_EVENT_LOOP))} if rank == 0 else {}

    def step_async():
        if world == 1:                      # the fused step: S6 and S7 run in the last CTA of the iteration's kernels,
            return g.step_enqueue(n, epl, w.seed, w.alpha)      # no memset, no separate refine kernel, no host round trip
        # this rank's shard, ONE all-reduce of the 8 + d*N partials, then S6 + S7 on every rank
        # (one kernel; the refinement's outcome is collected after the timed region)
        return S.iterate_sharded_enqueue(g, n, epl, w.seed, refine_alpha=w.alpha) + 1

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
    def step_blocking():
        if world == 1:
            g.iterate(n, epl, w.seed)                   # D2H: I, sigma, histogram
        else:
            S.iterate_sharded_enqueue(g, n, epl, w.seed)
            g.iterate_collect()                         # D2H: I, sigma, histogram
        g.refine(w.alpha)                               # D2H: status

    g.reset()
    for _ in range(args.warmup):
        step_blocking()
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        step_blocking()
    torch.cuda.synchronize(dev)
    e2e_ms = (time.perf_counter() - t0) * 1e3

    dev_ms, e2e_ms, iter_ms = max_over_ranks([dev_ms, e2e_ms, iter_ms], dev if args.dist_backend == "nccl" else "cpu")

    if rank == 0:
        total_events = float(n) * args.steps              # the whole job: every step is ONE n-event iteration
        value = aggregate_value(n, args.steps, dev_ms)
        dt = dtype_of(w)
        kern_s = iter_ms * 1e-3 / args.steps          # average duration of one iteration's kernels (this rank's shard)
        fpe = ALGO_FLOPS[args.workload]
        if isinstance(fpe, tuple):
            fpe = fpe[0] * pass_fraction + fpe[1] * (1.0 - pass_fraction)
        flops = fpe * count                           # one rank's launch processes its shard
        clock_hz = (clocks.get("sm_max_mhz") or info["sm_clock_khz"] / 1e3) * 1e6
        peak = info["sm_count"] * FP_LANES[dt] * 2 * clock_hz / 1e12
        achieved = flops / kern_s / 1e12
        fp_rate = pipes["dfma" if dt == "f64" else "ffma"]
        peak_measured = 2.0 * fp_rate / 1e12
        # ---- the co-bounds (SURVEY 8.d "Report all four"): fraction of each SM resource's peak that this kernel's own
        # instruction stream takes at the measured events/s; per-event counts from the ncu capture of the committed
        # kernel (profiles/r03_kernel_counts.csv), pipe rates from vegas_pipe_rate in this process.  The shared-memory
        # data pipe serves one wavefront per clock per SM; the issue stage one warp instruction per SM sub-partition
        # per clock.  `evidence` holds comparison figures that are NOT hardware ceilings.
        kc, kc_note = kernel_counts(args.workload, w, shape)
        ev_per_s = count / kern_s
        bounds, bound_detail, evidence = None, {"note": kc_note}, None
        if kc:
            issue_rate = info["sm_count"] * 4 * 32 * clock_hz
            bounds = {
                "fp_pipe": ev_per_s * kc["fp64" if dt == "f64" else "fp32"] / fp_rate,
                "int_wide": ev_per_s * kc["imad_wide"] / pipes["imad_wide"],
                "shared_pipe": ev_per_s * kc["smem_wavefronts"] / (info["sm_count"] * clock_hz),
                "issue": ev_per_s * kc["inst"] / issue_rate,
            }
            evidence = {
                # histogram updates that reach the accumulators (events that pass the cuts x d) against the rate of a
                # latency-chained microbenchmark of the same LDS + DADD + ATOMS.CAS update (vegas_pipe_rate SHARED_F64_ADD)
                "hist_updates_vs_cas_microbenchmark": ev_per_s * pass_fraction * w.dim / pipes["shared_f64_add"],
                # the kernel's instruction rate against that of a dependency-free synthetic stream of the event loop's
                # instruction ratio (vegas_pipe_rate MIX_EVENT_LOOP): a comparison stream, not a ceiling
                "instr_rate_vs_synthetic_mix": ev_per_s * kc["inst"] / pipes["mix_event_loop"],
            }
            bound_detail = {"per_event": {k: kc[k] for k in ("inst", "fp64", "fp32", "imad_wide", "imad", "lop3", "lds", "atoms", "smem_wavefronts")},
                            "hist_updates_per_event": w.dim * pass_fraction,
                            "source": "profiles/r03_kernel_counts.csv (ncu capture of %s, kernel sources %s)" % (kc["kernel"], kc["src_sha"]),
                            "meaning": "events/s x per-event count / peak rate of that resource (1.0 = saturated): fp_pipe and "
                                       "int_wide against the measured DFMA|FFMA and IMAD.WIDE rates, shared_pipe = shared-memory "
                                       "wavefronts against 1 per clock per SM, issue = warp instructions against 1 per clock per "
                                       "SM sub-partition"}
        at_full = (n == w.n_events and world == 1 and epl == n)
        out = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": dev_ms / args.steps, "higher_is_better": True, "scaling": "strong" if world > 1 else "weak",
            "vs_baseline": None,
            "dtype": dt, "data": "synthetic", "config": config_of(args, w, n, shape),
            "clocks": clocks,
            "e2e": {"value": total_events / (e2e_ms * 1e-3), "unit": UNIT, "h2d_bytes_per_step": 0,
                    "d2h_bytes_per_step": 16 + w.dim * w.nbins * 8 + 4,
                    "note": "vegas_iterate + vegas_refine with host result buffers, host wall clock"},
            "gpu_launches": launches,
            "roofline": {"bound": "alu", "achieved": achieved, "peak": peak, "unit": "TFLOP/s", "frac": achieved / peak,
                         "traffic": kc["dram_bytes"] if (kc and at_full) else None,
                         "traffic_unit": "bytes per launch: dram__bytes_read.sum + dram__bytes_write.sum of the ncu --set full capture in profiles/r03_kernel_counts.csv",
                         "kernel": "iterate_kernel", "kernel_ms": kern_s * 1e3,
                         "flops_per_event": fpe,
                         "peak_source": "SMs x %d %s lanes x 2 x max SM clock (B200 unit counts; DESIGN.md section 7)" % (FP_LANES[dt], dt),
                         "peak_measured": peak_measured, "frac_of_measured": achieved / peak_measured,
                         "peak_measured_source": "2 x vegas_pipe_rate(%s) in this process before the timed region" % ("DFMA" if dt == "f64" else "FFMA"),
                         "pipe_rates_thread_instr_per_s": pipes,
                         "bounds": bounds,
                         "co_bound": max(bounds, key=bounds.get) if bounds else None,
                         "evidence": evidence,
                         "bounds_detail": bound_detail},
            "result": {"integral": I, "error": s, "pass_fraction": pass_fraction},
        }
        if world == 1 and args.workload == "cfg2" and at_full and not args.no_other_configs:
            out["other_configs"] = other_configs(V, torch, info, clock_hz)
        if world > 1:
            out["config"]["parallelism"] = ("events sharded over %d ranks ([g n/N, (g+1) n/N), last rank takes the remainder); one "
                                            "all-reduce of %d doubles per iteration (%s); identical refine on every rank"
                                            % (world, 8 + w.dim * w.nbins, args.dist_backend))
            out["config"]["nccl"] = nccl_lines(nccl_log) if nccl_log else []
            for ln in out["config"]["nccl"]:
                print("[nccl] " + ln, file=sys.stderr)
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
