"""NEXT-2: one Vegas iteration sharded over G ranks with ONE all-reduce of the partials.

CPU (-m "not gpu"): the partition arithmetic and, under gloo with world size 2 and 3, the host flow
shard -> all-reduce -> finalize -> identical refine, with the oracle standing in for the kernels.
GPU (-m gpu, one device): G shards run one after the other into G contexts, their partials regions are added on the
device (what the all-reduce does), S6 runs from the sum: equal to the unsharded iteration and to the oracle.
"""
import os
import socket
import subprocess
import sys

import numpy as np
import pytest

from paper_2010_09341_b200 import sharded, workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
THREADS = max(1, min(32, len(os.sched_getaffinity(0))))


def test_shard_ranges_tile_the_event_range_exactly():
    for n in (0, 1, 2, 7, 10**6 + 3, 10**8, 2**33 + 5):
        for world in (1, 2, 3, 8, 72):
            at = 0
            for rank in range(world):
                first, count = sharded.shard_range(n, rank, world)
                assert first == at and count >= 0
                if rank < world - 1:
                    assert count == n // world
                at += count
            assert at == n                               # the last rank took the remainder
    with pytest.raises(ValueError):
        sharded.shard_range(10, 2, 2)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


@pytest.mark.parametrize("world", [2, 3])
def test_sharded_iteration_flow_gloo(world):
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(world),
           "--master-addr", "127.0.0.1", "--master-port", str(_free_port()), os.path.join("tests", "_gloo_shard_worker.py")]
    r = subprocess.run(cmd, cwd=ROOT, env=dict(os.environ, OMP_NUM_THREADS="1"), capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stderr[-3000:]
    assert "SHARD_OK world=%d" % world in r.stdout


# ------------------------------------------------------------------------------------------------- GPU
@pytest.fixture(scope="module")
def V():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2010_09341_b200 import vegas
    return vegas


def _close(gres, ores, rI=1e-12, rH=1e-10):
    gI, gs, gh = gres
    oI, os_, oh = ores
    assert abs(gI - oI) <= rI * abs(oI), (gI, oI)
    assert abs(gs - os_) <= rI * abs(os_), (gs, os_)
    assert np.array_equal(gh == 0.0, oh == 0.0)
    np.testing.assert_allclose(gh, oh, rtol=rH, atol=0.0)


@pytest.mark.gpu
@pytest.mark.parametrize("name,G,n,epl", [("cfg2", 2, 10**6 + 3, 0), ("cfg2", 3, 10**6 + 3, 100_000), ("cfg5", 8, 10**6 + 3, 0),
                                          ("cfg4", 3, 500_009, 70_001), ("cfg1", 8, 5, 0)])
def test_sharded_iteration_equals_unsharded_and_oracle(V, name, G, n, epl):
    from oracle import oracle as O
    w = W.ALL[name]()
    whole = V.from_workload(w)
    o = O.Oracle(w.dim, w.nbins, w.integrand_id, w.params, w.precision)
    ctxs = [V.from_workload(w) for _ in range(G)]
    for it in range(2):
        ores = o.iterate(n, w.seed, threads=THREADS)
        wres = whole.iterate(n, epl, w.seed)
        # the shards, one after the other, each into its own context
        for rank, c in enumerate(ctxs):
            first, count = sharded.shard_range(n, rank, G)
            c.iterate_shard_enqueue(n, first, count, epl or max(count, 1), w.seed)
            with pytest.raises(V.VegasError) as ei:
                c.iterate_collect(want_hist=False)       # a shard alone has no estimate
            assert ei.value.code == V.ESTATE
        # what the all-reduce does: every rank ends up with the sum of all partials regions
        parts = [c.partials_tensor() for c in ctxs]
        assert parts[0].numel() == 8 + w.dim * w.nbins and parts[0].data_ptr() % 256 == 0
        total = sum(p.clone() for p in parts)
        for p in parts:
            p.copy_(total)
        for c in ctxs:
            c.finalize_enqueue(n)
        res = [c.iterate_collect() for c in ctxs]
        for r in res:
            _close(r, ores)
            _close(r, wres, rI=1e-13, rH=1e-12)
            assert r[0] == res[0][0] and r[1] == res[0][1] and np.array_equal(r[2], res[0][2])
        if o.npass is not None:
            assert ctxs[-1].last_npass() == o.npass == whole.last_npass()
        # identical refinement everywhere
        o.refine(w.alpha); whole.refine(w.alpha)
        for c in ctxs:
            c.refine(w.alpha)
        e0 = ctxs[0].get_grid()
        assert all(np.array_equal(c.get_grid(), e0) for c in ctxs)
        assert np.max(np.abs(e0 - o.get_grid())) <= 1e-12
        assert ctxs[0].iteration == o.iteration == whole.iteration == it + 1


@pytest.mark.gpu
def test_sharded_iteration_two_ranks_one_gpu_non_default_stream(V):
    """The real binding under a process group (gloo, two ranks sharing the one GPU), contexts on a non-default stream:
    the all-reduce must be ordered on the context's stream (tests/_gloo_gpu_shard_worker.py)."""
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", str(_free_port()), os.path.join("tests", "_gloo_gpu_shard_worker.py")]
    r = subprocess.run(cmd, cwd=ROOT, env=dict(os.environ, OMP_NUM_THREADS="1"), capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stderr[-3000:]
    assert "GPU_SHARD_OK world=2" in r.stdout


@pytest.mark.gpu
@pytest.mark.parametrize("name,n", [("cfg2", 10**6 + 3), ("cfg4", 300_007)])
def test_finalize_step_is_finalize_plus_refine(V, name, n):
    """vegas_finalize_step_enqueue (S6 + S7 in one kernel after the all-reduce) against the oracle: two shards into two
    contexts, partials summed on the device, then the fused tail; I, sigma rel 1e-12, grid within 1e-12, two iterations."""
    from oracle import oracle as O
    w = W.ALL[name]()
    o = O.Oracle(w.dim, w.nbins, w.integrand_id, w.params, w.precision)
    ctxs = [V.from_workload(w) for _ in range(2)]
    for it in range(2):
        oI, os_, _ = o.iterate(n, w.seed, threads=THREADS)
        o.refine(w.alpha)
        for rank, c in enumerate(ctxs):
            first, count = sharded.shard_range(n, rank, 2)
            c.iterate_shard_enqueue(n, first, count, count, w.seed)
        parts = [c.partials_tensor() for c in ctxs]
        total = parts[0] + parts[1]
        for p, c in zip(parts, ctxs):
            p.copy_(total)
            c.finalize_step_enqueue(n, w.alpha)
            I, s, _ = c.iterate_collect(want_hist=False)
            c.refine_collect()
            assert abs(I - oI) <= 1e-12 * abs(oI) and abs(s - os_) <= 1e-12 * abs(os_)
            assert np.max(np.abs(c.get_grid() - o.get_grid())) <= 1e-12
            with pytest.raises(V.VegasError) as ei:
                c.iterate_collect(want_hist=True)            # consumed by the refinement
            assert ei.value.code == V.ESTATE
        assert np.array_equal(ctxs[0].get_grid(), ctxs[1].get_grid())
    with pytest.raises(V.VegasError) as ei:
        ctxs[0].finalize_step_enqueue(n, w.alpha)            # no shard pending
    assert ei.value.code == V.ESTATE


@pytest.mark.gpu
def test_bench_two_ranks_gloo_on_one_gpu_matches_the_oracle(V):
    """bench.py's N > 1 path (sharded strong scaling: shard, one all-reduce, fused S6 + S7 on every rank) under
    torch.distributed.run with two gloo ranks sharing the one GPU: its line says so and its result is the oracle's."""
    import json
    from oracle import oracle as O
    n, steps, warm = 2_000_003, 2, 1
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", str(_free_port()), "bench.py", "--gpus", "2", "--dist-backend", "gloo", "--workload", "cfg2",
           "--n-events", str(n), "--steps", str(steps), "--warmup", str(warm)]
    r = subprocess.run(cmd, cwd=ROOT, env=dict(os.environ, OMP_NUM_THREADS="1"), capture_output=True, text=True, timeout=900)
    assert r.returncode == 0, r.stderr[-3000:]
    line = json.loads([ln for ln in r.stdout.splitlines() if ln.startswith("{")][-1])
    assert line["n_gpus"] == 2 and line["scaling"] == "strong" and "parallelism" in line["config"]
    assert line["gpu_launches"] == 2 * steps
    w = W.cfg2()
    o = O.Oracle(w.dim, w.nbins, w.integrand_id, w.params, w.precision)
    for _ in range(warm + steps):                            # the device-timed region's last step, from a reset grid
        oI, os_, _ = o.iterate(n, w.seed, threads=THREADS)
        o.refine(w.alpha)
    assert abs(line["result"]["integral"] - oI) <= 1e-12 * abs(oI)
    assert abs(line["result"]["error"] - os_) <= 1e-12 * abs(os_)


@pytest.mark.gpu
def test_shard_argument_errors(V):
    w = W.cfg1()
    g = V.from_workload(w)
    with pytest.raises(V.VegasError) as ei:
        g.iterate_shard_enqueue(1000, 900, 200, 100, 0)      # runs past n_total
    assert ei.value.code == V.EINVAL
    with pytest.raises(V.VegasError) as ei:
        g.finalize_enqueue(1000)                             # no shard pending
    assert ei.value.code == V.ESTATE
    g.iterate_shard_enqueue(1000, 0, 0, 100, 0)              # an empty shard is fine: zeros
    assert float(g.partials_tensor().abs().sum()) == 0.0
    with pytest.raises(V.VegasError) as ei:
        g.refine(1.5)                                        # partial histogram: not before finalize
    assert ei.value.code == V.ESTATE
    g.finalize_enqueue(1000)
    I, s, h = g.iterate_collect()
    assert I == 0.0 and s == 0.0 and not h.any()


@pytest.mark.gpu
def test_run_integration_sharded_equals_the_library_driver_without_a_process_group(V):
    """Without a process group the sharded driver is the whole range on one rank: same estimates as
    vegas_run_integration (plain loop and graph replay)."""
    w = W.cfg1()
    a, b = V.from_workload(w), V.from_workload(w)
    m1, e1, c1, log1 = sharded.run_integration_sharded(a, 4, 50_000, 0, w.seed, w.alpha, n_warmup=2)
    m2, e2, c2, log2 = b.run_integration(4, 50_000, 0, w.seed, w.alpha, n_warmup=2)
    np.testing.assert_allclose(log1["integral"], log2["integral"], rtol=1e-12)
    np.testing.assert_allclose(log1["error"], log2["error"], rtol=1e-11)
    assert abs(m1 - m2) <= 1e-12 * abs(m2) and abs(e1 - e2) <= 1e-11 * e2 and abs(c1 - c2) <= 1e-8 * max(c2, 1e-30)
    np.testing.assert_allclose(a.get_grid(), b.get_grid(), rtol=0, atol=1e-12)
