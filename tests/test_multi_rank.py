"""The N > 1 host logic of bench.py on CPU (gloo, world_size 2): max-over-ranks timing, whole-job aggregation of the
sharded run, and the rule that only rank 0 prints (and, for --impl reference, only rank 0 works).  The sharded
iteration itself (partition, one all-reduce, finalize, identical refine) is covered by tests/test_sharding.py."""
import json
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _torchrun(args, nproc=2, timeout=300):
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(nproc),
           "--master-addr", "127.0.0.1", "--master-port", str(_free_port())] + args
    env = dict(os.environ, OMP_NUM_THREADS="1")
    return subprocess.run(cmd, cwd=ROOT, env=env, capture_output=True, text=True, timeout=timeout)


def test_max_over_ranks_and_aggregation_gloo_world2():
    r = _torchrun([os.path.join("tests", "_gloo_worker.py")])
    assert r.returncode == 0, r.stderr[-2000:]
    assert "GLOO_OK world=2 max=[11.0, 5.0, 7.0]" in r.stdout


def test_reference_arm_under_torchrun_prints_one_line_from_rank0():
    r = _torchrun(["bench.py", "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0",
                   "--workload", "cfg1", "--ref-sample", "20000"])
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["cpu_baseline"]["kind"] == "oracle"
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["value"] > 0


def test_single_process_max_over_ranks_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks([1.5, 2.5]) == [1.5, 2.5]
    assert bench.aggregate_value(100, 2, 1000.0) == 200.0
