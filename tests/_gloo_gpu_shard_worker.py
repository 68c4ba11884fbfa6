"""Worker of tests/test_sharding.py::test_sharded_iteration_two_ranks_one_gpu_non_default_stream: one of WORLD_SIZE gloo
ranks that all use cuda:0.  Unlike tests/_gloo_shard_worker.py (oracle stand-in, CPU) this drives the real binding --
Vegas.iterate_shard_enqueue, partials_tensor, finalize_enqueue through sharded.iterate_sharded_enqueue -- with the context
on a stream that is NOT torch's current stream, and checks each rank's result against the unsharded iteration of a
second context.  The ranks' kernels never wait on one another (the exchange is a host-side gloo all-reduce), so sharing
the one GPU is safe.  Shards are long enough (about a millisecond of kernel) that an all-reduce ordered on the wrong
stream would read unfinished partials."""
import os
import sys

import numpy as np
import torch
import torch.distributed as dist

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
from paper_2010_09341_b200 import sharded, vegas as V, workloads as W  # noqa: E402


def main():
    dist.init_process_group("gloo")
    rank, world = dist.get_rank(), dist.get_world_size()
    torch.cuda.set_device(0)
    w = W.cfg2()
    n = 60_000_007                                       # ragged: the last rank takes the remainder
    side = torch.cuda.Stream()
    ctx = V.from_workload(w, stream=side)                # its kernels run on `side`; the current stream stays the default
    assert ctx.stream is side and torch.cuda.current_stream() != side
    whole = V.from_workload(w)
    for it in range(2):
        launches = sharded.iterate_sharded_enqueue(ctx, n, 0, w.seed)
        assert launches == 1
        I, s, h = ctx.iterate_collect()
        rI, rs, rh = whole.iterate(n, 0, w.seed)
        assert abs(I - rI) <= 1e-13 * abs(rI) and abs(s - rs) <= 1e-13 * abs(rs), (rank, it, I, rI, s, rs)
        assert np.array_equal(h == 0.0, rh == 0.0)
        np.testing.assert_allclose(h, rh, rtol=1e-12, atol=0)
        ctx.refine(w.alpha); whole.refine(w.alpha)
        e = torch.from_numpy(ctx.get_grid().copy())
        lo, hi = e.clone(), e.clone()
        dist.all_reduce(lo, op=dist.ReduceOp.MIN); dist.all_reduce(hi, op=dist.ReduceOp.MAX)
        assert torch.equal(lo, hi)                       # identical grids on all ranks, bit for bit
        assert np.max(np.abs(ctx.get_grid() - whole.get_grid())) <= 1e-13
    dist.barrier()
    if rank == 0:
        print("GPU_SHARD_OK world=%d I=%.15g" % (world, I))
    dist.destroy_process_group()


if __name__ == "__main__":
    main()
