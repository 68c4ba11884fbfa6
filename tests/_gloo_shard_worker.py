"""Worker of tests/test_sharding.py: one of WORLD_SIZE gloo ranks on CPU.  The host flow of a sharded iteration
(paper_2010_09341_b200.sharded: partition, one all-reduce of the partials, finalize, identical refine on every rank)
with the CPU oracle standing in for the kernels: its range call plays vegas_iterate_shard_enqueue and its commit call
plays vegas_finalize_enqueue.  No GPU, no product kernels."""
import math
import os
import sys

import numpy as np
import torch
import torch.distributed as dist

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
from oracle import oracle as O  # noqa: E402
from paper_2010_09341_b200 import sharded, workloads as W  # noqa: E402


class OracleShard:
    """The three calls of the binding, on the CPU: partials = {S1.hi, S1.lo, S2.hi, S2.lo, npass, 0, 0, 0, H}."""

    def __init__(self, w):
        self.o = O.Oracle(w.dim, w.nbins, w.integrand_id, w.params, w.precision)
        self.t = torch.zeros(8 + w.dim * w.nbins, dtype=torch.float64)
        self.result = None

    def iterate_shard_enqueue(self, n_total, first, count, epl, seed):
        self.t.zero_()
        if count:
            sums, hs, hc, npass = self.o.iterate_range(first, count, seed)
            self.t[0:4] = torch.from_numpy(sums)
            self.t[4] = float(npass)
            self.t[8:] = torch.from_numpy((hs + hc).reshape(-1))
        return -(-count // epl)

    def partials_tensor(self):
        return self.t

    def finalize_enqueue(self, n_total):
        p = self.t.numpy()
        h = p[8:].reshape(self.o.dim, self.o.nbins).copy()
        I, s = self.o.commit(n_total, math.fsum(p[0:2]), math.fsum(p[2:4]), h)
        self.result = (I, s, h, int(p[4]))


def main():
    dist.init_process_group("gloo")
    rank, world = dist.get_rank(), dist.get_world_size()
    w = W.cfg5()
    n = 200_003                                          # ragged: the last rank takes the remainder
    ctx = OracleShard(w)
    ref = O.Oracle(w.dim, w.nbins, w.integrand_id, w.params, w.precision)
    for it in range(2):
        launches = sharded.iterate_sharded_enqueue(ctx, n, 30_000, w.seed)
        first, count = sharded.shard_range(n, rank, world)
        assert launches == -(-count // 30_000)
        I, s, h, npass = ctx.result
        ref_npass = ref.iterate_range(0, n, w.seed)[3]   # (a range call changes no state)
        rI, rs, rh = ref.iterate(n, w.seed)              # the unsharded iteration, single-threaded
        assert abs(I - rI) <= 1e-13 * abs(rI) and abs(s - rs) <= 1e-13 * abs(rs), (rank, I, rI, s, rs)
        np.testing.assert_allclose(h, rh, rtol=1e-12, atol=0)
        assert npass == ref_npass
        ctx.o.refine(w.alpha)                            # every rank refines from the same reduced histogram
        ref.refine(w.alpha)
        ctx.o.set_iteration(ref.iteration)               # (the stand-in's range call does not count iterations)
        # identical grids on all ranks, bit for bit, with no further communication
        e = torch.from_numpy(ctx.o.get_grid().copy())
        lo, hi = e.clone(), e.clone()
        dist.all_reduce(lo, op=dist.ReduceOp.MIN); dist.all_reduce(hi, op=dist.ReduceOp.MAX)
        assert torch.equal(lo, hi)
        assert np.max(np.abs(ctx.o.get_grid() - ref.get_grid())) <= 1e-13
    dist.barrier()
    if rank == 0:
        print("SHARD_OK world=%d I=%.15g" % (world, I))
    dist.destroy_process_group()


if __name__ == "__main__":
    main()
