"""Worker of tests/test_multi_rank.py: one of WORLD_SIZE gloo ranks on CPU (no GPU, no kernels)."""
import os
import sys

import torch.distributed as dist

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
import bench  # noqa: E402


def main():
    dist.init_process_group("gloo")
    rank, world = dist.get_rank(), dist.get_world_size()
    # each rank "measured" different times: everyone must end up with the element-wise maximum
    got = bench.max_over_ranks([10.0 + rank, 5.0 - rank, 7.0])
    want = [10.0 + world - 1, 5.0, 7.0]
    assert got == want, (rank, got, want)
    v = bench.aggregate_value(10**8, 4, got[0])          # sharded run: every step is ONE n-event iteration
    assert abs(v - 10**8 * 4 / (want[0] * 1e-3)) < 1e-3
    dist.barrier()
    if rank == 0:
        print("GLOO_OK world=%d max=%s" % (world, got))
    dist.destroy_process_group()


if __name__ == "__main__":
    main()
