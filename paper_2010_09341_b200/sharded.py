"""NEXT-2 ("ensure that all GPUs ... receive a share"): one Vegas iteration
sharded over the ranks of a torch.distributed process group.

Host logic only -- the partition of the event range and the order of the calls; every step of the arithmetic runs in
the library's kernels.  Events are counter-indexed (global event index e in [0, n)), so rank g of G runs the events
[first_g, first_g + count_g) and the ONLY exchange per iteration is one all-reduce (sum) of the unreduced partials
{S1.hi, S1.lo, S2.hi, S2.lo, npass, 0, 0, 0, H[dim][nbins]} -- 8 + dim*nbins doubles, NCCL over NVLink on GPUs; after
it every rank holds the same sums, runs S6 (vegas_finalize_enqueue) and the identical refinement, so the grids stay
bit-identical on all ranks with no further communication.

`ctx` is anything with the binding's three calls (paper_2010_09341_b200.vegas.Vegas, or a stand-in in the CPU tests):
iterate_shard_enqueue(n_total, first, count, events_per_launch, seed), partials_tensor(), finalize_enqueue(n_total);
if it has a `stream` attribute (the torch stream its kernels run on) the all-reduce is issued on that stream.
Never run on more than one device so far (one GPU per box): covered by gloo tests, on CPU and with two ranks on one GPU.
"""
from __future__ import annotations


def shard_range(n_events: int, rank: int, world: int):
    """(first, count) of rank's share of [0, n_events): equal shares of n // world events, the last rank also takes the
    remainder.  The shares tile [0, n_events) exactly, in rank order."""
    if not (0 <= rank < world) or n_events < 0:
        raise ValueError("rank %d of %d, n_events %d" % (rank, world, n_events))
    base = n_events // world
    first = rank * base
    count = base if rank < world - 1 else n_events - first
    return first, count


def iterate_sharded_enqueue(ctx, n_events: int, events_per_launch: int = 0, seed: int = 0, group=None,
                            rank: int | None = None, world: int | None = None, refine_alpha: float | None = None):
    """One sharded iteration: this rank's shard, ONE all-reduce of the partials, S6.  Returns the number of kernels this
    rank launched for its shard.  Without an initialised process group (or world == 1) the shard is the whole range and
    no collective runs.  Results are read afterwards with ctx.iterate_collect() like after a plain iteration.
    With refine_alpha the identical refinement of every rank is part of the call -- S6 and S7 run as one kernel after
    the all-reduce (ctx.finalize_step_enqueue) -- and its outcome is read with ctx.refine_collect()."""
    import torch.distributed as dist
    have_pg = dist.is_available() and dist.is_initialized()
    if world is None:
        world = dist.get_world_size(group) if have_pg else 1
    if rank is None:
        rank = dist.get_rank(group) if have_pg else 0
    first, count = shard_range(int(n_events), rank, world)
    epl = int(events_per_launch) if events_per_launch else max(count, 1)
    launches = ctx.iterate_shard_enqueue(int(n_events), first, count, epl, seed)
    if world > 1:
        # The iteration's one exchange.  The collective orders itself against torch's CURRENT stream, while the shard
        # kernels before it and S6 after it run on the stream the context was created with: make that stream current
        # for the call, else the sum could read partials the last CTA has not written yet (or S6 read them before the
        # sum landed) whenever the two streams differ.
        part = ctx.partials_tensor()
        stream = getattr(ctx, "stream", None)
        if stream is not None and part.is_cuda:
            import torch
            with torch.cuda.stream(stream):
                dist.all_reduce(part, op=dist.ReduceOp.SUM, group=group)
        else:
            dist.all_reduce(part, op=dist.ReduceOp.SUM, group=group)
    if refine_alpha is None:
        ctx.finalize_enqueue(int(n_events))
    else:
        ctx.finalize_step_enqueue(int(n_events), float(refine_alpha))
    return launches


def run_integration_sharded(ctx, n_iter: int, n_events: int, events_per_launch: int = 0, seed: int = 0, alpha: float = 1.5,
                            n_warmup: int = 0, group=None):
    """PAPER.md:L79 `run_integration` over the ranks of a process group (the paper's multi-GPU mode, L53-L57):
    (n_warmup + n_iter) x {sharded iteration, identical refinement on every rank}, then the classic inverse-variance
    combination of the last n_iter iterations (the library's host routine vegas_combine_iterations).  Every rank returns
    the same (mean, error, chi2_dof, {integral, error}); one all-reduce per iteration is the only communication.  A
    refinement rejected for a non-monotone grid leaves the grid unchanged on every rank alike and the run goes on."""
    import numpy as np
    from . import vegas as V
    total = int(n_iter) + int(n_warmup)
    I, s = np.empty(total), np.empty(total)
    for it in range(total):
        iterate_sharded_enqueue(ctx, n_events, events_per_launch, seed, group=group)
        I[it], s[it], _ = ctx.iterate_collect(want_hist=False)
        try:
            ctx.refine(alpha)
        except V.VegasError as e:
            if e.code != V.EGRID:
                raise
    mean, err, chi2 = V.combine_iterations(I[n_warmup:], s[n_warmup:])
    return mean, err, chi2, dict(integral=I, error=s)
