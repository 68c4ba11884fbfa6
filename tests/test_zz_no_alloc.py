"""vegas_refine_static_enqueue -- the refinement for callers that cannot allocate device memory.

Who these callers are: code that runs as a guest inside another program (a plug-in, a framework callback, a custom
operator).  It is handed device buffers for its inputs and outputs; the host program's memory pool owns the rest of the
GPU, so the guest's own cudaMalloc can fail outright, it has no handle on the pool to ask it instead, and a
cudaMalloc / cudaFree in the middle of the host's pipelined work would stall the whole device.  Such a caller cannot
build the workspace vegas_create wants, so this one entry point keeps its working memory in an array compiled into the
library (one per device, shared by all calls, dim*(nbins+1) <= 8192 edges).

What is checked: on several calls in a row -- the array keeps the previous call's contents, so a later call must not see
the leftovers of an earlier one -- the new entry point returns the grid that the existing path (vegas_set_grid +
vegas_set_histogram / vegas_iterate + vegas_refine on a context with a workspace) commits for the same inputs, within
the tolerance the refinement's parity tests use (|dE| <= 1e-12; in fact it is the same device function in the same
launch geometry).  Calls in between are a rejected refinement (status 1, grid handed back unchanged) and a grid of
another shape.  The size limit and the argument checks need no GPU.

This file sorts last on purpose (pytest -x stops at the first failure: a failure here hides nothing); it passes alone in
a fresh process (the first call on a device does the one-time set-up) and after the other GPU tests.
"""
import ctypes as C

import numpy as np
import pytest

from paper_2010_09341_b200 import workloads as W

EDGE_TOL = 1e-12          # north_star: "refined grid edges must agree within an absolute 1e-12"

# the rejection case of tests/test_refine_kernel.py: the middle bin is one ulp wide and two new edges land in it
EG_N = 8
EG_EDGES = np.array([0.0, 0.2, 0.4, 0.5, 0.5 + 2.0 ** -53, 0.7, 0.8, 0.9, 1.0])
EG_HIST = np.array([0.0, 0.0, 0.0, 1.0, 0.0, 0.0, 0.0, 0.0])


def test_static_entry_point_refuses_what_it_cannot_hold_before_touching_the_device():
    """The capacity limit and the argument checks are host logic: they come before any CUDA call."""
    from paper_2010_09341_b200 import vegas
    L = vegas.lib()
    p = C.c_void_p(256)                                   # never dereferenced: every case fails validation first
    call = L.vegas_refine_static_enqueue
    assert vegas.STATIC_MAX_EDGES == 8192
    assert call(32, 4095, 1.5, p, p, p, p, None) == vegas.EINVAL          # 131072 edges
    msg = L.vegas_last_error().decode()
    assert "8192" in msg and "131072" in msg and "vegas_create" in msg      # says what the limit is and what to use instead
    assert call(32, 256, 1.5, p, p, p, p, None) == vegas.EINVAL           # 32 * 257 = 8224: just over
    assert call(0, 50, 1.5, p, p, p, p, None) == vegas.EINVAL
    assert call(33, 50, 1.5, p, p, p, p, None) == vegas.EINVAL
    assert call(4, 1, 1.5, p, p, p, p, None) == vegas.EINVAL
    assert call(4, 50, -1.0, p, p, p, p, None) == vegas.EINVAL
    assert call(4, 50, float("nan"), p, p, p, p, None) == vegas.EINVAL
    assert call(4, 50, 1.5, None, p, p, p, None) == vegas.EINVAL
    assert call(4, 50, 1.5, p, p, p, None, None) == vegas.EINVAL
    assert call(4, 50, 1.5, C.c_void_p(260), p, p, p, None) == vegas.EINVAL   # doubles need 8-byte alignment
    assert call(4, 50, 1.5, p, p, p, C.c_void_p(258), None) == vegas.EINVAL   # the status word 4-byte alignment


# ---------------------------------------------------------------------------------------------- GPU
gpu = pytest.mark.gpu


@pytest.fixture(scope="module")
def V():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2010_09341_b200 import vegas
    return vegas


def existing_path(V, dim, N, edges, hist, alpha):
    """The grid vegas_refine commits (context + caller-allocated workspace), or None if it rejects."""
    g = V.Vegas(dim, N, W.TOY_SUM, ())
    g.set_grid(edges)
    g.set_histogram(hist)
    try:
        g.refine(alpha)
    except V.VegasError as e:
        assert e.code == V.EGRID
        return None
    finally:
        E = g.get_grid()
        g.close()
    return E


def static_path(V, dim, N, edges, hist, alpha, in_place=False):
    """The same through vegas_refine_static_enqueue.  torch only supplies the caller's input and output buffers here
    (what the host program would hand to a guest); the entry point itself allocates nothing."""
    import torch
    dev = torch.device("cuda:0")
    e_in = torch.from_numpy(np.ascontiguousarray(edges, dtype=np.float64)).to(dev)
    h_in = torch.from_numpy(np.ascontiguousarray(hist, dtype=np.float64)).to(dev)
    e_out = e_in if in_place else torch.full_like(e_in, float("nan"))
    status = torch.full((1,), -7, dtype=torch.int32, device=dev)
    before = (edges.copy(), hist.copy())
    V.refine_static_enqueue(dim, N, alpha, e_in, h_in, e_out, status, torch.cuda.current_stream(dev))
    torch.cuda.synchronize(dev)
    if not in_place:                                      # the inputs are read-only
        assert np.array_equal(e_in.cpu().numpy(), before[0])
    assert np.array_equal(h_in.cpu().numpy(), before[1])
    return e_out.cpu().numpy(), int(status.item())


def random_case(rng, dim, N):
    edges = np.stack([np.concatenate([[0.0], np.sort(rng.uniform(0, 1, N - 1)), [1.0]]) for _ in range(dim)])
    hist = rng.uniform(0, 1, (dim, N)) ** 4
    return edges, hist


@gpu
def test_static_refine_equals_the_workspace_path_on_calls_in_a_row(V):
    rng = np.random.default_rng(20101)
    # call 1: the shape of configs[0] (d = 4, 50 bins), one dimension with nothing to adapt to
    E1, h1 = random_case(rng, 4, 50)
    h1[2] = 0.0
    want1 = existing_path(V, 4, 50, E1, h1, 1.5)
    got1, st1 = static_path(V, 4, 50, E1, h1, 1.5)
    assert st1 == 0 and want1 is not None
    assert np.max(np.abs(got1 - want1)) <= EDGE_TOL
    assert np.array_equal(got1[2], E1[2])
    # call 2, straight after it on the same array: the shape of configs[3] (d = 20, 100 bins) -- more cells than call 1
    # wrote, and the first call's leftovers underneath
    E2, h2 = random_case(rng, 20, 100)
    want2 = existing_path(V, 20, 100, E2, h2, 1.5)
    got2, st2 = static_path(V, 20, 100, E2, h2, 1.5)
    assert st2 == 0 and np.max(np.abs(got2 - want2)) <= EDGE_TOL
    assert np.all(np.diff(got2, axis=1) > 0) and np.all(got2[:, 0] == 0.0) and np.all(got2[:, -1] == 1.0)
    # call 3: a refinement that is rejected (the existing path: VEGAS_EGRID, grid unchanged) -> status 1, edges handed back
    E3 = np.stack([EG_EDGES, np.linspace(0, 1, EG_N + 1)])
    h3 = np.stack([EG_HIST, np.arange(1.0, EG_N + 1)])
    assert existing_path(V, 2, EG_N, E3, h3, 1.5) is None
    got3, st3 = static_path(V, 2, EG_N, E3, h3, 1.5)
    assert st3 == 1 and np.array_equal(got3, E3)
    # call 4: the rejection must not stick (the outcome flags are part of what the array keeps between calls), smaller
    # shape than before, another alpha, written in place over the input edges
    E4, h4 = random_case(rng, 3, 50)
    want4 = existing_path(V, 3, 50, E4, h4, 0.7)
    got4, st4 = static_path(V, 3, 50, E4, h4, 0.7, in_place=True)
    assert st4 == 0 and np.max(np.abs(got4 - want4)) <= EDGE_TOL
    # call 5: call 1 again gives call 1's answer again, bit for bit
    got5, st5 = static_path(V, 4, 50, E1, h1, 1.5)
    assert st5 == 0 and np.array_equal(got5, got1)


@gpu
def test_static_refine_follows_an_iteration_like_vegas_refine(V):
    """Histogram from a real iteration (configs[0] at its stated size), then both refinements from the same grid."""
    w = W.cfg1()
    g = V.from_workload(w)
    E0 = g.get_grid()
    _, _, hist = g.iterate(w.n_events, 0, w.seed)
    got, st = static_path(V, w.dim, w.nbins, E0, hist, w.alpha)
    g.refine(w.alpha)
    assert st == 0 and np.max(np.abs(got - g.get_grid())) <= EDGE_TOL
    # second iteration through the refined grid, second call in a row
    E1 = g.get_grid()
    _, _, hist = g.iterate(w.n_events, 0, w.seed)
    got, st = static_path(V, w.dim, w.nbins, E1, hist, w.alpha)
    g.refine(w.alpha)
    assert st == 0 and np.max(np.abs(got - g.get_grid())) <= EDGE_TOL


@gpu
def test_static_refine_at_the_capacity_limit(V):
    """dim * (nbins + 1) = 8192 exactly (32 x 255 bins): the largest grid the array holds."""
    rng = np.random.default_rng(7)
    E, h = random_case(rng, 32, 255)
    want = existing_path(V, 32, 255, E, h, 1.5)
    got, st = static_path(V, 32, 255, E, h, 1.5)
    assert want is not None and st == 0 and np.max(np.abs(got - want)) <= EDGE_TOL
