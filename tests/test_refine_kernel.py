"""S7 on the GPU, fed hand-made histograms through the test hook vegas_set_histogram: the independent pins of the
refinement (tests/test_oracle_math.py: closed-form / mpmath expectations, the equal-damped-mass property) run through
refine_kernel itself, not only through histograms an iteration produced; plus the rejection path (step 7:
VEGAS_EGRID, grid and histogram unchanged) on both sides.
"""
import mpmath as mp
import numpy as np
import pytest

from paper_2010_09341_b200 import workloads as W

# a histogram row and an edge row that make step 7 fail: three equal-weight bins after smoothing, the middle one
# one ulp wide, so two of the seven new edges land on the same double (0.5)
EG_N = 8
EG_EDGES = np.array([0.0, 0.2, 0.4, 0.5, 0.5 + 2.0 ** -53, 0.7, 0.8, 0.9, 1.0])
EG_HIST = np.array([0.0, 0.0, 0.0, 1.0, 0.0, 0.0, 0.0, 0.0])


def oracle_with(N, hist, edges=None, dim=1):
    from oracle import oracle as O
    o = O.Oracle(dim, N, W.TOY_SUM)
    if edges is not None:
        o.set_grid(np.array(edges, dtype=np.float64).reshape(dim, N + 1))
    o.commit(10, 1.0, 1.0, np.array(hist, dtype=np.float64).reshape(dim, N))
    return o


def test_oracle_rejects_non_monotone_refinement_and_keeps_its_state():
    """The ORACLE_EGRID branch: grid bit-unchanged, histogram kept, a second refine gives the same answer, and a
    refinement that can succeed (alpha = 0 on the same histogram: all weights 1) then goes through."""
    from oracle import oracle as O
    o = oracle_with(EG_N, EG_HIST, EG_EDGES)
    for _ in range(2):
        with pytest.raises(O.OracleError) as ei:
            o.refine(1.5)
        assert ei.value.code == O.EGRID
        assert np.array_equal(o.get_grid()[0], EG_EDGES)
    # by hand: s = {0,0,1/3,1/3,1/3,0,0,0}, three equal weights m, delta = 3m/8, edges 3 and 4 both in the one-ulp bin
    # [0.5, 0.5 + 2^-53] at fractions 1/8 and 1/2 -> both round to 0.5
    o2 = oracle_with(EG_N, EG_HIST, np.linspace(0, 1, EG_N + 1))
    o2.refine(1.5)                                      # same histogram on a uniform grid is fine
    E = o2.get_grid()[0]
    assert np.all(np.diff(E) > 0) and abs(E[3] - (0.375 + 0.125 * 0.125)) < 1e-15 and abs(E[4] - (0.375 + 0.5 * 0.125)) < 1e-15


# ---------------------------------------------------------------------------------------------- GPU
gpu = pytest.mark.gpu


@pytest.fixture(scope="module")
def V():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2010_09341_b200 import vegas
    return vegas


def gpu_refine(V, N, hist, alpha, edges=None, dim=1, precision=W.FP64):
    g = V.Vegas(dim, N, W.TOY_SUM, (), precision)
    if edges is not None:
        g.set_grid(np.array(edges, dtype=np.float64).reshape(dim, N + 1))
    g.set_histogram(np.array(hist, dtype=np.float64).reshape(dim, N))
    g.refine(alpha)
    return g.get_grid()


@gpu
def test_gpu_refine_flat_histogram_keeps_uniform_grid(V):
    for N in (4, 50, 100, 511):
        E = gpu_refine(V, N, [1.0] * N, 1.5)[0]
        assert np.allclose(E, np.arange(N + 1) / N, rtol=0, atol=N * 3e-16)


@gpu
def test_gpu_refine_alpha_zero_is_identity_map_on_nonuniform_edges(V):
    E0 = np.array([0, 0.1, 0.15, 0.5, 1.0])
    E = gpu_refine(V, 4, [3.0, 1.0, 0.5, 9.0], 0.0, E0)[0]
    assert np.allclose(E, E0, rtol=0, atol=1e-15)


@gpu
def test_gpu_refine_hand_case_with_zero_weight_bins(V):
    """N=4, H={0,0,1,1}, alpha=1 against an mpmath evaluation of S7 (bin 0 has m = 0 and is skipped, reading R11)."""
    mp.mp.dps = 40
    r = [mp.mpf(0), mp.mpf(1) / 6, mp.mpf(1) / 3, mp.mpf(1) / 2]
    m = [mp.mpf(0)] + [(1 - ri) / mp.log(1 / ri) for ri in r[1:]]
    c = [mp.mpf(0)]
    for mi in m:
        c.append(c[-1] + mi)
    delta = c[-1] / 4
    want = [0.0]
    for j in (1, 2, 3):
        t = j * delta
        i = next(i for i in range(4) if c[i + 1] >= t and m[i] > 0)
        want.append(float(mp.mpf(i) / 4 + (t - c[i]) / m[i] * mp.mpf(1) / 4))
    want.append(1.0)
    E = gpu_refine(V, 4, [0.0, 0.0, 1.0, 1.0], 1.0)[0]
    assert np.allclose(E, want, rtol=0, atol=1e-15)
    assert E[1] > 0.25
    # {1,1,1,1}: unchanged
    assert np.allclose(gpu_refine(V, 4, [1.0] * 4, 1.0)[0], np.arange(5) / 4, rtol=0, atol=1e-15)


@gpu
def test_gpu_refine_tie_takes_the_lower_bin(V):
    """Reading R12: t = c_{i+1} exactly takes bin i, i.e. the new edge is E[i+1] itself.  N=4, alpha=0 (all m = 1):
    t_j = j lands exactly on c_j."""
    E0 = np.array([0, 0.125, 0.25, 0.625, 1.0])
    E = gpu_refine(V, 4, [1.0, 2.0, 3.0, 4.0], 0.0, E0)[0]
    assert np.array_equal(E, E0)


@gpu
def test_gpu_refine_equalises_damped_weight(V):
    """The defining property of the rebinning with random edges and a random histogram (50 and 300 bins; several
    dimensions at once, one of them with an all-zero histogram that must stay as it is)."""
    rng = np.random.default_rng(3)
    for N in (50, 300):
        d = 3
        E0 = np.stack([np.concatenate([[0.0], np.sort(rng.uniform(0, 1, N - 1)), [1.0]]) for _ in range(d)])
        h = rng.uniform(0, 1, (d, N)) ** 4
        h[1] = 0.0
        alpha = 1.5
        E = gpu_refine(V, N, h, alpha, E0, dim=d)
        assert np.array_equal(E[1], E0[1])              # nothing to adapt to: dimension unchanged
        for k in (0, 2):
            s = np.empty(N)
            s[0] = (h[k, 0] + h[k, 1]) / 2; s[-1] = (h[k, -2] + h[k, -1]) / 2
            s[1:-1] = (h[k, :-2] + h[k, 1:-1] + h[k, 2:]) / 3
            r = s / s.sum()
            m = ((1 - r) / np.log(1 / r)) ** alpha
            cum = np.concatenate([[0], np.cumsum(m)])
            mass = np.diff(np.interp(E[k], E0[k], cum))
            assert np.allclose(mass, cum[-1] / N, rtol=1e-10)
            assert np.all(np.diff(E[k]) > 0)
        # and the oracle agrees to 1e-12 on the same inputs
        o = oracle_with(N, h, E0, dim=d)
        o.refine(alpha)
        assert np.max(np.abs(E - o.get_grid())) <= 1e-12


@gpu
def test_gpu_refine_rejection_leaves_grid_and_histogram_and_agrees_with_the_oracle(V):
    """Step 7 fails (two new edges collide inside a one-ulp bin) in one of two dimensions: VEGAS_EGRID, the whole grid
    bit-unchanged (all-or-nothing), the same answer from a second refine, the histogram still there -- on both sides."""
    from oracle import oracle as O
    N, d = EG_N, 2
    E0 = np.stack([EG_EDGES, np.linspace(0, 1, N + 1)])
    h = np.stack([EG_HIST, np.arange(1.0, N + 1)])
    o = oracle_with(N, h, E0, dim=d)
    g = V.Vegas(d, N, W.TOY_SUM, ())
    g.set_grid(E0)
    g.set_histogram(h)
    for _ in range(2):
        with pytest.raises(O.OracleError) as eo:
            o.refine(1.5)
        with pytest.raises(V.VegasError) as eg:
            g.refine(1.5)
        assert eo.value.code == O.EGRID and eg.value.code == V.EGRID
        assert np.array_equal(g.get_grid(), E0) and np.array_equal(o.get_grid(), E0)
    # the histogram survived the rejections: alpha = 0 (all weights 1 where the smoothed histogram is positive) succeeds
    # on the second dimension's account and still fails on the first -> still EGRID; replace the first row and it works
    h2 = h.copy(); h2[0] = 1.0
    g.set_histogram(h2); o.commit(10, 1.0, 1.0, h2)
    g.refine(1.5); o.refine(1.5)
    assert np.max(np.abs(g.get_grid() - o.get_grid())) <= 1e-12
    with pytest.raises(V.VegasError) as eg:
        g.refine(1.5)                                   # consumed by the successful refinement
    assert eg.value.code == V.ESTATE


@gpu
def test_gpu_async_rejection_is_reported_and_gives_the_histogram_back(V):
    g = V.Vegas(1, EG_N, W.TOY_SUM, ())
    g.set_grid(EG_EDGES[None, :])
    g.set_histogram(EG_HIST[None, :])
    g.refine_enqueue(1.5)
    with pytest.raises(V.VegasError) as eg:
        g.refine_collect()
    assert eg.value.code == V.EGRID
    assert np.array_equal(g.get_grid()[0], EG_EDGES)
    g.refine_enqueue(0.0)                               # the histogram is still there; this one is rejected as well
    with pytest.raises(V.VegasError) as eg:
        g.refine(0.0)                                   # ... and a blocking refine reports the pending rejection
    assert eg.value.code in (V.EGRID, V.ESTATE)
    g.refine_collect()
