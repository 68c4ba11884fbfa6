"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element, on the same
seeded inputs.  Tolerances are those of BASELINE.json north_star: bins / pass / mapped point bit-exact,
I and sigma rel 1e-12, histogram rel 1e-10 per cell (zero cells zero on both sides), refined edges abs
1e-12 after 5 iterations.  Per-event integrand values: bit-exact where the arithmetic is fully specified
(fp32 genz_osc_peak, toy_sum), a few ulp where a libm exp() is involved (glibc vs CUDA).
"""
import os

import numpy as np
import pytest

from paper_2010_09341_b200 import workloads as W

pytestmark = pytest.mark.gpu

THREADS = max(1, min(32, len(os.sched_getaffinity(0))))
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def V():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2010_09341_b200 import vegas
    return vegas


@pytest.fixture(scope="module")
def O():
    from oracle import oracle
    return oracle


def small_workloads():
    return {
        "cfg1": W.cfg1(), "cfg2": W.cfg2(), "cfg4": W.cfg4(), "cfg5": W.cfg5(), "toy": W.toy(),
        # run-time-dimension instances
        "gauss_sym_d2": W.Workload("gs2", 2, 37, W.GAUSS_SYM, (0.1, 0.5), W.FP64, 10**5, 3),
        "gauss_double_d5": W.Workload("gd5", 5, 64, W.GAUSS_DOUBLE, (0.1, 1 / 3, 2 / 3), W.FP64, 10**5, 3),
        "genz_d7": W.cfg4(dim=7),
        "toy_d32": W.Workload("toy32", 32, 50, W.TOY_SUM, (), W.FP64, 10**5, 3),
        "toy_f32_d9": W.Workload("toyf9", 9, 100, W.TOY_SUM, (), W.FP32_EVAL, 10**5, 3),
        # 32-bit-uniform stream mode (extra; reading R3): tuned and generic instances
        "cfg5_tab": W.cfg5_tab(),                        # NEXT-4: tabulated PDF
        "cfg2_u32": W.cfg2_u32(),
        "lo_u32": W.Workload("lo_u32", 3, 50, W.LO_2TO2, (13000.0, 50.0, 0.9, 1.1, 5.0), W.FP64_U32, 10**5, 3),
        "gauss_sym_d5_u32": W.Workload("gs5u", 5, 33, W.GAUSS_SYM, (0.1, 0.5), W.FP64_U32, 10**5, 3),
        "toy_d7_u32": W.Workload("toy7u", 7, 50, W.TOY_SUM, (), W.FP64_U32, 10**5, 3),
    }


F_RTOL = {W.GAUSS_SYM: 2e-15, W.GAUSS_DOUBLE: 2e-15, W.GENZ_OSC_PEAK: 0.0, W.LO_2TO2: 2e-14, W.TOY_SUM: 0.0,
          W.LO_2TO2_TAB: 2e-14}


def make_pair(V, O, w):
    g, o = V.from_workload(w), O.Oracle(w.dim, w.nbins, w.integrand_id, w.params, w.precision)
    if w.integrand_id == W.LO_2TO2_TAB:                 # the tabulated PDF is input data for both sides
        g.set_table(W.pdf_table()); o.set_table(W.pdf_table())
    return g, o


def assert_events_equal(g, o, w):
    np.testing.assert_array_equal(g["bins"], o["bins"])
    np.testing.assert_array_equal(g["passed"], o["passed"])
    np.testing.assert_array_equal(g["x"], o["x"])            # bit-exact mapped point (S2)
    np.testing.assert_array_equal(g["jac"], o["jac"])
    rt = F_RTOL[w.integrand_id]
    if rt == 0.0:
        np.testing.assert_array_equal(g["f"], o["f"])
        np.testing.assert_array_equal(g["wf"], o["wf"])
    else:
        np.testing.assert_allclose(g["f"], o["f"], rtol=rt, atol=0.0)
        np.testing.assert_allclose(g["wf"], o["wf"], rtol=rt, atol=0.0)


def assert_iteration_close(gres, ores):
    gI, gs, gh = gres
    oI, os_, oh = ores
    assert abs(gI - oI) <= 1e-12 * abs(oI), (gI, oI)
    assert abs(gs - os_) <= 1e-12 * abs(os_), (gs, os_)
    assert np.array_equal(gh == 0.0, oh == 0.0)
    np.testing.assert_allclose(gh, oh, rtol=1e-10, atol=0.0)


# ---------------------------------------------------------------------------------------------------
# per-event parity (S1-S4)
# ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("name", list(small_workloads()))
def test_events_uniform_grid(V, O, name):
    w = small_workloads()[name]
    g, o = make_pair(V, O, w)
    for first, count in [(0, 5000), (99_990_000, 777), (2**32 - 300, 300), (2**32, 129), (2**40 + 12345, 64)]:
        assert_events_equal(g.debug_events(first, count, seed=w.seed), o.events(first, count, w.seed), w)
    # another seed and iteration counter
    g.set_iteration(7); o.set_iteration(7)
    assert_events_equal(g.debug_events(1000, 2000, seed=0xDEADBEEF12345678), o.events(1000, 2000, 0xDEADBEEF12345678), w)


@pytest.mark.parametrize("name", ["cfg1", "cfg2", "cfg4", "cfg5", "gauss_double_d5", "cfg2_u32"])
def test_events_adapted_grid(V, O, name):
    """Cascade-free: load the oracle's refined grid into the library, then compare events."""
    w = small_workloads()[name]
    g, o = make_pair(V, O, w)
    for _ in range(2):
        o.iterate(200_000, w.seed, threads=THREADS)
        o.refine(w.alpha)
    g.set_grid(o.get_grid())
    g.set_iteration(o.iteration)
    np.testing.assert_array_equal(g.get_grid(), o.get_grid())
    assert_events_equal(g.debug_events(0, 20_000, seed=w.seed), o.events(0, 20_000, w.seed), w)
    if w.integrand_id not in (W.TOY_SUM,):
        assert np.any(o.events(0, 100, w.seed)["jac"] != 1.0)


@pytest.mark.parametrize("alpha", [0.3, 0.05, 0.02])
def test_events_exp_ranges(V, O, alpha):
    """The kernels' own exp (exp_f64: |argument| < 700) and the library routine it hands over to beyond that, against
    the oracle's libm: narrow Gaussians drive the arguments of exp from 0 down past -708 (subnormal results) to total
    underflow.  Normal results agree to 2e-15 relative, subnormal ones to one unit of the subnormal grid."""
    for wl in (W.Workload("gs_exp", 4, 50, W.GAUSS_SYM, (alpha, 0.5), W.FP64, 10**5, 1),
               W.Workload("gd_exp", 8, 50, W.GAUSS_DOUBLE, (alpha, 1 / 3, 2 / 3), W.FP64, 10**5, 1)):
        g, o = make_pair(V, O, wl)
        eg, eo = g.debug_events(0, 50_000, seed=3), o.events(0, 50_000, 3)
        np.testing.assert_array_equal(eg["x"], eo["x"])
        fg, fo = eg["f"], eo["f"]
        normal = fo >= 1e-290
        np.testing.assert_allclose(fg[normal], fo[normal], rtol=2e-15, atol=0.0)
        np.testing.assert_allclose(fg[~normal], fo[~normal], rtol=0.0, atol=1e-290 * 2e-15)
        if alpha == 0.02:
            assert np.any(fo == 0.0) and np.any(normal)     # both regimes are present
        n = 200_003
        assert_iteration_close(g.iterate(n, 0, 3), o.iterate(n, 3, threads=THREADS))


def test_exp_f64_against_mpmath(V):
    """The kernels' exp against 50-digit arithmetic (not against another libm): a one-dimensional Gaussian,
    f = fl(C exp(t)) with t = -fl(fl((x - mu)^2) / alpha^2 ...) rebuilt here operation by operation from the mapped
    point the library reports, so that the only unknown is exp itself.  Arguments from 0 down to -625."""
    import mpmath
    mpmath.mp.prec = 200
    for alpha in (0.1, 0.02):
        g = V.Vegas(1, 50, W.GAUSS_SYM, (alpha, 0.5), W.FP64)
        ev = g.debug_events(0, 4000, seed=11)
        x, f = ev["x"][:, 0], ev["f"]
        b = np.float64(alpha) * np.sqrt(np.float64(np.pi))
        Cc = np.float64(1.0) / b                                  # C = (alpha sqrt(pi))^-1: one division for d = 1
        a2 = np.float64(1.0) / (np.float64(alpha) * np.float64(alpha))
        dx = x - np.float64(0.5)
        s = dx * dx                                               # fma(dx, dx, 0) = fl(dx^2)
        t = -(s * a2)
        worst = 0.0
        for ti, fi in zip(t, f):
            if ti <= -700.0:
                continue
            e = mpmath.exp(mpmath.mpf(float(ti)))
            want = mpmath.mpf(float(Cc)) * e
            ulp = abs(float(want)) * 2.0 ** -52
            worst = max(worst, float(abs(mpmath.mpf(float(fi)) - want)) / ulp)
        assert worst <= 1.5, worst                                # measured 0.90: exp within ~1 ulp + the rounding of the product
        g.close()


# ---------------------------------------------------------------------------------------------------
# one iteration (S1-S6): several tiles + a ragged tail, several launch splits
# ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("name", list(small_workloads()))
def test_iteration_parity(V, O, name):
    w = small_workloads()[name]
    g, o = make_pair(V, O, w)
    n = 1_000_003
    ores = o.iterate(n, w.seed, threads=THREADS)
    for epl in (0, 65_537, 300_000):
        g.reset()
        gres = g.iterate(n, epl, w.seed)
        assert_iteration_close(gres, ores)
        S1, S2, _ = g.last_sums()
        oS1, oS2 = o.last_sums()
        assert abs(S1 - oS1) <= 1e-12 * abs(oS1) and abs(S2 - oS2) <= 1e-12 * abs(oS2)
        # invariant P4: every dimension's histogram sums to S2
        np.testing.assert_allclose(gres[2].sum(axis=1), S2, rtol=1e-12)
    if o.npass is not None:
        assert g.last_npass() == o.npass


def test_iteration_launch_shapes(V, O):
    """Results do not depend on the launch shape or replica count beyond summation order."""
    w = W.cfg2()
    g, o = make_pair(V, O, w)
    n = 500_009
    ores = o.iterate(n, 3, threads=THREADS)
    for ctas, threads, reps in [(1, 1024, 32), (2, 512, 16), (4, 256, 8), (1, 128, 1), (8, 64, 2)]:
        g.reset()
        g.set_launch_shape(ctas, threads)
        g.set_hist_replicas(reps)
        assert g.launch_shape()["hist_replicas"] == reps
        assert_iteration_close(g.iterate(n, 0, 3), ores)


@pytest.mark.parametrize("graph", [True, False])
def test_batch_size_independence(V, O, graph):
    """Reading R16: the event index is global, so events_per_launch changes nothing but summation order.  Every batch
    size is compared with the oracle (200 / 20 / 2 / 1 launches: the 1/4- and 1/2-of-the-SMs geometries, with and without
    the CUDA-graph replay of many-launch iterations) and with the first run."""
    w = W.cfg2()
    g, o = make_pair(V, O, w)
    g.use_cuda_graph(graph)
    n = 2 * 10**6
    ores = o.iterate(n, 0, threads=THREADS)
    ref = None
    for epl in (10**4, 10**5, 10**6, 2 * 10**6):
        g.reset()
        I, s, h = g.iterate(n, epl, 0)
        assert_iteration_close((I, s, h), ores)
        if ref is None:
            ref = (I, s, h)
        assert abs(I - ref[0]) <= 1e-13 * abs(ref[0]) and abs(s - ref[1]) <= 1e-13 * abs(ref[1])
        np.testing.assert_allclose(h, ref[2], rtol=1e-12)
    # a second replay of the cached graph runs the next iteration counter, not the captured one
    g.reset(); o.reset()
    for it in range(2):
        ores = o.iterate(n, 0, threads=THREADS)
        assert_iteration_close(g.iterate(n, 10**4, 0), ores)
        assert g.iteration == o.iteration == it + 1


# ---------------------------------------------------------------------------------------------------
# iterate + refine cascades (S7)
# ---------------------------------------------------------------------------------------------------
def run_cascade(g, o, w, n, n_iter, epl=0):
    for it in range(n_iter):
        ores = o.iterate(n, w.seed, threads=THREADS)
        gres = g.iterate(n, epl, w.seed)
        assert_iteration_close(gres, ores)
        o.refine(w.alpha)
        g.refine(w.alpha)
        ge, oe = g.get_grid(), o.get_grid()
        assert np.all(np.diff(ge, axis=1) > 0) and np.all(ge[:, 0] == 0) and np.all(ge[:, -1] == 1)
        assert np.max(np.abs(ge - oe)) <= 1e-12, (it, np.max(np.abs(ge - oe)))
    assert g.iteration == o.iteration == n_iter


def test_cfg1_full_five_iterations(V, O):
    """BASELINE.json configs[0] at full size: 1e5 events x 5 iterations, alpha = 1.5, seed 0."""
    w = W.cfg1()
    g, o = make_pair(V, O, w)
    run_cascade(g, o, w, w.n_events, w.n_iter)


@pytest.mark.parametrize("name", ["cfg2", "cfg4", "cfg5", "toy", "gauss_sym_d2", "toy_f32_d9", "cfg2_u32", "lo_u32", "cfg5_tab"])
def test_cascade_reduced(V, O, name):
    w = small_workloads()[name]
    g, o = make_pair(V, O, w)
    run_cascade(g, o, w, 400_000, 5, epl=w.events_per_launch)


def test_refine_alpha_zero_and_flat(V, O):
    w = W.Workload("toy3", 3, 16, W.TOY_SUM, (), W.FP64, 10**5, 1)
    g, o = make_pair(V, O, w)
    o.iterate(50_000, 1); g.iterate(50_000, 0, 1)
    o.refine(0.0); g.refine(0.0)
    assert np.max(np.abs(g.get_grid() - o.get_grid())) <= 1e-15
    # alpha = 0: all damped weights are 1 -> the grid stays uniform
    assert np.max(np.abs(g.get_grid() - np.linspace(0, 1, 17)[None, :])) <= 1e-15


def test_all_events_cut_away(V, O):
    """Degenerate: cos_cut = 0 rejects every event: I = sigma = 0, H = 0, refine leaves the grid unchanged."""
    w = W.Workload("lo_cut", 3, 50, W.LO_2TO2, (13000.0, 50.0, 0.0, 1.1, 5.0), W.FP64, 10**5, 1)
    g, o = make_pair(V, O, w)
    I, s, h = g.iterate(100_000, 0, 0)
    oI, os_, oh = o.iterate(100_000, 0)
    assert I == oI == 0.0 and s == os_ == 0.0 and not h.any() and not oh.any()
    assert g.last_npass() == 0
    before = g.get_grid()
    g.refine(1.5); o.refine(1.5)
    np.testing.assert_array_equal(g.get_grid(), before)
    np.testing.assert_array_equal(o.get_grid(), before)


def test_extreme_sizes(V, O):
    """Minimum n, one event per launch, maximum bin counts (fp64 4095, fp32 511), dim 32."""
    w = W.Workload("toy1", 1, 4095, W.TOY_SUM, (), W.FP64, 10**5, 1)
    g, o = make_pair(V, O, w)
    assert_iteration_close(g.iterate(300_001, 0, 5), o.iterate(300_001, 5, threads=THREADS))
    g.refine(1.5); o.refine(1.5)
    assert np.max(np.abs(g.get_grid() - o.get_grid())) <= 1e-12
    g.set_grid(o.get_grid())          # cascade-free: refined edges agree to 1e-12, not bit for bit (libm pow/log)
    assert_events_equal(g.debug_events(0, 3000, 5), o.events(0, 3000, 5), w)

    w = W.Workload("toyf", 2, 511, W.TOY_SUM, (), W.FP32_EVAL, 10**5, 1)
    g, o = make_pair(V, O, w)
    assert_iteration_close(g.iterate(200_001, 0, 5), o.iterate(200_001, 5, threads=THREADS))
    g.refine(1.5); o.refine(1.5)
    assert np.max(np.abs(g.get_grid() - o.get_grid())) <= 1e-12
    g.set_grid(o.get_grid())          # cascade-free: refined edges agree to 1e-12, not bit for bit (libm pow/log)
    assert_events_equal(g.debug_events(0, 3000, 5), o.events(0, 3000, 5), w)

    w = W.cfg1()
    g, o = make_pair(V, O, w)
    assert_iteration_close(g.iterate(2, 0, 0), o.iterate(2, 0))
    g.reset(); o.reset()
    assert_iteration_close(g.iterate(64, 1, 0), o.iterate(64, 0))         # 64 launches of one event


# ---------------------------------------------------------------------------------------------------
# API state machine and error behaviour (include/vegas_b200.h)
# ---------------------------------------------------------------------------------------------------
def test_api_state_and_errors(V):
    w = W.cfg1()
    g = V.from_workload(w)
    with pytest.raises(V.VegasError) as ei:
        g.refine(1.5)                                   # no histogram yet
    assert ei.value.code == V.ESTATE
    with pytest.raises(V.VegasError) as ei:
        g.last_sums()
    assert ei.value.code == V.ESTATE
    with pytest.raises(V.VegasError) as ei:
        g.iterate(1)
    assert ei.value.code == V.EINVAL
    g.iterate(10_000)
    assert g.iteration == 1
    with pytest.raises(V.VegasError) as ei:
        g.refine(-1.0)
    assert ei.value.code == V.EINVAL
    with pytest.raises(V.VegasError) as ei:
        g.refine(float("nan"))
    assert ei.value.code == V.EINVAL
    g.refine(1.5)
    with pytest.raises(V.VegasError) as ei:
        g.refine(1.5)                                   # histogram was consumed
    assert ei.value.code == V.ESTATE
    e = g.get_grid()
    g.set_grid(e)
    np.testing.assert_array_equal(g.get_grid(), e)      # identity (P4)
    bad = e.copy(); bad[1, 10] = bad[1, 11]
    with pytest.raises(V.VegasError) as ei:
        g.set_grid(bad)
    assert ei.value.code == V.EGRID
    np.testing.assert_array_equal(g.get_grid(), e)      # unchanged
    bad = e.copy(); bad[0, -1] = 0.999
    with pytest.raises(V.VegasError) as ei:
        g.set_grid(bad)
    assert ei.value.code == V.EGRID
    g.reset()
    assert g.iteration == 0
    u = g.get_grid()
    np.testing.assert_array_equal(u[0], np.array([i / 50 for i in range(50)] + [1.0]))
    with pytest.raises(V.VegasError) as ei:
        g.set_launch_shape(1, 100)
    assert ei.value.code == V.EINVAL
    info = g.device_info()
    assert info["sm_count"] >= 100


def test_uniform_grid_jacobian_is_one(V):
    """P4 / reading R6: on the uniform grid J == 1 exactly for N = 50, 100."""
    for w in (W.cfg2(), W.cfg4()):
        g = V.from_workload(w)
        ev = g.debug_events(0, 10_000, 0)
        assert np.all(ev["jac"] == 1.0)
        assert ev["bins"].min() >= 0 and ev["bins"].max() < w.nbins
        assert np.all((ev["x"] >= 0) & (ev["x"] <= 1))


def test_estimates_within_4_sigma_of_closed_form(V, golden_dir):
    """P3 on the GPU path alone: adapted estimates land within 4 sigma of the exact integrals."""
    from conftest import read_golden
    exact = read_golden(os.path.join(golden_dir, "closed_forms.txt"))
    for name, key in [("cfg1", "cfg1"), ("cfg5", "cfg5"), ("toy", None)]:
        w = small_workloads()[name]
        target = float(exact[key][0]) if key else w.dim / 2.0
        g = V.from_workload(w)
        for _ in range(6):
            I, s, _ = g.iterate(10**6, 0, w.seed)
            g.refine(w.alpha)
        assert abs(I - target) <= 4 * s, (name, I, s)


# ---------------------------------------------------------------------------------------------------
# BASELINE.json full sizes, in the launch configuration bench.py times (one launch per iteration, the
# instance's default shape)
# ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("name", ["cfg2", "cfg4", "cfg5", "cfg2_u32", "cfg5_tab"])
def test_full_size_iteration_parity(V, O, name):
    """1e8 events: iteration 0 on the uniform grid and iteration 1 on the oracle's refined grid
    (cascade-free), I / sigma rel 1e-12, every histogram cell rel 1e-10, pass count exact, plus sampled events
    from the far end of the index range compared one by one."""
    w = small_workloads()[name]
    assert w.n_events == 10**8
    g, o = make_pair(V, O, w)
    for it in range(2):
        ores = o.iterate(w.n_events, w.seed, threads=THREADS)
        gres = g.iterate(w.n_events, 0, w.seed)
        assert g.launch_shape()["ctas_per_sm"] * g.launch_shape()["threads_per_cta"] >= 512
        assert_iteration_close(gres, ores)
        if o.npass is not None:
            assert g.last_npass() == o.npass
        S2 = g.last_sums()[1]
        np.testing.assert_allclose(gres[2].sum(axis=1), S2, rtol=1e-12)
        g.set_iteration(it)
        o.set_iteration(it)
        assert_events_equal(g.debug_events(w.n_events - 4096, 4096, seed=w.seed),
                            o.events(w.n_events - 4096, 4096, w.seed), w)
        g.set_iteration(it + 1)
        o.set_iteration(it + 1)
        o.refine(w.alpha)
        g.refine(w.alpha)
        assert np.max(np.abs(g.get_grid() - o.get_grid())) <= 1e-12
        g.set_grid(o.get_grid())


_CASCADE = {}


def oracle_cascade(O, name):
    """The oracle's own free-running full-size run of a configuration -- its n_iter iterations of 1e8 events, a refinement
    after each -- computed once per test session and shared by the tests that hold different GPU paths against it (the
    blocking calls, the un-synchronised fused steps bench.py times).  Rows: I, sigma, H, npass, the grid after the refine."""
    if name not in _CASCADE:
        w = small_workloads()[name]
        _, o = None, O.Oracle(w.dim, w.nbins, w.integrand_id, w.params, w.precision)
        rows = []
        for _ in range(w.n_iter):
            I, s, h = o.iterate(w.n_events, w.seed, threads=THREADS)
            npass = o.npass
            o.refine(w.alpha)
            rows.append(dict(I=I, s=s, h=h.copy(), npass=npass, grid=o.get_grid().copy()))
        _CASCADE[name] = rows
    return _CASCADE[name]


@pytest.mark.parametrize("name", ["cfg2", "cfg4", "cfg5"])
def test_full_size_cascade(V, O, name):
    """BASELINE.json acceptance at the stated sizes: the configuration's 10 free-running iterations of 1e8 events (the
    GPU grid is never re-seeded from the oracle), refine after each.  I, sigma rel 1e-12, every H cell rel 1e-10, the
    pass count exact in every iteration; refined edges within 1e-12 (absolute) of the oracle's after every refinement:
    the fifth, which the acceptance names, and all the way to the tenth."""
    w = small_workloads()[name]
    assert w.n_events == 10**8 and w.n_iter == 10
    rows = oracle_cascade(O, name)
    g = V.from_workload(w)
    for it in range(w.n_iter):
        r = rows[it]
        gres = g.iterate(w.n_events, 0, w.seed)
        assert_iteration_close(gres, (r["I"], r["s"], r["h"]))
        if r["npass"] is not None:
            assert g.last_npass() == r["npass"]
        g.refine(w.alpha)
        ge, oe = g.get_grid(), r["grid"]
        assert np.all(np.diff(ge, axis=1) > 0) and np.all(ge[:, 0] == 0) and np.all(ge[:, -1] == 1)
        assert np.max(np.abs(ge - oe)) <= 1e-12, (it, np.max(np.abs(ge - oe)))
    assert g.iteration == w.n_iter


BENCH_PATH_STEPS = 5


def bench_path(V, w, steps=BENCH_PATH_STEPS):
    """Exactly the sequence bench.py times: reset, then `steps` fused steps of the full size enqueued back to back with NO
    collect or synchronisation in between (every kernel carries the programmatic-dependent-launch attribute, so step i+1's
    prologue runs under step i's S6/S7 tail), and only then the read-back."""
    g = V.from_workload(w)
    g.reset()
    launches = [g.step_enqueue(w.n_events, w.n_events, w.seed, w.alpha) for _ in range(steps)]
    g.refine_collect()                                   # raises if a refinement was rejected
    I, s, _ = g.iterate_collect(want_hist=False)
    return dict(I=I, s=s, grid=g.get_grid(), npass=g.last_npass(), launches=launches, iteration=g.iteration)


def assert_bench_path(res, rows, w, steps=BENCH_PATH_STEPS):
    last = rows[steps - 1]                               # a right grid after five steps implies right earlier steps
    assert res["launches"] == [1] * steps and res["iteration"] == steps
    assert abs(res["I"] - last["I"]) <= 1e-12 * abs(last["I"]), (res["I"], last["I"])
    assert abs(res["s"] - last["s"]) <= 1e-12 * abs(last["s"]), (res["s"], last["s"])
    if last["npass"] is not None:
        assert res["npass"] == last["npass"]
    assert np.max(np.abs(res["grid"] - last["grid"])) <= 1e-12, np.max(np.abs(res["grid"] - last["grid"]))


@pytest.mark.parametrize("name", ["cfg2", "cfg4", "cfg5"])
def test_bench_path_parity(V, O, name):
    """The path bench.py's device-timed region runs (un-synchronised chain of fused steps, 1e8 events each, one launch
    per step, programmatic dependent launch live) against five free-running oracle steps at the stated tolerances:
    I, sigma of the fifth step rel 1e-12, pass count exact, the grid after the fifth refinement within 1e-12."""
    w = small_workloads()[name]
    assert w.n_events == 10**8
    assert_bench_path(bench_path(V, w), oracle_cascade(O, name), w)


@pytest.mark.parametrize("name", ["cfg2", "cfg4", "cfg5"])
def test_bench_path_parity_without_pdl(V, O, name):
    """The same chain with VEGAS_NO_PDL=1 (plain stream order between the steps' kernels; the switch is read when the
    library is loaded, hence the subprocess): same numbers against the oracle."""
    import json
    import subprocess
    import sys
    w = small_workloads()[name]
    code = ("import json, sys; sys.path[:0] = [%r, %r]\n"
            "from test_gpu_parity import bench_path, small_workloads\n"
            "from paper_2010_09341_b200 import vegas as V\n"
            "r = bench_path(V, small_workloads()[%r]); r['grid'] = r['grid'].tolist()\n"
            "print('RESULT ' + json.dumps(r))\n") % (ROOT, os.path.join(ROOT, "tests"), name)
    out = subprocess.run([sys.executable, "-c", code], cwd=ROOT, env=dict(os.environ, VEGAS_NO_PDL="1"),
                         capture_output=True, text=True, timeout=600)
    assert out.returncode == 0, out.stderr[-3000:]
    res = json.loads([ln for ln in out.stdout.splitlines() if ln.startswith("RESULT ")][-1][7:])
    res["grid"] = np.array(res["grid"])
    assert_bench_path(res, oracle_cascade(O, name), w)


@pytest.mark.parametrize("epl", [0, 300_000])
def test_shard_across_2pow32(V, O, epl):
    """The global event index is 64 bits wide (S1: counter words 0 and 1) and a launch never straddles a multiple of 2^32
    (its kernels keep the high word uniform): a shard [2^32 - 5e5, 2^32 + 5e5) of an iteration of 2^32 + 1e6 events, as one
    requested launch (cut in two at 2^32) and as launches of 3e5 (cut at 2^32 as well), against the oracle's range call:
    S1, S2, the pass count and every histogram cell."""
    w = W.cfg2()
    n_total, first, count = 2**32 + 10**6, 2**32 - 5 * 10**5, 10**6
    g = V.from_workload(w)
    o = O.Oracle(w.dim, w.nbins, w.integrand_id, w.params, w.precision)
    sums, hs, hc, npass = o.iterate_range(first, count, w.seed)
    launches = g.iterate_shard_enqueue(n_total, first, count, epl or count, w.seed)
    assert launches == (2 if not epl else 4)             # 5e5 | 5e5   and   3e5, 2e5 | 3e5, 2e5
    p = g.partials_tensor().cpu().numpy()
    import math
    S1, S2, oS1, oS2 = math.fsum(p[0:2]), math.fsum(p[2:4]), math.fsum(sums[0:2]), math.fsum(sums[2:4])
    assert abs(S1 - oS1) <= 1e-12 * abs(oS1) and abs(S2 - oS2) <= 1e-12 * abs(oS2)
    assert int(p[4]) == npass == count
    gh, oh = p[8:].reshape(w.dim, w.nbins), hs + hc
    assert np.array_equal(gh == 0.0, oh == 0.0)
    np.testing.assert_allclose(gh, oh, rtol=1e-10, atol=0.0)
    g.finalize_enqueue(n_total)
    I, s, _ = g.iterate_collect()
    oI, os_ = o.commit(n_total, oS1, oS2, oh.copy())
    assert abs(I - oI) <= 1e-12 * abs(oI) and abs(s - os_) <= 1e-12 * abs(os_)
    # the events on both sides of the boundary, one by one (iteration counter as during the shard)
    g.set_iteration(0); o.set_iteration(0)
    for at in (2**32 - 64, 2**32):                       # (the parity hook takes ranges on one side of a multiple of 2^32)
        assert_events_equal(g.debug_events(at, 64, seed=w.seed), o.events(at, 64, w.seed), w)


def test_cfg3_sweep_parity(V, O):
    """BASELINE.json configs[2]: 1e8 events of the d=8 double Gaussian split into launches of 1e4 ... 1e8 events; every
    split is compared with ONE oracle iteration (not with another GPU run).  The launches are dealt to up to 128 internal
    streams with the grid the library's wave model picks (10 000 launches of one CTA each -- two for every third --, 1 000 of
    two, 100 of sixteen, 10 of 59, 1 of all), as a replayed CUDA graph and, for 1e4 / 1e5, also as plain launches."""
    w = W.cfg3()
    g, o = make_pair(V, O, w)
    ores = o.iterate(w.n_events, w.seed, threads=THREADS)
    for epl, graph in [(e, True) for e in w.batch_sizes] + [(10**4, False), (10**5, False)]:
        g.reset()
        g.use_cuda_graph(graph)
        gres = g.iterate(w.n_events, epl, w.seed)
        assert_iteration_close(gres, ores)
        S1, S2, _ = g.last_sums()
        oS1, oS2 = o.last_sums()
        assert abs(S1 - oS1) <= 1e-12 * abs(oS1) and abs(S2 - oS2) <= 1e-12 * abs(oS2)
        np.testing.assert_allclose(gres[2].sum(axis=1), S2, rtol=1e-12)
    # and the cascade of the sweep's smallest batch: 3 free-running iterations at 1e5 events per launch
    g.reset(); o.reset()
    g.use_cuda_graph(True)
    for it in range(3):
        ores = o.iterate(w.n_events, w.seed, threads=THREADS)
        assert_iteration_close(g.iterate(w.n_events, 10**5, w.seed), ores)
        o.refine(w.alpha); g.refine(w.alpha)
        assert np.max(np.abs(g.get_grid() - o.get_grid())) <= 1e-12


def test_two_contexts_of_one_generic_instance_interleaved(V, O):
    """Two live contexts that share one run-time-shaped kernel instance with different shapes (different nbins, hence
    different dynamic shared memory) do not disturb each other (the shared-memory limit is a per-function attribute)."""
    wa = W.Workload("gsa", 3, 400, W.GAUSS_SYM, (0.1, 0.5), W.FP64, 10**5, 1)     # large histogram
    ga, oa = make_pair(V, O, wa)
    wb = W.Workload("gsb", 3, 8, W.GAUSS_SYM, (0.1, 0.5), W.FP64, 10**5, 1)       # small one, created afterwards
    gb, ob = make_pair(V, O, wb)
    assert ga.launch_shape()["smem_bytes"] > 48 * 1024 > gb.launch_shape()["smem_bytes"]
    ra, rb = oa.iterate(200_003, 1, threads=THREADS), ob.iterate(200_003, 1, threads=THREADS)
    for _ in range(2):
        ga.reset(); gb.reset()
        assert_iteration_close(ga.iterate(200_003, 0, 1), ra)
        assert_iteration_close(gb.iterate(200_003, 0, 1), rb)


def test_state_after_graph_run_set_grid_and_consumed_histogram(V):
    """State-machine holes: last_sums() after a graph-replayed run on a fresh context, set_grid dropping the histogram,
    the histogram being unavailable after a successful refine."""
    w = W.cfg1()
    g = V.from_workload(w)
    m, e, c2, log = g.run_integration(3, 50_000, 0, w.seed, w.alpha)
    S1, S2, ms = g.last_sums()                          # the run's average step time, not an unrecorded event pair
    assert ms > 0 and np.all(log["kernel_ms"] > 0)
    assert abs(ms - log["kernel_ms"].mean()) < 0.5 * ms
    g.iterate(50_000, 0, w.seed)
    g.set_grid(g.get_grid())
    with pytest.raises(V.VegasError) as ei:
        g.refine(w.alpha)                               # H was sampled through the grid that set_grid replaced
    assert ei.value.code == V.ESTATE
    g.iterate(50_000, 0, w.seed)
    g.refine(w.alpha)
    with pytest.raises(V.VegasError) as ei:
        g.iterate_collect(want_hist=True)               # consumed (cleared) by the refinement
    assert ei.value.code == V.ESTATE
    I, s, _ = g.iterate_collect(want_hist=False)
    assert s > 0
    with pytest.raises(V.VegasError) as ei:
        g.iterate(10**8, 10, w.seed)                    # 1e7 launches: refused up front
    assert ei.value.code == V.EINVAL


def test_batch_size_study_shape(V):
    """configs[2] / PAPER.md:L65: throughput suffers when the batch is too small and reaches a plateau.
    Loose, timing-based: 1e4-event launches (1000 of them, replayed as a CUDA graph over 128 internal streams) are at
    least 1.2x slower per event than 1e7-event launches, and 1e6-event launches are within a factor 2.5 of them."""
    w = W.cfg2(n_events=10**7)
    g = V.from_workload(w)
    ms = {}
    for epl in (10**4, 10**6, 10**7):
        g.reset()
        g.iterate(w.n_events, epl, w.seed, want_hist=False)          # warm-up
        best = 1e30
        for _ in range(3):
            g.iterate(w.n_events, epl, w.seed, want_hist=False)
            best = min(best, g.last_sums()[2])
        ms[epl] = best
    assert ms[10**4] > 1.2 * ms[10**7], ms
    assert ms[10**6] >= 0.95 * ms[10**7] and ms[10**6] < 2.5 * ms[10**7], ms


def test_tune_events_per_launch_leaves_state_alone_and_prefers_large_batches(V, O):
    w = W.cfg2(n_events=10**7)
    g, o = make_pair(V, O, w)
    g.iterate(200_000, 0, w.seed); g.refine(w.alpha)
    o.iterate(200_000, w.seed, threads=THREADS); o.refine(w.alpha)
    grid, it = g.get_grid(), g.iteration
    best, ms = g.tune_events_per_launch(w.n_events, [10**4, 10**5, 10**6, 10**7], seed=w.seed)
    assert best in (10**6, 10**7) and ms[10**4] > ms[10**7] and all(v > 0 for v in ms.values())
    np.testing.assert_array_equal(g.get_grid(), grid)
    assert g.iteration == it
    with pytest.raises(V.VegasError) as ei:
        g.refine(w.alpha)                               # the histogram on the device is a tuning run's
    assert ei.value.code == V.ESTATE
    g.set_grid(o.get_grid())
    assert_iteration_close(g.iterate(300_000, best, w.seed), o.iterate(300_000, w.seed, threads=THREADS))


@pytest.mark.parametrize("name,n,epl", [("cfg1", 10**5, 0), ("cfg2", 400_003, 0), ("cfg2", 400_003, 60_000), ("cfg2", 400_003, 20_000),
                                        ("cfg4", 300_000, 0), ("cfg5", 300_000, 100_000), ("toy_d32", 200_000, 0), ("toy_f32_d9", 200_000, 0)])
def test_fused_step_equals_iterate_plus_refine_and_the_oracle(V, O, name, n, epl):
    """vegas_step_enqueue (S1-S7 in one kernel per launch: the last CTA finalizes, refines, commits and clears the
    accumulators; no memset between steps) against the oracle, five free-running steps, single launch / several launches /
    graph-replayed many launches."""
    w = small_workloads()[name]
    g, o = make_pair(V, O, w)
    for it in range(5):
        oI, os_, _ = o.iterate(n, w.seed, threads=THREADS)
        launches = g.step_enqueue(n, epl, w.seed, w.alpha)
        assert launches == (1 if not epl else -(-n // epl))
        gI, gs, _ = g.iterate_collect(want_hist=False)
        assert abs(gI - oI) <= 1e-12 * abs(oI) and abs(gs - os_) <= 1e-12 * abs(os_), (it, gI, oI, gs, os_)
        if o.npass is not None:
            assert g.last_npass() == o.npass
        with pytest.raises(V.VegasError) as ei:
            g.iterate_collect(want_hist=True)           # consumed by the fused refinement
        assert ei.value.code == V.ESTATE
        o.refine(w.alpha)
        g.refine_collect()
        assert np.max(np.abs(g.get_grid() - o.get_grid())) <= 1e-12, (it, np.max(np.abs(g.get_grid() - o.get_grid())))
    # a plain iteration after fused steps starts from clean accumulators as well
    assert_iteration_close(g.iterate(n, epl, w.seed), o.iterate(n, w.seed, threads=THREADS))
    # ... and a fused step after a plain iteration (dirty accumulators: the memset comes back)
    o.refine(w.alpha); g.refine(w.alpha)
    g.step_enqueue(n, epl, w.seed, w.alpha); g.refine_collect()
    oI, os_, _ = o.iterate(n, w.seed, threads=THREADS); o.refine(w.alpha)
    gI, gs, _ = g.iterate_collect(want_hist=False)
    assert abs(gI - oI) <= 1e-12 * abs(oI) and abs(gs - os_) <= 1e-12 * abs(os_)
    assert np.max(np.abs(g.get_grid() - o.get_grid())) <= 1e-12


def test_async_step_equals_blocking_step(V):
    """vegas_iterate_enqueue + vegas_refine_enqueue (bench.py's device-timed step) against the blocking calls."""
    w = W.cfg1()
    a, b = V.from_workload(w), V.from_workload(w)
    for _ in range(3):
        a.iterate_enqueue(w.n_events, 30_000, w.seed)
        a.refine_enqueue(w.alpha)
        b.iterate(w.n_events, 30_000, w.seed)
        b.refine(w.alpha)
    a.refine_collect()
    np.testing.assert_allclose(a.get_grid(), b.get_grid(), rtol=0, atol=1e-13)   # (H is summed in a different order in the two runs)
    Ia, sa, ha = a.iterate(w.n_events, 0, w.seed)
    Ib, sb, hb = b.iterate(w.n_events, 0, w.seed)
    assert abs(Ia - Ib) <= 1e-13 * abs(Ib) and abs(sa - sb) <= 1e-12 * sb
    assert all(a.iteration_kernel_ms(k) > 0 for k in range(4))
    with pytest.raises(V.VegasError) as ei:
        a.iteration_kernel_ms(4)
    assert ei.value.code == V.EINVAL
    with pytest.raises(V.VegasError) as ei:
        a.refine_enqueue(w.alpha); a.refine_enqueue(w.alpha)       # second one has no histogram
    assert ei.value.code == V.ESTATE
    a.refine_collect()
