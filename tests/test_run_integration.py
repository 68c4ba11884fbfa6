"""run_integration: the combination of iteration estimates pinned against exact
rational arithmetic on both sides (oracle and library: host arithmetic, no GPU needed), the oracle's multi-iteration
driver against the closed form, and (gpu) the library's driver against the oracle's."""
import math
from fractions import Fraction

import numpy as np
import pytest

from paper_2010_09341_b200 import workloads as W


def exact_combine(I, s):
    I = [Fraction(x) for x in I]
    w = [1 / (Fraction(x) ** 2) for x in s]
    sw = sum(w)
    mean = sum(wi * Ii for wi, Ii in zip(w, I)) / sw
    chi2 = sum(wi * (Ii - mean) ** 2 for wi, Ii in zip(w, I))
    return float(mean), math.sqrt(float(1 / sw)), float(chi2 / (len(I) - 1)) if len(I) > 1 else 0.0


LATE_RTOL = 1e-12          # iterations 6..20 of the 20-iteration graph test (see there)

CASES = [([1.0, 2.0, 4.0], [1.0, 2.0, 4.0]),            # hand case: mean 4/3, error sqrt(16/21), chi2/dof 1/3
         ([0.5, 0.25, 0.75, 0.625], [0.125, 0.5, 0.25, 1.0]),
         ([3.0], [0.5]),
         ([1.0000001, 0.9999999, 1.0, 1.00000005], [1e-7, 2e-7, 4e-7, 1e-7])]


@pytest.mark.parametrize("I,s", CASES)
def test_combination_matches_exact_rationals_on_both_sides(I, s):
    from oracle import oracle as O
    from paper_2010_09341_b200 import vegas as V
    want = exact_combine(I, s)
    for got in (O.combine(I, s), V.combine_iterations(I, s)):
        assert got[0] == pytest.approx(want[0], rel=1e-15)
        assert got[1] == pytest.approx(want[1], rel=1e-15)
        assert got[2] == pytest.approx(want[2], rel=1e-9, abs=1e-300)
    assert exact_combine([1, 2, 4], [1, 2, 4]) == pytest.approx((4 / 3, math.sqrt(16 / 21), 1 / 3), rel=1e-15)


def test_combination_degenerate_weights():
    from oracle import oracle as O
    from paper_2010_09341_b200 import vegas as V
    for f in (O.combine, V.combine_iterations):
        assert f([2.0, 4.0], [0.0, 0.0]) == (3.0, 0.0, 0.0)                  # no weight anywhere: plain average
        m, e, c = f([2.0, 5.0, 7.0], [0.0, 0.5, float("inf")])               # only the middle one carries weight
        assert (m, e) == (5.0, 0.5) and c == 0.0
        m, e, c = f([1.0, 3.0], [1.0, 1.0])
        assert (m, c) == (2.0, 2.0) and e == pytest.approx(math.sqrt(0.5))


def test_oracle_run_integration_cfg1_and_paper_example():
    from oracle import oracle as O
    w = W.cfg1()
    o = O.Oracle(w.dim, w.nbins, w.integrand_id, w.params, w.precision)
    mean, err, chi2, I, s = o.run_integration(4, w.n_events, w.seed, w.alpha, n_warmup=1, threads=4)
    exact = math.erf(5.0) ** 4
    assert len(I) == 5 and o.iteration == 5
    assert abs(mean - exact) <= 4 * err and err < s[1:].min() and chi2 < 5.0
    assert (mean, err, chi2) == O.combine(I[1:], s[1:])
    t = W.toy()                                                                # PAPER.md:L72-L79, exact d/2 = 5
    o = O.Oracle(t.dim, t.nbins, t.integrand_id, t.params, t.precision)
    mean, err, chi2, I, s = o.run_integration(t.n_iter, 10**5, t.seed, t.alpha, threads=4)
    assert abs(mean - 5.0) <= 4 * err


@pytest.mark.gpu
@pytest.mark.parametrize("name,n,epl,warm", [("cfg1", 10**5, 0, 1), ("toy", 10**6, 10**5, 0), ("cfg5", 300_000, 0, 2)])
def test_run_integration_parity(name, n, epl, warm):
    import torch
    assert torch.cuda.is_available()
    from oracle import oracle as O
    from paper_2010_09341_b200 import vegas as V
    w = W.ALL[name]()
    g = V.from_workload(w)
    o = O.Oracle(w.dim, w.nbins, w.integrand_id, w.params, w.precision)
    gm, ge, gc, info = g.run_integration(4, n, epl, w.seed, w.alpha, n_warmup=warm)
    om, oe, oc, oI, os_ = o.run_integration(4, n, w.seed, w.alpha, n_warmup=warm, threads=8)
    np.testing.assert_allclose(info["integral"], oI, rtol=1e-12)     # north_star's tolerance: at most 6 iterations here
    np.testing.assert_allclose(info["error"], os_, rtol=1e-12)
    assert gm == pytest.approx(om, rel=1e-12) and ge == pytest.approx(oe, rel=1e-12)
    assert gc == pytest.approx(oc, rel=1e-6, abs=1e-9)
    assert g.iteration == o.iteration == 4 + warm and np.all(info["kernel_ms"] > 0)
    assert np.max(np.abs(g.get_grid() - o.get_grid())) <= 1e-12
    # the plain loop of blocking calls (no CUDA graph) gives the same numbers, and a second graph run continues
    h = V.from_workload(w)
    h.use_cuda_graph(False)
    hm, he, hc, hinfo = h.run_integration(4, n, epl, w.seed, w.alpha, n_warmup=warm)
    np.testing.assert_allclose(hinfo["integral"], info["integral"], rtol=1e-12)
    np.testing.assert_allclose(hinfo["error"], info["error"], rtol=1e-11)
    assert hm == pytest.approx(gm, rel=1e-12) and h.iteration == g.iteration
    g.run_integration(2, n, epl, w.seed, w.alpha)
    h.run_integration(2, n, epl, w.seed, w.alpha)
    assert g.iteration == h.iteration == 6 + warm
    assert np.max(np.abs(g.get_grid() - h.get_grid())) <= 1e-12
    I1, s1, _ = g.iterate(n, epl, w.seed)               # blocking calls keep working after graph replays
    I2, s2, _ = h.iterate(n, epl, w.seed)
    assert I1 == pytest.approx(I2, rel=1e-12)


@pytest.mark.gpu
def test_run_integration_parity_across_a_multi_step_graph():
    """20 iterations of cfg1 (1e5 events, one launch each): run_integration replays one CUDA graph of 16 consecutive
    steps -- their kernels linked by programmatic dependent launch -- and four single-step graphs; every iteration is
    compared with the oracle's free-running driver."""
    import torch
    assert torch.cuda.is_available()
    from oracle import oracle as O
    from paper_2010_09341_b200 import vegas as V
    w = W.cfg1()
    g = V.from_workload(w)
    o = O.Oracle(w.dim, w.nbins, w.integrand_id, w.params, w.precision)
    gm, ge, gc, info = g.run_integration(18, w.n_events, 0, w.seed, w.alpha, n_warmup=2)
    om, oe, oc, oI, os_ = o.run_integration(18, w.n_events, w.seed, w.alpha, n_warmup=2, threads=8)
    dI = np.abs(info["integral"] - oI) / np.abs(oI)
    ds = np.abs(info["error"] - os_) / np.abs(os_)
    dE = np.max(np.abs(g.get_grid() - o.get_grid()))
    print("16-step graph, cfg1 x20: max rel dev I %.2e sigma %.2e over the first 5 | I %.2e sigma %.2e over all 20 | edges %.2e"
          % (dI[:5].max(), ds[:5].max(), dI.max(), ds.max(), dE))
    # the five iterations configs[0] states, at north_star's tolerance ...
    assert dI[:5].max() <= 1e-12 and ds[:5].max() <= 1e-12
    # ... and the fifteen beyond them, where the adaptive feedback amplifies last-bit differences of the histogram sums
    # from refinement to refinement: measured I 7e-16, sigma 6e-14, edges 4e-14 by iteration 20, so
    # the same tolerance still holds with a factor 16 to spare
    assert dI.max() <= LATE_RTOL and ds.max() <= LATE_RTOL
    assert gm == pytest.approx(om, rel=LATE_RTOL) and ge == pytest.approx(oe, rel=LATE_RTOL)
    assert g.iteration == o.iteration == 20 and np.all(info["kernel_ms"] > 0)
    assert dE <= LATE_RTOL


@pytest.mark.gpu
def test_run_integration_graph_many_iterations_and_speed():
    """More iterations than the device-side result ring holds (64), and the graph replay is not slower than
    the loop of blocking calls on the latency-bound configuration (cfg1)."""
    import time
    from paper_2010_09341_b200 import vegas as V
    w = W.cfg1()
    g, h = V.from_workload(w), V.from_workload(w)
    h.use_cuda_graph(False)
    g.run_integration(3, w.n_events, 0, w.seed, w.alpha); h.run_integration(3, w.n_events, 0, w.seed, w.alpha)
    t0 = time.perf_counter(); gm = g.run_integration(150, w.n_events, 0, w.seed, w.alpha); tg = time.perf_counter() - t0
    t0 = time.perf_counter(); hm = h.run_integration(150, w.n_events, 0, w.seed, w.alpha); th = time.perf_counter() - t0
    # the first iterations agree to rounding; over 150 refinements the last-bit differences of the atomically
    # accumulated histograms are amplified by the adaptive feedback (observed ~4e-7 by iteration 150), so the
    # later ones are compared statistically
    np.testing.assert_allclose(gm[3]["integral"][:8], hm[3]["integral"][:8], rtol=1e-11)
    np.testing.assert_allclose(gm[3]["integral"], hm[3]["integral"], rtol=1e-4)
    assert gm[0] == pytest.approx(hm[0], rel=1e-5) and g.iteration == h.iteration == 153
    assert abs(gm[0] - math.erf(5.0) ** 4) <= 5 * gm[1]
    print("run_integration cfg1 x150: graph %.2f ms, blocking loop %.2f ms" % (tg * 1e3, th * 1e3))
    assert tg < 1.2 * th
