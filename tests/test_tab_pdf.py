"""lo_2to2_tab: the tabulated-PDF variant of BASELINE.json configs[4].  Oracle pins: the
four-point Lagrange interpolation reproduces cubics, converges to the analytic PDF, the integrand agrees with the
analytic lo_2to2 to interpolation accuracy, and the estimate lands on the cfg5 closed form."""
import os

import numpy as np
import pytest

from paper_2010_09341_b200 import workloads as W

EXACT_CFG5 = 0.20588619982410909          # tests/golden/closed_forms.txt


def test_interpolation_reproduces_cubics_and_clamps_at_the_ends():
    from oracle import oracle as O
    M = 37
    v = 1.0 - np.arange(M) / (M - 1.0)
    cubic = lambda t: 2.0 + 3.0 * t - t * t + 0.5 * t ** 3
    G = cubic(v)
    for t in (0.0, 1e-9, 0.013, 0.25, 0.5, 0.77, 0.987, 1.0 - 1e-12, 1.0):
        assert O.tab_interp(G, t) == pytest.approx(cubic(t), rel=0, abs=2e-14)
    for j in range(M):                                   # knots are hit exactly
        assert O.tab_interp(G, v[j]) == pytest.approx(G[j], rel=1e-15)
    # a quartic is not reproduced: error ~ h^4 f''''/24 * max|s(s-1)(s+1)(s-2)| = h^4 * (9/16) at mid-interval
    Q = v ** 4
    h = 1.0 / (M - 1)
    mid = 0.5 * (v[10] + v[11])
    assert abs(O.tab_interp(Q, mid) - mid ** 4) == pytest.approx(9.0 / 16.0 * h ** 4, rel=1e-6)


def test_table_converges_to_the_analytic_pdf():
    from oracle import oracle as O
    import math
    tau = (50.0 / 13000.0) ** 2
    errs = []
    for M in (256, 1024):
        G = W.pdf_table(M)
        e = 0.0
        for t in np.linspace(0.1, 0.999, 400):          # x <= tau^0.1 = 0.33; towards x -> 1 g -> 0 steeply
            x = math.exp(t * math.log(tau))
            g = x ** -1.1 * (1 - x) ** 5
            e = max(e, abs(O.tab_interp(G, t) - g) / g)
        errs.append(e)
    assert errs[1] < 5e-8 and errs[0] / errs[1] > 100       # fourth order: 4^4 = 256


def test_tabulated_integrand_matches_the_analytic_one_and_the_closed_form():
    from oracle import oracle as O
    w = W.cfg5_tab()
    t = O.Oracle(w.dim, w.nbins, w.integrand_id, w.params, w.precision)
    with_nan = t.events(0, 50, 0)["f"]
    assert np.isnan(with_nan[t.events(0, 50, 0)["passed"] == 1]).all()      # no table yet
    t.set_table(W.pdf_table())
    a = O.Oracle(3, 50, W.LO_2TO2, (13000.0, 50.0, 0.9, 1.1, 5.0), W.FP64)
    et, ea = t.events(0, 20000, 0), a.events(0, 20000, 0)
    np.testing.assert_array_equal(et["bins"], ea["bins"])
    np.testing.assert_array_equal(et["passed"], ea["passed"])
    np.testing.assert_array_equal(et["x"], ea["x"])
    ok = ea["f"] > 0
    # away from x -> 1 (where g -> 0 and the relative interpolation error grows) the two agree to 1e-7
    far = ok & (ea["x"][:, 0] > 0.1) & (ea["x"][:, 1] > 0.1)
    np.testing.assert_allclose(et["f"][far], ea["f"][far], rtol=1e-7)
    np.testing.assert_allclose(et["f"][ok], ea["f"][ok], rtol=1e-3, atol=1e-6)      # x -> 1: g -> 0, absolute error only
    assert far.sum() > 5000
    mean, err, chi2, I, s = t.run_integration(4, 400_000, 0, 1.5, n_warmup=2, threads=max(1, min(8, len(os.sched_getaffinity(0)))))
    assert abs(mean - EXACT_CFG5) <= 4 * err and err < 3e-3 * EXACT_CFG5
