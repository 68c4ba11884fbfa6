"""Oracle against the mathematics (no GPU): closed-form integrals (P3), invariants (P4), brute-force
quadrature of the grid-mapped integrand (P5), refinement properties and hand cases (P6).

Exact values are recomputed here with mpmath/erf from the *definitions* of the configs in BASELINE.json;
tests/golden/closed_forms.txt records the cited numbers and is cross-checked too.
"""
import math
import os

import mpmath as mp
import numpy as np
import pytest

from conftest import read_golden
from oracle import oracle as O
from paper_2010_09341_b200 import workloads as W

ALPHA = 1.5


def make(wl):
    return O.Oracle(wl.dim, wl.nbins, wl.integrand_id, wl.params, wl.precision)


# ---------------------------------------------------------------------------------------- exact values
def exact_cfg1(d=4, alpha=0.1):
    return math.erf(0.5 / alpha) ** d


def exact_gauss_double(d=8, alpha=0.1):
    mp.mp.dps = 40
    a = mp.mpf(alpha)
    g = lambda mu: (mp.erf((1 - mu) / a) + mp.erf(mu / a)) / 2
    return float((g(mp.mpf(1) / 3) ** d + g(mp.mpf(2) / 3) ** d) / 2)


def exact_genz(cs, phase_fraction=0.3):
    mp.mp.dps = 30
    prod = mp.mpf(1); s = mp.mpf(0)
    for c in cs:
        c = mp.mpf(c)
        prod *= mp.quad(lambda t: mp.cos(c * t) / (c ** -2 + t * t), [-0.5, 0, 0.5])
        s += c / 2
    return float(mp.cos(2 * mp.pi * mp.mpf(phase_fraction) + s) * prod)


def exact_lo2to2():
    mp.mp.dps = 40
    s = mp.mpf(13000) ** 2; tau = mp.mpf(50) ** 2 / s
    cang = mp.quad(lambda c: (4 + (1 + c) ** 2) / (1 - c) ** 2, [-0.9, 0, 0.9])
    h = lambda x: x ** mp.mpf("-2.1") * (1 - x) ** 5
    Hint = lambda a: sum(mp.binomial(5, k) * (-1) ** k * (1 - a ** (k - mp.mpf("1.1"))) / (k - mp.mpf("1.1")) for k in range(6))
    X = mp.quad(lambda x1: h(x1) * Hint(tau / x1), [tau, 1e-4, 1e-3, 1e-2, 1e-1, 1])
    return float(X * cang / (2 * s))


def test_closed_forms_match_cited_values(golden_dir):
    g = read_golden(os.path.join(golden_dir, "closed_forms.txt"))
    assert exact_cfg1() == pytest.approx(float(g["cfg1"][0]), rel=1e-14)
    assert exact_gauss_double() == pytest.approx(float(g["cfg2"][0]), rel=1e-14)
    assert exact_lo2to2() == pytest.approx(float(g["cfg5"][0]), rel=1e-12)
    c32 = [float(np.float32(c)) for c in W.genz_c(0, 20)]
    assert exact_genz(c32) == pytest.approx(float(g["cfg4_fp32c"][0]), rel=1e-10)


# ---------------------------------------------------------------------------------------- P3: 4 sigma
def run(wl, n, iters, seed, threads=4):
    o = make(wl)
    out = []
    for _ in range(iters):
        I, s, h = o.iterate(n, seed, threads=threads)
        out.append((I, s))
        o.refine(ALPHA)
    return o, out


def test_cfg1_full_size_within_4_sigma_and_adapts():
    """BASELINE.json configs[0] at full size: 1e5 events x 5 iterations, seeds 0,1,2."""
    exact = exact_cfg1()
    for seed in (0, 1, 2):
        o, res = run(W.cfg1(), 10**5, 5, seed, threads=1)
        for I, s in res[1:]:
            assert abs(I - exact) < 4 * s
        # "every iteration informs the subsequent run": the error collapses after adapting
        assert res[-1][1] < 0.1 * res[0][1]
        assert 1.0e-3 < res[-1][1] < 2.5e-3


def test_gauss_double_d8_within_4_sigma_and_rejects_other_reading():
    """configs[1] at n=1e6: consistent with the reading N(x)=exp(-(x-mu)^2/a^2)/(a sqrt(pi)) (R13)."""
    exact = exact_gauss_double()
    o, res = run(W.cfg2(), 10**6, 6, 0)
    I, s = res[-1]
    assert abs(I - exact) < 4 * s
    assert s < 0.25
    # inverse-variance combination of the adapted iterations discriminates against the sigma=alpha pdf reading
    w = np.array([1 / s ** 2 for _, s in res[2:]]); v = np.array([I for I, _ in res[2:]])
    comb, cs = float((w * v).sum() / w.sum()), float(w.sum() ** -0.5)
    assert abs(comb - exact) < 4 * cs


def test_gauss_low_dim_tight():
    """I0/I1 in d=1,2 where sigma is tiny: a dropped factor or a wrong mu shows at once."""
    for d in (1, 2):
        wl = W.Workload("g", d, 50, W.GAUSS_SYM, (0.1, 0.5), W.FP64, 0, 0)
        o, res = run(wl, 200_000, 4, 1)
        assert abs(res[-1][0] - exact_cfg1(d)) < 4 * res[-1][1] and res[-1][1] < 2e-3
        wl = W.Workload("g2", d, 50, W.GAUSS_DOUBLE, (0.1, 1 / 3, 2 / 3), W.FP64, 0, 0)
        o, res = run(wl, 200_000, 4, 2)
        assert abs(res[-1][0] - exact_gauss_double(d)) < 4 * res[-1][1] and res[-1][1] < 4e-3


def test_genz_low_dim_within_4_sigma():
    """I2 (fp32) in d=4 where the cancellation is mild: pins cos_f32, c_k, w_k and the division."""
    wl = W.cfg4(dim=4)
    exact = exact_genz([float(np.float32(c)) for c in wl.params[1:]])
    o, res = run(wl, 400_000, 4, 0)
    I, s = res[-1]
    assert abs(I - exact) < 4 * s
    assert s < 0.01 * abs(exact)


def test_genz_d20_within_4_sigma():
    wl = W.cfg4()
    exact = exact_genz([float(np.float32(c)) for c in wl.params[1:]])
    o, res = run(wl, 10**6, 3, 0)
    for I, s in res:
        assert abs(I - exact) < 4 * s


def test_lo_2to2_within_4_sigma():
    exact = exact_lo2to2()
    o, res = run(W.cfg5(), 10**6, 4, 0)
    for I, s in res[1:]:
        assert abs(I - exact) < 4 * s
    assert res[-1][1] < 5e-3 * exact * 2


def test_toy_sum_paper_example():
    """f=sum x_i, n_dim=10, 1e6 events, 5 iterations; exact integral d/2."""
    o, res = run(W.toy(10), 10**6, 2, 0)
    for I, s in res:
        assert abs(I - 5.0) < 4 * s and s < 2e-3


# ---------------------------------------------------------------------------------------- P4: invariants
def test_invariants_after_each_refine():
    for wl, n in ((W.cfg1(), 10**5), (W.cfg5(), 2 * 10**5), (W.cfg4(dim=4), 10**5)):
        o = make(wl)
        for it in range(4):
            I, s, h = o.iterate(n, 0, threads=2)
            S1, S2 = o.last_sums()
            # every event lands in exactly one bin of every dimension: row sums equal S2
            for k in range(wl.dim):
                assert math.fsum(h[k]) == pytest.approx(S2, rel=1e-13)
            o.refine(ALPHA)
            E = o.get_grid()
            assert np.all(E[:, 0] == 0.0) and np.all(E[:, -1] == 1.0)
            assert np.all(np.diff(E, axis=1) > 0)
            lo, wd, g = o.get_table()
            if wl.precision == W.FP64:
                assert np.array_equal(lo, E[:, :-1]) and np.array_equal(wd, np.diff(E, axis=1))
                assert np.array_equal(g, wl.nbins * wd)
            else:
                assert np.array_equal(lo, E[:, :-1].astype(np.float32).astype(np.float64))
                assert np.array_equal(wd, np.diff(E, axis=1).astype(np.float32).astype(np.float64))


def test_bin_occupancy_is_uniform_whatever_the_grid():
    """Bin index = floor(u N) of a uniform u, independent of the grid: chi^2 over bins."""
    wl = W.cfg1()
    o = make(wl)
    o.iterate(10**5, 0); o.refine(ALPHA)
    ev = o.events(0, 200_000, 9)
    for k in range(wl.dim):
        cnt = np.bincount(ev["bins"][:, k], minlength=wl.nbins)
        chi2 = ((cnt - 4000.0) ** 2 / 4000.0).sum()
        assert chi2 < 49 + 6 * math.sqrt(2 * 49)


def test_set_get_grid_identity_and_validation():
    wl = W.cfg1()
    o = make(wl)
    o.iterate(10**4, 0); o.refine(ALPHA)
    E = o.get_grid()
    p = make(wl)
    p.set_grid(E)
    assert np.array_equal(p.get_grid(), E)
    p.set_iteration(1)
    a = o.events(5, 50, 0); b = p.events(5, 50, 0)
    assert all(np.array_equal(a[k], b[k]) for k in a)
    bad = E.copy(); bad[1, 7] = bad[1, 6]
    with pytest.raises(O.OracleError) as ei:
        p.set_grid(bad)
    assert ei.value.code == O.EGRID
    bad = E.copy(); bad[0, 0] = 1e-9
    with pytest.raises(O.OracleError):
        p.set_grid(bad)


def test_result_does_not_depend_on_range_split():
    """R16: the event index is global, so any split of the range gives the same real-number sums."""
    wl = W.cfg1()
    o = make(wl)
    whole = o.iterate_range(0, 30_000, 0)
    a = o.iterate_range(0, 12_345, 0); b = o.iterate_range(12_345, 30_000 - 12_345, 0)
    assert whole[0][0] + whole[0][1] == pytest.approx(a[0][0] + a[0][1] + b[0][0] + b[0][1], rel=1e-15)
    assert np.allclose(whole[1] + whole[2], a[1] + a[2] + b[1] + b[2], rtol=1e-15, atol=0)


def test_error_codes():
    with pytest.raises(O.OracleError):
        O.Oracle(0, 50, W.TOY_SUM)
    with pytest.raises(O.OracleError):
        O.Oracle(4, 4096, W.TOY_SUM)
    with pytest.raises(O.OracleError):
        O.Oracle(4, 512, W.TOY_SUM, precision=O.FP32_EVAL)
    with pytest.raises(O.OracleError):
        O.Oracle(4, 50, W.GAUSS_SYM, (0.1,))
    o = O.Oracle(2, 4, W.TOY_SUM)
    with pytest.raises(O.OracleError) as ei:
        o.refine(1.5)
    assert ei.value.code == O.ESTATE


# ---------------------------------------------------------------------------------------- P5: quadrature
def gl_nodes(n):
    x, w = np.polynomial.legendre.leggauss(n)
    return (x + 1) / 2, w / 2


def mapped_quadrature(o, d, N, nodes=32):
    """sum over bins of Gauss-Legendre of J(y) f(x(y)) dy, y in [0,1]^d, through the oracle's S2-S4 at
    caller-chosen mantissas m=floor(y 2^52)."""
    t, w = gl_nodes(nodes)
    y1 = ((np.arange(N)[:, None] + t[None, :]) / N).ravel()          # N*nodes points
    w1 = np.tile(w / N, N)
    if d == 1:
        Y = y1[:, None]; Wt = w1
    else:
        A, B = np.meshgrid(y1, y1, indexing="ij")
        Y = np.stack([A.ravel(), B.ravel()], axis=1); Wt = np.outer(w1, w1).ravel()
    m = np.floor(Y * 2.0**52).astype(np.uint64)
    r = o.map_eval(m)
    return math.fsum(Wt * r["jac"] * r["f"]), r


def test_mapped_integrand_quadrature_equals_closed_form():
    """Validates map + Jacobian on an *adapted* grid independently of sampling: the change of variables
    must leave the integral unchanged."""
    for d in (1, 2):
        for ident, params, exact in ((W.GAUSS_SYM, (0.1, 0.5), exact_cfg1(d)),
                                     (W.GAUSS_DOUBLE, (0.1, 1 / 3, 2 / 3), exact_gauss_double(d))):
            o = O.Oracle(d, 50, ident, params)
            for _ in range(3):
                o.iterate(50_000, 0); o.refine(ALPHA)
            E = o.get_grid()
            assert np.ptp(np.diff(E, axis=1)) > 1e-3            # the grid really is non-uniform
            val, r = mapped_quadrature(o, d, 50)
            assert val == pytest.approx(exact, rel=1e-11)
            # x(y) is the piecewise-linear interpolation of the edges
            y = (r["bins"] + 0.5) / 50
            assert np.all(r["x"] >= E[np.arange(d)[None, :], r["bins"]])
            assert np.all(r["x"] <= E[np.arange(d)[None, :], r["bins"] + 1])


def test_lo_2to2_integrand_quadrature_equals_closed_form():
    """I3 by deterministic quadrature over the allowed region (v1+v2<1, |2 v3-1|<0.9) on the uniform grid:
    pins the PDFs, matrix element, flux, Jacobian and L against the closed form C_ang X/(2s)."""
    wl = W.cfg5()
    o = make(wl)
    t, w = gl_nodes(24)
    # panels in v1, Duffy map v2=(1-v1) u, v3 in [0.05,0.95]
    p1 = np.linspace(0, 1, 9); vs = []; ws = []
    for a, b in zip(p1[:-1], p1[1:]):
        for ti, wi in zip(t, w):
            v1 = a + (b - a) * ti
            for a2, b2 in zip(p1[:-1], p1[1:]):
                for tj, wj in zip(t, w):
                    u = a2 + (b2 - a2) * tj
                    vs.append((v1, (1 - v1) * u)); ws.append(wi * (b - a) * wj * (b2 - a2) * (1 - v1))
    vs = np.array(vs); ws = np.array(ws)
    t3, w3 = gl_nodes(24)
    total = 0.0
    p3 = [0.05, 0.5, 0.8, 0.9, 0.95]                      # panels refine towards the t-channel pole at cos=1
    for a3, b3 in zip(p3[:-1], p3[1:]):
        for tk, wk in zip(t3, w3):
            v3 = a3 + (b3 - a3) * tk
            Y = np.column_stack([vs, np.full(len(vs), v3)])
            r = o.map_eval(np.floor(Y * 2.0**52).astype(np.uint64))
            assert np.all(r["jac"] == 1.0)
            total += (b3 - a3) * wk * math.fsum(ws * r["f"])
    assert total == pytest.approx(exact_lo2to2(), rel=1e-9)
    # outside the cuts the integrand is exactly zero
    out = o.map_eval(np.floor(np.array([[0.6, 0.5, 0.5], [0.2, 0.2, 0.99], [0.2, 0.2, 0.01]]) * 2.0**52).astype(np.uint64))
    assert np.all(out["f"] == 0.0)


def test_genz_integrand_pointwise_vs_mpmath():
    """I2 at fixed points against an mpmath evaluation of the formula in BASELINE.json configs[3]."""
    mp.mp.dps = 30
    wl = W.cfg4(dim=6)
    o = make(wl)
    c = [mp.mpf(float(np.float32(v))) for v in wl.params[1:]]
    rng = np.random.default_rng(5)
    m = rng.integers(0, 2**23, size=(200, 6)).astype(np.uint64)
    r = o.map_eval(m)
    for n in range(200):
        x = [mp.mpf(float(v)) for v in r["x"][n]]
        ref = mp.cos(2 * mp.pi * mp.mpf("0.3") + sum(ci * xi for ci, xi in zip(c, x)))
        den = mp.mpf(1)
        for ci, xi in zip(c, x):
            den *= ci ** -2 + (xi - mp.mpf("0.5")) ** 2
        # fp32 evaluation: absolute error of cos ~1e-6 (argument rounding), relative error of the product ~1e-6
        assert abs(float(r["f"][n]) - float(ref / den)) <= 4e-6 * float(1 / den)


# ---------------------------------------------------------------------------------------- S7 refine
def refine_with(N, hist, alpha, edges=None):
    o = O.Oracle(1, N, W.TOY_SUM)
    if edges is not None:
        o.set_grid(np.array([edges]))
    o.commit(10, 1.0, 1.0, np.array([hist], dtype=np.float64))
    o.refine(alpha)
    return o.get_grid()[0]


def test_refine_flat_histogram_keeps_uniform_grid():
    for N in (4, 50, 100):
        E = refine_with(N, [1.0] * N, 1.5)
        assert np.allclose(E, np.arange(N + 1) / N, rtol=0, atol=1e-14)   # N sequential prefix adds


def test_refine_alpha_zero_is_identity_map():
    E0 = np.array([0, 0.1, 0.15, 0.5, 1.0])
    E = refine_with(4, [3.0, 1.0, 0.5, 9.0], 0.0, E0)       # all m_i = 1: new edges = old edges
    assert np.allclose(E, E0, rtol=0, atol=1e-15)


def test_refine_hand_case_with_zero_weight_bins():
    """N=4, H={0,0,1,1}, alpha=1: smoothing s={0,1/3,2/3,1}, r=s/2, m_i=(1-r)/ln(1/r), bin 0 has m=0 and
    is skipped (reading R11)."""
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
    E = refine_with(4, [0.0, 0.0, 1.0, 1.0], 1.0)
    assert np.allclose(E, want, rtol=0, atol=1e-15)
    assert E[1] > 0.25                                      # nothing is placed inside the empty bin


def test_refine_equalises_damped_weight():
    """Defining property of the rebinning: with density m_i/(E_{i+1}-E_i) on old bin i, every new bin
    holds the same mass delta (checked by integrating the piecewise-constant density over new bins)."""
    rng = np.random.default_rng(3)
    N = 50
    E0 = np.concatenate([[0.0], np.sort(rng.uniform(0, 1, N - 1)), [1.0]])
    h = rng.uniform(0, 1, N) ** 4
    alpha = 1.5
    E = refine_with(N, h, alpha, E0)
    s = np.empty(N)
    s[0] = (h[0] + h[1]) / 2; s[-1] = (h[-2] + h[-1]) / 2; s[1:-1] = (h[:-2] + h[1:-1] + h[2:]) / 3
    r = s / s.sum()
    m = ((1 - r) / np.log(1 / r)) ** alpha
    cum = np.concatenate([[0], np.cumsum(m)])
    F = lambda x: np.interp(x, E0, cum)                     # cumulative damped weight at position x
    mass = np.diff(F(E))
    assert np.allclose(mass, cum[-1] / N, rtol=1e-11)
    assert np.all(np.diff(E) > 0)


def test_refine_unchanged_when_histogram_is_empty():
    E0 = np.array([0, 0.3, 0.35, 0.9, 1.0])
    E = refine_with(4, [0.0] * 4, 1.5, E0)
    assert np.array_equal(E, E0)
