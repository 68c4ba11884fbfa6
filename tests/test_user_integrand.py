"""User integrands compiled at run time (vegas_create_custom; PAPER.md:L72-L78 `compile(integrand)`; SURVEY 8.f
NEXT-3).  The same C source is compiled by gcc for the oracle and by NVRTC for the GPU.  CPU: the oracle's hook
against closed forms.  GPU: event-by-event and iteration parity, a built-in integrand restated as user code,
compile errors."""
import math

import numpy as np
import pytest

from paper_2010_09341_b200 import workloads as W

# the paper's example integrand (tf.reduce_sum(xarr, axis=1)), with a scale parameter
SUM_SRC = """
VEGAS_INTEGRAND double vegas_user_integrand(const double* x, int dim, const double* params)
{
    double s = 0.0;
    for (int k = 0; k < dim; ++k) s = s + x[k];
    return params[0] * s;
}
"""

# a peaked, non-separable integrand with a helper function and libm calls:
#   f = exp(-|x - c|^2 / w^2) * (1 + 0.5 cos(2 pi x_0 x_1)),  c = params[0], w = params[1]
PEAK_SRC = """
VEGAS_INTEGRAND double sq(double v) { return v * v; }
VEGAS_INTEGRAND double vegas_user_integrand(const double* x, int dim, const double* params)
{
    double r2 = 0.0;
    for (int k = 0; k < dim; ++k) r2 = r2 + sq(x[k] - params[0]);
    return exp(-r2 / (params[1] * params[1])) * (1.0 + 0.5 * cos(6.283185307179586 * x[0] * x[1]));
}
"""


def test_oracle_user_hook_matches_builtin_toy_and_closed_form():
    from oracle import oracle as O
    u = O.Oracle.custom(10, 50, SUM_SRC, (1.0,))
    t = O.Oracle(10, 50, W.TOY_SUM, ())
    eu, et = u.events(0, 2000, 3), t.events(0, 2000, 3)
    for k in ("bins", "x", "jac", "f", "wf"):
        np.testing.assert_array_equal(eu[k], et[k])
    mean, err, chi2, I, s = u.run_integration(4, 100_000, 0, 1.5, n_warmup=1, threads=4)
    assert abs(mean - 5.0) <= 4 * err
    g = O.Oracle.custom(2, 40, PEAK_SRC, (0.5, 0.2))
    mean, err, chi2, I, s = g.run_integration(5, 200_000, 1, 1.5, n_warmup=2, threads=4)
    # reference value by tensor Gauss-Legendre quadrature (numpy), independent of the sampler
    xs, ws = np.polynomial.legendre.leggauss(200)
    xs, ws = 0.5 * (xs + 1), 0.5 * ws
    X, Y = np.meshgrid(xs, xs, indexing="ij")
    ref = np.sum(np.outer(ws, ws) * np.exp(-((X - 0.5) ** 2 + (Y - 0.5) ** 2) / 0.04) * (1 + 0.5 * np.cos(2 * np.pi * X * Y)))
    assert abs(mean - ref) <= 4 * err and err < 2e-3 * ref


@pytest.mark.gpu
@pytest.mark.parametrize("src,dim,nbins,params,prec,frtol", [
    (SUM_SRC, 10, 50, (1.5,), W.FP64, 0.0),
    (PEAK_SRC, 4, 64, (0.4, 0.25), W.FP64, 4e-15),
    (PEAK_SRC, 3, 50, (0.6, 0.3), W.FP64_U32, 4e-15),
])
def test_user_integrand_parity(src, dim, nbins, params, prec, frtol):
    import torch
    assert torch.cuda.is_available()
    from oracle import oracle as O
    from paper_2010_09341_b200 import vegas as V
    g = V.Vegas(dim, nbins, V.USER, params, prec, source=src)
    o = O.Oracle.custom(dim, nbins, src, params, prec)
    eg, eo = g.debug_events(0, 5000, 9), o.events(0, 5000, 9)
    np.testing.assert_array_equal(eg["bins"], eo["bins"])
    np.testing.assert_array_equal(eg["x"], eo["x"])
    np.testing.assert_array_equal(eg["jac"], eo["jac"])
    if frtol == 0.0:
        np.testing.assert_array_equal(eg["f"], eo["f"])
    else:
        np.testing.assert_allclose(eg["f"], eo["f"], rtol=frtol, atol=0.0)
    for it in range(4):
        gI, gs, gh = g.iterate(300_007, 70_000, 9)
        oI, os_, oh = o.iterate(300_007, 9, threads=8)
        assert abs(gI - oI) <= 1e-12 * abs(oI) and abs(gs - os_) <= 1e-12 * abs(os_)
        np.testing.assert_allclose(gh, oh, rtol=1e-10, atol=0.0)
        g.refine(1.5); o.refine(1.5)
        assert np.max(np.abs(g.get_grid() - o.get_grid())) <= 1e-12
    gm, ge, gc, _ = g.run_integration(3, 100_000, 0, 9, 1.5)
    om, oe, oc, _, _ = o.run_integration(3, 100_000, 9, 1.5, threads=8)
    assert gm == pytest.approx(om, rel=1e-12) and ge == pytest.approx(oe, rel=1e-12)


@pytest.mark.gpu
def test_user_integrand_equals_builtin_and_reports_compile_errors():
    from paper_2010_09341_b200 import vegas as V
    u = V.Vegas(10, 50, V.USER, (1.0,), V.FP64, source=SUM_SRC)
    t = V.Vegas(10, 50, V.TOY_SUM, (), V.FP64)
    a, b = u.iterate(500_000, 0, 4), t.iterate(500_000, 0, 4)
    assert a[0] == pytest.approx(b[0], rel=1e-13) and a[1] == pytest.approx(b[1], rel=1e-12)
    np.testing.assert_allclose(a[2], b[2], rtol=1e-12)
    with pytest.raises(V.VegasError) as ei:
        V.Vegas(3, 50, V.USER, (), V.FP64, source="VEGAS_INTEGRAND double vegas_user_integrand(const double* x, int d, const double* p) { return undefined_symbol(x[0]); }")
    assert ei.value.code == V.EUNSUPPORTED and "undefined_symbol" in str(ei.value)
    with pytest.raises(V.VegasError) as ei:
        V.Vegas(3, 50, V.USER, (), V.FP32_EVAL, source=SUM_SRC)
    assert ei.value.code == V.EINVAL
    with pytest.raises(V.VegasError) as ei:
        V.Vegas(3, 50, V.USER, (), V.FP64)                      # USER without source goes through vegas_create
    assert ei.value.code == V.EINVAL
