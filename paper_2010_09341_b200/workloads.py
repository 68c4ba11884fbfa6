"""Seeded, synthetic workload definitions (BASELINE.json configs[0..4] + the paper's toy example).

This module serves both the CUDA path and the oracle (the tests and bench.py pass what it returns to
each side).  It holds no Vegas arithmetic: only the configuration tables and the parameter draw of
config 4 ("c_i drawn uniform in [1,5] from the seed", BASELINE.json configs[3]).  That draw uses its own
small counter-based generator (the published Philox4x32-10 recipe, parameter stream j=0xFFFFFFFF,
SURVEY.md 8.c I2); the CUDA path and the oracle each carry their own independent implementation for the
event stream.  It imports neither the binding nor the oracle.

Stand-ins: cfg3 stands in for the batch-size study of PAPER.md Fig. 2
(L57-L65) and cfg5 for its LO hadronic integrand (L49, L63); the real single-top integrand and its PDF
set are not available.  No dataset is read; every event is generated from (seed, iteration, event index).
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Tuple

# integrand ids and precisions of the C ABI (include/vegas_b200.h)
GAUSS_SYM, GAUSS_DOUBLE, GENZ_OSC_PEAK, LO_2TO2, TOY_SUM, USER, LO_2TO2_TAB = 0, 1, 2, 3, 4, 5, 6
FP64, FP32_EVAL, FP64_U32 = 0, 1, 2

_M32 = 0xFFFFFFFF


def _philox4x32_10(ctr, key):
    c = list(ctr)
    k = list(key)
    for _ in range(10):
        p0 = 0xD2511F53 * c[0]
        p1 = 0xCD9E8D57 * c[2]
        c = [((p1 >> 32) ^ c[1] ^ k[0]) & _M32, p1 & _M32, ((p0 >> 32) ^ c[3] ^ k[1]) & _M32, p0 & _M32]
        k = [(k[0] + 0x9E3779B9) & _M32, (k[1] + 0xBB67AE85) & _M32]
    return c


def genz_c(seed: int, dim: int):
    """c_k = 1 + 4 u_k, u_k the 52-bit uniform from words r0,r1 of Philox(counter=(k,0,0,0xFFFFFFFF), key=seed)."""
    out = []
    for k in range(dim):
        r = _philox4x32_10([k, 0, 0, 0xFFFFFFFF], [seed & _M32, (seed >> 32) & _M32])
        m = ((r[1] << 32) | r[0]) >> 12
        out.append(1.0 + 4.0 * (m * 2.0 ** -52))
    return out


@dataclass(frozen=True)
class Workload:
    name: str
    dim: int
    nbins: int
    integrand_id: int
    params: Tuple[float, ...]
    precision: int
    n_events: int            # events per iteration at full size
    n_iter: int
    alpha: float = 1.5       # refinement damping exponent
    seed: int = 0
    events_per_launch: int = 0   # 0 = whole iteration in one launch
    note: str = ""
    batch_sizes: Tuple[int, ...] = field(default=())


def cfg1():
    return Workload("cfg1_gauss_sym_d4", 4, 50, GAUSS_SYM, (0.1, 0.5), FP64, 10**5, 5,
                    note="BASELINE.json configs[0]")


def cfg2(n_events=10**8, n_iter=10):
    return Workload("cfg2_gauss_double_d8", 8, 50, GAUSS_DOUBLE, (0.1, 1.0 / 3.0, 2.0 / 3.0), FP64,
                    n_events, n_iter, note="BASELINE.json configs[1] (headline)")


def cfg2_u32(n_events=10**8, n_iter=10):
    """configs[1] driven by the 32-bit-uniform stream (precision FP64_U32): an extra mode, reported separately."""
    w = cfg2(n_events, n_iter)
    return Workload("cfg2_gauss_double_d8_u32", w.dim, w.nbins, w.integrand_id, w.params, FP64_U32, n_events, n_iter,
                    note="BASELINE.json configs[1] with 32-bit uniforms (extra mode, DESIGN.md R3)")


def cfg3():
    w = cfg2(10**8, 5)
    return Workload("cfg3_batch_sweep_d8", w.dim, w.nbins, w.integrand_id, w.params, w.precision, 10**8, 5,
                    batch_sizes=(10**4, 10**5, 10**6, 10**7, 10**8), note="BASELINE.json configs[2]")


def cfg4(n_events=10**8, n_iter=10, seed=0, dim=20):
    return Workload("cfg4_genz_osc_peak_d%d" % dim, dim, 100, GENZ_OSC_PEAK, (0.3, *genz_c(seed, dim)),
                    FP32_EVAL, n_events, n_iter, seed=seed, note="BASELINE.json configs[3]")


def cfg5(n_events=10**8, n_iter=10):
    return Workload("cfg5_lo_2to2_d3", 3, 50, LO_2TO2, (13000.0, 50.0, 0.9, 1.1, 5.0), FP64,
                    n_events, n_iter, note="BASELINE.json configs[4]")


def pdf_table(n_knots=1024, sqrt_s=13000.0, sqrt_shat_min=50.0, a=1.1, b=5):
    """Synthetic PDF grid for lo_2to2_tab: values[j] = g(x_j) = x_j^-a (1-x_j)^b at x_j = tau^(1 - j/(n-1)) -- the toy PDF
    of BASELINE.json configs[4] tabulated on knots uniform in ln x (a stand-in for a PDFFlow/LHAPDF grid, which is not
    available).  Input data only: the interpolation is done by the CUDA path and by the oracle, each on its own."""
    import math
    tau = (sqrt_shat_min / sqrt_s) ** 2
    out = []
    for j in range(n_knots):
        x = 1.0 if j == n_knots - 1 else math.exp((1.0 - j / (n_knots - 1.0)) * math.log(tau))
        out.append(x ** (-a) * (1.0 - x) ** b)
    return out


def cfg5_tab(n_events=10**8, n_iter=10):
    """NEXT-4: configs[4] with the PDF looked up in a 1024-knot table instead of evaluated analytically."""
    return Workload("cfg5_lo_2to2_tab_d3", 3, 50, LO_2TO2_TAB, (13000.0, 50.0, 0.9), FP64, n_events, n_iter,
                    note="BASELINE.json configs[4] with a tabulated PDF (SURVEY 8.f NEXT-4)")


def toy(dim=10):
    """f = sum_i x_i, n_dim=10, n_events=1e6, events_limit=1e5, n_iter=5."""
    return Workload("toy_sum_d%d" % dim, dim, 50, TOY_SUM, (), FP64, 10**6, 5, events_per_launch=10**5,
                    note="PAPER.md:L72-L79 usage example")


ALL = {"cfg1": cfg1, "cfg2": cfg2, "cfg2_u32": cfg2_u32, "cfg5_tab": cfg5_tab, "cfg3": cfg3, "cfg4": cfg4, "cfg5": cfg5, "toy": toy}
