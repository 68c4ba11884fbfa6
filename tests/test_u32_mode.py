"""The 32-bit-uniform stream mode (precision FP64_U32; reading R3: an extra, reported separately).
Oracle pins: the mantissa rule against the Philox known-answer words, the exact-rational bin rule, invariants,
closed forms.  GPU parity for this mode runs with the other workloads in tests/test_gpu_parity.py."""
import math
from fractions import Fraction

import numpy as np

from paper_2010_09341_b200 import workloads as W

# Philox4x32-10, seed 0, iteration 0, event 0: blocks j = 0 and j = 1 (SURVEY 8.c P1 layout pins / P2 fp32 draws)
BLOCK0 = [0x6627E8D5, 0xE169C58D, 0xBC57AC4C, 0x9B00DBD8]
BLOCK1 = [0x2DCE73E5, 0x1348E23F, 0xFCF8E0EC, 0xA287AADB]


def make(dim=8, nbins=50, integrand=W.GAUSS_DOUBLE, params=(0.1, 1 / 3, 2 / 3)):
    from oracle import oracle as O
    return O, O.Oracle(dim, nbins, integrand, params, W.FP64_U32)


def test_mantissas_are_the_philox_words():
    O, o = make()
    assert [int(v) for v in o.mantissas(0, 0, 0)] == BLOCK0 + BLOCK1
    # any other event: word k&3 of block k>>2, from the (KAT-pinned) Philox function itself
    for e, it, seed in [(1, 0, 0), (2**32 + 5, 3, 0xDEADBEEF12345678)]:
        want = []
        for j in range(2):
            want += [int(v) for v in O.philox4x32_10([e & 0xFFFFFFFF, e >> 32, it, j], [seed & 0xFFFFFFFF, seed >> 32])]
        assert [int(v) for v in o.mantissas(seed, it, e)] == want


def test_bin_rule_is_exact_and_x_is_within_an_ulp_of_u():
    O, o = make()
    ev = o.events(0, 1, 0)
    want_bins = [int(Fraction(w * 50, 2**32)) for w in BLOCK0 + BLOCK1]
    assert want_bins == [19, 44, 36, 30, 8, 3, 49, 31]
    assert ev["bins"][0].tolist() == want_bins
    ev = o.events(123456, 4000, 7)
    for n in range(0, 4000, 97):
        m = o.mantissas(7, 0, 123456 + n)
        for k in range(8):
            u = Fraction(int(m[k]), 2**32)
            assert ev["bins"][n, k] == int(u * 50)
            assert abs(Fraction(float(ev["x"][n, k])) - u) <= Fraction(float(np.spacing(float(u))))   # uniform grid
    assert np.all(ev["jac"] == 1.0)


def test_gauss_sym_u32_within_4_sigma_and_invariants():
    O, o = make(4, 50, W.GAUSS_SYM, (0.1, 0.5))
    exact = math.erf(5.0) ** 4
    for it in range(5):
        I, s, h = o.iterate(100_000, 0, threads=4)
        S1, S2 = o.last_sums()
        np.testing.assert_allclose(h.sum(axis=1), S2, rtol=1e-12)
        o.refine(1.5)
        e = o.get_grid()
        assert np.all(np.diff(e, axis=1) > 0) and np.all(e[:, 0] == 0) and np.all(e[:, -1] == 1)
    assert abs(I - exact) <= 4 * s and s < 3e-3


def test_u32_stream_differs_from_the_52_bit_stream_but_agrees_statistically():
    from oracle import oracle as O
    a = O.Oracle(3, 50, W.LO_2TO2, (13000.0, 50.0, 0.9, 1.1, 5.0), W.FP64)
    b = O.Oracle(3, 50, W.LO_2TO2, (13000.0, 50.0, 0.9, 1.1, 5.0), W.FP64_U32)
    Ia, sa, _ = a.iterate(400_000, 0, threads=4)
    Ib, sb, _ = b.iterate(400_000, 0, threads=4)
    assert Ia != Ib and abs(Ia - Ib) <= 4 * math.hypot(sa, sb)


def test_modes_that_do_not_exist_are_refused():
    import pytest
    from oracle import oracle as O
    with pytest.raises(O.OracleError):
        O.Oracle(20, 100, W.GENZ_OSC_PEAK, W.cfg4().params, W.FP64_U32)       # the fp32 integrand has no fp64 stream mode
