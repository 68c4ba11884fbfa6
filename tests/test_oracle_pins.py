"""Pins of the CPU oracle against things other than itself (no GPU).

P1 Philox known answers and counter/key layout, P2 worked example (exact-rational values from
SURVEY.md 8.c), P6 estimator by exact rational arithmetic, P7 cos_f32 against fp64 cos, constants
against mpmath.  Every expected value here is either a cited fixture under tests/golden/ or computed in
the test by arithmetic independent of oracle/ (Python integers, fractions, mpmath, math).
"""
import math
import os
import struct
from fractions import Fraction as Fr

import mpmath as mp
import numpy as np
import pytest

from conftest import read_golden
from oracle import oracle as O
from paper_2010_09341_b200 import workloads as W


def f32(x):
    return struct.unpack("f", struct.pack("f", x))[0]


# ------------------------------------------------------------------------------------------------ P1
def test_philox_known_answers(golden_dir):
    g = read_golden(os.path.join(golden_dir, "philox_kat.txt"))
    for name in ("kat_zero", "kat_ones", "kat_pi"):
        w = [int(t, 16) for t in g[name]]
        assert O.philox4x32_10(w[0:4], w[4:6]) == w[6:10], name


def test_philox_layout_pins(golden_dir):
    """key=(seed lo, seed hi); counter=(e lo, e hi, it, j) -- a swapped word fails one of these."""
    g = read_golden(os.path.join(golden_dir, "philox_kat.txt"))
    for name in ("layout_e1", "layout_j1", "layout_it1", "layout_e2p32", "layout_seed1"):
        t = g[name]
        seed, it, e, j = int(t[0]), int(t[1]), int(t[2]), int(t[3])
        want = [int(v, 16) for v in t[4:8]]
        got = O.philox4x32_10([e & 0xFFFFFFFF, e >> 32, it, j], [seed & 0xFFFFFFFF, seed >> 32])
        assert got == want, name


def test_philox_matches_independent_python_integers():
    """Same recipe in unbounded Python integers (written for the input generator, not for the oracle)."""
    rng = np.random.default_rng(7)
    for _ in range(200):
        ctr = [int(v) for v in rng.integers(0, 2**32, 4)]
        key = [int(v) for v in rng.integers(0, 2**32, 2)]
        assert O.philox4x32_10(ctr, key) == W._philox4x32_10(ctr, key)


def test_mantissa_rule_fp64_and_fp32():
    """S1: 52-bit m from word pairs (r0,r1),(r2,r3) of block k>>1; 23-bit m = r[k&3]>>9 of block k>>2."""
    seed, it, e = 0x123456789ABCDEF, 3, 2**33 + 17
    key = [seed & 0xFFFFFFFF, seed >> 32]
    o64 = O.Oracle(5, 50, W.TOY_SUM)
    m = o64.mantissas(seed, it, e)
    for k in range(5):
        r = W._philox4x32_10([e & 0xFFFFFFFF, e >> 32, it, k >> 1], key)
        a = 2 * (k & 1)
        assert m[k] == ((r[a + 1] << 32) | r[a]) >> 12
    o32 = O.Oracle(7, 100, W.TOY_SUM, precision=O.FP32_EVAL)
    m = o32.mantissas(seed, it, e)
    for k in range(7):
        r = W._philox4x32_10([e & 0xFFFFFFFF, e >> 32, it, k >> 2], key)
        assert m[k] == r[k & 3] >> 9


# ------------------------------------------------------------------------------------------------ P2
def test_worked_example_cfg1(golden_dir):
    g = read_golden(os.path.join(golden_dir, "worked_example_cfg1.txt"))
    w = W.cfg1()
    o = O.Oracle(w.dim, w.nbins, w.integrand_id, w.params)
    lo, wd, gg = o.get_table()
    assert np.all(wd == float.fromhex(g["wd"][0]))
    assert np.all(gg == 1.0)                                   # uniform grid: Jacobian exactly 1
    C, a2 = o.gauss_consts()
    assert C == float.fromhex(g["C"][0]) and a2 == float.fromhex(g["a2"][0])
    assert o.mantissas(0, 0, 0) == [int(t, 16) for t in g["e0_m"]]
    ev = o.events(0, 2, 0)
    assert ev["bins"][0].tolist() == [int(t) for t in g["e0_bins"]]
    assert ev["bins"][1].tolist() == [int(t) for t in g["e1_bins"]]
    assert [float(v) for v in ev["x"][0]] == [float.fromhex(t) for t in g["e0_x"]]
    assert [float(v) for v in ev["x"][1]] == [float.fromhex(t) for t in g["e1_x"]]
    assert ev["jac"][0] == 1.0 and ev["jac"][1] == 1.0
    assert ev["f"][0] == pytest.approx(float(g["e0_f"][0]), rel=1e-13)
    assert ev["f"][1] == pytest.approx(float(g["e1_f"][0]), rel=1e-13)
    last = o.events(99999, 1, 0)
    assert last["bins"][0].tolist() == [int(t) for t in g["e99999_bins"]]
    assert last["f"][0] == pytest.approx(float(g["e99999_f"][0]), rel=1e-13)
    # frac and s recomputed from the dumped x: s = fma chain of (x-mu)^2 in exact rationals
    for tag, row in (("e0", ev["x"][0]), ("e1", ev["x"][1])):
        s = 0.0
        for xv in row:
            dx = float(xv) - 0.5
            s = float(Fr(dx) * Fr(dx) + Fr(s))
        assert s == float.fromhex(g[tag + "_s"][0])
    fr = [float.fromhex(t) for t in g["e0_frac"]]
    for k in range(4):
        p = int(g["e0_m"][k], 16) * 50
        assert p >> 52 == int(g["e0_bins"][k]) and (p & (2**52 - 1)) * 2.0**-52 == fr[k]
        assert float(Fr(fr[k]) * Fr(float.fromhex(g["wd"][0])) + Fr(int(g["e0_bins"][k]) / 50)) == float(ev["x"][0][k])


def test_worked_example_fp32_draws(golden_dir):
    g = read_golden(os.path.join(golden_dir, "worked_example_cfg1.txt"))
    w = W.cfg4()
    o = O.Oracle(w.dim, w.nbins, w.integrand_id, w.params, w.precision)
    m = o.mantissas(0, 0, 0)[:6]
    assert m == [int(t, 16) for t in g["f32_m"]]
    ev = o.events(0, 1, 0)
    assert ev["bins"][0][:6].tolist() == [int(t) for t in g["f32_bins"]]
    lo, wd, gg = o.get_table()
    assert np.all(gg == 1.0) and np.all(wd == f32(0.01))
    for k in range(6):
        frac = int(g["f32_frac_2p23"][k]) * 2.0**-23
        want = f32(float(Fr(frac) * Fr(f32(0.01)) + Fr(f32(int(g["f32_bins"][k]) / 100))))
        assert float(ev["x"][0][k]) == want


def test_exact_bin_rule_vs_rational_and_uniform_x_within_one_ulp():
    """S2: i=floor(m N / 2^B) exactly; on the uniform grid x is within 1 ulp of u=m/2^B and J==1."""
    o = O.Oracle(6, 50, W.TOY_SUM)
    for e in range(0, 4000, 7):
        m = o.mantissas(5, 0, e)
        ev = o.events(e, 1, 5)
        for k in range(6):
            assert int(ev["bins"][0][k]) == (m[k] * 50) >> 52
            u = m[k] * 2.0**-52
            assert abs(float(ev["x"][0][k]) - u) <= np.spacing(max(u, 2.0**-10))
        assert ev["jac"][0] == 1.0
    # explicit boundary mantissas: the largest m maps to the last bin, m=0 to bin 0, x stays in [0,1]
    top = 2**52 - 1
    r = o.map_eval(np.array([[0, top, top // 2, top // 50, top // 50 + 1, 1]], dtype=np.uint64))
    assert r["bins"][0].tolist()[:3] == [0, 49, 24]
    assert r["bins"][0][3] == 0 and r["bins"][0][4] == 1
    assert np.all(r["x"] >= 0.0) and np.all(r["x"] <= 1.0)


# ------------------------------------------------------------------------------------------------ constants
def test_constants_against_mpmath():
    mp.mp.dps = 50
    # I0/I1 constants: b=fl(alpha sqrt(fl64(pi))), C=1 then d divisions, a2=fl(1/fl(alpha alpha)).
    # DESIGN.md reading R19: sqrt of the *rounded* pi (0x1.c5bf891b4ef6ap+0, one ulp below the correctly
    # rounded sqrt(pi)) -- the value the cited worked example (P2, C for d=4) was computed with.
    alpha = 0.1
    sqrt_pi = float(mp.sqrt(mp.mpf(float(mp.pi))))
    assert sqrt_pi.hex() == "0x1.c5bf891b4ef6ap+0"
    b = alpha * sqrt_pi
    C = 1.0
    for _ in range(8):
        C = C / b
    o = O.Oracle(8, 50, W.GAUSS_DOUBLE, (alpha, 1 / 3, 2 / 3))
    assert o.gauss_consts() == (C, 1.0 / (alpha * alpha))
    # the correctly rounded C of the real constant is within a few ulp
    assert o.gauss_consts()[0] == pytest.approx(float((mp.mpf(alpha) * mp.sqrt(mp.pi)) ** -8), rel=4e-15)


def test_genz_parameters_match_cited_values(golden_dir):
    g = read_golden(os.path.join(golden_dir, "closed_forms.txt"))
    want = [float(t) for t in g["genz_c64"]]
    got = W.genz_c(0, 20)
    assert got == want
    assert got[0].hex() == "0x1.3a3bfcddcc97cp+2" and got[1].hex() == "0x1.121390a983d2ap+2"
    assert all(1.0 <= c < 5.0 for c in W.genz_c(3, 20))


# ------------------------------------------------------------------------------------------------ P7
def test_cos_f32_constants():
    mp.mp.dps = 60
    half_pi = mp.pi / 2
    C1 = f32(float(half_pi)); C2 = f32(float(half_pi - mp.mpf(C1))); C3 = f32(float(half_pi - mp.mpf(C1) - mp.mpf(C2)))
    assert (C1, C2, C3) == (float.fromhex("0x1.921fb6p+0"), float.fromhex("-0x1.777a5cp-25"), float.fromhex("-0x1.ee59dap-50"))
    assert f32(float(2 / mp.pi)) == float.fromhex("0x1.45f306p-1")
    # exact multiples of pi/2 pin the quadrant logic and the reduction constants
    a = np.array([0.0, float(mp.pi), float(2 * mp.pi), float(mp.pi / 2), float(3 * mp.pi / 2)], dtype=np.float32)
    got = O.cos_f32(a).astype(np.float64)
    want = np.array([float(mp.cos(mp.mpf(float(v)))) for v in a])
    assert np.allclose(got, want, atol=2e-7)
    assert got[0] == 1.0


def test_cos_f32_within_2ulp_of_fp64_cos():
    rng = np.random.default_rng(11)
    a = np.concatenate([rng.uniform(-128, 128, 4_000_000), rng.uniform(0, 103, 4_000_000),
                        np.linspace(-128, 128, 2_000_001)]).astype(np.float32)
    got = O.cos_f32(a).astype(np.float64)
    ref = np.cos(a.astype(np.float64))
    ulp = np.spacing(np.abs(ref).astype(np.float32)).astype(np.float64)
    err = np.abs(got - ref) / ulp
    assert err.max() <= 2.0, err.max()
    assert np.all(np.abs(got) <= 1.0)


def test_cos_f32_taylor_coefficients_are_rounded_factorials():
    """The polynomial coefficients typed into the oracle are rnd32(+-1/k!): check through cos_f32 on
    small arguments where the reduction is the identity (q=0) against mpmath evaluation of the same
    truncated series in high precision (bounds a mistyped coefficient)."""
    mp.mp.dps = 40
    a = np.linspace(-0.78, 0.78, 20001).astype(np.float32)
    got = O.cos_f32(a).astype(np.float64)
    ref = np.array([float(mp.cos(mp.mpf(float(v)))) for v in a[::50]])
    assert np.max(np.abs(got[::50] - ref)) <= 1.2e-7


# ------------------------------------------------------------------------------------------------ P6
def test_estimator_exact_rational_tiny_n():
    """S4-S6 with n=8 events: S1, S2, H recomputed exactly (fractions) from the dumped J and f."""
    for wl in (W.cfg1(), W.cfg5(), W.toy(3), W.cfg4(dim=4)):
        o = O.Oracle(wl.dim, wl.nbins, wl.integrand_id, wl.params, wl.precision)
        n = 8
        ev = o.events(0, n, 42)
        I, sig, h = o.iterate(n, 42)
        wf = [float(j) * float(f) for j, f in zip(ev["jac"], ev["f"])]           # one fp64 multiply (S4)
        assert wf == [float(v) for v in ev["wf"]]
        q = [v * v for v in wf]
        S1 = Fr(0); S2 = Fr(0)
        for a, b in zip(wf, q):
            S1 += Fr(a); S2 += Fr(b)
        S1f, S2f = float(S1), float(S2)
        assert o.last_sums() == (S1f, S2f)
        Iw = S1f / n
        V = (S2f / n - Iw * Iw) / (n - 1)
        assert I == Iw and sig == math.sqrt(max(V, 0.0))
        H = [[Fr(0)] * wl.nbins for _ in range(wl.dim)]
        for e in range(n):
            for k in range(wl.dim):
                H[k][int(ev["bins"][e][k])] += Fr(q[e])
        for k in range(wl.dim):
            for i in range(wl.nbins):
                assert h[k][i] == float(H[k][i])
        assert o.iteration == 1


def test_threaded_ranges_equal_single_thread():
    wl = W.cfg5()
    a = O.Oracle(wl.dim, wl.nbins, wl.integrand_id, wl.params)
    b = O.Oracle(wl.dim, wl.nbins, wl.integrand_id, wl.params)
    Ia, sa, ha = a.iterate(200_000, 3)
    Ib, sb, hb = b.iterate(200_000, 3, threads=4)
    assert Ia == pytest.approx(Ib, rel=1e-15) and sa == pytest.approx(sb, rel=1e-14)
    assert np.allclose(ha, hb, rtol=1e-15, atol=0)
    assert 0.40 < b.npass / 200_000 < 0.50        # ~45 % of events pass the cuts on the uniform grid


def test_compensated_sum_beats_naive_on_cancelling_stream():
    """S5 asks for the real-number sum: the oracle's S1 must match math.fsum of the dumped wf."""
    wl = W.cfg4(dim=20)
    o = O.Oracle(wl.dim, wl.nbins, wl.integrand_id, wl.params, wl.precision)
    n = 50_000
    ev = o.events(0, n, 0)
    I, sig, h = o.iterate(n, 0)
    S1, S2 = o.last_sums()
    assert S1 == pytest.approx(math.fsum(ev["wf"]), rel=1e-15)
    assert S2 == pytest.approx(math.fsum(ev["wf"] ** 2), rel=1e-15)
