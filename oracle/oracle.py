"""ctypes wrapper of the CPU oracle (oracle/vegas_oracle.c).

TEST INFRASTRUCTURE, NOT PRODUCT CODE.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs may import this module.  It shares nothing with the CUDA path
(paper_2010_09341_b200/): no source, no header, no table or constant generator; neither imports the other.

The arithmetic lives entirely in the C file; this wrapper only builds it with gcc, marshals numpy arrays,
and (optionally) runs disjoint event ranges of one iteration on several host threads and adds the
compensated partial sums with math.fsum (events are counter-indexed, so the
real-number sums do not depend on the split).
"""
from __future__ import annotations

import ctypes as C
import math
import os
import subprocess
import threading
from concurrent.futures import ThreadPoolExecutor

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "vegas_oracle.c")
_LIB = os.path.join(_HERE, "liboracle_vegas.so")
CFLAGS = ["-O2", "-std=c11", "-ffp-contract=off", "-fno-fast-math", "-fPIC", "-shared"]

OK, EINVAL, ENOMEM, ESTATE, EUNSUPPORTED, EGRID = 0, -1, -3, -4, -5, -6
FP64, FP32_EVAL, FP64_U32 = 0, 1, 2

_lock = threading.Lock()
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (building the checker is not using it)."""
    with _lock:
        stale = (not os.path.exists(_LIB)) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC)
        if force or stale:
            tmp = _LIB + ".tmp.%d" % os.getpid()
            subprocess.run(["gcc", *CFLAGS, "-o", tmp, _SRC, "-lm"], check=True)
            os.replace(tmp, _LIB)
    return _LIB


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        u32p, u64p, i32p = C.POINTER(C.c_uint32), C.POINTER(C.c_uint64), C.POINTER(C.c_int32)
        dp, fp, vp = C.POINTER(C.c_double), C.POINTER(C.c_float), C.c_void_p
        L.oracle_philox4x32_10.argtypes = [u32p, u32p, u32p]
        L.oracle_philox4x32_10.restype = None
        L.oracle_mantissas.argtypes = [vp, C.c_uint64, C.c_uint32, C.c_uint64, u64p]
        L.oracle_mantissas.restype = None
        L.oracle_cos_f32.argtypes = [C.c_float]
        L.oracle_cos_f32.restype = C.c_float
        L.oracle_cos_f32_batch.argtypes = [fp, fp, C.c_uint64]
        L.oracle_cos_f32_batch.restype = None
        L.oracle_create.argtypes = [C.POINTER(vp), C.c_int, C.c_int, C.c_int, dp, C.c_int, C.c_int]
        L.oracle_destroy.argtypes = [vp]
        L.oracle_destroy.restype = None
        L.oracle_reset.argtypes = [vp]
        L.oracle_set_iteration.argtypes = [vp, C.c_uint32]
        L.oracle_get_iteration.argtypes = [vp]
        L.oracle_get_iteration.restype = C.c_uint32
        L.oracle_get_grid.argtypes = [vp, dp]
        L.oracle_set_grid.argtypes = [vp, dp]
        L.oracle_events.argtypes = [vp, C.c_uint64, C.c_uint32, C.c_uint64, i32p, dp, dp, dp, dp, i32p]
        L.oracle_map_eval.argtypes = [vp, u64p, C.c_uint32, i32p, dp, dp, dp]
        L.oracle_iterate_range.argtypes = [vp, C.c_uint64, C.c_uint64, C.c_uint64, dp, dp, dp, u64p]
        L.oracle_commit.argtypes = [vp, C.c_uint64, C.c_double, C.c_double, dp, dp, dp]
        L.oracle_iterate.argtypes = [vp, C.c_uint64, C.c_uint64, dp, dp, dp]
        L.oracle_last_sums.argtypes = [vp, dp, dp]
        L.oracle_refine.argtypes = [vp, C.c_double]
        L.oracle_get_table.argtypes = [vp, dp, dp, dp]
        L.oracle_get_gauss_consts.argtypes = [vp, dp]
        L.oracle_combine.argtypes = [C.c_int, dp, dp, dp, dp, dp]
        L.oracle_set_user_integrand.argtypes = [vp, vp]
        L.oracle_set_table.argtypes = [vp, dp, C.c_int]
        L.oracle_tab_interp.argtypes = [dp, C.c_int, C.c_double]
        L.oracle_tab_interp.restype = C.c_double
        _lib = L
    return _lib


class OracleError(RuntimeError):
    def __init__(self, code, what):
        super().__init__("oracle %s failed with status %d" % (what, code))
        self.code = code


def _chk(code, what):
    if code != OK:
        raise OracleError(code, what)


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def philox4x32_10(ctr, key):
    c = (C.c_uint32 * 4)(*[int(v) & 0xFFFFFFFF for v in ctr])
    k = (C.c_uint32 * 2)(*[int(v) & 0xFFFFFFFF for v in key])
    o = (C.c_uint32 * 4)()
    lib().oracle_philox4x32_10(c, k, o)
    return [int(v) for v in o]


def cos_f32(a: np.ndarray) -> np.ndarray:
    a = np.ascontiguousarray(a, dtype=np.float32)
    out = np.empty_like(a)
    fp = C.POINTER(C.c_float)
    lib().oracle_cos_f32_batch(a.ctypes.data_as(fp), out.ctypes.data_as(fp), a.size)
    return out


class Oracle:
    """One Vegas integrator state on the CPU (grid, iteration counter, last histogram)."""

    def __init__(self, dim, nbins, integrand_id, params=(), precision=FP64):
        self._h = C.c_void_p()
        p = np.ascontiguousarray(np.asarray(params, dtype=np.float64))
        rc = lib().oracle_create(C.byref(self._h), dim, nbins, integrand_id,
                                 _dp(p) if p.size else None, int(p.size), precision)
        if rc != OK:
            self._h = None
            raise OracleError(rc, "create")
        self.dim, self.nbins, self.integrand_id, self.precision = dim, nbins, integrand_id, precision
        self.npass = None

    @classmethod
    def custom(cls, dim, nbins, c_source, params=(), precision=FP64):
        """ID_USER: compiles `c_source` (plain C defining vegas_user_integrand(x, dim, params); the prefix macro
        VEGAS_INTEGRAND expands to nothing) with gcc -O2 -ffp-contract=off and plugs it into S3."""
        import hashlib
        import tempfile
        tag = hashlib.sha1(c_source.encode()).hexdigest()[:16]
        d = os.path.join(tempfile.gettempdir(), "vegas_oracle_user")
        os.makedirs(d, exist_ok=True)
        so = os.path.join(d, "user_%s.so" % tag)
        if not os.path.exists(so):
            src = os.path.join(d, "user_%s.c" % tag)
            with open(src, "w") as f:
                f.write("#include <math.h>\n#define VEGAS_INTEGRAND\n" + c_source + "\n")
            subprocess.run(["gcc", "-O2", "-std=c11", "-ffp-contract=off", "-fno-fast-math", "-fPIC", "-shared", src,
                            "-o", so + ".tmp", "-lm"], check=True)
            os.replace(so + ".tmp", so)
        ulib = C.CDLL(so)
        self = cls(dim, nbins, 5, params, precision)
        self._user_lib = ulib                                  # keep the code mapped
        _chk(lib().oracle_set_user_integrand(self._h, C.cast(ulib.vegas_user_integrand, C.c_void_p)), "set_user")
        return self

    def close(self):
        if getattr(self, "_h", None):
            lib().oracle_destroy(self._h)
            self._h = None

    __del__ = close

    # ---- state -------------------------------------------------------------------------------
    def reset(self):
        _chk(lib().oracle_reset(self._h), "reset")

    def set_iteration(self, it):
        _chk(lib().oracle_set_iteration(self._h, it), "set_iteration")

    @property
    def iteration(self):
        return int(lib().oracle_get_iteration(self._h))

    def get_grid(self):
        e = np.empty((self.dim, self.nbins + 1), dtype=np.float64)
        _chk(lib().oracle_get_grid(self._h, _dp(e)), "get_grid")
        return e

    def set_grid(self, edges):
        e = np.ascontiguousarray(edges, dtype=np.float64)
        assert e.shape == (self.dim, self.nbins + 1)
        _chk(lib().oracle_set_grid(self._h, _dp(e)), "set_grid")

    def get_table(self):
        lo = np.empty((self.dim, self.nbins)); wd = np.empty_like(lo); g = np.empty_like(lo)
        _chk(lib().oracle_get_table(self._h, _dp(lo), _dp(wd), _dp(g)), "get_table")
        return lo, wd, g

    def gauss_consts(self):
        o = np.empty(2)
        _chk(lib().oracle_get_gauss_consts(self._h, _dp(o)), "gauss_consts")
        return float(o[0]), float(o[1])

    # ---- per-event hooks ---------------------------------------------------------------------
    def mantissas(self, seed, it, e):
        m = (C.c_uint64 * self.dim)()
        lib().oracle_mantissas(self._h, seed, it, e, m)
        return [int(v) for v in m]

    def events(self, first, count, seed):
        d = self.dim
        bins = np.empty((count, d), dtype=np.int32)
        x = np.empty((count, d)); jac = np.empty(count); f = np.empty(count); wf = np.empty(count)
        ps = np.empty(count, dtype=np.int32)
        i32p = C.POINTER(C.c_int32)
        _chk(lib().oracle_events(self._h, first, count, seed, bins.ctypes.data_as(i32p), _dp(x), _dp(jac),
                                 _dp(f), _dp(wf), ps.ctypes.data_as(i32p)), "events")
        return dict(bins=bins, x=x, jac=jac, f=f, wf=wf, passed=ps)

    def map_eval(self, m):
        m = np.ascontiguousarray(m, dtype=np.uint64)
        count = m.shape[0]
        assert m.shape == (count, self.dim)
        bins = np.empty((count, self.dim), dtype=np.int32)
        x = np.empty((count, self.dim)); jac = np.empty(count); f = np.empty(count)
        _chk(lib().oracle_map_eval(self._h, m.ctypes.data_as(C.POINTER(C.c_uint64)), count,
                                   bins.ctypes.data_as(C.POINTER(C.c_int32)), _dp(x), _dp(jac), _dp(f)),
             "map_eval")
        return dict(bins=bins, x=x, jac=jac, f=f)

    # ---- one iteration -----------------------------------------------------------------------
    def iterate_range(self, first, count, seed):
        cells = (self.dim, self.nbins)
        sums = np.empty(4); hs = np.empty(cells); hc = np.empty(cells)
        np_ = C.c_uint64(0)
        _chk(lib().oracle_iterate_range(self._h, first, count, seed, _dp(sums), _dp(hs), _dp(hc),
                                        C.byref(np_)), "iterate_range")
        return sums, hs, hc, int(np_.value)

    def iterate(self, n_events, seed, threads=1):
        """S1-S6 for one iteration.  threads=1 is the plain single-threaded C loop; threads>1 runs
        disjoint ranges concurrently and combines the compensated pieces exactly (math.fsum)."""
        n_events = int(n_events)
        if threads <= 1:
            I = C.c_double(); s = C.c_double()
            h = np.empty((self.dim, self.nbins))
            _chk(lib().oracle_iterate(self._h, n_events, seed, C.byref(I), C.byref(s), _dp(h)), "iterate")
            self.npass = None
            return I.value, s.value, h
        nchunk = min(threads * 4, max(1, n_events // 1024))
        bounds = [n_events * i // nchunk for i in range(nchunk + 1)]
        with ThreadPoolExecutor(max_workers=threads) as ex:
            parts = list(ex.map(lambda i: self.iterate_range(bounds[i], bounds[i + 1] - bounds[i], seed),
                                range(nchunk)))
        S1 = math.fsum(v for p in parts for v in (p[0][0], p[0][1]))
        S2 = math.fsum(v for p in parts for v in (p[0][2], p[0][3]))
        stack = np.stack([a for p in parts for a in (p[1], p[2])])          # (2*nchunk, d, N)
        h = np.array([[math.fsum(stack[:, k, i]) for i in range(self.nbins)] for k in range(self.dim)])
        self.npass = sum(p[3] for p in parts)
        return (*self.commit(n_events, S1, S2, h), h)

    def commit(self, n_events, S1, S2, hist):
        h = np.ascontiguousarray(hist, dtype=np.float64)
        I = C.c_double(); s = C.c_double()
        _chk(lib().oracle_commit(self._h, int(n_events), S1, S2, _dp(h), C.byref(I), C.byref(s)), "commit")
        return I.value, s.value

    def last_sums(self):
        a = C.c_double(); b = C.c_double()
        _chk(lib().oracle_last_sums(self._h, C.byref(a), C.byref(b)), "last_sums")
        return a.value, b.value

    def refine(self, alpha):
        _chk(lib().oracle_refine(self._h, float(alpha)), "refine")

    def set_table(self, values):
        """ID_LO_2TO2_TAB: the tabulated PDF G_j = g(x_j), x_j = tau^(1 - j/(M-1))."""
        v = np.ascontiguousarray(values, dtype=np.float64)
        _chk(lib().oracle_set_table(self._h, _dp(v), int(v.size)), "set_table")

    def run_integration(self, n_iter, n_events, seed, alpha, n_warmup=0, threads=1):
        """(n_warmup + n_iter) x (iterate, refine); combination of the last n_iter (oracle_combine).
        A refine rejected for a non-monotone grid (EGRID) leaves the grid unchanged and the run goes on."""
        I, s = [], []
        for _ in range(n_warmup + n_iter):
            res = self.iterate(n_events, seed, threads=threads)
            I.append(res[0]); s.append(res[1])
            try:
                self.refine(alpha)
            except OracleError as e:
                if e.code != EGRID:
                    raise
        return (*combine(I[n_warmup:], s[n_warmup:]), np.array(I), np.array(s))


def combine(integral, sigma):
    """oracle_combine: inverse-variance average, its error and chi2/dof."""
    I = np.ascontiguousarray(integral, dtype=np.float64)
    s = np.ascontiguousarray(sigma, dtype=np.float64)
    m, e, c2 = C.c_double(), C.c_double(), C.c_double()
    _chk(lib().oracle_combine(int(I.size), _dp(I), _dp(s), C.byref(m), C.byref(e), C.byref(c2)), "combine")
    return m.value, e.value, c2.value


def tab_interp(values, v):
    """The four-point Lagrange interpolation of oracle_set_table's table at v (scalar)."""
    t = np.ascontiguousarray(values, dtype=np.float64)
    return float(lib().oracle_tab_interp(_dp(t), int(t.size), float(v)))
