"""ctypes binding of libvegas_b200.so -- same names as include/vegas_b200.h, argument marshalling only.

Every step of the path (S1-S7) runs in the library's CUDA kernels.  PyTorch supplies the device
workspace (``torch.empty(..., dtype=uint8, device='cuda')``) and the stream
(``torch.cuda.current_stream().cuda_stream``), nothing else.  If the library cannot be built/loaded or
there is no CUDA device, calls raise: there is no CPU fallback.
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from . import build as _build

OK, EINVAL, ECUDA, ENOMEM, ESTATE, EUNSUPPORTED, EGRID = 0, -1, -2, -3, -4, -5, -6
FP64, FP32_EVAL, FP64_U32 = 0, 1, 2
GAUSS_SYM, GAUSS_DOUBLE, GENZ_OSC_PEAK, LO_2TO2, TOY_SUM, USER, LO_2TO2_TAB = 0, 1, 2, 3, 4, 5, 6

_vp, _dp, _ip = C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_int)
_i32p, _u32p, _u64p, _szp = C.POINTER(C.c_int32), C.POINTER(C.c_uint32), C.POINTER(C.c_uint64), C.POINTER(C.c_size_t)

# name -> (restype, argtypes): every symbol include/vegas_b200.h declares
SIGNATURES = {
    "vegas_workspace_bytes": (C.c_size_t, [C.c_int, C.c_int]),
    "vegas_create": (C.c_int, [C.POINTER(_vp), C.c_int, C.c_int, C.c_int, _dp, C.c_int, C.c_int, _vp, C.c_size_t, _vp]),
    "vegas_create_custom": (C.c_int, [C.POINTER(_vp), C.c_int, C.c_int, C.c_char_p, _dp, C.c_int, C.c_int, _vp, C.c_size_t, _vp]),
    "vegas_iterate": (C.c_int, [_vp, C.c_uint64, C.c_uint64, C.c_uint64, _dp, _dp, _dp]),
    "vegas_refine": (C.c_int, [_vp, C.c_double]),
    "vegas_refine_enqueue": (C.c_int, [_vp, C.c_double]),
    "vegas_refine_collect": (C.c_int, [_vp]),
    "vegas_step_enqueue": (C.c_int, [_vp, C.c_uint64, C.c_uint64, C.c_uint64, C.c_double, _ip]),
    "vegas_iteration_kernel_ms": (C.c_int, [_vp, C.c_int, _dp]),
    "vegas_set_table": (C.c_int, [_vp, _dp, C.c_int]),
    "vegas_get_grid": (C.c_int, [_vp, _dp]),
    "vegas_set_grid": (C.c_int, [_vp, _dp]),
    "vegas_reset": (C.c_int, [_vp]),
    "vegas_set_iteration": (C.c_int, [_vp, C.c_uint32]),
    "vegas_get_iteration": (C.c_int, [_vp, _u32p]),
    "vegas_debug_events": (C.c_int, [_vp, C.c_uint64, C.c_uint32, C.c_uint64, _i32p, _dp, _dp, _dp, _dp, _i32p]),
    "vegas_last_sums": (C.c_int, [_vp, _dp, _dp, _dp]),
    "vegas_last_npass": (C.c_int, [_vp, _u64p]),
    "vegas_iterate_enqueue": (C.c_int, [_vp, C.c_uint64, C.c_uint64, C.c_uint64, _ip]),
    "vegas_iterate_collect": (C.c_int, [_vp, _dp, _dp, _dp]),
    "vegas_iterate_shard_enqueue": (C.c_int, [_vp, C.c_uint64, C.c_uint64, C.c_uint64, C.c_uint64, C.c_uint64, _ip]),
    "vegas_partials": (C.c_int, [_vp, C.POINTER(_vp), _szp]),
    "vegas_finalize_enqueue": (C.c_int, [_vp, C.c_uint64]),
    "vegas_finalize_step_enqueue": (C.c_int, [_vp, C.c_uint64, C.c_double]),
    "vegas_set_histogram": (C.c_int, [_vp, _dp]),
    "vegas_set_launch_shape": (C.c_int, [_vp, C.c_int, C.c_int]),
    "vegas_set_hist_replicas": (C.c_int, [_vp, C.c_int]),
    "vegas_get_launch_shape": (C.c_int, [_vp, _ip, _ip, _ip, _szp]),
    "vegas_device_info": (C.c_int, [_vp, _ip, _ip]),
    "vegas_pipe_rate": (C.c_int, [C.c_int, _vp, _dp]),
    "vegas_run_integration": (C.c_int, [_vp, C.c_int, C.c_int, C.c_uint64, C.c_uint64, C.c_uint64, C.c_double, _dp, _dp,
                                        _dp, _dp, _dp, _dp]),
    "vegas_tune_events_per_launch": (C.c_int, [_vp, C.c_uint64, C.c_uint64, _u64p, C.c_int, _u64p, _dp]),
    "vegas_use_cuda_graph": (C.c_int, [_vp, C.c_int]),
    "vegas_plan_launches": (C.c_int, [C.c_uint64, C.c_uint64, C.c_int, C.c_int, _ip, _ip, _ip, _ip]),
    "vegas_combine_iterations": (C.c_int, [C.c_int, _dp, _dp, _dp, _dp, _dp]),
    "vegas_refine_static_enqueue": (C.c_int, [C.c_int, C.c_int, C.c_double, _vp, _vp, _vp, _vp, _vp]),
    "vegas_destroy": (None, [_vp]),
    "vegas_last_error": (C.c_char_p, []),
}

_lib = None


def lib():
    """Load (building first if the sources are newer) libvegas_b200.so.  Raises if that fails."""
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build())
        for name, (res, args) in SIGNATURES.items():
            fn = getattr(L, name)          # AttributeError if the library does not export it
            fn.restype, fn.argtypes = res, args
        _lib = L
    return _lib


class VegasError(RuntimeError):
    def __init__(self, code, what):
        msg = lib().vegas_last_error()
        super().__init__("%s failed with status %d: %s" % (what, code, msg.decode() if msg else ""))
        self.code = code


def _chk(code, what):
    if code != OK:
        raise VegasError(code, what)


def _d(a):
    return a.ctypes.data_as(_dp)


def workspace_bytes(dim, nbins):
    return int(lib().vegas_workspace_bytes(dim, nbins))


def plan_launches(n_events, events_per_launch, threads_per_cta, cta_slots):
    """(launches, stream lanes, CTAs per launch, every how many launches one CTA more) of an iteration cut into
    launches: the library's wave model (vegas_plan_launches; host arithmetic only)."""
    nl, lanes, grid, extra = C.c_int(), C.c_int(), C.c_int(), C.c_int()
    _chk(lib().vegas_plan_launches(int(n_events), int(events_per_launch), int(threads_per_cta), int(cta_slots),
                                   C.byref(nl), C.byref(lanes), C.byref(grid), C.byref(extra)), "vegas_plan_launches")
    return nl.value, lanes.value, grid.value, extra.value


class Vegas:
    """One integrator state on the GPU: VegasFlow(n_dim, ...) + compile(integrand) of PAPER.md:L77-L78."""

    def __init__(self, dim, nbins, integrand_id, params=(), precision=FP64, stream=None, device="cuda:0", source=None):
        """integrand_id: a built-in integrand, or USER with `source` = C source of
        `VEGAS_INTEGRAND double vegas_user_integrand(const double* x, int dim, const double* params)`
        (vegas_create_custom: compiled at run time, the paper's compile(integrand))."""
        import torch  # device memory and stream only

        L = lib()
        self._h = None
        nbytes = workspace_bytes(dim, nbins)
        p = np.ascontiguousarray(np.asarray(params, dtype=np.float64))
        if nbytes == 0 or not torch.cuda.is_available():
            # let the library report the error (EINVAL ranges first, then ECUDA: no CPU fallback)
            h = _vp()
            rc = L.vegas_create(C.byref(h), dim, nbins, integrand_id, _d(p) if p.size else None, int(p.size),
                                precision, None if nbytes == 0 else _vp(256), max(nbytes, 1), None)
            raise VegasError(rc if rc != OK else ECUDA, "vegas_create")
        self._dev = torch.device(device)
        torch.cuda.set_device(self._dev)
        self._ws = torch.empty(nbytes + 256, dtype=torch.uint8, device=self._dev)
        ptr = (self._ws.data_ptr() + 255) & ~255
        self._stream = stream if stream is not None else torch.cuda.current_stream(self._dev)
        h = _vp()
        if source is not None:
            _chk(L.vegas_create_custom(C.byref(h), dim, nbins, source.encode(), _d(p) if p.size else None, int(p.size),
                                       precision, _vp(ptr), nbytes, _vp(self._stream.cuda_stream)), "vegas_create_custom")
        else:
            _chk(L.vegas_create(C.byref(h), dim, nbins, integrand_id, _d(p) if p.size else None, int(p.size), precision,
                                _vp(ptr), nbytes, _vp(self._stream.cuda_stream)), "vegas_create")
        self._h = h
        self.dim, self.nbins, self.integrand_id, self.precision = dim, nbins, integrand_id, precision

    @property
    def stream(self):
        """The torch stream every kernel of this context runs on (the one given at construction, else the stream that
        was current then).  Work that reads or writes the context's device memory -- the all-reduce of
        partials_tensor() -- must be ordered on it."""
        return self._stream

    def close(self):
        if getattr(self, "_h", None):
            lib().vegas_destroy(self._h)
            self._h = None

    __del__ = close

    # ---- the three calls of BASELINE.json north_star ------------------------------------------------
    def iterate(self, n_events, events_per_launch=0, seed=0, want_hist=True):
        n_events = int(n_events)
        epl = int(events_per_launch) if events_per_launch else n_events
        I, s = C.c_double(), C.c_double()
        h = np.empty((self.dim, self.nbins)) if want_hist else None
        _chk(lib().vegas_iterate(self._h, n_events, epl, int(seed), C.byref(I), C.byref(s),
                                 _d(h) if want_hist else None), "vegas_iterate")
        return I.value, s.value, h

    def refine(self, alpha):
        _chk(lib().vegas_refine(self._h, float(alpha)), "vegas_refine")

    def run_integration(self, n_iter, n_events, events_per_launch=0, seed=0, alpha=1.5, n_warmup=0):
        """PAPER.md:L79 run_integration: returns (mean, error, chi2_dof, per-iteration dict).  kernel_ms[i] is the
        device time of iteration i: with CUDA-graph replay (the default) from the end of iteration i-1 (the start of
        the run for i = 0) to the end of iteration i, refinement i-1 included (device time stamps); with
        use_cuda_graph(False) the CUDA-event time of iteration i's kernels alone."""
        n_events = int(n_events)
        epl = int(events_per_launch) if events_per_launch else n_events
        tot = n_iter + n_warmup
        m, e, c2 = C.c_double(), C.c_double(), C.c_double()
        I, s, ms = np.empty(tot), np.empty(tot), np.empty(tot)
        _chk(lib().vegas_run_integration(self._h, int(n_iter), int(n_warmup), n_events, epl, int(seed), float(alpha),
                                         C.byref(m), C.byref(e), C.byref(c2), _d(I), _d(s), _d(ms)),
             "vegas_run_integration")
        return m.value, e.value, c2.value, dict(integral=I, error=s, kernel_ms=ms)

    def use_cuda_graph(self, enable=True):
        _chk(lib().vegas_use_cuda_graph(self._h, 1 if enable else 0), "vegas_use_cuda_graph")

    def tune_events_per_launch(self, n_events, candidates, seed=0):
        """The batch-size study of PAPER.md:L57-L65 on this GPU: (best candidate, {candidate: ms})."""
        cand = (C.c_uint64 * len(candidates))(*[int(v) for v in candidates])
        best = C.c_uint64()
        ms = np.empty(len(candidates))
        _chk(lib().vegas_tune_events_per_launch(self._h, int(n_events), int(seed), cand, len(candidates),
                                                C.byref(best), _d(ms)), "vegas_tune_events_per_launch")
        return int(best.value), {int(k): float(v) for k, v in zip(candidates, ms)}

    # ---- asynchronous form (timing) ------------------------------------------------------------------
    def iterate_enqueue(self, n_events, events_per_launch=0, seed=0):
        n_events = int(n_events)
        epl = int(events_per_launch) if events_per_launch else n_events
        nl = C.c_int()
        _chk(lib().vegas_iterate_enqueue(self._h, n_events, epl, int(seed), C.byref(nl)), "vegas_iterate_enqueue")
        return nl.value

    def step_enqueue(self, n_events, events_per_launch=0, seed=0, alpha=1.5):
        """One fused step (iteration + refinement in the same kernels); returns the number of kernels launched."""
        n_events = int(n_events)
        epl = int(events_per_launch) if events_per_launch else n_events
        nl = C.c_int()
        _chk(lib().vegas_step_enqueue(self._h, n_events, epl, int(seed), float(alpha), C.byref(nl)), "vegas_step_enqueue")
        return nl.value

    def refine_enqueue(self, alpha):
        _chk(lib().vegas_refine_enqueue(self._h, float(alpha)), "vegas_refine_enqueue")

    def refine_collect(self):
        _chk(lib().vegas_refine_collect(self._h), "vegas_refine_collect")

    def iteration_kernel_ms(self, back=0):
        v = C.c_double()
        _chk(lib().vegas_iteration_kernel_ms(self._h, int(back), C.byref(v)), "vegas_iteration_kernel_ms")
        return v.value

    def iterate_collect(self, want_hist=True):
        I, s = C.c_double(), C.c_double()
        h = np.empty((self.dim, self.nbins)) if want_hist else None
        _chk(lib().vegas_iterate_collect(self._h, C.byref(I), C.byref(s), _d(h) if want_hist else None),
             "vegas_iterate_collect")
        return I.value, s.value, h

    # ---- NEXT-2: one shard of an iteration, the partials region, S6 after the all-reduce --------------
    def iterate_shard_enqueue(self, n_total, first, count, events_per_launch=0, seed=0):
        epl = int(events_per_launch) if events_per_launch else max(int(count), 1)
        nl = C.c_int()
        _chk(lib().vegas_iterate_shard_enqueue(self._h, int(n_total), int(first), int(count), epl, int(seed),
                                               C.byref(nl)), "vegas_iterate_shard_enqueue")
        return nl.value

    def partials(self):
        """(device pointer, number of doubles) of {S1.hi, S1.lo, S2.hi, S2.lo, npass, 0, 0, 0, H[dim][nbins]}."""
        ptr, n = _vp(), C.c_size_t()
        _chk(lib().vegas_partials(self._h, C.byref(ptr), C.byref(n)), "vegas_partials")
        return int(ptr.value), int(n.value)

    def partials_tensor(self):
        """The partials region as a float64 torch tensor sharing the workspace's memory (for all_reduce)."""
        import torch
        ptr, n = self.partials()
        off = ptr - self._ws.data_ptr()
        return self._ws[off:off + 8 * n].view(torch.float64)

    def finalize_enqueue(self, n_total):
        _chk(lib().vegas_finalize_enqueue(self._h, int(n_total)), "vegas_finalize_enqueue")

    def finalize_step_enqueue(self, n_total, alpha):
        """S6 from the summed partials and the refinement, one kernel (the tail of a sharded step)."""
        _chk(lib().vegas_finalize_step_enqueue(self._h, int(n_total), float(alpha)), "vegas_finalize_step_enqueue")

    def set_histogram(self, hist):
        h = np.ascontiguousarray(hist, dtype=np.float64)
        assert h.shape == (self.dim, self.nbins)
        _chk(lib().vegas_set_histogram(self._h, _d(h)), "vegas_set_histogram")

    # ---- state ---------------------------------------------------------------------------------------
    def get_grid(self):
        e = np.empty((self.dim, self.nbins + 1))
        _chk(lib().vegas_get_grid(self._h, _d(e)), "vegas_get_grid")
        return e

    def set_grid(self, edges):
        e = np.ascontiguousarray(edges, dtype=np.float64)
        assert e.shape == (self.dim, self.nbins + 1)
        _chk(lib().vegas_set_grid(self._h, _d(e)), "vegas_set_grid")

    def set_table(self, values):
        v = np.ascontiguousarray(values, dtype=np.float64)
        _chk(lib().vegas_set_table(self._h, _d(v), int(v.size)), "vegas_set_table")

    def reset(self):
        _chk(lib().vegas_reset(self._h), "vegas_reset")

    def set_iteration(self, it):
        _chk(lib().vegas_set_iteration(self._h, int(it)), "vegas_set_iteration")

    @property
    def iteration(self):
        v = C.c_uint32()
        _chk(lib().vegas_get_iteration(self._h, C.byref(v)), "vegas_get_iteration")
        return v.value

    def debug_events(self, first, count, seed=0):
        d = self.dim
        bins = np.empty((count, d), dtype=np.int32)
        x = np.empty((count, d)); jac = np.empty(count); f = np.empty(count); wf = np.empty(count)
        ps = np.empty(count, dtype=np.int32)
        _chk(lib().vegas_debug_events(self._h, int(first), int(count), int(seed), bins.ctypes.data_as(_i32p), _d(x),
                                      _d(jac), _d(f), _d(wf), ps.ctypes.data_as(_i32p)), "vegas_debug_events")
        return dict(bins=bins, x=x, jac=jac, f=f, wf=wf, passed=ps)

    def last_sums(self):
        a, b, ms = C.c_double(), C.c_double(), C.c_double()
        _chk(lib().vegas_last_sums(self._h, C.byref(a), C.byref(b), C.byref(ms)), "vegas_last_sums")
        return a.value, b.value, ms.value

    def last_npass(self):
        v = C.c_uint64()
        _chk(lib().vegas_last_npass(self._h, C.byref(v)), "vegas_last_npass")
        return v.value

    def set_launch_shape(self, ctas_per_sm=0, threads_per_cta=0):
        _chk(lib().vegas_set_launch_shape(self._h, ctas_per_sm, threads_per_cta), "vegas_set_launch_shape")

    def set_hist_replicas(self, replicas=0):
        _chk(lib().vegas_set_hist_replicas(self._h, replicas), "vegas_set_hist_replicas")

    def launch_shape(self):
        a, b, r, s = C.c_int(), C.c_int(), C.c_int(), C.c_size_t()
        _chk(lib().vegas_get_launch_shape(self._h, C.byref(a), C.byref(b), C.byref(r), C.byref(s)),
             "vegas_get_launch_shape")
        return dict(ctas_per_sm=a.value, threads_per_cta=b.value, hist_replicas=r.value, smem_bytes=s.value)

    def device_info(self):
        a, b = C.c_int(), C.c_int()
        _chk(lib().vegas_device_info(self._h, C.byref(a), C.byref(b)), "vegas_device_info")
        return dict(sm_count=a.value, sm_clock_khz=b.value)


PIPE_DFMA, PIPE_FFMA, PIPE_IMAD_WIDE, PIPE_LOP3, PIPE_SHARED_F64_ADD = 0, 1, 2, 3, 4
PIPE_SHARED_F64_ADD_R8, PIPE_SHARED_F64_RMW_PLAIN, PIPE_SHARED_U32_ADD = 5, 6, 7   # evidence only
PIPE_DFMA_3REG, PIPE_MIX_EVENT_LOOP = 8, 9                                            # evidence only: issue-rate bound


def pipe_rate(pipe, stream=None):
    """Measured thread-instructions/s of one SM pipe (vegas_pipe_rate): the roofline denominators."""
    v = C.c_double()
    _chk(lib().vegas_pipe_rate(int(pipe), _vp(stream.cuda_stream) if stream is not None else None, C.byref(v)),
         "vegas_pipe_rate")
    return v.value


STATIC_MAX_EDGES = 8192   # VEGAS_STATIC_MAX_EDGES


def _dev_ptr(t):
    return _vp(int(t.data_ptr()) if hasattr(t, "data_ptr") else int(t))


def refine_static_enqueue(dim, nbins, alpha, dev_edges, dev_hist, dev_new_edges, dev_status, stream=None):
    """vegas_refine_static_enqueue: the refinement for callers that cannot allocate device memory -- guests of
    another program (plug-ins, framework callbacks) that are handed device buffers while the host's pool owns the
    rest of the GPU.  No context, no workspace: the working memory is an array compiled into the library (one per
    device, shared by all calls: do not let two of these calls overlap on a device; dim*(nbins+1) <= STATIC_MAX_EDGES).
    The buffers are device memory given as torch tensors (float64 edges [dim][nbins+1] and hist [dim][nbins] in,
    float64 new edges and one int32 status out) or raw addresses.  Enqueues one kernel and returns."""
    _chk(lib().vegas_refine_static_enqueue(int(dim), int(nbins), float(alpha), _dev_ptr(dev_edges), _dev_ptr(dev_hist),
                                           _dev_ptr(dev_new_edges), _dev_ptr(dev_status),
                                           _vp(stream.cuda_stream) if stream is not None else None),
         "vegas_refine_static_enqueue")


def combine_iterations(integral, error):
    """Inverse-variance combination of iteration estimates (vegas_combine_iterations; host arithmetic, no GPU)."""
    I = np.ascontiguousarray(integral, dtype=np.float64)
    s = np.ascontiguousarray(error, dtype=np.float64)
    assert I.shape == s.shape and I.ndim == 1
    m, e, c2 = C.c_double(), C.c_double(), C.c_double()
    _chk(lib().vegas_combine_iterations(int(I.size), _d(I), _d(s), C.byref(m), C.byref(e), C.byref(c2)),
         "vegas_combine_iterations")
    return m.value, e.value, c2.value


def from_workload(w, **kw):
    """Vegas(...) for a paper_2010_09341_b200.workloads.Workload."""
    return Vegas(w.dim, w.nbins, w.integrand_id, w.params, w.precision, **kw)
