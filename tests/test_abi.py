"""Host-side checks of the boundary that need no GPU: the C-ABI library builds, loads and exports every
function include/vegas_b200.h declares; the ctypes binding covers each of them; argument validation that
happens before any device work; and the product path fails loudly (no CPU fallback) without a CUDA device.
"""
import ctypes as C
import os
import re
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_functions():
    text = open(os.path.join(ROOT, "include", "vegas_b200.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)           # drop comments
    return sorted(set(re.findall(r"\b(vegas_[a-z0-9_]+)\s*\(", text)))


def test_header_declares_the_north_star_calls():
    names = declared_functions()
    for must in ("vegas_create", "vegas_iterate", "vegas_refine", "vegas_destroy", "vegas_last_error"):
        assert must in names
    assert len(names) >= 20


def test_library_exports_every_declared_symbol_and_binding_covers_it():
    from paper_2010_09341_b200 import build, vegas
    path = build.build()
    raw = C.CDLL(path)
    for name in declared_functions():
        assert hasattr(raw, name), "libvegas_b200.so does not export %s" % name
        assert name in vegas.SIGNATURES, "binding lacks %s" % name
    assert sorted(vegas.SIGNATURES) == declared_functions()
    vegas.lib()                                                  # resolves every symbol with its signature


def test_library_is_sm100a_only_and_has_no_oracle_symbols():
    from paper_2010_09341_b200 import build
    path = build.build()
    out = subprocess.run(["cuobjdump", "-lelf", path], capture_output=True, text=True).stdout
    assert "sm_100a" in out and not re.search(r"sm_(?!100a)\d+", out)
    syms = subprocess.run(["nm", "-D", "--defined-only", path], capture_output=True, text=True).stdout
    assert "oracle_" not in syms


def test_workspace_bytes_and_ranges():
    from paper_2010_09341_b200 import vegas
    assert vegas.workspace_bytes(8, 50) > 8 * 50 * 8 * 3
    assert vegas.workspace_bytes(0, 50) == 0 and vegas.workspace_bytes(33, 50) == 0
    assert vegas.workspace_bytes(4, 1) == 0 and vegas.workspace_bytes(4, 4096) == 0
    assert vegas.workspace_bytes(20, 100) % 256 == 0


def _no_gpu():
    import torch
    return not torch.cuda.is_available()


def test_argument_errors_before_device_work():
    from paper_2010_09341_b200 import vegas
    L = vegas.lib()
    h = C.c_void_p()
    p = (C.c_double * 3)(0.1, 1 / 3, 2 / 3)
    fake = C.c_void_p(256)
    # ranges and parameter counts are checked before the device is touched
    assert L.vegas_create(C.byref(h), 0, 50, 1, p, 3, 0, fake, 1 << 20, None) == vegas.EINVAL
    assert L.vegas_create(C.byref(h), 8, 5000, 1, p, 3, 0, fake, 1 << 20, None) == vegas.EINVAL
    assert L.vegas_create(C.byref(h), 8, 600, 4, None, 0, 1, fake, 1 << 20, None) == vegas.EINVAL   # fp32: N < 512
    assert L.vegas_create(C.byref(h), 8, 50, 1, p, 2, 0, fake, 1 << 20, None) == vegas.EINVAL
    assert L.vegas_create(C.byref(h), 8, 50, 99, p, 3, 0, fake, 1 << 20, None) == vegas.EUNSUPPORTED
    assert L.vegas_create(C.byref(h), 4, 50, 3, p, 3, 0, fake, 1 << 20, None) in (vegas.EINVAL, vegas.EUNSUPPORTED)
    assert L.vegas_create(C.byref(h), 8, 50, 1, p, 3, 0, C.c_void_p(260), 1 << 20, None) == vegas.EINVAL  # alignment
    assert L.vegas_create(C.byref(h), 8, 50, 1, p, 3, 0, fake, 16, None) == vegas.ENOMEM
    assert L.vegas_create(None, 8, 50, 1, p, 3, 0, fake, 1 << 20, None) == vegas.EINVAL
    assert L.vegas_last_error()                                   # a message was recorded
    assert L.vegas_iterate(None, 10, 10, 0, None, None, None) == vegas.EINVAL
    assert L.vegas_refine(None, 1.5) == vegas.EINVAL
    v = C.c_double()
    assert L.vegas_pipe_rate(99, None, C.byref(v)) in (vegas.EINVAL, vegas.ECUDA)
    assert L.vegas_pipe_rate(0, None, None) == vegas.EINVAL


@pytest.mark.skipif(not _no_gpu(), reason="checks the behaviour without a CUDA device")
def test_no_cpu_fallback_without_a_device():
    from paper_2010_09341_b200 import vegas, workloads
    with pytest.raises(vegas.VegasError) as ei:
        vegas.from_workload(workloads.cfg1())
    assert ei.value.code == vegas.ECUDA
    v = C.c_double()
    assert vegas.lib().vegas_pipe_rate(0, None, C.byref(v)) == vegas.ECUDA


def test_product_package_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2010_09341_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", text, flags=re.M), f
                assert "vegas_oracle" not in text and '#include "../../oracle' not in text, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            text = open(os.path.join(ROOT, "oracle", f)).read()
            assert not re.search(r"^\s*(from|import)\s+paper_2010_09341_b200\b", text, flags=re.M), f
            assert not re.search(r'#include\s+"[^"]*(csrc|vegas_b200)', text), f


def test_plan_launches_wave_model():
    """The launch geometry of many-launch iterations (host arithmetic, no GPU): the grids DESIGN.md section 7 tabulates
    for the batch-size sweep of configs[2] on 148 SMs x 768 threads, and the model's invariants."""
    from paper_2010_09341_b200 import vegas
    n = 10**8
    assert vegas.plan_launches(n, 10**4, 768, 148) == (10000, 128, 1, 3)
    assert vegas.plan_launches(n, 10**5, 768, 148) == (1000, 128, 2, 0)
    assert vegas.plan_launches(n, 10**6, 768, 148) == (100, 100, 16, 0)
    assert vegas.plan_launches(n, 10**7, 768, 148) == (10, 10, 59, 0)
    assert vegas.plan_launches(n, n, 768, 148) == (1, 1, 148, 0)
    assert vegas.plan_launches(n, 2 * n, 768, 148) == (1, 1, 148, 0)          # events_per_launch is capped at n_events
    for epl in (1, 7, 999, 12345, 10**6 + 3):
        for threads, slots in ((64, 148), (1024, 296), (256, 2048)):
            m = 10**6 + 3
            if (m + epl - 1) // epl > 2**20:
                continue
            nl, lanes, grid, extra = vegas.plan_launches(m, epl, threads, slots)
            assert nl == (m + epl - 1) // epl and 1 <= lanes <= min(nl, 128) and 1 <= grid <= slots
            assert extra >= 0 and (extra == 0 or lanes * grid < slots)
            assert lanes * (grid + 1) <= 16384                                       # slot regions of the workspace
    # the model's cost is never worse than the two extreme grids
    import math
    def cost(L, per_thread, g, slots, lanes): return math.ceil(L * g / min(slots, lanes * g)) * (3.0 + per_thread / g)
    nl, lanes, grid, _ = vegas.plan_launches(n, 10**6, 768, 148)
    assert cost(nl, 1e6 / 768, grid, 148, lanes) <= min(cost(nl, 1e6 / 768, 1, 148, lanes), cost(nl, 1e6 / 768, 148, 148, lanes))
    L = vegas.lib()
    assert L.vegas_plan_launches(0, 1, 768, 148, None, None, None, None) == vegas.EINVAL
    assert L.vegas_plan_launches(10, 0, 768, 148, None, None, None, None) == vegas.EINVAL
    assert L.vegas_plan_launches(10, 1, 16, 148, None, None, None, None) == vegas.EINVAL
    assert L.vegas_plan_launches(10**8, 1, 768, 148, None, None, None, None) == vegas.EINVAL      # 1e8 launches
    assert L.vegas_plan_launches(10, 5, 768, 148, None, None, None, None) == vegas.OK
