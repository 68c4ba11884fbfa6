"""Host logic of bench.py that needs no GPU: the table of per-event counts an ncu capture yields
(profiles/r03_kernel_counts.csv) is only used for the co-bounds while it still describes the running kernels."""
import importlib.util
import os

from paper_2010_09341_b200 import build as B, workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def load_bench():
    spec = importlib.util.spec_from_file_location("bench_under_test", os.path.join(ROOT, "bench.py"))
    m = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(m)
    return m


def test_committed_counts_match_the_committed_kernel_sources():
    """The committed table carries the hash of the committed kernel headers: a kernel edit without a new capture fails
    here (and bench.py would print bounds: null)."""
    bench = load_bench()
    shape = {"ctas_per_sm": 1, "threads_per_cta": 768, "hist_replicas": 32}
    kc, note = bench.kernel_counts("cfg2", W.cfg2(), shape)
    assert note is None and kc["src_sha"] == B.kernel_source_sha()
    assert 400 < kc["inst"] < 520 and 2.0 < kc["smem_wavefronts"] < 3.5 and kc["dram_bytes"] < 1e6
    for name in ("cfg1", "cfg4", "cfg5"):
        assert bench.kernel_counts(name)[0] is not None


def test_stale_or_foreign_counts_are_refused(tmp_path, monkeypatch):
    bench = load_bench()
    w = W.cfg2()
    shape = {"ctas_per_sm": 1, "threads_per_cta": 768, "hist_replicas": 32}
    # another launch shape than the captured instance <GaussDouble, 8, 50, RS=5, 8, 4, MAXT=768, 1>
    assert bench.kernel_counts("cfg2", w, dict(shape, hist_replicas=16))[0] is None
    assert bench.kernel_counts("cfg2", w, dict(shape, threads_per_cta=1024))[0] is None
    assert "not the running shape" in bench.kernel_counts("cfg2", w, dict(shape, hist_replicas=16))[1]
    assert bench.kernel_counts("cfg2", W.cfg4(), shape)[0] is None               # another dim / bin count
    assert bench.kernel_counts("no_such_workload")[0] is None
    # a table captured from other kernel sources
    text = open(bench.KERNEL_COUNTS_CSV).read().replace(B.kernel_source_sha(), "0123456789abcdef")
    stale = tmp_path / "stale.csv"
    stale.write_text(text)
    monkeypatch.setattr(bench, "KERNEL_COUNTS_CSV", str(stale))
    kc, note = bench.kernel_counts("cfg2", w, shape)
    assert kc is None and "recapture" in note
    monkeypatch.setattr(bench, "KERNEL_COUNTS_CSV", str(tmp_path / "missing.csv"))
    assert bench.kernel_counts("cfg2", w, shape)[0] is None
