"""the oracle under AddressSanitizer and UndefinedBehaviorSanitizer.  oracle/vegas_oracle.c is
compiled together with a small C driver (-fsanitize=address,undefined, no recovery) and runs one iteration + refinement
of configs[0] (d = 4 Gaussian) and of configs[4] (d = 3, cuts: events are rejected) at a reduced event count, twice
each, plus the fp32 path of configs[3]; any out-of-bounds access, misaligned load, signed overflow or invalid shift
aborts the run.  The driver also prints the estimates, which must equal the normally built oracle's bit for bit
(sanitizer instrumentation does not change IEEE arithmetic at -ffp-contract=off)."""
import os
import shutil
import subprocess

import numpy as np
import pytest

from paper_2010_09341_b200 import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
N_EVENTS = 20_000

DRIVER = r"""
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>
typedef struct oracle_ctx oracle_ctx;
int oracle_create(oracle_ctx **out, int dim, int nbins, int integrand_id, const double *params, int n_params, int precision);
int oracle_iterate(oracle_ctx *c, uint64_t n_events, uint64_t seed, double *integral, double *error, double *hist);
int oracle_refine(oracle_ctx *c, double alpha);
int oracle_get_grid(const oracle_ctx *c, double *edges);
void oracle_destroy(oracle_ctx *c);
int main(int argc, char **argv)
{
    /* argv: dim nbins id precision n_events seed alpha params... */
    int dim = atoi(argv[1]), nbins = atoi(argv[2]), id = atoi(argv[3]), prec = atoi(argv[4]);
    uint64_t n = strtoull(argv[5], 0, 10), seed = strtoull(argv[6], 0, 10);
    double alpha = atof(argv[7]);
    int np = argc - 8;
    double *params = malloc(sizeof(double) * (np > 0 ? np : 1));
    for (int i = 0; i < np; ++i) params[i] = strtod(argv[8 + i], 0);
    oracle_ctx *c = 0;
    if (oracle_create(&c, dim, nbins, id, params, np, prec)) return 2;
    double *hist = malloc(sizeof(double) * dim * nbins), *edges = malloc(sizeof(double) * dim * (nbins + 1));
    for (int it = 0; it < 2; ++it) {
        double I, s;
        if (oracle_iterate(c, n, seed, &I, &s, hist)) return 3;
        if (oracle_refine(c, alpha)) return 4;
        if (oracle_get_grid(c, edges)) return 5;
        printf("%a %a %a\n", I, s, edges[dim * (nbins + 1) / 2]);
    }
    oracle_destroy(c);
    free(params); free(hist); free(edges);
    return 0;
}
"""


@pytest.fixture(scope="module")
def sanitized(tmp_path_factory):
    if shutil.which("gcc") is None:
        pytest.skip("gcc not available")
    d = tmp_path_factory.mktemp("asan")
    drv = d / "driver.c"
    drv.write_text(DRIVER)
    exe = d / "oracle_asan"
    cmd = ["gcc", "-O1", "-g", "-std=c11", "-ffp-contract=off", "-fno-fast-math", "-fsanitize=address,undefined",
           "-fno-sanitize-recover=all", "-fno-omit-frame-pointer", "-o", str(exe), str(drv),
           os.path.join(ROOT, "oracle", "vegas_oracle.c"), "-lm"]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0 and "asan" in (r.stderr or "").lower():
        pytest.skip("sanitizer runtime not installed: " + r.stderr[-300:])
    assert r.returncode == 0, r.stderr[-3000:]
    return str(exe)


@pytest.mark.parametrize("name", ["cfg1", "cfg5", "cfg4"])
def test_oracle_runs_clean_under_asan_and_ubsan(sanitized, name):
    from oracle import oracle as O
    w = W.ALL[name]()
    args = [sanitized, str(w.dim), str(w.nbins), str(w.integrand_id), str(w.precision), str(N_EVENTS), str(w.seed),
            repr(float(w.alpha))] + [float(p).hex() for p in w.params]
    r = subprocess.run(args, capture_output=True, text=True, timeout=600,
                       env=dict(os.environ, ASAN_OPTIONS="detect_leaks=1:abort_on_error=0", UBSAN_OPTIONS="print_stacktrace=1"))
    assert r.returncode == 0, (r.returncode, r.stderr[-3000:])
    assert "runtime error" not in r.stderr and "AddressSanitizer" not in r.stderr
    rows = [[float.fromhex(t) for t in ln.split()] for ln in r.stdout.splitlines()]
    assert len(rows) == 2
    o = O.Oracle(w.dim, w.nbins, w.integrand_id, w.params, w.precision)
    for I_s, s_s, e_s in rows:
        I, s, _ = o.iterate(N_EVENTS, w.seed)
        o.refine(w.alpha)
        e = o.get_grid().reshape(-1)[w.dim * (w.nbins + 1) // 2]
        assert (I, s, e) == (I_s, s_s, e_s)
