"""The C oracle under AddressSanitizer + UndefinedBehaviorSanitizer (the CPU half of the sanitizer
evidence; compute-sanitizer is not available on the GPU pool).

`oracle/sg_oracle.c` is compiled, unchanged, together with a small driver into an instrumented executable
(-fsanitize=address,undefined, no recovery: the first finding aborts with a non-zero exit code) and run on a dense case,
a case with a truncated l3max, the degenerate lmax = 0 case, the spin-1 sums and one 3j family.  The values it prints
must be those of the ordinary build, so the run that is clean is a run of the same arithmetic.
"""
import os
import shutil
import subprocess

import numpy as np
import pytest

import oracle

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

DRIVER = r"""
#include <stdio.h>
#include <stdlib.h>
int oracle_3j_family(int j2, int j3, int m2, int m3, double *out, int *jmin_out, int *jmax_out);
int oracle_coupling_pairs(int l3max, const double *Wtt, const double *Wtp, const double *Wpp, long npairs,
                          const int *l1s, const int *l2s, double *TT, double *TE, double *EE, double *EB);
int oracle_coupling_spin1_pairs(int l3max, const double *W01, const double *W11, long npairs, const int *l1s,
                                const int *l2s, double *K01, double *K11p, double *K11m);

static int run(int lmax, int l3max)
{
    long n = (long)(lmax + 1) * (lmax + 1), q = 0;
    double *W = malloc(sizeof(double) * 3 * (size_t)(l3max + 1));
    int *l1 = malloc(sizeof(int) * (size_t)n), *l2 = malloc(sizeof(int) * (size_t)n);
    double *o = malloc(sizeof(double) * 7 * (size_t)n);
    if (!W || !l1 || !l2 || !o) return 10;
    for (int k = 0; k < 3; ++k)
        for (int l = 0; l <= l3max; ++l) W[k * (l3max + 1) + l] = ((l * 7 + k * 3) % 11 - 5) / (1.0 + l);   /* signed */
    for (int a = 0; a <= lmax; ++a)
        for (int b = 0; b <= lmax; ++b) { l1[q] = a; l2[q] = b; ++q; }
    if (oracle_coupling_pairs(l3max, W, W + (l3max + 1), W + 2 * (l3max + 1), n, l1, l2, o, o + n, o + 2 * n, o + 3 * n)) return 11;
    if (oracle_coupling_spin1_pairs(l3max, W + (l3max + 1), W + 2 * (l3max + 1), n, l1, l2, o + 4 * n, o + 5 * n, o + 6 * n)) return 12;
    /* partial requests: NULL outputs with NULL windows */
    if (oracle_coupling_pairs(l3max, W, NULL, NULL, n, l1, l2, o, NULL, NULL, NULL)) return 13;
    for (int k = 0; k < 7; ++k) {
        double s = 0.0, sa = 0.0;
        for (long i = 0; i < n; ++i) { s += o[k * n + i] * (1.0 + (double)(i % 5)); sa += o[k * n + i] < 0 ? -o[k * n + i] : o[k * n + i]; }
        printf("%d %d %d %.17g %.17g\n", lmax, l3max, k, s, sa);
    }
    free(W); free(l1); free(l2); free(o);
    return 0;
}

int main(void)
{
    int rc;
    if ((rc = run(40, 80))) return rc;      /* dense */
    if ((rc = run(37, 23))) return rc;      /* truncated l3max */
    if ((rc = run(0, 0))) return rc;        /* degenerate */
    if ((rc = run(1, 2))) return rc;
    double fam[64];
    int jmin, jmax;
    if (oracle_3j_family(20, 17, 2, -2, fam, &jmin, &jmax)) return 20;
    printf("fam %d %d %.17g %.17g\n", jmin, jmax, fam[0], fam[jmax - jmin]);
    return 0;
}
"""


def _expected_lines():
    out = []
    for lmax, l3max in ((40, 80), (37, 23), (0, 0), (1, 2)):
        W = np.array([[((l * 7 + k * 3) % 11 - 5) / (1.0 + l) for l in range(l3max + 1)] for k in range(3)])
        l1, l2 = (a.ravel().astype(np.int32) for a in np.indices((lmax + 1, lmax + 1)))
        K = oracle.coupling_pairs(l3max, W[0], W[1], W[2], l1, l2)
        S = oracle.spin1_pairs(l3max, W[1], W[2], l1, l2)
        wgt = 1.0 + (np.arange(l1.size) % 5)
        for k, v in enumerate((K["TT"], K["TE"], K["EE"], K["EB"], S["K01"], S["K11p"], S["K11m"])):
            out.append((lmax, l3max, k, float(np.sum(v * wgt)), float(np.sum(np.abs(v)))))
    return out


def test_oracle_is_clean_under_asan_and_ubsan(tmp_path):
    if shutil.which("gcc") is None:
        pytest.skip("no gcc")
    drv = tmp_path / "driver.c"
    drv.write_text(DRIVER)
    exe = tmp_path / "oracle_san"
    cmd = ["gcc", "-std=c11", "-O1", "-g", "-fopenmp", "-fsanitize=address,undefined", "-fno-sanitize-recover=all",
           "-fno-omit-frame-pointer", "-Wall", "-Wextra", str(drv), os.path.join(ROOT, "oracle", "sg_oracle.c"),
           "-o", str(exe), "-lm"]
    b = subprocess.run(cmd, capture_output=True, text=True)
    if b.returncode != 0 and ("asan" in b.stderr.lower() or "ubsan" in b.stderr.lower() or "sanitize" in b.stderr.lower()):
        pytest.skip("sanitizer runtime not installed: " + b.stderr.strip().splitlines()[-1])
    assert b.returncode == 0, b.stderr
    env = dict(os.environ, OMP_NUM_THREADS="4", ASAN_OPTIONS="detect_leaks=1:abort_on_error=0", UBSAN_OPTIONS="print_stacktrace=1")
    p = subprocess.run([str(exe)], capture_output=True, text=True, env=env, timeout=600)
    assert p.returncode == 0, (p.returncode, p.stderr[-3000:])
    assert "runtime error" not in p.stderr and "AddressSanitizer" not in p.stderr and "LeakSanitizer" not in p.stderr, p.stderr[-3000:]
    lines = [ln.split() for ln in p.stdout.strip().splitlines()]
    got = [(int(a), int(b_), int(c), float(d), float(e)) for a, b_, c, d, e in (ln for ln in lines if ln[0] != "fam")]
    want = _expected_lines()
    assert len(got) == len(want) == 28
    for g, w in zip(got, want):
        assert g[:3] == w[:3]
        # same arithmetic at another optimisation level; the sums here are taken in a different order than numpy's
        assert abs(g[3] - w[3]) <= 1e-12 * max(w[4] * 5.0, 1e-300), (g, w)
        assert abs(g[4] - w[4]) <= 1e-12 * max(w[4], 1e-300), (g, w)
    fam = [ln for ln in lines if ln[0] == "fam"][0]
    jmin, vals = oracle.three_j_family(20, 17, 2, -2)
    assert (int(fam[1]), int(fam[2])) == (jmin, jmin + vals.size - 1) == (3, 37)
    assert float(fam[3]) == vals[0] and float(fam[4]) == vals[-1]
