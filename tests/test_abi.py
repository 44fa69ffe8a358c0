"""The C-ABI library builds, loads and exports every symbol include/tj.h declares (no compute calls:
this runs without a GPU), and its host-side integer helpers agree with the oracle's bookkeeping."""
import ctypes
import os
import re

import numpy as np
import pytest

import oracle
from paper_2602_15605_b200 import binding, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    build.build()
    return binding.load_library()


def _header_symbols():
    src = open(os.path.join(ROOT, "include", "tj.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(tj_[a-z0-9_]+)\s*\(", src)))


def test_every_declared_symbol_is_exported(lib):
    declared = _header_symbols()
    assert declared == sorted(binding.SYMBOLS)
    for name in declared:
        assert hasattr(lib, name), name
        assert ctypes.cast(getattr(lib, name), ctypes.c_void_p).value


def test_strerror(lib):
    assert lib.tj_strerror(0) == b"ok"
    assert b"invalid" in lib.tj_strerror(-1)
    n = ctypes.c_longlong(-1)
    assert lib.tj_profile_launches(ctypes.byref(n)) == 0 and n.value >= 0
    assert lib.tj_profile_launches(None) == binding.TJ_EINVAL


def test_argument_errors_without_gpu(lib):
    # argument validation happens before any CUDA call
    h = ctypes.c_void_p()
    assert lib.tj_build_tables(-1, 0, None, ctypes.byref(h)) == binding.TJ_EINVAL
    assert lib.tj_build_tables(10, 21, None, ctypes.byref(h)) == binding.TJ_EINVAL
    assert lib.tj_build_tables(10, 20, None, None) == binding.TJ_EINVAL
    assert lib.tj_coupling_tt(None, None, 1, None, None) == binding.TJ_EINVAL
    assert lib.tj_l3_range(-1, 0, 0, 0, None, None, None) == binding.TJ_EINVAL
    assert lib.tj_l3_range(1, 1, 5, 2, None, None, None) == binding.TJ_EINVAL


def test_l3_range_matches_oracle_bookkeeping(lib):
    """Bit-exact triangle / l3-range bookkeeping (north_star): all pairs of a small case, random
    pairs at the sizes of the other configs incl. truncated l3max and the band cut."""
    rng = np.random.default_rng(7)
    cases = [(l1, l2, 512) for l1 in range(0, 257, 5) for l2 in range(0, 257, 3)]
    for lmax, l3max in ((2000, 4000), (5000, 10000), (10000, 20000), (15000, 300), (300, 17), (40, 0)):
        l1 = rng.integers(0, lmax + 1, 4000)
        l2 = rng.integers(0, lmax + 1, 4000)
        near = np.clip(l1 + rng.integers(-l3max - 3, l3max + 4, 4000), 0, lmax)
        cases += [(int(a), int(b), l3max) for a, b in zip(l1, l2)]
        cases += [(int(a), int(b), l3max) for a, b in zip(l1, near)]
    for l1, l2, l3max in cases:
        for parity in (0, 1):
            o = oracle.l3_range(l1, l2, l3max, parity)
            g = binding.l3_range(l1, l2, l3max, parity)
            assert o[2] == g[2], (l1, l2, l3max, parity, o, g)
            if o[2] > 0:
                assert o == g, (l1, l2, l3max, parity, o, g)
            else:
                assert g[0] > g[1]
        te_lo, te_hi, to_lo, to_hi = binding.sweep_counts(l1, l2, l3max)
        s = l1 + l2
        even = [s - 2 * t for t in range(te_lo, te_hi + 1)]
        odd = [s - 2 * t - 1 for t in range(to_lo, to_hi + 1)]
        lo, hi, n = oracle.l3_range(l1, l2, l3max, 0)
        assert len(even) == n and (n == 0 or (min(even), max(even)) == (lo, hi))
        lo, hi, n = oracle.l3_range(l1, l2, l3max, 1)
        assert len(odd) == n and (n == 0 or (min(odd), max(odd)) == (lo, hi))


def test_binding_fails_loudly_without_library(monkeypatch, tmp_path):
    monkeypatch.setattr(binding, "_LIB", None)
    monkeypatch.setattr(binding, "_SO", str(tmp_path / "nope.so"))
    with pytest.raises(binding.TJError):
        binding.load_library()


def test_header_is_plain_c_and_links(tmp_path):
    """include/tj.h compiles as C (no torch or C++ types at the boundary) and a C program links against libtj.so
    and calls the host-side entry points."""
    import subprocess
    src = tmp_path / "use_tj.c"
    src.write_text(
        '#include "tj.h"\n#include <stdio.h>\n'
        "int main(void) {\n"
        "  int lo, hi, n;\n"
        "  if (tj_l3_range(3, 5, 100, 0, &lo, &hi, &n) != TJ_OK) return 1;\n"
        "  if (lo != 2 || hi != 8 || n != 4) return 2;\n"
        "  if (tj_l3_range(3, 5, 100, 1, &lo, &hi, &n) != TJ_OK || lo != 3 || hi != 7 || n != 3) return 3;\n"
        "  if (tj_build_tables(-1, 0, 0, 0) != TJ_EINVAL) return 4;\n"
        '  printf("%s\\n", tj_strerror(TJ_OK));\n'
        "  return 0;\n}\n")
    exe = tmp_path / "use_tj"
    libdir = os.path.dirname(binding.library_path())
    inc = os.path.join(os.path.dirname(libdir), "include")
    subprocess.run(["gcc", "-std=c99", "-Wall", "-Werror", "-I", inc, str(src), "-o", str(exe), "-L", libdir, "-l:libtj.so",
                    "-Wl,-rpath," + libdir], check=True)
    p = subprocess.run([str(exe)], capture_output=True, text=True)
    assert p.returncode == 0 and p.stdout.strip() == "ok", (p.returncode, p.stdout, p.stderr)
