"""CPU-side checks of the boundary: the C-ABI library loads and exports every symbol include/sht.h declares
(no compute calls without a GPU), and its pure host helpers agree with the layout definition."""
import ctypes
import os
import re
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    sys.path.insert(0, ROOT)
    from paper_2208_10154_b200 import build
    path = build.build()
    return ctypes.CDLL(path)


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "sht.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(sht_[a-z0-9_]+)\s*\(", text)))


def test_every_declared_symbol_is_exported(lib):
    syms = _declared_symbols()
    assert len(syms) >= 16
    for s in syms:
        assert hasattr(lib, s), "libsht_b200.so does not export %s" % s
    from paper_2208_10154_b200 import binding
    assert sorted(binding.EXPORTED) == syms


def test_host_helpers(lib):
    lib.sht_npix.restype = ctypes.c_longlong
    lib.sht_nalm.restype = ctypes.c_longlong
    lib.sht_alm_index.restype = ctypes.c_longlong
    assert lib.sht_npix(512) == 3145728 and lib.sht_nalm(1535) == 1180416
    lmax = 7
    seen = []
    for m in range(lmax + 1):
        for l in range(m, lmax + 1):
            seen.append(lib.sht_alm_index(lmax, l, m))
    assert seen == list(range(lib.sht_nalm(lmax)))                 # m-major, dense
    assert lib.sht_alm_index(lmax, 3, 4) == -1 and lib.sht_alm_index(lmax, 8, 0) == -1
    lib.sht_status_string.restype = ctypes.c_char_p
    assert lib.sht_status_string(0) == b"ok" and lib.sht_status_string(-4) == b"CUDA error"


def test_plan_create_fails_loudly_without_gpu_or_on_bad_args(lib):
    h = ctypes.c_void_p()
    assert lib.sht_plan_create(ctypes.byref(h), 0, 5, 1, 0) == -1           # nside < 1
    assert lib.sht_plan_create(ctypes.byref(h), 4, 5, 1, 1) == -1           # spin not in {0,2}
    assert lib.sht_plan_create(ctypes.byref(h), 4, 1, 1, 2) == -1           # spin 2 needs lmax >= 2
    assert lib.sht_plan_create(None, 4, 5, 1, 0) == -5
    import torch
    if not torch.cuda.is_available():
        assert lib.sht_plan_create(ctypes.byref(h), 4, 5, 1, 0) == -4       # no CPU fallback
        assert not h.value
    assert lib.sht_plan_destroy(None) == 0


def test_no_product_import_of_oracle():
    """the product package must not import, load, link, include or execute anything under oracle/ (the word may
    appear in prose): every statement that could pull code or data in is matched by a regex"""
    import re
    pkg = os.path.join(ROOT, "paper_2208_10154_b200")
    pulls = re.compile(
        r"^\s*(from|import)\s+[\w.]*oracle"                      # python imports
        r"|(__import__|import_module)\s*\([^)]*oracle"           # dynamic imports
        r"|(CDLL|LoadLibrary|dlopen|PyDLL)\s*\([^)]*oracle"      # shared-library loads
        r"|#\s*include\s*[<\"][^>\"]*oracle"                     # C / CUDA includes
        r"|(open|fopen|exec|system|Popen|check_call|check_output|run)\s*\([^)]*oracle"   # reads / runs
        r"|liboracle|sht_oracle",                               # its artefacts by name
        re.IGNORECASE | re.MULTILINE)
    checked = 0
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".h", ".cuh", ".c", ".cpp")):
                txt = open(os.path.join(dirpath, f)).read()
                hit = pulls.search(txt)
                assert hit is None, (f, hit.group(0))
                checked += 1
    assert checked >= 10
    # the shared library links nothing but the CUDA runtime and the C/C++ runtimes
    import subprocess
    so = os.path.join(pkg, "libsht_b200.so")
    needed = subprocess.run(["objdump", "-p", so], capture_output=True, text=True).stdout
    libs = [ln.split()[1] for ln in needed.splitlines() if ln.strip().startswith("NEEDED")]
    assert libs and all(not re.search("oracle|cufft|cublas", x, re.IGNORECASE) for x in libs), libs


def test_bench_and_entry_use_the_oracle_only_where_allowed():
    """bench.py may execute oracle/ only in its cpu_baseline / --impl reference leg (one function), __graft_entry__
    only in smoke() (and build(), which compiles it)"""
    import re
    txt = open(os.path.join(ROOT, "bench.py")).read()
    lines = [i for i, ln in enumerate(txt.splitlines()) if re.search(r"^\s*(from|import)\s+[\w.]*oracle", ln)]
    assert len(lines) == 1
    body = txt.splitlines()
    start = max(i for i in range(lines[0]) if body[i].startswith("def "))
    assert body[start].startswith("def oracle_timed_sample("), body[start]
