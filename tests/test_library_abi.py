"""CPU checks of the C-ABI boundary: the library builds for sm_100a, loads without a GPU, and exports
every symbol include/meb.h declares; the Python structs mirror the C structs; the product path never
touches the oracle."""
import ctypes
import os
import re
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def meb():
    import paper_2605_31425_b200 as meb
    if not os.path.exists(meb.LIB_PATH):
        meb.build()
    return meb


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "meb.h")).read()
    return sorted(set(re.findall(r"MEB_API\s+[\w\s\*]+?\b(meb_\w+)\s*\(", text)))


def test_header_symbols_are_exported(meb):
    names = _declared_symbols()
    assert len(names) >= 17 and "meb_solve" in names and "meb_screen_compact" in names
    lib = ctypes.CDLL(meb.LIB_PATH)
    for n in names:
        assert hasattr(lib, n), n
    assert sorted(meb.EXPORTS) == names
    out = subprocess.run(["nm", "-D", "--defined-only", meb.LIB_PATH], capture_output=True, text=True).stdout
    exported = sorted(l.split()[-1] for l in out.splitlines() if " T " in l and "meb_" in l)
    assert exported == names                      # nothing else leaks out of the library


def test_no_compute_calls_without_gpu_but_pure_calls_work(meb):
    lib = meb.load()
    assert lib.meb_version() == 100
    assert meb.strerror(0) == "ok" and "capacity" in meb.strerror(meb.MEB_E_CAPACITY)
    p = meb.meb_default_params()
    assert (p.rho, p.sigma0, p.kappa, p.tau, p.tol_lo, p.tol_red_factor) == (0.5, 1.0, 3.0, 1.0, 1e-2, 0.02)
    assert (p.armijo_max_halvings, p.cg_max, p.dense_d_max, p.inner_max, p.sample_rows) == (30, 500, 128, 50, 1024)
    # argument errors are reported before anything touches a device
    assert lib.meb_create(None, 0, None, 10, 10) == meb.MEB_E_ARG
    assert lib.meb_destroy(None) == meb.MEB_E_ARG


def test_struct_sizes_match_header(meb):
    src = r'''
    #include <stdio.h>
    #include "meb.h"
    int main(void) { printf("%zu %zu %d\n", sizeof(meb_params), sizeof(meb_stats), MEB_EVAL_NSCALARS); return 0; }
    '''
    import tempfile
    with tempfile.TemporaryDirectory() as td:
        cpath = os.path.join(td, "s.c")
        open(cpath, "w").write(src)
        exe = os.path.join(td, "s")
        subprocess.run(["gcc", "-I", os.path.join(ROOT, "include"), cpath, "-o", exe], check=True)
        a, b, c = subprocess.run([exe], capture_output=True, text=True).stdout.split()
    assert int(a) == ctypes.sizeof(meb.meb_params) and int(b) == ctypes.sizeof(meb.meb_stats)
    assert int(c) == meb.MEB_EVAL_NSCALARS


def test_product_never_imports_oracle():
    pkg = os.path.join(ROOT, "paper_2605_31425_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".sh")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith(".py"):
            text = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_2605_31425_b200" not in text and "from paper_2605_31425_b200" not in text, f
            assert "import ctypes" not in text and "import torch" not in text, f


def test_missing_library_fails_loudly(meb, monkeypatch):
    from paper_2605_31425_b200 import binding
    monkeypatch.setattr(binding, "_lib", None)
    monkeypatch.setattr(binding, "LIB_PATH", "/nonexistent/libmeb_b200.so")
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        binding.load()
