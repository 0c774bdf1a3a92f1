"""CPU-only checks of the boundary: the C-ABI library builds/loads, exports every symbol that
include/hawkes.h declares, and fails loudly (no fallback) when there is no CUDA device."""
import ctypes
import os
import re

import pytest

import paper_2103_03348_b200 as hp
from paper_2103_03348_b200 import _lib

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "hawkes.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(hawkes_[a-z0-9_]+)\s*\(", text)))


def test_header_declares_the_north_star_calls():
    syms = declared_symbols()
    for name in ("hawkes_loglik", "hawkes_grad", "hawkes_hessian", "hawkes_eval", "hawkes_create", "hawkes_destroy"):
        assert name in syms


def test_library_exports_every_declared_symbol():
    lib = hp.load()
    syms = declared_symbols()
    assert len(syms) >= 14
    for name in syms:
        assert hasattr(lib, name), f"{name} declared in include/hawkes.h but not exported"
    assert set(syms) == set(_lib.SYMBOLS), "binding and header disagree on the symbol list"


def test_library_is_in_tree_and_sm100a():
    path = hp.lib_path()
    assert os.path.dirname(path) == os.path.join(ROOT, "paper_2103_03348_b200")
    assert os.path.exists(path)


def test_strerror_and_argument_errors_without_a_device():
    lib = hp.load()
    assert lib.hawkes_strerror(0) == b"ok"
    assert b"unknown" not in lib.hawkes_strerror(-3)
    h = ctypes.c_void_p()
    assert lib.hawkes_create(ctypes.byref(h), 0, 2, 0) == hp.ERR_ARG
    assert lib.hawkes_create(ctypes.byref(h), 10, 4, 0) == hp.ERR_UNSUPPORTED
    assert lib.hawkes_launch_count(None) == 0
    # NULL context: every evaluation entry point refuses
    p = hp.Params(0.3, 10, 14, 0.7, 1, 1 / 3)
    assert lib.hawkes_loglik(None, 1, None, None, None, ctypes.byref(p), None, None) == hp.ERR_ARG
    assert lib.hawkes_eval(None, 1, None, None, None, ctypes.byref(p), 1, None, None, None, None, None, None, None) == hp.ERR_ARG


def test_no_cpu_fallback(has_cuda):
    if has_cuda:
        pytest.skip("this check is for machines without a GPU")
    with pytest.raises(hp.HawkesError):
        hp.HawkesContext(100, 2, 0)


def test_product_package_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2103_03348_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".h", ".cuh", ".inc")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text and "hawkes_ref" not in text, f


def test_build_returns_the_library_path_when_nothing_is_stale():
    """build() with an up-to-date library takes its early return (it used to raise UnboundLocalError there)."""
    from paper_2103_03348_b200 import build as b
    hp.load()                       # builds if needed
    assert b.up_to_date()
    assert b.build() == b.LIB


def test_loader_refuses_a_library_without_its_source_stamp(tmp_path, monkeypatch):
    """A .so whose .srchash is missing and that cannot be rebuilt is an ImportError (it used to load with a warning that
    no test run turns into a failure); HAWKES_B200_ALLOW_UNSTAMPED=1 is the explicit override."""
    import shutil
    import warnings
    from paper_2103_03348_b200 import build as b
    real = hp.lib_path()
    fake = str(tmp_path / "libhawkes_b200.so")
    shutil.copy(real, fake)                                   # copied without its stamp
    monkeypatch.setattr(b, "LIB", fake)
    monkeypatch.setattr(b, "nvcc", lambda: (_ for _ in ()).throw(RuntimeError("nvcc not found")))
    monkeypatch.setattr(_lib, "_lib", None)
    with pytest.raises(ImportError, match="no source stamp"):
        _lib.load()
    monkeypatch.setenv("HAWKES_B200_ALLOW_UNSTAMPED", "1")
    with warnings.catch_warnings(record=True) as w:
        warnings.simplefilter("always")
        lib = _lib.load()
    assert lib.hawkes_strerror(0) == b"ok" and any("HAWKES_B200_ALLOW_UNSTAMPED" in str(x.message) for x in w)
    monkeypatch.setattr(_lib, "_lib", None)                   # the next load() takes the real library again
