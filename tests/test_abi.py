"""The C-ABI library loads and exports every symbol include/dbie.h declares; argument errors are
reported before any launch; without a CUDA device the compute entry points fail loudly
(DBIE_ECUDA) instead of falling back to the CPU.  No GPU needed."""
import ctypes as C
import os
import re

import numpy as np
import pytest

import paper_1306_1122_b200 as dbie
from paper_1306_1122_b200 import build as dbuild

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    dbuild.build_lib()
    return dbie.load()


def _declared_functions():
    text = open(os.path.join(ROOT, "include", "dbie.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(dbie_[a-z0-9_]+)\s*\(", text)))


def test_every_declared_symbol_is_exported(lib):
    names = _declared_functions()
    assert {"dbie_create", "dbie_eval", "dbie_solve", "dbie_destroy", "dbie_strerror"} <= set(names)
    assert len(names) >= 15
    for n in names:
        assert hasattr(lib, n), f"{n} declared in include/dbie.h but not exported"


def test_library_is_self_contained():
    """No torch types / libraries behind the ABI: the .so depends on libc (+ static cudart) only."""
    import subprocess
    out = subprocess.check_output(["ldd", dbie.LIB_PATH]).decode()
    assert "torch" not in out and "c10" not in out


def test_solve_opts_layout_and_defaults(lib):
    o = dbie.default_opts()
    assert (o.method, o.maxiter, o.n_trial, o.n_level, o.use_eq12, o.analytic) == (0, 200, 8, 10, 1, 0)
    assert (o.delta, o.cell, o.w_g, o.eps_f, o.eps_g) == (1e-3, 1.0, 1.0, 1e-3, 1e-4)
    assert (o.lam0, o.step, o.xtol, o.ftol, o.lam_max) == (0.05, 0.05, 1e-4, 1e-6, 0.4)
    with pytest.raises(TypeError):
        dbie.default_opts(nonsense=1)


def test_strerror_and_version(lib):
    assert lib.dbie_strerror(0) == b"ok"
    for s in range(1, 5):
        assert len(lib.dbie_strerror(s)) > 3
    assert b"sm_100a" in lib.dbie_version()
    assert lib.dbie_last_cuda_error(None) is not None


def test_argument_errors_before_any_launch(lib):
    h = C.c_void_p()
    a = np.zeros(4)
    p = C.c_void_p(a.ctypes.data)
    E = dbie.DBIE_EINVAL
    assert lib.dbie_create_host(None, 2, 2, 1.0, 0.0, 0.0, p, p, p, 0) == E
    assert lib.dbie_create_host(C.byref(h), 0, 2, 1.0, 0.0, 0.0, p, p, p, 0) == E
    assert lib.dbie_create_host(C.byref(h), 2, 2, 1.0, 0.0, 0.0, None, p, p, 0) == E
    assert lib.dbie_create(C.byref(h), 2, 2, -1.0, 0.0, 0.0, p, p, p, 0) == E
    assert lib.dbie_create(C.byref(h), 2, 2, float("nan"), 0.0, 0.0, p, p, p, 0) == E
    assert lib.dbie_eval(None, 1, p, p, p, p, p, None) == E
    assert lib.dbie_solve(None, 1, p, p, p, None, p, p, p, p, p, None) == E
    assert lib.dbie_probe_dfma_rate(0.0, None, None) == E
    assert lib.dbie_probe_fp64_operands(C.c_double(0.0), None) == E
    lib.dbie_destroy(None)   # no-op


def test_no_cpu_fallback_without_a_device(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    a = np.ones(4)
    with pytest.raises(dbie.DBIEError) as ei:
        dbie.DBIE(2, 2, 1.0, 0.0, 0.0, a, a, a)
    assert ei.value.status in (dbie.DBIE_ECUDA, dbie.DBIE_ENOMEM)


def test_missing_library_fails_loudly(monkeypatch):
    monkeypatch.setattr(dbie, "_lib", None)
    monkeypatch.setattr(dbie, "LIB_PATH", "/nonexistent/libdbie_b200.so")
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        dbie.load()


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_1306_1122_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text, f
                assert "dbie_oracle" not in text and "liboracle" not in text, f
    otext = open(os.path.join(ROOT, "oracle", "__init__.py")).read()
    assert "paper_1306_1122_b200" not in otext.replace("`paper_1306_1122_b200`", "")
