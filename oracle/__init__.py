"""ORACLE — TEST INFRASTRUCTURE, NOT PRODUCT CODE.

ctypes front-end of `oracle/dbie_oracle.c`, the plain CPU implementation of
the DBIE hot path written from the paper (see the header of that file for the
passage each function follows and for the pins).  Only `tests/`,
`__graft_entry__.smoke()` and `bench.py`'s cpu_baseline / `--impl reference`
legs may import this package; the product (`paper_1306_1122_b200`) never does,
and this package never imports the product.
"""
from __future__ import annotations

import ctypes as C
import dataclasses
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "dbie_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")
_lib = None

_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int)


class _Boundary(C.Structure):
    _fields_ = [("nx", C.c_int), ("ny", C.c_int), ("h", C.c_double), ("x0", C.c_double),
                ("y0", C.c_double), ("bx", _dp), ("by", _dp), ("bz", _dp), ("xs", _dp), ("ys", _dp)]


class _Opts(C.Structure):
    _fields_ = [("method", C.c_int), ("delta", C.c_double), ("cell", C.c_double),
                ("w_g", C.c_double), ("eps_f", C.c_double), ("eps_g", C.c_double),
                ("lam0", C.c_double), ("step", C.c_double), ("xtol", C.c_double),
                ("ftol", C.c_double), ("maxiter", C.c_int), ("n_trial", C.c_int),
                ("n_level", C.c_int), ("lam_max", C.c_double), ("use_eq12", C.c_int),
                ("analytic", C.c_int)]


@dataclasses.dataclass
class Opts:
    """Solver options; defaults are the DESIGN.md readings A-5..A-9, O-4."""
    method: int = 0
    delta: float = 1e-3
    cell: float = 1.0
    w_g: float = 1.0
    eps_f: float = 1e-3
    eps_g: float = 1e-4
    lam0: float = 0.05
    step: float = 0.05
    xtol: float = 1e-4
    ftol: float = 1e-6
    maxiter: int = 200
    n_trial: int = 8
    n_level: int = 10
    lam_max: float = 0.4
    use_eq12: int = 1
    analytic: int = 0     # O-5: analytic gradient instead of Eq. 13's finite differences (NM only)

    def _c(self) -> _Opts:
        return _Opts(*[getattr(self, f.name) for f in dataclasses.fields(self)])


def build(force: bool = False) -> str:
    """Compile the C oracle (gcc -O2 -ffp-contract=off -fopenmp)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(["gcc", "-O2", "-ffp-contract=off", "-fno-fast-math", "-fopenmp",
                               "-shared", "-fPIC", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.orc_max_threads.restype = C.c_int
        _lib.orc_q9_count.restype = C.c_int
        _lib.orc_q9_count.argtypes = [C.c_int]
        _lib.orc_q9_stage.restype = C.c_int
    return _lib


def max_threads() -> int:
    return int(_load().orc_max_threads())


def _d(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a, a.ctypes.data_as(_dp)


def _boundary(wl):
    """The boundary of a workload; `wl.quad == 9` selects the 9-node element quadrature (O-6):
    the nodal data are staged once into the tensor grid of weighted Gauss-point sources."""
    keep = []
    ptrs = []
    for name in ("bx", "by", "bz"):
        a, p = _d(getattr(wl, name))
        assert a.size == wl.nx * wl.ny
        keep.append(a)
        ptrs.append(p)
    nodal = _Boundary(wl.nx, wl.ny, wl.h, wl.x0, wl.y0, *ptrs, None, None)
    if getattr(wl, "quad", 0) != 9:
        return nodal, keep
    lib = _load()
    nsx, nsy = lib.orc_q9_count(wl.nx), lib.orc_q9_count(wl.ny)
    xs, ys = np.empty(nsx), np.empty(nsy)
    sv = [np.empty(nsx * nsy) for _ in range(3)]
    rc = lib.orc_q9_stage(C.byref(nodal), xs.ctypes.data_as(_dp), ys.ctypes.data_as(_dp),
                          *[a.ctypes.data_as(_dp) for a in sv])
    if rc != 0:
        raise ValueError("9-node elements need at least 3 x 3 nodes")
    keep += [xs, ys] + sv
    return _Boundary(nsx, nsy, wl.h, wl.x0, wl.y0, *[a.ctypes.data_as(_dp) for a in sv],
                     xs.ctypes.data_as(_dp), ys.ctypes.data_as(_dp)), keep


def q9_sources(wl):
    """O-6 staging alone: (xs, ys, sx, sy, sz) of the weighted Gauss-point source grid."""
    import copy
    w9 = copy.copy(wl)
    w9.quad = 9
    b, keep = _boundary(w9)
    return keep[3], keep[4], keep[5], keep[6], keep[7]


def eval(wl, x=None, y=None, z=None, lam=None, nthreads: int = 0) -> np.ndarray:
    """O-1: B[3, M] at points (x, y, z) with per-point per-component lambda[3, M]."""
    lib = _load()
    b, keep = _boundary(wl)
    x, px = _d(wl.x if x is None else x)
    y, py = _d(wl.y if y is None else y)
    z, pz = _d(wl.z if z is None else z)
    M = x.size
    lam = np.zeros((3, M)) if lam is None and wl.lam is None else (wl.lam if lam is None else lam)
    lam, pl = _d(np.asarray(lam).reshape(3, M))
    B = np.empty((3, M))
    lib.orc_eval(C.byref(b), C.c_long(M), px, py, pz, pl, B.ctypes.data_as(_dp), C.c_int(nthreads))
    return B


def residual(wl, lam, opts: Opts | None = None, x=None, y=None, z=None, nthreads: int = 0):
    """O-2: dict with B[3,M], f, g, J[3,M], div, phi at the given lambda triples."""
    lib = _load()
    o = (opts or Opts())._c()
    b, keep = _boundary(wl)
    x, px = _d(wl.x if x is None else x)
    y, py = _d(wl.y if y is None else y)
    z, pz = _d(wl.z if z is None else z)
    M = x.size
    lam, pl = _d(np.asarray(lam).reshape(3, M))
    out = np.empty((9, M))
    phi = np.empty(M)
    lib.orc_residual(C.byref(b), C.byref(o), C.c_long(M), px, py, pz, pl,
                     out.ctypes.data_as(_dp), phi.ctypes.data_as(_dp), C.c_int(nthreads))
    return {"B": out[0:3], "f": out[3], "g": out[4], "J": out[5:8], "div": out[8], "phi": phi}


def gradient(wl, lam=None, x=None, y=None, z=None, nthreads: int = 0):
    """O-5: B (3, M) and the nine dB_p/dx_j (3, 3, M) from the analytic derivative of Eq. 6."""
    lib = _load()
    b, keep = _boundary(wl)
    x, px = _d(wl.x if x is None else x)
    y, py = _d(wl.y if y is None else y)
    z, pz = _d(wl.z if z is None else z)
    M = x.size
    lam = np.ascontiguousarray(wl.lam if lam is None else lam, dtype=np.float64).reshape(3, M)
    B = np.empty((3, M)); G = np.empty((3, 3, M))
    lib.orc_gradient(C.byref(b), C.c_long(M), px, py, pz, lam.ctypes.data_as(_dp),
                     B.ctypes.data_as(_dp), G.ctypes.data_as(_dp), C.c_int(nthreads))
    return B, G


def _solve(fn_name, wl, opts, x, y, z, nthreads):
    lib = _load()
    o = (opts or Opts())._c()
    b, keep = _boundary(wl)
    x, px = _d(wl.x if x is None else x)
    y, py = _d(wl.y if y is None else y)
    z, pz = _d(wl.z if z is None else z)
    M = x.size
    B = np.empty((3, M)); lam = np.empty((3, M)); resid = np.empty((2, M))
    iters = np.empty(M, dtype=np.int32); status = np.empty(M, dtype=np.int32)
    margin = np.empty(M); phi = np.empty(M)
    nfev = np.zeros(M, dtype=np.int32)
    common = [C.byref(b), C.byref(o), C.c_long(M), px, py, pz, B.ctypes.data_as(_dp),
              lam.ctypes.data_as(_dp), resid.ctypes.data_as(_dp), iters.ctypes.data_as(_ip),
              status.ctypes.data_as(_ip), margin.ctypes.data_as(_dp)]
    if fn_name == "orc_solve_nm":
        lib.orc_solve_nm(*common, nfev.ctypes.data_as(_ip), phi.ctypes.data_as(_dp),
                         C.c_int(nthreads))
    else:
        lib.orc_solve_grid(*common, phi.ctypes.data_as(_dp), C.c_int(nthreads))
    return {"B": B, "lam": lam, "f": resid[0], "g": resid[1], "iters": iters, "status": status,
            "margin": margin, "nfev": nfev, "phi": phi}


def solve_nm(wl, opts: Opts | None = None, x=None, y=None, z=None, nthreads: int = 0):
    """O-3: per-point Nelder-Mead search on (lambda_x, lambda_y, lambda_z)."""
    return _solve("orc_solve_nm", wl, opts, x, y, z, nthreads)


def solve_grid(wl, opts: Opts | None = None, x=None, y=None, z=None, nthreads: int = 0):
    """O-4: per-point separable grid refinement (BASELINE config 5 reading)."""
    return _solve("orc_solve_grid", wl, opts, x, y, z, nthreads)


_OBJ3 = C.CFUNCTYPE(C.c_double, _dp)


def nm_generic(fn, simplex, xtol: float, ftol: float, maxiter: int):
    """The oracle's Nelder-Mead driver on a Python objective of 3 variables (pin S-1)."""
    lib = _load()

    def _cb(p):
        return float(fn(np.array([p[0], p[1], p[2]])))

    cb = _OBJ3(_cb)
    simplex, ps = _d(np.asarray(simplex).reshape(4, 3))
    trace = np.full((maxiter + 1, 3), np.nan)
    fs = np.empty((4, 3)); ff = np.empty(4)
    it = C.c_int(); nf = C.c_int(); st = C.c_int(); mg = C.c_double()
    lib.orc_nm_generic(cb, ps, C.c_double(xtol), C.c_double(ftol), C.c_int(maxiter),
                       trace.ctypes.data_as(_dp), fs.ctypes.data_as(_dp), ff.ctypes.data_as(_dp),
                       C.byref(it), C.byref(nf), C.byref(st), C.byref(mg))
    return {"trace": trace[: it.value + 1], "simplex": fs, "f": ff, "iters": it.value,
            "nfev": nf.value, "status": st.value, "margin": mg.value}
