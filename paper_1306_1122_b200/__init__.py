"""paper_1306_1122_b200 — Python binding of libdbie_b200.so (include/dbie.h).

Argument marshalling only: every step of the hot path (boundary staging, the M x N
point-pixel interaction sums of PAPER.md Eq. 6/16, the residuals of Eq. 8/9/13/14 and the
per-point Downhill Simplex search) runs in the CUDA kernels behind the C ABI.
PyTorch supplies device memory and streams.  There is no CPU fallback: if the shared library is
missing, or there is no CUDA device, the calls raise.

    ctx = DBIE(nx, ny, h, x0, y0, bx, by, bz)         # torch CUDA tensors (or numpy -> _host)
    B = ctx.eval(x, y, z, lam)                         # (3, M) torch.float64 on the device
    out = ctx.solve(x, y, z)                           # dict: B, lam, f, g, iters, status
"""
from __future__ import annotations

import ctypes as C
import dataclasses
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libdbie_b200.so")
_lib = None

DBIE_OK, DBIE_EINVAL, DBIE_ENOMEM, DBIE_ECUDA, DBIE_ESTATE = range(5)
DBIE_WITH_FP32 = 1
DBIE_QUAD_9NODE = 2
DBIE_EVAL_REDUCED_SINCOS = 4


class DBIEError(RuntimeError):
    def __init__(self, status: int, msg: str):
        super().__init__(f"dbie status {status}: {msg}")
        self.status = status


class SolveOpts(C.Structure):
    """Mirror of dbie_solve_opts (include/dbie.h)."""
    _fields_ = [("method", C.c_int), ("delta", C.c_double), ("cell", C.c_double),
                ("w_g", C.c_double), ("eps_f", C.c_double), ("eps_g", C.c_double),
                ("lam0", C.c_double), ("step", C.c_double), ("xtol", C.c_double),
                ("ftol", C.c_double), ("maxiter", C.c_int), ("n_trial", C.c_int),
                ("n_level", C.c_int), ("lam_max", C.c_double), ("use_eq12", C.c_int),
                ("analytic", C.c_int)]


class TraceOpts(C.Structure):
    """Mirror of dbie_trace_opts (include/dbie.h)."""
    _fields_ = [("ds", C.c_double), ("max_steps", C.c_int), ("direction", C.c_int), ("current", C.c_int),
                ("fixed_lambda", C.c_int), ("lam", C.c_double * 3), ("z_min", C.c_double), ("z_max", C.c_double)]


_vp = C.c_void_p


def load() -> C.CDLL:
    """dlopen libdbie_b200.so; raises if it has not been built (python -m paper_1306_1122_b200.build)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(f"{LIB_PATH} is missing: build it with "
                           "`python -m paper_1306_1122_b200.build` (there is no CPU fallback)")
    lib = C.CDLL(LIB_PATH)
    lib.dbie_create.argtypes = [C.POINTER(_vp), C.c_int, C.c_int, C.c_double, C.c_double, C.c_double,
                                _vp, _vp, _vp, C.c_uint]
    lib.dbie_create_host.argtypes = lib.dbie_create.argtypes
    lib.dbie_destroy.argtypes = [_vp]
    lib.dbie_destroy.restype = None
    lib.dbie_eval.argtypes = [_vp, C.c_longlong, _vp, _vp, _vp, _vp, _vp, _vp]
    lib.dbie_eval_host.argtypes = [_vp, C.c_longlong, _vp, _vp, _vp, _vp, _vp]
    lib.dbie_eval_f32.argtypes = [_vp, C.c_longlong, _vp, _vp, _vp, _vp, _vp, _vp]
    lib.dbie_eval_f32_host.argtypes = [_vp, C.c_longlong, _vp, _vp, _vp, _vp, _vp]
    lib.dbie_eval_noalloc.argtypes = [_vp, C.c_longlong, _vp, _vp, _vp, _vp, _vp, _vp]
    lib.dbie_noalloc_max_points.argtypes = []
    lib.dbie_noalloc_max_points.restype = C.c_longlong
    lib.dbie_set_f32_sfu_mask.argtypes = [_vp, C.c_int]
    lib.dbie_debug_set_batch_limit.argtypes = [_vp, C.c_longlong]
    lib.dbie_solve_default_opts.argtypes = [C.POINTER(SolveOpts)]
    lib.dbie_solve_default_opts.restype = None
    lib.dbie_solve.argtypes = [_vp, C.c_longlong, _vp, _vp, _vp, C.POINTER(SolveOpts), _vp, _vp, _vp,
                               _vp, _vp, _vp]
    lib.dbie_solve_host.argtypes = [_vp, C.c_longlong, _vp, _vp, _vp, C.POINTER(SolveOpts), _vp, _vp,
                                    _vp, _vp, _vp]
    lib.dbie_residual.argtypes = [_vp, C.c_longlong, _vp, _vp, _vp, _vp, C.POINTER(SolveOpts), _vp, _vp,
                                  _vp]
    lib.dbie_trace_default_opts.argtypes = [C.POINTER(TraceOpts)]
    lib.dbie_trace_default_opts.restype = None
    lib.dbie_trace.argtypes = [_vp, C.c_longlong, _vp, _vp, _vp, C.POINTER(SolveOpts), C.POINTER(TraceOpts), _vp, _vp,
                               _vp, _vp]
    lib.dbie_last_counters.argtypes = [_vp, C.POINTER(C.c_double), C.POINTER(C.c_longlong),
                                       C.POINTER(C.c_longlong)]
    lib.dbie_profile.argtypes = [_vp, C.c_int]
    lib.dbie_last_kernel_time.argtypes = [_vp, C.POINTER(C.c_double), C.POINTER(C.c_longlong)]
    lib.dbie_last_pass_trace.argtypes = [_vp, C.c_int, C.POINTER(C.c_longlong), C.POINTER(C.c_double),
                                         C.POINTER(C.c_int)]
    lib.dbie_probe_fp64_operands.argtypes = [C.c_double, C.POINTER(C.c_double)]
    lib.dbie_probe_dfma_rate.argtypes = [C.c_double, C.POINTER(C.c_double), C.POINTER(C.c_double)]
    lib.dbie_strerror.argtypes = [C.c_int]
    lib.dbie_strerror.restype = C.c_char_p
    lib.dbie_last_cuda_error.argtypes = [_vp]
    lib.dbie_last_cuda_error.restype = C.c_char_p
    lib.dbie_version.restype = C.c_char_p
    _lib = lib
    return lib


def default_opts(**kw) -> SolveOpts:
    o = SolveOpts()
    load().dbie_solve_default_opts(C.byref(o))
    for k, v in kw.items():
        if not hasattr(o, k):
            raise TypeError(f"unknown solve option {k!r}")
        setattr(o, k, v)
    return o


def default_trace_opts(**kw) -> TraceOpts:
    """dbie_trace_default_opts, then keyword overrides; lam=(lx, ly, lz) also sets fixed_lambda = 1."""
    o = TraceOpts()
    load().dbie_trace_default_opts(C.byref(o))
    for k, v in kw.items():
        if k == "lam":
            o.lam[0], o.lam[1], o.lam[2] = (float(t) for t in v)
            o.fixed_lambda = 1
        elif not hasattr(o, k):
            raise TypeError(f"unknown trace option {k!r}")
        else:
            setattr(o, k, v)
    return o


def version() -> str:
    return load().dbie_version().decode()


def noalloc_max_points() -> int:
    """DBIE_NOALLOC_MAX_POINTS of the loaded library: the most points one eval_noalloc call takes."""
    return int(load().dbie_noalloc_max_points())


def probe_dfma_rate(millis: float = 200.0) -> tuple[float, float]:
    """Measured (DFMA/s, FFMA/s) lane-instruction rates of the device (dbie_probe_dfma_rate)."""
    d, f = C.c_double(), C.c_double()
    st = load().dbie_probe_dfma_rate(float(millis), C.byref(d), C.byref(f))
    if st != DBIE_OK:
        raise DBIEError(st, load().dbie_last_cuda_error(None).decode())
    return d.value, f.value


def probe_fp64_operands(millis: float = 100.0) -> dict:
    """Measured FP64 lane-instruction rates by operand pattern (dbie_probe_fp64_operands)."""
    r = (C.c_double * 4)()
    st = load().dbie_probe_fp64_operands(float(millis), r)
    if st != DBIE_OK:
        raise DBIEError(st, load().dbie_last_cuda_error(None).decode())
    return {"dfma_2reg_imm": r[0], "dfma_3reg": r[1], "dmul": r[2], "dfma_1reg_2reuse": r[3]}


def _torch():
    import torch
    return torch


def _dev_f64(t, n, name):
    torch = _torch()
    if not isinstance(t, torch.Tensor) or not t.is_cuda or t.dtype != torch.float64:
        raise TypeError(f"{name}: expected a CUDA float64 tensor")
    if not t.is_contiguous() or t.numel() != n:
        raise ValueError(f"{name}: expected {n} contiguous elements, got {tuple(t.shape)}")
    return _vp(t.data_ptr())


def _dev_f32(t, n, name):
    torch = _torch()
    if not isinstance(t, torch.Tensor) or not t.is_cuda or t.dtype != torch.float32:
        raise TypeError(f"{name}: expected a CUDA float32 tensor")
    if not t.is_contiguous() or t.numel() != n:
        raise ValueError(f"{name}: expected {n} contiguous elements, got {tuple(t.shape)}")
    return _vp(t.data_ptr())


def _host_f64(a, n, name):
    a = np.ascontiguousarray(a, dtype=np.float64)
    if a.size != n:
        raise ValueError(f"{name}: expected {n} elements, got {a.shape}")
    return a


def _stream_ptr(stream):
    torch = _torch()
    s = torch.cuda.current_stream() if stream is None else stream
    return _vp(s.cuda_stream)


class DBIE:
    """One boundary magnetogram staged on the device (dbie_create / dbie_destroy)."""

    def __init__(self, nx: int, ny: int, h: float, x0: float, y0: float, bx, by, bz, fp32: bool = False,
                 quad9: bool = False, reduced_sincos: bool = False):
        lib = load()
        self._lib = lib
        self._h = _vp()
        self.nx, self.ny, self.h, self.x0, self.y0 = int(nx), int(ny), float(h), float(x0), float(y0)
        self.N = self.nx * self.ny
        flags = ((DBIE_WITH_FP32 if fp32 else 0) | (DBIE_QUAD_9NODE if quad9 else 0)
                 | (DBIE_EVAL_REDUCED_SINCOS if reduced_sincos else 0))
        if isinstance(bx, np.ndarray):
            b = [_host_f64(a, self.N, n) for a, n in ((bx, "bx"), (by, "by"), (bz, "bz"))]
            st = lib.dbie_create_host(C.byref(self._h), nx, ny, h, x0, y0, *[_vp(a.ctypes.data) for a in b],
                                      flags)
        else:
            ptrs = [_dev_f64(a, self.N, n) for a, n in ((bx, "bx"), (by, "by"), (bz, "bz"))]
            st = lib.dbie_create(C.byref(self._h), nx, ny, h, x0, y0, *ptrs, flags)
        if st != DBIE_OK:
            self._h = _vp()
            raise DBIEError(st, f"{lib.dbie_strerror(st).decode()}: {lib.dbie_last_cuda_error(None).decode()}")

    @classmethod
    def from_workload(cls, wl, device=None, fp32: bool = False, reduced_sincos: bool = False) -> "DBIE":
        """Stage the boundary of a workloads.Workload (host arrays) on the current device."""
        return cls(wl.nx, wl.ny, wl.h, wl.x0, wl.y0, np.asarray(wl.bx), np.asarray(wl.by),
                   np.asarray(wl.bz), fp32=fp32, quad9=getattr(wl, "quad", 0) == 9, reduced_sincos=reduced_sincos)

    # -- lifetime
    def close(self):
        if getattr(self, "_h", None) and self._h.value:
            self._lib.dbie_destroy(self._h)
            self._h = _vp()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def _check(self, st):
        if st != DBIE_OK:
            raise DBIEError(st, f"{self._lib.dbie_strerror(st).decode()}: "
                                f"{self._lib.dbie_last_cuda_error(self._h).decode()}")

    # -- dbie_eval
    def eval(self, x, y, z, lam, out=None, stream=None):
        """B (3, M) = Eq. 6/16 at per-point per-component lambda (3, M).  Device tensors."""
        torch = _torch()
        M = x.numel()
        if out is None:
            out = torch.empty((3, M), dtype=torch.float64, device=x.device)
        self._check(self._lib.dbie_eval(self._h, M, _dev_f64(x, M, "x"), _dev_f64(y, M, "y"),
                                        _dev_f64(z, M, "z"), _dev_f64(lam, 3 * M, "lam"),
                                        _dev_f64(out, 3 * M, "out"), _stream_ptr(stream)))
        return out

    def eval_host(self, x, y, z, lam) -> np.ndarray:
        """dbie_eval_host: numpy in, numpy out; the copies are inside the call."""
        x = np.ascontiguousarray(x, dtype=np.float64)
        M = x.size
        y, z = _host_f64(y, M, "y"), _host_f64(z, M, "z")
        lam = _host_f64(lam, 3 * M, "lam")
        B = np.empty((3, M), dtype=np.float64)
        self._check(self._lib.dbie_eval_host(self._h, M, _vp(x.ctypes.data), _vp(y.ctypes.data),
                                             _vp(z.ctypes.data), _vp(lam.ctypes.data), _vp(B.ctypes.data)))
        return B

    # -- dbie_eval_noalloc
    def eval_noalloc(self, x, y, z, lam, out, stream=None):
        """dbie_eval_noalloc: dbie_eval for callers that must not allocate device memory (their own pool owns
        the GPU's memory, or cudaMalloc's device-wide synchronisation is not allowed where they run).  The
        partial sums go to a fixed 6 MiB array inside the library, so M <= noalloc_max_points() (16,384) per
        call, and `out` (3, M) must be passed in: this method creates no tensor.  Bit-identical to eval().
        Calls that may overlap on the GPU share that array and race; keep them on one stream."""
        M = x.numel()
        self._check(self._lib.dbie_eval_noalloc(self._h, M, _dev_f64(x, M, "x"), _dev_f64(y, M, "y"),
                                                _dev_f64(z, M, "z"), _dev_f64(lam, 3 * M, "lam"),
                                                _dev_f64(out, 3 * M, "out"), _stream_ptr(stream)))
        return out

    # -- dbie_eval_f32
    def eval_f32(self, x, y, z, lam, out=None, stream=None):
        """fp32-arithmetic variant: float32 device tensors in, B (3, M) float32 out."""
        torch = _torch()
        M = x.numel()
        if out is None:
            out = torch.empty((3, M), dtype=torch.float32, device=x.device)
        self._check(self._lib.dbie_eval_f32(self._h, M, _dev_f32(x, M, "x"), _dev_f32(y, M, "y"),
                                            _dev_f32(z, M, "z"), _dev_f32(lam, 3 * M, "lam"),
                                            _dev_f32(out, 3 * M, "out"), _stream_ptr(stream)))
        return out

    def eval_f32_host(self, x, y, z, lam) -> np.ndarray:
        """dbie_eval_f32_host: float32 numpy in, (3, M) float32 numpy out; the copies are inside the call."""
        x = np.ascontiguousarray(x, dtype=np.float32)
        M = x.size
        y, z = (np.ascontiguousarray(a, dtype=np.float32) for a in (y, z))
        lam = np.ascontiguousarray(lam, dtype=np.float32)
        if y.size != M or z.size != M or lam.size != 3 * M:
            raise ValueError("eval_f32_host: y, z need M elements and lam 3 M")
        B = np.empty((3, M), dtype=np.float32)
        self._check(self._lib.dbie_eval_f32_host(self._h, M, _vp(x.ctypes.data), _vp(y.ctypes.data),
                                                 _vp(z.ctypes.data), _vp(lam.ctypes.data), _vp(B.ctypes.data)))
        return B

    def set_f32_sfu_mask(self, mask: int):
        """dbie_set_f32_sfu_mask: which components take sin/cos from the SFU (0, 1, 3 or 7)."""
        self._check(self._lib.dbie_set_f32_sfu_mask(self._h, int(mask)))

    def set_batch_limit(self, points: int):
        """dbie_debug_set_batch_limit: internal batches of at most `points` points (0: defaults)."""
        self._check(self._lib.dbie_debug_set_batch_limit(self._h, int(points)))

    # -- dbie_residual
    def residual(self, x, y, z, lam, opts: SolveOpts | None = None, stream=None):
        torch = _torch()
        M = x.numel()
        out = torch.empty((9, M), dtype=torch.float64, device=x.device)
        phi = torch.empty((M,), dtype=torch.float64, device=x.device)
        o = opts if opts is not None else default_opts()
        self._check(self._lib.dbie_residual(self._h, M, _dev_f64(x, M, "x"), _dev_f64(y, M, "y"),
                                            _dev_f64(z, M, "z"), _dev_f64(lam, 3 * M, "lam"), C.byref(o),
                                            _vp(out.data_ptr()), _vp(phi.data_ptr()), _stream_ptr(stream)))
        return {"B": out[0:3], "f": out[3], "g": out[4], "J": out[5:8], "div": out[8], "phi": phi}

    # -- dbie_solve
    def solve(self, x, y, z, opts: SolveOpts | None = None, stream=None, with_current: bool = False):
        """dbie_solve.  with_current=True adds J = curl B (Eq. 14) and div B at the
        converged lambda by one more dbie_residual call with the same options."""
        torch = _torch()
        M = x.numel()
        dev = x.device
        B = torch.empty((3, M), dtype=torch.float64, device=dev)
        lam = torch.empty((3, M), dtype=torch.float64, device=dev)
        resid = torch.empty((2, M), dtype=torch.float64, device=dev)
        iters = torch.empty((M,), dtype=torch.int32, device=dev)
        status = torch.empty((M,), dtype=torch.int32, device=dev)
        o = opts if opts is not None else default_opts()
        self._check(self._lib.dbie_solve(self._h, M, _dev_f64(x, M, "x"), _dev_f64(y, M, "y"),
                                         _dev_f64(z, M, "z"), C.byref(o), _vp(B.data_ptr()),
                                         _vp(lam.data_ptr()), _vp(resid.data_ptr()), _vp(iters.data_ptr()),
                                         _vp(status.data_ptr()), _stream_ptr(stream)))
        out = {"B": B, "lam": lam, "f": resid[0], "g": resid[1], "iters": iters, "status": status}
        if with_current:
            r = self.residual(x, y, z, lam, o, stream=stream)
            out["J"], out["div"] = r["J"], r["div"]
        return out

    # -- dbie_trace
    def trace(self, x0, y0, z0, topts: TraceOpts | None = None, sopts: SolveOpts | None = None, stream=None):
        """Field lines (or current lines) through the seeds: dict path (3, S+1, L), npts (L,), status (L,)."""
        torch = _torch()
        L = x0.numel()
        t = topts if topts is not None else default_trace_opts()
        o = sopts if sopts is not None else default_opts()
        S = int(t.max_steps)
        path = torch.empty((3, S + 1, L), dtype=torch.float64, device=x0.device)
        npts = torch.empty((L,), dtype=torch.int32, device=x0.device)
        status = torch.empty((L,), dtype=torch.int32, device=x0.device)
        self._check(self._lib.dbie_trace(self._h, L, _dev_f64(x0, L, "x0"), _dev_f64(y0, L, "y0"),
                                         _dev_f64(z0, L, "z0"), C.byref(o), C.byref(t), _vp(path.data_ptr()),
                                         _vp(npts.data_ptr()), _vp(status.data_ptr()), _stream_ptr(stream)))
        return {"path": path, "npts": npts, "status": status}

    def solve_host(self, x, y, z, opts: SolveOpts | None = None):
        x = np.ascontiguousarray(x, dtype=np.float64)
        M = x.size
        y, z = _host_f64(y, M, "y"), _host_f64(z, M, "z")
        B = np.empty((3, M)); lam = np.empty((3, M)); resid = np.empty((2, M))
        iters = np.empty(M, dtype=np.int32); status = np.empty(M, dtype=np.int32)
        o = opts if opts is not None else default_opts()
        self._check(self._lib.dbie_solve_host(self._h, M, _vp(x.ctypes.data), _vp(y.ctypes.data),
                                              _vp(z.ctypes.data), C.byref(o), _vp(B.ctypes.data),
                                              _vp(lam.ctypes.data), _vp(resid.ctypes.data),
                                              _vp(iters.ctypes.data), _vp(status.ctypes.data)))
        return {"B": B, "lam": lam, "f": resid[0], "g": resid[1], "iters": iters, "status": status}

    def profile(self, enable: bool = True):
        """dbie_profile: CUDA-event pairs around every interaction-kernel launch of later calls."""
        self._check(self._lib.dbie_profile(self._h, int(bool(enable))))

    def kernel_time(self) -> dict:
        """dbie_last_kernel_time: device ms and launch count of the last call's interaction kernels."""
        a, b = C.c_double(), C.c_longlong()
        self._check(self._lib.dbie_last_kernel_time(self._h, C.byref(a), C.byref(b)))
        return {"interact_ms": a.value, "interact_launches": b.value}

    def pass_trace(self, cap: int = 4096) -> dict:
        """dbie_last_pass_trace (profile mode): active points and device ms of every pass of the last fused NM launch."""
        act = (C.c_longlong * cap)()
        ms = (C.c_double * cap)()
        n = C.c_int()
        self._check(self._lib.dbie_last_pass_trace(self._h, cap, act, ms, C.byref(n)))
        k = min(n.value, cap)
        return {"npass": n.value, "active": np.array(act[:k], dtype=np.int64), "ms": np.array(ms[:k])}

    def counters(self) -> dict:
        """dbie_last_counters: interactions, launches, objective evaluations of the last call."""
        a, b, c = C.c_double(), C.c_longlong(), C.c_longlong()
        self._check(self._lib.dbie_last_counters(self._h, C.byref(a), C.byref(b), C.byref(c)))
        return {"interactions": a.value, "launches": b.value, "objective_evals": c.value}


@dataclasses.dataclass
class DeviceWorkload:
    """Points (and lambda) of a workloads.Workload as device tensors."""
    x: object
    y: object
    z: object
    lam: object


def to_device(wl, device="cuda") -> DeviceWorkload:
    torch = _torch()
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64)).to(device)
    lam = None if wl.lam is None else t(wl.lam)
    return DeviceWorkload(t(wl.x), t(wl.y), t(wl.z), lam)
