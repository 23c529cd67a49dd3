"""Thin Python binding of include/gda.h (argument marshalling only; every step runs in the CUDA library).

Names mirror the C ABI: create_qubo_csr / create_qubo_dense / create_maxsat -> Problem;
Problem.run / run_host / grad / score / info / destroy.  PyTorch supplies device memory and streams.
The library is loaded from lib/libgda_b200.so; a missing library raises -- there is no fallback.
"""
from __future__ import annotations

import ctypes as C
from pathlib import Path
from typing import Optional

import numpy as np

import os

# GDA_B200_LIB points at another build of the same library (e.g. one compiled with different tuning macros)
_LIB_PATH = Path(os.environ.get("GDA_B200_LIB") or Path(__file__).resolve().parent / "lib" / "libgda_b200.so")
_lib = None

STATUS = {0: "GDA_OK", 1: "GDA_ERR_INVALID_ARG", 2: "GDA_ERR_ALLOC", 3: "GDA_ERR_CUDA", 4: "GDA_ERR_UNSUPPORTED"}
G_QUADRATIC, G_ENTROPY = 0, 1
DUAL_PER_VARIABLE, DUAL_SCALAR = 0, 1
DENSE_BF16 = 1
# gda_option keys of gda_set_option (per-handle launch options)
OPT_SPARSE_PATH, OPT_SPLIT_ALL_ROWS, OPT_NARROW_SPLIT, OPT_MAXSAT_NARROW, OPT_DENSE_SHAPE, OPT_GRAPHS, OPT_ROW_GROUPING = range(7)
SPARSE_PATH = {"auto": 0, "slab": 1, "stream": 2}


class GdaError(RuntimeError):
    def __init__(self, status: int, msg: str):
        super().__init__(f"{STATUS.get(status, status)}: {msg}")
        self.status = status


class Params(C.Structure):
    _fields_ = [("alpha", C.c_float), ("beta", C.c_float), ("delta", C.c_float), ("log_eps", C.c_float),
                ("iters", C.c_int32), ("eval_every", C.c_int32), ("gfun", C.c_int32), ("t0", C.c_int32),
                ("seed", C.c_uint64), ("dual", C.c_int32), ("reserved", C.c_int32)]


class Extra(C.Structure):
    _fields_ = [("x_final", C.c_void_p), ("lambda_final", C.c_void_p), ("best_obj", C.c_void_p),
                ("trace_best", C.c_void_p), ("trace_ns", C.c_void_p), ("trace_cap", C.c_int32), ("ones", C.c_void_p)]


class Info(C.Structure):
    _fields_ = [("kind", C.c_int32), ("n", C.c_int32), ("nnz", C.c_int64), ("m", C.c_int32),
                ("integral", C.c_int32), ("last_run_kernel_launches", C.c_int64),
                ("last_run_step_launches", C.c_int64)]


EXPORTS = ["gda_create_qubo_csr", "gda_create_qubo_dense", "gda_create_maxsat", "gda_create_maxkcut", "gda_destroy", "gda_run",
           "gda_run_host", "gda_grad", "gda_score", "gda_lagrangian", "gda_score_qubo_csr_static", "gda_set_option", "gda_get_info",
           "gda_last_error", "gda_version"]


def lib():
    """Load the C-ABI library (once).  Raises if it has not been built."""
    global _lib
    if _lib is None:
        if not _LIB_PATH.exists():
            raise ImportError(f"{_LIB_PATH} is missing: run `python -m paper_2509_21064_b200.build` "
                              "(there is no CPU fallback)")
        L = C.CDLL(str(_LIB_PATH))
        vp, i32, f32 = C.c_void_p, C.c_int32, C.c_float
        L.gda_create_qubo_csr.argtypes = [i32, vp, vp, vp, vp, C.POINTER(vp)]
        L.gda_create_qubo_dense.argtypes = [i32, vp, vp, i32, C.POINTER(vp)]
        L.gda_create_maxsat.argtypes = [i32, i32, vp, vp, vp, C.POINTER(vp)]
        L.gda_create_maxkcut.argtypes = [i32, i32, vp, vp, vp, C.POINTER(vp)]
        L.gda_destroy.argtypes = [vp]
        L.gda_destroy.restype = None
        L.gda_run.argtypes = [vp, i32, vp, vp, f32, C.POINTER(Params), vp, vp, vp, C.POINTER(Extra), vp]
        L.gda_run_host.argtypes = [vp, i32, vp, vp, f32, C.POINTER(Params), vp, vp, vp, vp]
        L.gda_grad.argtypes = [vp, i32, vp, vp, vp]
        L.gda_score.argtypes = [vp, i32, vp, vp, vp]
        L.gda_lagrangian.argtypes = [vp, i32, vp, vp, f32, i32, f32, vp, vp]
        L.gda_score_qubo_csr_static.argtypes = [i32, vp, vp, vp, vp, i32, vp, vp, vp]
        L.gda_set_option.argtypes = [vp, i32, i32]
        L.gda_get_info.argtypes = [vp, C.POINTER(Info)]
        L.gda_last_error.restype = C.c_char_p
        L.gda_version.restype = C.c_char_p
        for name in EXPORTS[:-2]:
            if name != "gda_destroy":
                getattr(L, name).restype = C.c_int
        _lib = L
    return _lib


def _check(status: int):
    if status != 0:
        raise GdaError(status, lib().gda_last_error().decode())


def _host(a, dt):
    return None if a is None else np.ascontiguousarray(a, dtype=dt)


def _hp(a):
    return None if a is None else a.ctypes.data


def make_params(alpha, beta, delta=1e-4, log_eps=1e-6, iters=0, eval_every=100, gfun=G_QUADRATIC, t0=0, seed=0,
                dual=DUAL_PER_VARIABLE) -> Params:
    return Params(alpha, beta, delta, log_eps, iters, eval_every, gfun, t0, seed, dual, 0)


class Problem:
    """Owns a gda_problem* handle."""

    def __init__(self, handle: int, n: int, k: int = 0):
        self._h = C.c_void_p(handle)
        self.n = n
        self.k = k          # Max-k-Cut: number of parts (x0 / x are then [k][n][B] logits); 0 otherwise

    # ---- constructors (gda_create_*) ----------------------------------------------------------
    @staticmethod
    def create_qubo_csr(n, rowptr, col, val, c=None) -> "Problem":
        rowptr, col, val, c = _host(rowptr, np.int32), _host(col, np.int32), _host(val, np.float32), _host(c, np.float32)
        h = C.c_void_p()
        _check(lib().gda_create_qubo_csr(n, _hp(rowptr), _hp(col), _hp(val), _hp(c), C.byref(h)))
        return Problem(h.value, n)

    @staticmethod
    def create_qubo_dense(n, Q, c=None, flags=DENSE_BF16) -> "Problem":
        Q, c = _host(Q, np.float32), _host(c, np.float32)
        h = C.c_void_p()
        _check(lib().gda_create_qubo_dense(n, _hp(Q), _hp(c), flags, C.byref(h)))
        return Problem(h.value, n)

    @staticmethod
    def create_maxsat(n, m, cptr, lit, w=None) -> "Problem":
        cptr, lit, w = _host(cptr, np.int32), _host(lit, np.int32), _host(w, np.float32)
        h = C.c_void_p()
        _check(lib().gda_create_maxsat(n, m, _hp(cptr), _hp(lit), _hp(w), C.byref(h)))
        return Problem(h.value, n)

    @staticmethod
    def create_maxkcut(n, k, rowptr, col, val) -> "Problem":
        rowptr, col, val = _host(rowptr, np.int32), _host(col, np.int32), _host(val, np.float32)
        h = C.c_void_p()
        _check(lib().gda_create_maxkcut(n, k, _hp(rowptr), _hp(col), _hp(val), C.byref(h)))
        return Problem(h.value, n, k)

    def set_option(self, key: int, value: int) -> "Problem":
        """gda_set_option: a launch option of THIS handle (OPT_* keys above); takes effect at the next call."""
        _check(lib().gda_set_option(self._h, key, value))
        return self

    def destroy(self):
        if self._h:
            lib().gda_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    # ---- gda_run --------------------------------------------------------------------------------
    def run(self, x0, lambda0, params: Params, *, want_final=False, trace_cap=0, want_ones=False, stream=None):
        """x0: CUDA float32 tensor [n][B]; lambda0: tensor [n][B] ([B] with params.dual = DUAL_SCALAR) or a float (y-bar).
        Returns dict of CUDA tensors: x_bin, obj, best_restart (+ x, lam, best_obj, ones, trace_best, trace_ns).
        Asynchronous on `stream` (default: torch's current stream)."""
        import torch
        assert x0.is_cuda and x0.dtype == torch.float32 and x0.is_contiguous()
        assert tuple(x0.shape[:-1]) == ((self.k, self.n) if self.k else (self.n,))
        n, B = self.n, x0.shape[-1]
        dev = x0.device
        self._last = (n, B, dev)
        l_ptr, l_scalar = None, 0.0
        if isinstance(lambda0, torch.Tensor):
            assert lambda0.is_cuda and lambda0.dtype == torch.float32 and lambda0.is_contiguous()
            assert lambda0.shape == ((B,) if params.dual == DUAL_SCALAR else (n, B))
            l_ptr = lambda0.data_ptr()
        else:
            l_scalar = float(lambda0)
        out = dict(x_bin=torch.empty((n, B), dtype=torch.uint8, device=dev),
                   obj=torch.empty(B, dtype=torch.float64, device=dev),
                   best_restart=torch.empty(1, dtype=torch.int32, device=dev))
        ex = Extra()
        if want_final:
            out["x"] = torch.empty_like(x0)                      # Max-k-Cut: the logits [k][n][B]
            out["lam"] = torch.empty((B,) if params.dual == DUAL_SCALAR else (n, B), dtype=torch.float32, device=dev)
            out["best_obj"] = torch.empty(1, dtype=torch.float64, device=dev)
            ex.x_final, ex.lambda_final, ex.best_obj = out["x"].data_ptr(), out["lam"].data_ptr(), out["best_obj"].data_ptr()
        if want_ones:
            out["ones"] = torch.empty(B, dtype=torch.int32, device=dev)
            ex.ones = out["ones"].data_ptr()
        if trace_cap > 0:
            out["trace_best"] = torch.full((trace_cap,), float("nan"), dtype=torch.float64, device=dev)
            out["trace_ns"] = torch.zeros(trace_cap, dtype=torch.int64, device=dev)
            ex.trace_best, ex.trace_ns, ex.trace_cap = out["trace_best"].data_ptr(), out["trace_ns"].data_ptr(), trace_cap
        s = torch.cuda.current_stream(dev).cuda_stream if stream is None else stream
        _check(lib().gda_run(self._h, B, x0.data_ptr(), l_ptr, l_scalar, C.byref(params), out["x_bin"].data_ptr(),
                             out["obj"].data_ptr(), out["best_restart"].data_ptr(), C.byref(ex), s))
        return out

    def resume(self, params: Params, out: dict, stream=None):
        """gda_run with x0 = NULL: continue the previous run on this handle for params.iters more steps,
        writing into the tensors of `out` (a dict returned by run())."""
        import torch
        n, B, dev = self._last
        s = torch.cuda.current_stream(dev).cuda_stream if stream is None else stream
        _check(lib().gda_run(self._h, B, None, None, 0.0, C.byref(params), out["x_bin"].data_ptr(),
                             out["obj"].data_ptr(), out["best_restart"].data_ptr(), None, s))
        return out

    def run_host(self, x0: np.ndarray, lambda0, params: Params, stream=None):
        """gda_run_host: NumPy (ideally pinned) buffers in and out; synchronous."""
        x0 = np.ascontiguousarray(x0, dtype=np.float32)
        n, B = x0.shape
        assert n == self.n
        l_arr, l_scalar = None, 0.0
        if isinstance(lambda0, np.ndarray):
            l_arr = np.ascontiguousarray(lambda0, dtype=np.float32)
        else:
            l_scalar = float(lambda0)
        x_bin = np.empty((n, B), dtype=np.uint8)
        obj = np.empty(B, dtype=np.float64)
        best = np.empty(1, dtype=np.int32)
        _check(lib().gda_run_host(self._h, B, x0.ctypes.data, _hp(l_arr), l_scalar, C.byref(params),
                                  x_bin.ctypes.data, obj.ctypes.data, best.ctypes.data, stream))
        return dict(x_bin=x_bin, obj=obj, best_restart=int(best[0]))

    def run_host_ptrs(self, B, x0_ptr, lambda0_scalar, params: Params, x_bin_ptr, obj_ptr, best_ptr, stream=None):
        """gda_run_host on raw host pointers (e.g. pinned torch tensors), no allocation on the way."""
        _check(lib().gda_run_host(self._h, B, x0_ptr, None, float(lambda0_scalar), C.byref(params),
                                  x_bin_ptr, obj_ptr, best_ptr, stream))

    # ---- gda_grad / gda_score ---------------------------------------------------------------------
    def grad(self, x, stream=None):
        """gda_grad: grad f(x) for x [n][B] (Max-k-Cut: x = the logits [k][n][B], the gradient of Tr(X W X^T) w.r.t. them)."""
        import torch
        assert x.is_cuda and x.dtype == torch.float32 and x.is_contiguous()
        assert tuple(x.shape[:-1]) == ((self.k, self.n) if self.k else (self.n,))
        G = torch.empty_like(x)
        s = torch.cuda.current_stream(x.device).cuda_stream if stream is None else stream
        _check(lib().gda_grad(self._h, x.shape[-1], x.data_ptr(), G.data_ptr(), s))
        return G

    def score(self, x, stream=None):
        """gda_score: x [n][B] (Max-k-Cut: the logits [k][n][B], scored by their argmax labels)."""
        import torch
        assert x.is_cuda and x.dtype == torch.float32 and x.is_contiguous()
        assert tuple(x.shape[:-1]) == ((self.k, self.n) if self.k else (self.n,))
        obj = torch.empty(x.shape[-1], dtype=torch.float64, device=x.device)
        s = torch.cuda.current_stream(x.device).cuda_stream if stream is None else stream
        _check(lib().gda_score(self._h, x.shape[-1], x.data_ptr(), obj.data_ptr(), s))
        return obj

    def lagrangian(self, x, lam, gfun=G_QUADRATIC, log_eps=1e-6, stream=None):
        """gda_lagrangian: L(x, y) = f(x) + sum_i y_i g(x_i) per restart; lam a CUDA tensor [n][B] or a float."""
        import torch
        assert x.is_cuda and x.dtype == torch.float32 and x.is_contiguous()
        assert tuple(x.shape[:-1]) == ((self.k, self.n) if self.k else (self.n,))      # Max-k-Cut: the logits [k][n][B]
        B = x.shape[-1]
        out = torch.empty(B, dtype=torch.float64, device=x.device)
        l_ptr, l_scalar = None, 0.0
        if isinstance(lam, torch.Tensor):
            assert lam.is_cuda and lam.dtype == torch.float32 and lam.is_contiguous() and tuple(lam.shape) == (self.n, B)
            l_ptr = lam.data_ptr()
        else:
            l_scalar = float(lam)
        s = torch.cuda.current_stream(x.device).cuda_stream if stream is None else stream
        _check(lib().gda_lagrangian(self._h, B, x.data_ptr(), l_ptr, l_scalar, gfun, log_eps, out.data_ptr(), s))
        return out

    def info(self) -> Info:
        inf = Info()
        _check(lib().gda_get_info(self._h, C.byref(inf)))
        return inf


STATIC_SCORE_MAX_B = 4096


def score_qubo_csr_static(n, rowptr, col, val, c, x, obj, stream=None):
    """gda_score_qubo_csr_static: obj[b] = F([x[:, b] > 1/2]) of the QUBO given as DEVICE CSR tensors, for callers that must
    not allocate device memory (a host process whose pool owns all of the HBM, a loop that cannot afford cudaMalloc's
    device-wide synchronisation, code restricted to the buffers it was handed).  No handle, and nothing is allocated on the
    way -- not by the library (its partial sums live in a fixed 4 MiB array inside its image) and not here: every tensor,
    the output `obj` (float64 [B]) included, is the caller's.  rowptr / col int32, val / c float32 (c may be None),
    x float32 [n][B] with B <= STATIC_SCORE_MAX_B.  One array per GPU serves all calls: calls on different streams or
    threads that overlap on the GPU race on it; calls on one stream are ordered.  The first call on a GPU does the one-time
    address look-up and should happen at start-up, outside any stream capture."""
    import torch
    for t, dt in ((rowptr, torch.int32), (col, torch.int32), (val, torch.float32), (x, torch.float32), (obj, torch.float64)):
        assert t.is_cuda and t.dtype == dt and t.is_contiguous()
    assert c is None or (c.is_cuda and c.dtype == torch.float32 and c.is_contiguous() and c.numel() == n)
    assert rowptr.numel() == n + 1 and x.dim() == 2 and x.shape[0] == n and obj.numel() == x.shape[1]
    s = torch.cuda.current_stream(x.device).cuda_stream if stream is None else stream
    _check(lib().gda_score_qubo_csr_static(n, rowptr.data_ptr(), col.data_ptr(), val.data_ptr(),
                                           None if c is None else c.data_ptr(), x.shape[1], x.data_ptr(), obj.data_ptr(), s))
    return obj


def create_from_workload(P) -> Problem:
    """Problem from a workloads.QuboCSR / QuboDense / MaxSat container."""
    from . import workloads as wl
    if isinstance(P, wl.QuboCSR):
        return Problem.create_qubo_csr(P.n, P.rowptr, P.col, P.val, P.c)
    if isinstance(P, wl.QuboDense):
        return Problem.create_qubo_dense(P.n, P.Q, P.c)
    if isinstance(P, wl.MaxSat):
        return Problem.create_maxsat(P.n, P.m, P.cptr, P.lit, P.w)
    if isinstance(P, wl.MaxKCut):
        return Problem.create_maxkcut(P.n, P.k, P.rowptr, P.col, P.val)
    raise TypeError(type(P))


def params_from_hyper(h, **over) -> Params:
    d = dict(alpha=h.alpha, beta=h.beta, delta=h.delta, log_eps=h.log_eps, iters=h.iters,
             eval_every=h.eval_every, gfun=h.gfun, t0=0, seed=h.seed, dual=getattr(h, "dual", DUAL_PER_VARIABLE))
    d.update(over)
    return make_params(**d)
