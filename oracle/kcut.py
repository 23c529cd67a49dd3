"""ctypes front end of oracle/kcut_oracle.c (PDBO on Max-k-Cut).  TEST INFRASTRUCTURE ONLY:
imported by tests/, __graft_entry__.smoke() and bench.py's oracle legs, never by the CUDA library or its binding."""
from __future__ import annotations

import ctypes as C

import numpy as np

from . import pdbo

G_QUADRATIC, G_ENTROPY = 0, 1


class _Problem(C.Structure):
    _fields_ = [("n", C.c_int32), ("k", C.c_int32), ("rowptr", C.c_void_p), ("col", C.c_void_p), ("val", C.c_void_p)]


class _Params(C.Structure):
    _fields_ = [("alpha", C.c_double), ("beta", C.c_double), ("log_eps", C.c_double),
                ("gfun", C.c_int32), ("iters", C.c_int32), ("eval_every", C.c_int32)]


class Problem:
    """Symmetric weight matrix W as CSR (both directions stored, zero diagonal) and the number of parts k."""

    def __init__(self, n, k, rowptr, col, val):
        self.n, self.k = int(n), int(k)
        self.rowptr = np.ascontiguousarray(rowptr, dtype=np.int32)
        self.col = np.ascontiguousarray(col, dtype=np.int32)
        self.val = np.ascontiguousarray(val, dtype=np.float64)
        self.struct = _Problem(self.n, self.k, self.rowptr.ctypes.data, self.col.ctypes.data, self.val.ctypes.data)


def objective(P: Problem, labels: np.ndarray) -> np.ndarray:
    """out[b] = Tr(Xh W Xh^T) for the one-hot matrix of labels[:, b] (uint8 [n][B]); the k-cut is (sum W - out) / 2."""
    labels = np.ascontiguousarray(labels, dtype=np.uint8)
    assert labels.ndim == 2 and labels.shape[0] == P.n and labels.max(initial=0) < P.k
    out = np.empty(labels.shape[1], dtype=np.float64)
    rc = pdbo._lib("f64").kcut_objective_batch(C.byref(P.struct), C.c_int32(labels.shape[1]),
                                               C.c_void_p(labels.ctypes.data), C.c_void_p(out.ctypes.data))
    assert rc == 0
    return out


def lagrangian(P: Problem, Z: np.ndarray, Y, gfun: int = G_QUADRATIC, precision: str = "f64") -> np.ndarray:
    """out[b] = L(SoftMax(Z[:,:,b]), Y[:,b]) = Tr(X W X^T) + sum_i y_i g(X_:,i).  Y [n][B] or a scalar."""
    rt = pdbo._real(precision)
    Z = np.ascontiguousarray(Z, dtype=rt)
    k, n, B = Z.shape
    assert k == P.k and n == P.n
    Ya = np.full((n, B), Y, dtype=rt) if np.isscalar(Y) else np.ascontiguousarray(Y, dtype=rt)
    out = np.empty(B, dtype=np.float64)
    rc = pdbo._lib(precision).kcut_lagrangian_batch(C.byref(P.struct), C.c_int32(B), C.c_void_p(Z.ctypes.data),
                                                    C.c_void_p(Ya.ctypes.data), C.c_int32(gfun), C.c_void_p(out.ctypes.data))
    assert rc == 0
    return out


def grad(P: Problem, Z: np.ndarray, precision: str = "f64") -> np.ndarray:
    """grad_Z of Tr(X W X^T) at X = SoftMax(Z), [k][n][B] (the softmax chain rule of PAPER.md:816-824)."""
    rt = pdbo._real(precision)
    Z = np.ascontiguousarray(Z, dtype=rt)
    k, n, B = Z.shape
    assert k == P.k and n == P.n
    out = np.empty_like(Z)
    rc = pdbo._lib(precision).kcut_grad_batch(C.byref(P.struct), C.c_int32(B), C.c_void_p(Z.ctypes.data), C.c_void_p(out.ctypes.data))
    assert rc == 0
    return out


def run(P: Problem, Z0: np.ndarray, Y0, *, alpha: float, beta: float, gfun: int = G_QUADRATIC, log_eps: float = 1e-6,
        iters: int, eval_every: int, precision: str = "f64", nthreads: int = 1):
    """GDA on L(SoftMax(Z), y) for every restart.  Z0 [k][n][B] logits, Y0 an [n][B] array or a scalar.
    Returns dict(labels, obj, best_restart, z, x, y)."""
    rt = pdbo._real(precision)
    Z0 = np.ascontiguousarray(Z0, dtype=rt)
    k, n, B = Z0.shape
    assert k == P.k and n == P.n
    Y0a = np.full((n, B), Y0, dtype=rt) if np.isscalar(Y0) else np.ascontiguousarray(Y0, dtype=rt)
    assert Y0a.shape == (n, B)
    hp = _Params(alpha, beta, log_eps, gfun, iters, eval_every)
    labels = np.zeros((n, B), dtype=np.uint8)
    obj = np.empty(B, dtype=np.float64)
    best = C.c_int32(0)
    Zf, Xf, Yf = np.empty_like(Z0), np.empty_like(Z0), np.empty_like(Y0a)
    rc = pdbo._lib(precision).kcut_run(C.byref(P.struct), C.c_int32(B), C.c_void_p(Z0.ctypes.data),
                                       C.c_void_p(Y0a.ctypes.data), C.byref(hp), C.c_void_p(labels.ctypes.data),
                                       C.c_void_p(obj.ctypes.data), C.byref(best), C.c_void_p(Zf.ctypes.data),
                                       C.c_void_p(Yf.ctypes.data), C.c_void_p(Xf.ctypes.data), C.c_int32(nthreads))
    assert rc == 0
    return dict(labels=labels, obj=obj, best_restart=int(best.value), z=Zf, x=Xf, y=Yf)
