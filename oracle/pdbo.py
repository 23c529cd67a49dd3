"""oracle/pdbo.py -- Python front end of the CPU oracle (oracle/pdbo_oracle.c).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this.  It imports nothing from the CUDA package.  It builds pdbo_oracle.c with gcc into
oracle/_build/ (fp64 and fp32 variants; reading R12) and marshals NumPy arrays through ctypes.

Also here, in plain NumPy, are the DEFINITIONS the C code is pinned against in tests/ (never used by
the C code itself):
  * enumerate_f      -- Def. 2.2: f(x) = sum_xi P_x(xi) F(xi), by enumeration
  * F_qubo_dense / cut_value / unsat_weight -- objective definitions written independently
"""
from __future__ import annotations

import ctypes as C
import itertools
import os
import subprocess
from pathlib import Path
from typing import Optional

import numpy as np

_HERE = Path(__file__).resolve().parent
_BUILD = _HERE / "_build"
_SRC = _HERE / "pdbo_oracle.c"
_SRC_KCUT = _HERE / "kcut_oracle.c"

KIND_QUBO_CSR, KIND_QUBO_DENSE, KIND_MAXSAT = 0, 1, 2
G_QUADRATIC, G_ENTROPY = 0, 1
DUAL_PER_VARIABLE, DUAL_SCALAR = 0, 1


class _Problem(C.Structure):
    _fields_ = [("kind", C.c_int32), ("n", C.c_int32),
                ("rowptr", C.c_void_p), ("col", C.c_void_p), ("val", C.c_void_p),
                ("Qd", C.c_void_p), ("Qt", C.c_void_p), ("c", C.c_void_p),
                ("m", C.c_int32), ("cptr", C.c_void_p), ("lit", C.c_void_p), ("w", C.c_void_p)]


class _Params(C.Structure):
    _fields_ = [("alpha", C.c_double), ("beta", C.c_double), ("delta", C.c_double),
                ("log_eps", C.c_double), ("gfun", C.c_int32), ("iters", C.c_int32),
                ("eval_every", C.c_int32), ("t0", C.c_int32), ("seed", C.c_uint64), ("dual", C.c_int32)]


def build(force: bool = False) -> None:
    """Compile the oracle (gcc -O2, no fast-math) into oracle/_build/liboracle_{f64,f32}.so."""
    _BUILD.mkdir(exist_ok=True)
    for tag, real in (("f64", "double"), ("f32", "float")):
        out = _BUILD / f"liboracle_{tag}.so"
        if out.exists() and not force and out.stat().st_mtime >= max(_SRC.stat().st_mtime, _SRC_KCUT.stat().st_mtime):
            continue
        tmp = out.with_suffix(f".tmp{os.getpid()}.so")
        cmd = ["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-fopenmp", f"-DREAL={real}",
               "-o", str(tmp), str(_SRC), str(_SRC_KCUT), "-lm"]
        subprocess.run(cmd, check=True)
        os.replace(tmp, out)


_libs: dict = {}


def _lib(precision: str):
    if precision not in ("f64", "f32"):
        raise ValueError("precision must be 'f64' or 'f32'")
    if precision not in _libs:
        build()
        lib = C.CDLL(str(_BUILD / f"liboracle_{precision}.so"))
        lib.pdbo_side_bit.argtypes = [C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint32]
        lib.pdbo_side_bit.restype = C.c_int
        assert lib.pdbo_sizeof_real() == (8 if precision == "f64" else 4)
        _libs[precision] = lib
    return _libs[precision]


def max_threads() -> int:
    return int(_lib("f64").pdbo_max_threads())


class Problem:
    """Host-side problem for the oracle.  Keeps the arrays alive for the ctypes struct."""

    def __init__(self, kind: int, n: int, **arrs):
        self.kind, self.n = kind, int(n)
        self._keep = {}
        s = _Problem()
        s.kind, s.n, s.m = kind, int(n), int(arrs.pop("m", 0))
        for name, (arr, dt) in arrs.items():
            if arr is None:
                setattr(s, name, None)
                continue
            a = np.ascontiguousarray(arr, dtype=dt)
            self._keep[name] = a
            setattr(s, name, a.ctypes.data)
        self.struct = s

    # ---- constructors -------------------------------------------------------------------------
    @staticmethod
    def qubo_csr(n, rowptr, col, val, c=None) -> "Problem":
        """F(x) = x^T Q x + c^T x, Q given as CSR triplets (any square Q)."""
        return Problem(KIND_QUBO_CSR, n, rowptr=(rowptr, np.int32), col=(col, np.int32),
                       val=(val, np.float64), c=(c, np.float64))

    @staticmethod
    def qubo_dense(n, Q, c=None) -> "Problem":
        Q = np.asarray(Q, dtype=np.float64).reshape(n, n)
        return Problem(KIND_QUBO_DENSE, n, Qd=(Q, np.float64), Qt=(Q.T.copy(), np.float64),
                       c=(c, np.float64))

    @staticmethod
    def maxsat(n, m, cptr, lit, w=None) -> "Problem":
        return Problem(KIND_MAXSAT, n, m=m, cptr=(cptr, np.int32), lit=(lit, np.int32), w=(w, np.float64))


def _real(precision):
    return np.float64 if precision == "f64" else np.float32


def grad(P: Problem, X: np.ndarray, precision: str = "f64") -> np.ndarray:
    """G[:,b] = grad f(X[:,b]).  X is [n][B]."""
    rt = _real(precision)
    X = np.ascontiguousarray(X, dtype=rt)
    n, B = X.shape
    G = np.empty_like(X)
    rc = _lib(precision).pdbo_grad(C.byref(P.struct), C.c_int32(B), C.c_void_p(X.ctypes.data),
                                   C.c_void_p(G.ctypes.data))
    assert rc == 0
    return G


def f_ext(P: Problem, X: np.ndarray, precision: str = "f64") -> np.ndarray:
    """out[b] = f(X[:,b]): closed form of the multilinear extension (Prop. 2.4)."""
    rt = _real(precision)
    X = np.ascontiguousarray(X, dtype=rt)
    out = np.empty(X.shape[1], dtype=np.float64)
    rc = _lib(precision).pdbo_f(C.byref(P.struct), C.c_int32(X.shape[1]), C.c_void_p(X.ctypes.data),
                                C.c_void_p(out.ctypes.data))
    assert rc == 0
    return out


def lagrangian(P: Problem, X: np.ndarray, Y, gfun: int = G_QUADRATIC, precision: str = "f64") -> np.ndarray:
    """out[b] = L(X[:,b], Y[:,b]) = f(x) + sum_i y_i g(x_i).  Y an [n][B] array or a scalar."""
    rt = _real(precision)
    X = np.ascontiguousarray(X, dtype=rt)
    Ya = np.full(X.shape, Y, dtype=rt) if np.isscalar(Y) else np.ascontiguousarray(Y, dtype=rt)
    assert Ya.shape == X.shape
    out = np.empty(X.shape[1], dtype=np.float64)
    rc = _lib(precision).pdbo_lagrangian(C.byref(P.struct), C.c_int32(X.shape[1]), C.c_void_p(X.ctypes.data),
                                         C.c_void_p(Ya.ctypes.data), C.c_int32(gfun), C.c_void_p(out.ctypes.data))
    assert rc == 0
    return out


def F_binary(P: Problem, Xh: np.ndarray) -> np.ndarray:
    """out[b] = F(Xh[:,b]) for binary columns (uint8 [n][B])."""
    Xh = np.ascontiguousarray(Xh, dtype=np.uint8)
    assert Xh.ndim == 2 and Xh.shape[0] == P.n and Xh.max(initial=0) <= 1
    out = np.empty(Xh.shape[1], dtype=np.float64)
    rc = _lib("f64").pdbo_F(C.byref(P.struct), C.c_int32(Xh.shape[1]), C.c_void_p(Xh.ctypes.data),
                            C.c_void_p(out.ctypes.data))
    assert rc == 0
    return out


def run(P: Problem, X0: np.ndarray, Y0, *, alpha: float, beta: float, delta: float = 1e-4,
        gfun: int = G_QUADRATIC, log_eps: float = 1e-6, iters: int, eval_every: int, seed: int = 0,
        t0: int = 0, col_ids: Optional[np.ndarray] = None, precision: str = "f64", nthreads: int = 1,
        dual: int = DUAL_PER_VARIABLE):
    """Algorithm 1 for every column of X0.  Y0 is an [n][B] array or a scalar (y-bar).
    dual = DUAL_SCALAR runs PDBO-s (reading R14): one multiplier per restart, Y0 a scalar or a
    [B] array, and the returned y is [B].  Returns dict(x_bin, obj, best_restart, x, y)."""
    rt = _real(precision)
    X0 = np.ascontiguousarray(X0, dtype=rt)
    n, B = X0.shape
    assert n == P.n
    if dual == DUAL_SCALAR and not np.isscalar(Y0):
        Y0 = np.broadcast_to(np.asarray(Y0, dtype=rt).reshape(1, B), (n, B))
    Y0a = np.full((n, B), Y0, dtype=rt) if np.isscalar(Y0) else np.ascontiguousarray(Y0, dtype=rt)
    assert Y0a.shape == (n, B)
    hp = _Params(alpha, beta, delta, log_eps, gfun, iters, eval_every, t0, seed, dual)
    x_bin = np.zeros((n, B), dtype=np.uint8)
    obj = np.empty(B, dtype=np.float64)
    best = C.c_int32(-1)
    Xf, Yf = np.empty_like(X0), np.empty_like(X0)
    ids = None if col_ids is None else np.ascontiguousarray(col_ids, dtype=np.int32)
    rc = _lib(precision).pdbo_run(
        C.byref(P.struct), C.c_int32(B), C.c_void_p(X0.ctypes.data), C.c_void_p(Y0a.ctypes.data),
        C.c_void_p(None if ids is None else ids.ctypes.data), C.byref(hp),
        C.c_void_p(x_bin.ctypes.data), C.c_void_p(obj.ctypes.data), C.byref(best),
        C.c_void_p(Xf.ctypes.data), C.c_void_p(Yf.ctypes.data), C.c_int32(nthreads))
    assert rc == 0
    if dual == DUAL_SCALAR:
        assert (Yf == Yf[0:1]).all()                     # the multiplier stays one number per restart
        Yf = Yf[0].copy()
    return dict(x_bin=x_bin, obj=obj, best_restart=int(best.value), x=Xf, y=Yf)


def side_bit(seed: int, t: int, i: int, b: int) -> int:
    return int(_lib("f64").pdbo_side_bit(seed, t, i, b))


# ------------------------------------------------------------------------------------------------
# Definitions in plain NumPy, used only by tests to pin the C code (never called by it)
# ------------------------------------------------------------------------------------------------
def enumerate_f(F_of_bits, n: int, x: np.ndarray) -> float:
    """Def. 2.2: f(x) = sum over xi in {0,1}^n of prod_i x_i^xi_i (1-x_i)^(1-xi_i) * F(xi)."""
    total = 0.0
    for bits in itertools.product((0, 1), repeat=n):
        p = 1.0
        for i, bi in enumerate(bits):
            p *= x[i] if bi else (1.0 - x[i])
        total += p * F_of_bits(np.array(bits, dtype=np.uint8))
    return total


def F_qubo_dense(Q: np.ndarray, c: np.ndarray, xh: np.ndarray) -> float:
    """x^T Q x + c^T x by the matrix formula."""
    v = xh.astype(np.float64)
    return float(v @ np.asarray(Q, np.float64) @ v + np.asarray(c, np.float64) @ v)


def cut_value(edges: np.ndarray, w: np.ndarray, xh: np.ndarray) -> float:
    """sum over edges of W_ij (x_i + x_j - 2 x_i x_j)."""
    xi = xh[edges[:, 0]].astype(np.int64)
    xj = xh[edges[:, 1]].astype(np.int64)
    return float(np.sum(np.asarray(w, np.float64) * (xi + xj - 2 * xi * xj)))


def unsat_weight(cptr, lit, w, xh: np.ndarray) -> float:
    """Weight of clauses with every literal false, by literal truth values."""
    total = 0.0
    for j in range(len(cptr) - 1):
        sat = False
        for l in lit[cptr[j]:cptr[j + 1]]:
            v = bool(xh[abs(int(l)) - 1])
            if (v if l > 0 else not v):
                sat = True
                break
        if not sat:
            total += 1.0 if w is None else float(w[j])
    return total
