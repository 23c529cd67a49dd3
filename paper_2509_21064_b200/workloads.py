"""Seeded synthetic inputs shaped like the paper's workloads.

This module holds NO arithmetic of the method (no f, no gradient, no GDA step): it only draws
problem data and start points.  It is the one module that both the CPU oracle's tests and the CUDA
path's tests/bench import, so that the two sides see identical arrays.

Shapes follow BASELINE.json `configs` and SURVEY.md section 8(d):
  cfg1  Max-Cut  G(20, p=0.5), unit weights, B=64           (brute-force checkable)
  cfg2  Max-Cut  G(800, m=19176), unit weights, B=1024      (stands in for the 800-node Gset family)
  cfg3  Max-Cut  G(20000, m=40000), weights +-1, B=256      (stands in for G81)
  cfg4  dense QUBO n=4096, N(0,1) entries bf16-representable, B=4096
  cfg5  weighted Max-3-SAT n=10000, m=42600, w in 1..10, B=512  (stands in for the 3-CNF set)
Max-Cut is handed to the solvers in the paper's minimisation form F(x) = x^T W x - 1^T W x
(PAPER.md:146, 604), i.e. Q = W (symmetric, both directions stored) and c = -W 1; cut(x) = -F(x).
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Optional

import numpy as np


# --------------------------------------------------------------------------------------------
# problem containers (plain arrays; host memory)
# --------------------------------------------------------------------------------------------
@dataclass
class QuboCSR:
    """F(x) = x^T Q x + c^T x, Q symmetric, given as CSR with both (i,j) and (j,i) stored."""
    n: int
    rowptr: np.ndarray  # int32 [n+1]
    col: np.ndarray     # int32 [nnz]
    val: np.ndarray     # float32 [nnz]
    c: np.ndarray       # float32 [n]
    edges: Optional[np.ndarray] = None  # int64 [m,2] (i<j) when the instance is a Max-Cut graph
    edge_w: Optional[np.ndarray] = None  # float32 [m]


@dataclass
class QuboDense:
    """F(x) = x^T Q x + c^T x, Q symmetric row-major [n,n] float32 (bf16-representable values)."""
    n: int
    Q: np.ndarray  # float32 [n,n]
    c: np.ndarray  # float32 [n]


@dataclass
class MaxSat:
    """F(x) = sum_j w_j [clause j unsatisfied]; lit = +-(var+1), DIMACS sign convention."""
    n: int
    m: int
    cptr: np.ndarray  # int32 [m+1]
    lit: np.ndarray   # int32 [L]
    w: np.ndarray     # float32 [m]


@dataclass
class MaxKCut:
    """Max-k-Cut: symmetric weight matrix W as CSR (both directions), k parts."""
    n: int
    k: int
    rowptr: np.ndarray
    col: np.ndarray
    val: np.ndarray
    edges: np.ndarray = None
    edge_w: np.ndarray = None


@dataclass
class Hyper:
    """(y-bar, alpha, beta, delta, g) and run lengths for one config (Table 6; R7)."""
    lambda0: float
    alpha: float
    beta: float
    delta: float = 1e-4
    gfun: int = 0          # 0 quadratic x^2-x, 1 entropy
    log_eps: float = 1e-6
    iters: int = 1000
    eval_every: int = 100
    seed: int = 0
    dual: int = 0          # 0 per-variable multipliers (PDBO), 1 one multiplier per restart (PDBO-s)


@dataclass
class Workload:
    name: str
    kind: str              # "qubo_csr" | "qubo_dense" | "maxsat"
    problem: object
    B: int
    hyper: Hyper
    x0_seed: int
    note: str = ""
    extra: dict = field(default_factory=dict)


# --------------------------------------------------------------------------------------------
# graph / matrix / formula generators
# --------------------------------------------------------------------------------------------
def edges_gnp(n: int, p: float, seed: int) -> np.ndarray:
    """Erdos-Renyi G(n,p): one Bernoulli(p) draw per unordered pair, upper triangle, row-major."""
    rng = np.random.Generator(np.random.PCG64(seed))
    iu, ju = np.triu_indices(n, k=1)
    keep = rng.random(iu.shape[0]) < p
    return np.stack([iu[keep], ju[keep]], axis=1).astype(np.int64)


def edges_gnm(n: int, m: int, seed: int) -> np.ndarray:
    """G(n,m): m distinct unordered pairs i<j, uniform (oversample, dedupe, keep the first m)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    total = n * (n - 1) // 2
    if m > total:
        raise ValueError("m exceeds the number of pairs")
    chosen = np.empty(0, dtype=np.int64)
    while chosen.shape[0] < m:
        a = rng.integers(0, n, size=2 * m + 16, dtype=np.int64)
        b = rng.integers(0, n, size=2 * m + 16, dtype=np.int64)
        ok = a != b
        lo = np.minimum(a[ok], b[ok])
        hi = np.maximum(a[ok], b[ok])
        code = np.concatenate([chosen, lo * n + hi])
        _, first = np.unique(code, return_index=True)
        chosen = code[np.sort(first)]          # keep draw order, drop repeats
    chosen = chosen[:m]
    return np.stack([chosen // n, chosen % n], axis=1).astype(np.int64)


def edge_weights(m: int, seed: int, kind: str) -> np.ndarray:
    rng = np.random.Generator(np.random.PCG64(seed + 7919))
    if kind == "unit":
        return np.ones(m, dtype=np.float32)
    if kind == "pm1":
        return (2 * rng.integers(0, 2, size=m) - 1).astype(np.float32)
    raise ValueError(kind)


def maxcut_as_qubo(n: int, edges: np.ndarray, w: np.ndarray) -> QuboCSR:
    """Q = W (symmetric CSR, zero diagonal, columns sorted), c = -W 1  (reading R8)."""
    i = np.concatenate([edges[:, 0], edges[:, 1]])
    j = np.concatenate([edges[:, 1], edges[:, 0]])
    v = np.concatenate([w, w]).astype(np.float32)
    order = np.lexsort((j, i))
    i, j, v = i[order], j[order], v[order]
    rowptr = np.zeros(n + 1, dtype=np.int64)
    np.add.at(rowptr, i + 1, 1)
    rowptr = np.cumsum(rowptr)
    wdeg = np.zeros(n, dtype=np.float64)
    np.add.at(wdeg, i, v.astype(np.float64))
    return QuboCSR(n=n, rowptr=rowptr.astype(np.int32), col=j.astype(np.int32), val=v,
                   c=(-wdeg).astype(np.float32), edges=edges, edge_w=w.astype(np.float32))


def edges_regular(n: int, d: int, seed: int) -> np.ndarray:
    """A simple d-regular graph on n vertices (n * d even) as the union of d perfect matchings (n even) drawn one
    after the other; pairs that repeat an earlier edge are re-drawn among themselves and a few fresh pairs until
    none is left.  Shape of the d-RRGs of the paper's MIS experiment, not a uniform sample."""
    if n % 2 or d >= n:
        raise ValueError("edges_regular needs an even n and d < n")
    rng = np.random.Generator(np.random.PCG64(seed))
    seen = set()
    out = []
    for _ in range(d):
        perm = rng.permutation(n)
        a, b = perm[0::2].copy(), perm[1::2].copy()
        for _try in range(10000):
            lo, hi = np.minimum(a, b), np.maximum(a, b)
            code = lo.astype(np.int64) * n + hi
            bad = np.array([c in seen for c in code.tolist()], dtype=bool)
            if not bad.any():
                break
            pick = bad.copy()
            pick[rng.integers(0, a.shape[0], size=max(4, int(bad.sum())))] = True      # some freedom to re-pair
            verts = rng.permutation(np.concatenate([a[pick], b[pick]]))
            a[pick], b[pick] = verts[0::2], verts[1::2]
        else:
            raise RuntimeError("edges_regular: could not complete a matching")
        seen.update(code.tolist())
        out.append(np.stack([lo, hi], axis=1))
    return np.concatenate(out).astype(np.int64)


def mis_as_qubo(n: int, edges: np.ndarray, lam: float = 4.0) -> QuboCSR:
    """Maximum independent set as the QUBO  min -sum_i x_i + lam sum_{(i,j) in E} x_i x_j  (PAPER.md:1026-1028,
    lam = 4): Q = (lam/2) A with A the symmetric adjacency matrix, c = -1.  For binary x,
    F(x) = -|S| + lam * (number of edges inside S): S is independent iff F(x) = -|S|."""
    i = np.concatenate([edges[:, 0], edges[:, 1]])
    j = np.concatenate([edges[:, 1], edges[:, 0]])
    order = np.lexsort((j, i))
    i, j = i[order], j[order]
    rowptr = np.zeros(n + 1, dtype=np.int64)
    np.add.at(rowptr, i + 1, 1)
    return QuboCSR(n=n, rowptr=np.cumsum(rowptr).astype(np.int32), col=j.astype(np.int32),
                   val=np.full(i.shape[0], 0.5 * lam, dtype=np.float32), c=np.full(n, -1.0, dtype=np.float32),
                   edges=edges, edge_w=np.full(edges.shape[0], lam, dtype=np.float32))


def mis(n: int, d: int, B: int = 12, seed: int = 106, iters: int = 5000) -> Workload:
    """MIS on a d-regular graph (d in {3, 100}, n in {1e4, 5e4}); Table 6: ybar = 5,
    alpha = beta = 0.02, B = 10 (12 here: restarts come in multiples of 4).  With lam = 4 and degree d the no-flip
    rule of reading R7 asks for alpha (lam d + ybar) < 1, which Table 6's alpha meets for d = 3 only; for larger d
    alpha is scaled to 0.4 / (lam d / 2 + ybar)."""
    P = mis_as_qubo(n, edges_regular(n, d, seed), 4.0)
    alpha = 0.02 if d <= 8 else 0.4 / (2.0 * d + 5.0)
    return Workload(f"mis_n{n}_d{d}", "qubo_csr", P, B, Hyper(5.0, alpha, 0.02, 1e-4, 0, 1e-6, iters, 100, seed),
                    1000 + seed, f"MIS as QUBO (lam=4) on a {d}-regular graph")


def round_to_bf16(a: np.ndarray) -> np.ndarray:
    """Round float32 values to the nearest bf16-representable value (ties to even), kept as float32."""
    u = np.ascontiguousarray(a, dtype=np.float32).view(np.uint32).astype(np.uint64)
    u = (u + 0x7FFF + ((u >> 16) & 1)) & 0xFFFF0000
    return u.astype(np.uint32).view(np.float32).reshape(a.shape)


def dense_qubo(n: int, seed: int) -> QuboDense:
    """Q = triu(A,1) + triu(A,1)^T + diag(d), A,d ~ N(0,1), rounded to bf16 (reading R13); c ~ N(0,1)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    A = rng.standard_normal((n, n), dtype=np.float32)
    d = rng.standard_normal(n, dtype=np.float32)
    c = rng.standard_normal(n, dtype=np.float32)
    U = np.triu(A, 1)
    Q = U + U.T
    Q[np.arange(n), np.arange(n)] = d
    return QuboDense(n=n, Q=round_to_bf16(Q), c=c)


def random_ksat(n: int, m: int, k: int, seed: int, wmax: int = 10) -> MaxSat:
    """m clauses of k DISTINCT variables (uniform), uniform signs, integer weights uniform in 1..wmax."""
    rng = np.random.Generator(np.random.PCG64(seed))
    var = rng.integers(0, n, size=(m, k), dtype=np.int64)
    while True:
        s = np.sort(var, axis=1)
        bad = np.nonzero((s[:, 1:] == s[:, :-1]).any(axis=1))[0]
        if bad.size == 0:
            break
        var[bad] = rng.integers(0, n, size=(bad.size, k), dtype=np.int64)
    sign = 2 * rng.integers(0, 2, size=(m, k), dtype=np.int64) - 1
    w = rng.integers(1, wmax + 1, size=m).astype(np.float32)
    lit = (sign * (var + 1)).astype(np.int32).reshape(-1)
    cptr = (np.arange(m + 1, dtype=np.int64) * k).astype(np.int32)
    return MaxSat(n=n, m=m, cptr=cptr, lit=lit, w=w)


def random_pubo(n: int, m: int, kmax: int, seed: int, wmax: int = 6) -> MaxSat:
    """A polynomial in literal-product form with SIGNED integer weights: m terms of 1..kmax distinct variables, uniform
    literal signs, weights uniform in {-wmax..wmax} without 0 (Prop. 2.4: the extension of a polynomial)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    lits, cptr = [], [0]
    for _ in range(m):
        k = int(rng.integers(1, kmax + 1))
        v = rng.choice(n, size=k, replace=False)
        lits += list((2 * rng.integers(0, 2, size=k) - 1) * (v + 1))
        cptr.append(len(lits))
    w = rng.integers(1, wmax + 1, size=m) * (2 * rng.integers(0, 2, size=m) - 1)
    return MaxSat(n=n, m=m, cptr=np.array(cptr, np.int32), lit=np.array(lits, np.int32), w=w.astype(np.float32))


def qubo_as_literal_products(n: int, Q: np.ndarray, c: np.ndarray) -> MaxSat:
    """x^T Q x + c^T x on binary x as weighted literal products: {not i, not j} with weight Q_ij + Q_ji for i < j and
    {not i} with weight Q_ii + c_i (x_i^2 = x_i); zero terms are dropped."""
    lits, cptr, w = [], [0], []
    for i in range(n):
        d = float(Q[i, i] + c[i])
        if d != 0.0:
            lits.append(-(i + 1)); cptr.append(len(lits)); w.append(d)
        for j in range(i + 1, n):
            q = float(Q[i, j] + Q[j, i])
            if q != 0.0:
                lits += [-(i + 1), -(j + 1)]; cptr.append(len(lits)); w.append(q)
    return MaxSat(n=n, m=len(w), cptr=np.array(cptr, np.int32), lit=np.array(lits, np.int32), w=np.array(w, np.float32))


def binary_mrf_grid(rows: int, cols: int, seed: int, scale: int = 4) -> MaxSat:
    """MAP inference on a binary pairwise MRF as a polynomial in literal-product form: a rows x cols
    grid, integer energies theta_i(a) and theta_ij(a, b) uniform in {-scale..scale}; every table entry is the weight of the
    indicator of its assignment, i.e. of the clause that assignment falsifies (a positive literal is false at 0)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    n = rows * cols
    lits, cptr, w = [], [0], []
    lit_false_at = lambda v, a: (v + 1) if a == 0 else -(v + 1)      # the literal of variable v that is false when x_v = a
    def add(term, weight):
        if weight != 0:
            lits.extend(term); cptr.append(len(lits)); w.append(float(weight))
    for v in range(n):
        for a in (0, 1):
            add([lit_false_at(v, a)], int(rng.integers(-scale, scale + 1)))
    for r in range(rows):
        for q in range(cols):
            v = r * cols + q
            for u in ([v + 1] if q + 1 < cols else []) + ([v + cols] if r + 1 < rows else []):
                for a in (0, 1):
                    for b in (0, 1):
                        add([lit_false_at(v, a), lit_false_at(u, b)], int(rng.integers(-scale, scale + 1)))
    return MaxSat(n=n, m=len(w), cptr=np.array(cptr, np.int32), lit=np.array(lits, np.int32), w=np.array(w, np.float32))


def x0_uniform(n: int, B: int, seed: int) -> np.ndarray:
    """x0 ~ U[0,1)^(n x B), float32, layout [n][B]."""
    rng = np.random.Generator(np.random.PCG64(seed))
    return rng.random((n, B), dtype=np.float32)


# --------------------------------------------------------------------------------------------
# the five BASELINE.json configs (1-based like SURVEY.md section 8(d))
# --------------------------------------------------------------------------------------------
def config(idx: int, B: Optional[int] = None, n_scale: float = 1.0, n_exact: Optional[int] = None) -> Workload:
    """Build config `idx` (1..5).  `B` overrides the restart count; `n_scale` shrinks n (and m)
    proportionally for quick tests while keeping density / degree / clause ratio; `n_exact` (config 4 only) sets n
    to any value, e.g. one that is not a multiple of the GEMM tile."""
    if idx == 1:
        n = 20
        e = edges_gnp(n, 0.5, 101)
        P = maxcut_as_qubo(n, e, edge_weights(e.shape[0], 101, "unit"))
        return Workload("cfg1_maxcut_n20", "qubo_csr", P, B or 64,
                        Hyper(6.0, 0.025, 0.025, 1e-4, 0, 1e-6, 1000, 50, 101), 1101,
                        "Max-Cut G(20,0.5), unit weights; brute force 2^20")
    if idx == 2:
        n = max(8, int(round(800 * n_scale)))
        m = int(round(19176 * n_scale * n_scale)) if n_scale != 1.0 else 19176
        e = edges_gnm(n, m, 102)
        P = maxcut_as_qubo(n, e, edge_weights(m, 102, "unit"))
        return Workload("cfg2_maxcut_n800", "qubo_csr", P, B or 1024,
                        Hyper(6.0, 0.008, 0.025, 1e-4, 0, 1e-6, 5000, 100, 102), 1102,
                        "Max-Cut G(800,19176), unit weights; alpha per reading R7")
    if idx == 3:
        n = max(8, int(round(20000 * n_scale)))
        m = 2 * n
        e = edges_gnm(n, m, 103)
        P = maxcut_as_qubo(n, e, edge_weights(m, 103, "pm1"))
        return Workload("cfg3_maxcut_n20000", "qubo_csr", P, B or 256,
                        Hyper(6.0, 0.025, 0.025, 1e-4, 0, 1e-6, 10000, 100, 103), 1103,
                        "Max-Cut G(20000,40000), weights +-1")
    if idx == 4:
        n = n_exact or max(256, int(round(4096 * n_scale)) // 256 * 256)
        P = dense_qubo(n, 104)
        s = 2.0 * np.sqrt(n)                      # spectral scale of the N(0,1) matrix (reading R7)
        lam = 1.75 * s
        return Workload("cfg4_dense_n4096", "qubo_dense", P, B or 4096,
                        Hyper(float(lam), float(1.0 / (4.0 * (s + lam))), float(4.0 * lam / 1000.0),
                              1e-4, 0, 1e-6, 2000, 100, 104), 1104,
                        "dense QUBO N(0,1), bf16-representable Q")
    if idx == 5:
        n = max(8, int(round(10000 * n_scale)))
        m = int(round(4.26 * n))
        P = random_ksat(n, m, 3, 105)
        return Workload("cfg5_max3sat_n10000", "maxsat", P, B or 512,
                        Hyper(2.0, 0.01, 0.005, 1e-4, 1, 1e-6, 5000, 100, 105), 1105,
                        "weighted Max-3-SAT ratio 4.26, w in 1..10, entropy g")
    raise ValueError("config index must be 1..5")


def maxkcut(n: int, m: int, k: int = 3, B: int = 128, seed: int = 107, weights: str = "unit", iters: int = 5000) -> Workload:
    """Max-k-Cut on G(n, m).  Table 6: B = 100, ybar = 6, alpha = beta = 0.01; the initial logits are
    Z^0 ~ U[0,1)^(k x n x B) (reading K2; `z0_uniform`)."""
    e = edges_gnm(n, m, seed)
    w = edge_weights(m, seed, weights)
    q = maxcut_as_qubo(n, e, w)                          # same symmetric CSR of W
    P = MaxKCut(n=n, k=k, rowptr=q.rowptr, col=q.col, val=q.val, edges=e, edge_w=w)
    return Workload(f"max{k}cut_n{n}", "maxkcut", P, B, Hyper(6.0, 0.01, 0.01, 0.0, 0, 1e-6, iters, 100, seed), 1000 + seed,
                    f"Max-{k}-Cut G({n},{m}), {weights} weights")


def z0_uniform(k: int, n: int, B: int, seed: int) -> np.ndarray:
    """Initial logits Z^0 ~ U[0,1)^(k x n x B), float32, layout [k][n][B] (reading K2)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    return rng.random((k, n, B), dtype=np.float32)


def pdbo_s_variant(w: Workload) -> Workload:
    """The same instance run as PDBO-s (reading R14): one multiplier per restart,
    mu+ = mu + beta_s sum_i g(x_i).  The paper gives no step size for it; beta_s = beta / n keeps the multiplier's
    rate of decrease equal to the average of the per-variable rates of PDBO."""
    import copy
    v = copy.deepcopy(w)
    v.name = w.name + "_pdbo_s"
    v.hyper.dual = 1
    v.hyper.beta = w.hyper.beta / w.problem.n
    v.note = w.note + "; PDBO-s (scalar dual, beta_s = beta/n)"
    return v
