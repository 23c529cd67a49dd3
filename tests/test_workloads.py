"""Input generators: shapes, determinism, structure (CPU only)."""
from pathlib import Path

import numpy as np

from paper_2509_21064_b200 import workloads as wl

GOLD = Path(__file__).parent / "golden"


def table6():
    rows = {}
    for line in (GOLD / "table6_hyperparameters.txt").read_text().splitlines():
        if line.startswith("#") or not line.strip():
            continue
        name, B, y, a, b = line.split()
        rows[name] = (int(B), float(y), float(a), float(b))
    return rows


def test_defaults_follow_table_6():
    t = table6()
    for idx, key in ((1, "Max-Cut"), (3, "Max-Cut"), (5, "Max-k-SAT")):
        h = wl.config(idx, B=4, n_scale=0.01 if idx != 1 else 1.0).hyper
        assert (h.lambda0, h.alpha, h.beta) == t[key][1:]
    h2 = wl.config(2, B=4, n_scale=0.1).hyper          # reading R7: smaller alpha, rest from Table 6
    assert (h2.lambda0, h2.beta) == (t["Max-Cut"][1], t["Max-Cut"][3]) and h2.alpha < t["Max-Cut"][2]
    assert wl.config(5, B=4, n_scale=0.01).hyper.gfun == 1      # entropy g for Max-k-SAT


def test_maxcut_csr_is_symmetric_zero_diagonal_and_c_is_minus_degree():
    w = wl.config(3, B=4, n_scale=0.02)
    P = w.problem
    n = P.n
    D = np.zeros((n, n))
    for i in range(n):
        cols = P.col[P.rowptr[i]:P.rowptr[i + 1]]
        assert np.all(np.diff(cols) > 0)                       # sorted, no duplicate edges
        D[i, cols] = P.val[P.rowptr[i]:P.rowptr[i + 1]]
    assert np.array_equal(D, D.T) and np.all(np.diag(D) == 0)
    assert np.array_equal(P.c, -D.sum(1).astype(np.float32))
    assert P.edges.shape[0] == 2 * n and set(np.unique(P.val)) <= {-1.0, 1.0}


def test_full_size_shapes_and_determinism():
    w2, w3, w5 = wl.config(2), wl.config(3), wl.config(5)
    assert (w2.problem.n, w2.problem.edges.shape[0], w2.B) == (800, 19176, 1024)
    assert (w3.problem.n, w3.problem.edges.shape[0], w3.B) == (20000, 40000, 256)
    assert (w5.problem.n, w5.problem.m, w5.problem.lit.shape[0], w5.B) == (10000, 42600, 127800, 512)
    v = np.abs(w5.problem.lit).reshape(-1, 3)
    assert np.all(v[:, 0] != v[:, 1]) and np.all(v[:, 0] != v[:, 2]) and np.all(v[:, 1] != v[:, 2])   # R2
    assert w5.problem.w.min() == 1 and w5.problem.w.max() == 10
    assert np.array_equal(wl.config(3).problem.col, w3.problem.col)
    x = wl.x0_uniform(7, 8, 5)
    assert x.dtype == np.float32 and x.shape == (7, 8) and np.array_equal(x, wl.x0_uniform(7, 8, 5))
    assert 0 <= x.min() and x.max() < 1


def test_dense_qubo_is_bf16_representable_and_symmetric():
    P = wl.config(4, B=4, n_scale=0.0625).problem
    assert P.n == 256 and np.array_equal(P.Q, P.Q.T)
    assert np.all((P.Q.view(np.uint32) & 0xFFFF) == 0)          # low 16 mantissa bits are zero: exact in bf16
    r = wl.round_to_bf16(np.array([1.0, 1.00390625, 1.01171875, 3.14159], dtype=np.float32))
    assert r[0] == 1.0 and r[1] == 1.0 and r[2] == 1.015625     # ties to even


def test_regular_graph_and_mis_qubo():
    for n, d in ((60, 3), (40, 12)):
        e = wl.edges_regular(n, d, 5)
        assert e.shape == (n * d // 2, 2) and (e[:, 0] < e[:, 1]).all()
        assert len({(int(a), int(b)) for a, b in e}) == e.shape[0]              # simple graph
        assert (np.bincount(e.ravel(), minlength=n) == d).all()                 # d-regular
        assert np.array_equal(e, wl.edges_regular(n, d, 5))                     # seeded
        P = wl.mis_as_qubo(n, e, 4.0)
        # F(x) = -|S| + lam * (edges inside S), checked by the edge list on random sets
        rng = np.random.default_rng(0)
        Q = np.zeros((n, n))
        for i in range(n):
            Q[i, P.col[P.rowptr[i]:P.rowptr[i + 1]]] = P.val[P.rowptr[i]:P.rowptr[i + 1]]
        assert np.array_equal(Q, Q.T)
        for _ in range(20):
            x = (rng.random(n) < 0.3).astype(np.float64)
            inside = int((x[e[:, 0]] * x[e[:, 1]]).sum())
            assert x @ Q @ x + P.c @ x == -x.sum() + 4.0 * inside
