"""Pins of the Max-k-Cut oracle (oracle/kcut_oracle.c) against what the paper and the mathematics
fix: the objective by the edge list over all k^n labelings, k = 2 against the Max-Cut QUBO, the gradient of the
Lagrangian by finite differences of its definition typed out here, the invariants of the softmax parameterisation,
and a whole run against brute force."""
import itertools

import numpy as np
import pytest

from paper_2509_21064_b200 import workloads as wl
from tests.helpers import oracle_problem

kcut = pytest.importorskip("oracle.kcut")


def small_graph(n, m, seed, weights="pm"):
    e = wl.edges_gnm(n, m, seed)
    rng = np.random.default_rng(seed)
    w = rng.integers(1, 4, size=m).astype(np.float64) * (rng.choice([-1.0, 1.0], size=m) if weights == "pm" else 1.0)
    W = np.zeros((n, n))
    W[e[:, 0], e[:, 1]] = W[e[:, 1], e[:, 0]] = w
    rowptr, col, val = [0], [], []
    for i in range(n):
        nz = np.nonzero(W[i])[0]
        col += list(nz); val += list(W[i, nz]); rowptr.append(len(col))
    return e, w, W, (np.array(rowptr, np.int32), np.array(col, np.int32), np.array(val))


def test_objective_is_total_weight_minus_twice_the_cut_for_all_labelings():
    n, k = 7, 3
    e, w, W, csr = small_graph(n, 12, 3)
    P = kcut.Problem(n, k, *csr)
    labs = np.array(list(itertools.product(range(k), repeat=n)), dtype=np.uint8).T      # [n][k^n]
    got = kcut.objective(P, labs)
    cut = (w[:, None] * (labs[e[:, 0]] != labs[e[:, 1]])).sum(axis=0)                 # PAPER.md:788, by the edge list
    assert np.array_equal(got, W.sum() - 2.0 * cut)
    onehot = np.eye(k)[labs.T]                                                       # [k^n][n][k]; Tr(X W X^T)
    assert np.allclose(got, np.einsum("bik,ij,bjk->b", onehot, W, onehot))


def test_two_parts_is_the_maxcut_qubo(oracle):
    w2 = wl.config(1)                                            # Max-Cut n = 20 as a QUBO: F(x) = -cut(x)
    Pq = w2.problem
    val = Pq.val.astype(np.float64)
    P = kcut.Problem(Pq.n, 2, Pq.rowptr, Pq.col, val)
    rng = np.random.default_rng(1)
    labs = (rng.random((Pq.n, 50)) < 0.5).astype(np.uint8)
    F = oracle.F_binary(oracle_problem(Pq), labs)
    assert np.array_equal(kcut.objective(P, labs), 2.0 * F + val.sum())              # Tr = 2 x^T W x - 2 1^T W x + 1^T W 1


def lagrangian(W, Z, y, gfun):
    """L(SoftMax(Z), y) = Tr(X W X^T) + sum_i y_i g(X_:,i), typed from PAPER.md:802-824.  Z [k][n], y [n]."""
    X = np.exp(Z - Z.max(axis=0))
    X /= X.sum(axis=0)
    g = (X * X).sum(axis=0) - 1.0 if gfun == 0 else (X * np.log(X)).sum(axis=0)
    return np.trace(X @ W @ X.T) + (y * g).sum(), X, g


@pytest.mark.parametrize("gfun", [0, 1])
def test_one_step_is_gda_on_the_lagrangian(gfun):
    n, k = 6, 4
    e, w, W, csr = small_graph(n, 9, 5)
    P = kcut.Problem(n, k, *csr)
    rng = np.random.default_rng(2)
    Z, y = rng.normal(size=(k, n)), rng.uniform(0.5, 3.0, size=n)
    alpha, beta = 1e-3, 0.4
    r = kcut.run(P, Z.reshape(k, n, 1), y.reshape(n, 1), alpha=alpha, beta=beta, gfun=gfun, iters=1, eval_every=1)
    gradZ = (Z - r["z"][:, :, 0]) / alpha
    _, X, g = lagrangian(W, Z, y, gfun)
    h = 1e-6
    for j in range(k):
        for i in range(n):
            E = np.zeros((k, n)); E[j, i] = h
            fd = (lagrangian(W, Z + E, y, gfun)[0] - lagrangian(W, Z - E, y, gfun)[0]) / (2 * h)
            assert gradZ[j, i] == pytest.approx(fd, rel=2e-6, abs=2e-7)
    assert np.allclose((r["y"][:, 0] - y) / beta, g, rtol=1e-12)                     # dual ascent on g(X^t)
    assert np.allclose(r["x"][:, :, 0].sum(axis=0), 1.0)                             # columns stay on the simplex
    lab = r["labels"][:, 0]
    assert np.array_equal(lab, np.argmax(r["z"][:, :, 0], axis=0))                   # rounding = argmax (K4)


@pytest.mark.parametrize("gfun", [0, 1])
def test_lagrangian_and_gradient_functions(gfun):
    """kcut.lagrangian against L(SoftMax(Z), y) typed out above and, at one-hot points, against the
    objective; kcut.grad against central differences of that L with y = 0, and against the softmax Jacobian's null space."""
    n, k, B = 7, 3, 5
    e, w, W, csr = small_graph(n, 11, 8)
    P = kcut.Problem(n, k, *csr)
    rng = np.random.default_rng(6)
    Z, Y = rng.normal(size=(k, n, B)), rng.uniform(0.0, 3.0, size=(n, B))
    got = kcut.lagrangian(P, Z, Y, gfun)
    for b in range(B):
        assert got[b] == pytest.approx(lagrangian(W, Z[:, :, b], Y[:, b], gfun)[0], rel=1e-12, abs=1e-12)
    assert np.allclose(kcut.lagrangian(P, Z, 2.0, gfun), kcut.lagrangian(P, Z, np.full((n, B), 2.0), gfun), rtol=0, atol=1e-12)
    labs = rng.integers(0, k, size=(n, B)).astype(np.uint8)                          # one-hot columns: g = 0, L = the objective
    Zh = 60.0 * np.eye(k)[labs.T].transpose(2, 1, 0)                                 # [k][n][B], margin 60 between logits
    assert np.allclose(kcut.lagrangian(P, Zh, Y, gfun), kcut.objective(P, labs), rtol=0, atol=1e-9)
    G = kcut.grad(P, Z)
    h = 1e-6
    for b in range(2):
        for j in range(k):
            for i in range(n):
                E = np.zeros((k, n)); E[j, i] = h
                fd = (lagrangian(W, Z[:, :, b] + E, np.zeros(n), 0)[0] - lagrangian(W, Z[:, :, b] - E, np.zeros(n), 0)[0]) / (2 * h)
                assert G[j, i, b] == pytest.approx(fd, rel=2e-6, abs=2e-7)
    assert np.abs(G.sum(axis=0)).max() <= 1e-12                                      # shifts of a column's logits change nothing


def test_softmax_invariants_along_a_run():
    n, k = 30, 3
    e, w, W, csr = small_graph(n, 70, 7, weights="unit")
    P = kcut.Problem(n, k, *csr)
    rng = np.random.default_rng(3)
    Z0 = rng.random((k, n, 4))
    kw = dict(alpha=0.01, beta=0.01, gfun=0, eval_every=10)
    a = kcut.run(P, Z0, 6.0, iters=60, **kw)
    # the softmax Jacobian annihilates constants: sum_j Z_ji never changes
    assert np.allclose(a["z"].sum(axis=0), Z0.sum(axis=0), rtol=0, atol=1e-12)
    # adding a constant to a node's logits changes nothing but that constant
    shift = rng.normal(size=(1, n, 4))
    b = kcut.run(P, Z0 + shift, 6.0, iters=60, **kw)
    assert np.allclose(b["x"], a["x"], atol=1e-12) and np.array_equal(b["labels"], a["labels"])
    # g <= 0 on the simplex for both choices of g: the multipliers never increase, by at most beta (1 - 1/k) per step
    y_prev = np.full((n, 4), 6.0)
    Z = Z0
    for t in range(20):
        r = kcut.run(P, Z, y_prev, iters=1, **dict(kw, eval_every=1))
        assert np.all(r["y"] <= y_prev + 1e-15) and np.all(r["y"] >= y_prev - 0.01 * (1 - 1 / k) - 1e-15)
        Z, y_prev = r["z"], r["y"]
    assert np.array_equal(kcut.objective(P, a["labels"]), a["obj"])                  # returned values are those of the returned labelings


def test_whole_run_against_brute_force():
    n, k = 10, 3
    e, w, W, csr = small_graph(n, 24, 11, weights="unit")
    P = kcut.Problem(n, k, *csr)
    labs = np.array(list(itertools.product(range(k), repeat=n)), dtype=np.uint8).T
    opt = (W.sum() - kcut.objective(P, labs).min()) / 2                              # best 3-cut by brute force (59 049 labelings)
    Z0 = np.random.default_rng(4).random((k, n, 32))
    r = kcut.run(P, Z0, 6.0, alpha=0.01, beta=0.01, gfun=0, iters=3000, eval_every=100, nthreads=4)   # Table 6: ybar 6, alpha = beta = 0.01
    cut = (W.sum() - r["obj"]) / 2
    assert cut.max() <= opt and cut.max() >= 0.95 * opt and cut.mean() >= 0.85 * opt
    assert r["best_restart"] == int(np.argmin(r["obj"]))
