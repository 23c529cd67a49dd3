"""Seeded differential tests: many small random instances of every problem kind, with random sizes, degrees and batch sizes,
so that every launch path the library may choose on its own (slab, warp per row, narrow with and without lane groups,
row-split, packed records, slot groups, padding restarts) is hit by SOME case without being forced.  Each case: one step from a
random state against the oracle (Eq. 6), then a short run whose returned points must score exactly."""
import numpy as np
import pytest

from paper_2509_21064_b200 import workloads as wl
from tests.helpers import oracle_problem, hyper_kwargs

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

TOL_STEP = 1e-5


@pytest.fixture(scope="module")
def api():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2509_21064_b200 import api as _api
    _api.lib()
    return _api


def f32(v):
    return float(np.float32(v))


def okw(h, **over):
    d = hyper_kwargs(h, **over)
    for k in ("alpha", "beta", "delta", "log_eps"):
        d[k] = f32(d[k])
    return d


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def random_sparse_qubo(rng):
    """Symmetric integer Q with a random degree profile (a few long rows, isolated rows, a diagonal, a linear term)."""
    n = int(rng.integers(1, 260))
    deg = int(rng.choice([0, 1, 3, 6, 9, 20, 50]))
    m = min(n * (n - 1) // 2, n * deg // 2)
    e = wl.edges_gnm(n, m, int(rng.integers(1 << 30))) if m > 0 else np.zeros((0, 2), dtype=np.int64)
    if n > 40 and rng.random() < 0.3:                           # a hub
        hub = np.stack([np.zeros(n - 1, dtype=np.int64), np.arange(1, n)], axis=1)
        e = np.unique(np.concatenate([e, hub]), axis=0)
    w = rng.integers(-3, 4, size=e.shape[0]).astype(np.float32)
    Q = np.zeros((n, n), dtype=np.float32)
    Q[e[:, 0], e[:, 1]] = Q[e[:, 1], e[:, 0]] = w
    Q[np.arange(n), np.arange(n)] = rng.integers(-2, 3, size=n)
    c = rng.integers(-3, 4, size=n).astype(np.float32)
    rowptr, col, val = [0], [], []
    for i in range(n):
        nz = np.nonzero(Q[i])[0]
        col += list(nz); val += list(Q[i, nz]); rowptr.append(len(col))
    return wl.QuboCSR(n, np.array(rowptr, np.int32), np.array(col, np.int32), np.array(val, np.float32), c)


@pytest.mark.parametrize("seed", range(60))
def test_random_sparse_qubo(api, oracle, seed):
    rng = np.random.default_rng(1000 + seed)
    Pw = random_sparse_qubo(rng)
    n = Pw.n
    B = int(rng.choice([1, 2, 5, 10, 12, 33, 64, 100, 130, 260]))
    dual = int(rng.random() < 0.3)
    scale = float(np.abs(Pw.val).sum() / max(n, 1) + 4.0)
    h = wl.Hyper(3.0, 0.2 / scale, (0.05 / n) if dual else 0.05, 1e-4, int(rng.integers(0, 2)), 1e-6, 120, 50, seed, dual)
    OP = oracle_problem(Pw)
    P = api.create_from_workload(Pw)
    X = rng.random((n, B), dtype=np.float32)
    X[:, 0] = np.round(X[:, 0])
    lam = 3.0 if dual or rng.random() < 0.5 else (3.0 * rng.random((n, B))).astype(np.float32)
    r1 = P.run(dev(X), lam if np.isscalar(lam) else dev(lam), api.params_from_hyper(h, iters=1, eval_every=1), want_final=True)
    ref = oracle.run(OP, X, f32(lam) if np.isscalar(lam) else lam, **okw(h, iters=1, eval_every=1))
    assert np.abs(r1["x"].cpu().numpy() - ref["x"]).max() <= TOL_STEP, (n, B, dual)
    tol_y = TOL_STEP * np.maximum(1.0, np.abs(ref["y"])) + (1e-6 * f32(h.beta) * n if dual else 0.0)
    assert (np.abs(r1["lam"].cpu().numpy() - ref["y"]) <= tol_y).all(), (n, B, dual)
    r = P.run(dev(X), 3.0, api.params_from_hyper(h), want_final=True)
    obj, xb = r["obj"].cpu().numpy(), r["x_bin"].cpu().numpy()
    assert np.array_equal(obj, oracle.F_binary(OP, xb)) and int(r["best_restart"].item()) == int(np.argmin(obj))
    G = P.grad(dev(X)).cpu().numpy()
    Gref = oracle.grad(OP, X.astype(np.float64))
    assert (np.abs(G - Gref).max(axis=0) <= TOL_STEP * np.maximum(np.abs(Gref).max(axis=0), 1.0)).all()
    P.destroy()


@pytest.mark.parametrize("seed", range(30))
def test_random_literal_products(api, oracle, seed):
    rng = np.random.default_rng(2000 + seed)
    n = int(rng.integers(2, 200))
    kmax = int(rng.integers(1, min(n, 7) + 1))
    S = wl.random_pubo(n, int(rng.integers(1, 6 * n)), kmax, 3000 + seed)
    if rng.random() < 0.5:
        S.w = np.abs(S.w)                                      # plain weighted MaxSAT
    B = int(rng.choice([1, 3, 10, 40, 64, 70, 132]))
    dual = int(rng.random() < 0.25)
    h = wl.Hyper(2.0, 0.01, (0.005 / n) if dual else 0.005, 1e-4, int(rng.integers(0, 2)), 1e-6, 120, 50, seed, dual)
    OP = oracle_problem(S)
    P = api.create_from_workload(S)
    X = rng.random((n, B), dtype=np.float32)
    X[:, 0] = np.round(X[:, 0])
    r1 = P.run(dev(X), 2.0, api.params_from_hyper(h, iters=1, eval_every=1), want_final=True)
    ref = oracle.run(OP, X, 2.0, **okw(h, iters=1, eval_every=1))
    gmax = max(1.0, float(np.abs(oracle.grad(OP, X.astype(np.float64))).max()))
    assert np.abs(r1["x"].cpu().numpy() - ref["x"]).max() <= TOL_STEP * max(1.0, f32(h.alpha) * gmax), (n, B, kmax, dual)
    r = P.run(dev(X), 2.0, api.params_from_hyper(h))
    obj = r["obj"].cpu().numpy()
    assert np.array_equal(obj, oracle.F_binary(OP, r["x_bin"].cpu().numpy()))
    P.destroy()


@pytest.mark.parametrize("seed", range(20))
def test_random_maxkcut(api, seed):
    kcut = pytest.importorskip("oracle.kcut")
    rng = np.random.default_rng(4000 + seed)
    n = int(rng.integers(4, 220))
    k = int(rng.integers(2, 6))
    m = int(min(n * (n - 1) // 2, n * int(rng.choice([1, 3, 10, 30])) // 2 + 1))
    w = wl.maxkcut(n, m, k, B=int(rng.choice([1, 6, 10, 64, 100, 132])), seed=5000 + seed, weights="pm1" if seed % 2 else "unit")
    Pw, h = w.problem, w.hyper
    OP = kcut.Problem(n, k, Pw.rowptr, Pw.col, Pw.val.astype(np.float64))
    P = api.create_from_workload(Pw)
    Z = (2.0 * rng.standard_normal((k, n, w.B))).astype(np.float32)
    r1 = P.run(dev(Z), h.lambda0, api.params_from_hyper(h, iters=1, eval_every=1), want_final=True)
    ref = kcut.run(OP, Z, f32(h.lambda0), alpha=f32(h.alpha), beta=f32(h.beta), gfun=h.gfun, log_eps=f32(h.log_eps), iters=1, eval_every=1)
    assert (np.abs(r1["x"].cpu().numpy() - ref["z"]) <= TOL_STEP * np.maximum(1.0, np.abs(ref["z"]))).all(), (n, k, m, w.B)
    r = P.run(dev(Z), h.lambda0, api.params_from_hyper(h, iters=120, eval_every=50))
    assert np.array_equal(r["obj"].cpu().numpy(), kcut.objective(OP, r["x_bin"].cpu().numpy()))
    P.destroy()


@pytest.mark.parametrize("seed", range(10))
def test_random_dense_qubo(api, oracle, seed):
    """Dense path at random (mostly ragged) sizes: zero padding of variables and restarts, every cluster shape the sizes allow.
    Tolerances: the north star's 1e-2 on the gradient (bf16 operand, reading R13) and what it implies for one step."""
    rng = np.random.default_rng(6000 + seed)
    n = int(rng.choice([1, 7, 100, 255, 256, 300, 513, 700]))
    B = int(rng.choice([1, 10, 128, 130, 256, 300, 512]))
    A = rng.standard_normal((n, n)).astype(np.float32)
    Q = np.triu(A, 1) + np.triu(A, 1).T + np.diag(rng.standard_normal(n)).astype(np.float32)
    Q = torch.from_numpy(Q).to(torch.bfloat16).to(torch.float32).numpy()          # bf16-representable (reading R13)
    c = rng.standard_normal(n).astype(np.float32)
    Pw = wl.QuboDense(n, Q, c)
    s = 2.0 * np.sqrt(n)
    h = wl.Hyper(1.75 * s, 1.0 / (4.0 * (s + 1.75 * s)), 4.0 * 1.75 * s / 1000.0, 1e-4, int(rng.integers(0, 2)), 1e-6, 120, 50, seed)
    OP = oracle_problem(Pw)
    P = api.create_from_workload(Pw)
    X = rng.random((n, B), dtype=np.float32)
    G = P.grad(dev(X)).cpu().numpy()
    Gref = oracle.grad(OP, X.astype(np.float64))
    gmax = np.maximum(np.abs(Gref).max(axis=0), 1.0)
    assert (np.abs(G - Gref).max(axis=0) <= 1e-2 * gmax).all(), (n, B)
    r1 = P.run(dev(X), h.lambda0, api.params_from_hyper(h, iters=1, eval_every=1), want_final=True)
    ref = oracle.run(OP, X, f32(h.lambda0), **okw(h, iters=1, eval_every=1))
    assert (np.abs(r1["x"].cpu().numpy() - ref["x"]).max(axis=0) <= f32(h.alpha) * 1e-2 * gmax + 1e-5).all(), (n, B)
    assert np.abs(r1["lam"].cpu().numpy() - ref["y"]).max() <= TOL_STEP * max(1.0, f32(h.lambda0))
    r = P.run(dev(X), h.lambda0, api.params_from_hyper(h))
    obj, Fref = r["obj"].cpu().numpy(), oracle.F_binary(OP, r["x_bin"].cpu().numpy())
    assert np.allclose(obj, Fref, rtol=1e-5, atol=1e-5 * max(1.0, float(np.abs(Q).sum()) / max(n, 1)) * n)
    assert int(r["best_restart"].item()) == int(np.argmin(obj))
    P.destroy()
