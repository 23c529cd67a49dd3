"""GPU parity of the Max-k-Cut path (gda_create_maxkcut) against oracle/kcut_oracle.c."""
import numpy as np
import pytest

from paper_2509_21064_b200 import workloads as wl

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu
kcut = pytest.importorskip("oracle.kcut")

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


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def okw(h, **over):
    d = dict(alpha=f32(h.alpha), beta=f32(h.beta), gfun=h.gfun, log_eps=f32(h.log_eps), iters=h.iters, eval_every=h.eval_every)
    d.update(over)
    return d


def cases():
    a = wl.maxkcut(300, 900, 3, B=132, seed=21, weights="pm1")          # ragged B, +-1 weights
    b = wl.maxkcut(200, 2400, 4, B=64, seed=22)                          # degree 24, k = 4
    c = wl.maxkcut(150, 500, 5, B=8, seed=23)
    c.hyper.gfun = 1                                                     # entropy g
    c.name += "_entropy"
    d = wl.maxkcut(120, 400, 2, B=16, seed=24)
    return [a, b, c, d]


CASES = cases()


@pytest.mark.parametrize("w", CASES, ids=lambda w: w.name)
def test_teacher_forced_steps(api, w):
    Pw, h = w.problem, w.hyper
    n, k, B = Pw.n, Pw.k, w.B
    OP = kcut.Problem(n, k, Pw.rowptr, Pw.col, Pw.val.astype(np.float64))
    P = api.create_from_workload(Pw)
    z = dev(wl.z0_uniform(k, n, B, w.x0_seed))
    lam = torch.full((n, B), h.lambda0, dtype=torch.float32, device="cuda")
    for hop in (0, 1, 40, 300):                                          # states along the GPU's own trajectory
        if hop:
            r = P.run(z, lam, api.params_from_hyper(h, iters=hop, eval_every=50), want_final=True)
            z, lam = r["x"], r["lam"]
        r1 = P.run(z, lam, api.params_from_hyper(h, iters=1, eval_every=1), want_final=True)
        ref = kcut.run(OP, z.cpu().numpy(), lam.cpu().numpy(), **okw(h, iters=1, eval_every=1))
        zg, yg = r1["x"].cpu().numpy().astype(np.float64), r1["lam"].cpu().numpy().astype(np.float64)
        assert (np.abs(zg - ref["z"]) <= TOL_STEP * np.maximum(1.0, np.abs(ref["z"]))).all(), (w.name, hop)
        assert (np.abs(yg - ref["y"]) <= TOL_STEP * np.maximum(1.0, np.abs(ref["y"]))).all(), (w.name, hop)
    P.destroy()


@pytest.mark.parametrize("w", CASES, ids=lambda w: w.name)
def test_rows_split_across_the_warps_of_a_block(api, w):
    """kcut_step_kernel<.., SPLIT>: a block of 8 warps per node (slices of 8 neighbours); forced with GDA_OPT_SPLIT_ALL_ROWS = 1,
    read at every launch.  One step against the oracle and against the warp-per-node kernel, exact objectives after a run."""
    import os
    Pw, h = w.problem, w.hyper
    n, k, B = Pw.n, Pw.k, w.B
    OP = kcut.Problem(n, k, Pw.rowptr, Pw.col, Pw.val.astype(np.float64))
    P = api.create_from_workload(Pw)
    Z0 = wl.z0_uniform(k, n, B, w.x0_seed)
    out = {}
    for sw in ("1", "0"):
        P.set_option(api.OPT_SPLIT_ALL_ROWS, int(sw))
        r1 = P.run(dev(Z0), h.lambda0, api.params_from_hyper(h, iters=1, eval_every=1), want_final=True)
        r = P.run(dev(Z0), h.lambda0, api.params_from_hyper(h, iters=230, eval_every=50))
        torch.cuda.synchronize()
        ref = kcut.run(OP, Z0, f32(h.lambda0), **okw(h, iters=1, eval_every=1))
        assert (np.abs(r1["x"].cpu().numpy() - ref["z"]) <= TOL_STEP * np.maximum(1.0, np.abs(ref["z"]))).all()
        assert (np.abs(r1["lam"].cpu().numpy() - ref["y"]) <= TOL_STEP * np.maximum(1.0, np.abs(ref["y"]))).all()
        assert np.array_equal(r["obj"].cpu().numpy(), kcut.objective(OP, r["x_bin"].cpu().numpy()))
        out[sw] = r1["x"].cpu().numpy()
    assert np.abs(out["1"] - out["0"]).max() <= 2 * TOL_STEP
    P.destroy()


@pytest.mark.parametrize("w", CASES, ids=lambda w: w.name)
def test_full_run_objective_labels_and_statistics(api, w):
    Pw, h = w.problem, w.hyper
    n, k, B = Pw.n, Pw.k, w.B
    OP = kcut.Problem(n, k, Pw.rowptr, Pw.col, Pw.val.astype(np.float64))
    P = api.create_from_workload(Pw)
    Z0 = wl.z0_uniform(k, n, B, w.x0_seed)
    r50 = P.run(dev(Z0), h.lambda0, api.params_from_hyper(h, iters=50, eval_every=50), want_final=True)
    ref50 = kcut.run(OP, Z0, f32(h.lambda0), **okw(h, iters=50, eval_every=50))
    assert np.abs(r50["x"].cpu().numpy() - ref50["z"]).max() <= 1e-3                 # (c) 50 free-running steps
    iters = 2000
    r = P.run(dev(Z0), h.lambda0, api.params_from_hyper(h, iters=iters, eval_every=100), want_final=True)
    obj, lab = r["obj"].cpu().numpy(), r["x_bin"].cpu().numpy()
    assert lab.max() < k
    assert np.array_equal(obj, kcut.objective(OP, lab))                              # (a) exact objective of the returned labelings
    E, ew = Pw.edges, Pw.edge_w.astype(np.float64)
    cut = (ew[:, None] * (lab[E[:, 0]] != lab[E[:, 1]])).sum(axis=0)                 # by the edge list
    assert np.array_equal(obj, 2.0 * ew.sum() - 2.0 * cut)
    assert int(r["best_restart"].item()) == int(np.argmin(obj))
    sub = slice(0, min(B, 32))
    ref = kcut.run(OP, Z0[:, :, sub], f32(h.lambda0), nthreads=4, **okw(h, iters=iters, eval_every=100))
    sd = float(np.sqrt(0.5 * (obj[sub].var() + ref["obj"].var())))                   # (d), as assert_statistics_close
    nb = obj[sub].shape[0]
    assert abs(obj[sub].mean() - ref["obj"].mean()) <= max(0.005 * abs(ref["obj"].mean()), 3.0 * sd * np.sqrt(2.0 / nb))
    assert abs(obj[sub].min() - ref["obj"].min()) <= max(0.005 * abs(ref["obj"].min()), sd)
    # a random labeling cuts (1 - 1/k) of the weight in expectation; the method must do clearly better on unit weights
    if (ew > 0).all():
        assert cut.min() > (1 - 1 / k) * ew.sum() * 1.02
    P.destroy()


def test_arguments_and_unsupported_calls(api):
    w = CASES[3]
    Pw = w.problem
    P = api.create_from_workload(Pw)
    z = dev(wl.z0_uniform(Pw.k, Pw.n, w.B, 1))
    with pytest.raises(api.GdaError) as e:
        P.run(z, 6.0, api.params_from_hyper(w.hyper, iters=1, dual=api.DUAL_SCALAR))
    assert e.value.status == 4
    for bad_k in (1, 9):
        with pytest.raises(api.GdaError) as e:
            api.Problem.create_maxkcut(Pw.n, bad_k, Pw.rowptr, Pw.col, Pw.val)
        assert e.value.status == 1
    val = Pw.val.copy()
    rowptr = np.array([0, 1, 1], np.int32)
    with pytest.raises(api.GdaError) as e:                               # a self loop
        api.Problem.create_maxkcut(2, 3, rowptr, np.array([0], np.int32), np.array([1.0], np.float32))
    assert e.value.status == 1
    # resume: 30 + 20 steps equal 50 steps bit for bit
    a = P.run(z, 6.0, api.params_from_hyper(w.hyper, iters=50, eval_every=10), want_final=True)
    za = a["x"].clone()
    b = P.run(z, 6.0, api.params_from_hyper(w.hyper, iters=30, eval_every=10), want_final=True)
    ex = api.Extra()
    ex.x_final = b["x"].data_ptr()
    prm = api.params_from_hyper(w.hyper, iters=20, eval_every=10)
    api._check(api.lib().gda_run(P._h, w.B, None, None, 0.0, api.C.byref(prm), b["x_bin"].data_ptr(), b["obj"].data_ptr(),
                                 b["best_restart"].data_ptr(), api.C.byref(ex), torch.cuda.current_stream().cuda_stream))
    torch.cuda.synchronize()
    assert torch.equal(b["x"], za)
    P.destroy()


def test_score_of_given_logits_matches_the_oracle(api):
    """gda_score on a Max-k-Cut problem: labels = argmax_j Z_ji (lowest j on ties, reading K4), objective Tr(Xh W Xh^T)."""
    from oracle import kcut
    w = CASES[0]
    Pw = w.problem
    P = api.create_from_workload(Pw)
    OK = kcut.Problem(Pw.n, Pw.k, Pw.rowptr, Pw.col, Pw.val.astype(np.float64))
    Z = wl.z0_uniform(Pw.k, Pw.n, w.B, 9)
    Z[:, :5, 0] = 0.25                                            # ties: label 0
    obj = P.score(dev(Z)).cpu().numpy()
    lab = Z.argmax(axis=0).astype(np.uint8)                       # numpy's argmax also takes the first maximum
    assert np.array_equal(obj, kcut.objective(OK, lab))
    P.destroy()


@pytest.mark.parametrize("w", CASES[:3] + [wl.maxkcut(90, 300, 3, B=10, seed=29)], ids=lambda w: f"{w.name}_B{w.B}")
def test_gradient_and_lagrangian_of_the_softmax_form(api, w):
    """gda_grad / gda_lagrangian on Max-k-Cut problems: grad_Z Tr(X W X^T) and L(SoftMax(Z), y)."""
    Pw = w.problem
    n, k, B = Pw.n, Pw.k, w.B
    OP = kcut.Problem(n, k, Pw.rowptr, Pw.col, Pw.val.astype(np.float64))
    P = api.create_from_workload(Pw)
    rng = np.random.default_rng(3)
    Z = (2.0 * rng.standard_normal((k, n, B))).astype(np.float32)
    G = P.grad(dev(Z)).cpu().numpy()
    Gref = kcut.grad(OP, Z.astype(np.float64))
    assert G.shape == Z.shape
    assert np.abs(G - Gref).max() <= TOL_STEP * max(1.0, np.abs(Gref).max())
    Y = (3.0 * rng.random((n, B))).astype(np.float32)
    for gfun in (0, 1):
        L = P.lagrangian(dev(Z), dev(Y), gfun=gfun).cpu().numpy()
        Lref = kcut.lagrangian(OP, Z.astype(np.float64), Y.astype(np.float64), gfun)
        assert L.shape == (B,) and (np.abs(L - Lref) <= 1e-5 * np.maximum(1.0, np.abs(Lref))).all()
        Ls = P.lagrangian(dev(Z), 1.5, gfun=gfun).cpu().numpy()
        assert (np.abs(Ls - kcut.lagrangian(OP, Z.astype(np.float64), 1.5, gfun)) <= 1e-5 * np.maximum(1.0, np.abs(Lref))).all()
    P.destroy()
