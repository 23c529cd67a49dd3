"""Any number of restarts B >= 1 (the paper runs B = 1, 10, 100, 1000: Table 6, 873-878 Table 10).

The kernels work on float4s of restarts (the dense path on 128-restart tiles), so the library pads the restart axis with
zero-initialised PADDING RESTARTS up to the next multiple of 4 (128) inside its workspace.  They run like any other restart
and must never be seen: not by the evaluation, the trace, the arg-best or the copies out.  Checked here, for every problem
kind and launch path, against the oracle AND against a run of the same columns at a multiple of 4 (restarts are independent,
PAPER.md:212, so the first B columns must agree bit for bit).
"""
import numpy as np
import pytest

from paper_2509_21064_b200 import workloads as wl
from tests.helpers import oracle_problem, hyper_kwargs, create_problem

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


@pytest.fixture(scope="module")
def oracle():
    from oracle import pdbo
    pdbo.build()
    return pdbo


def f32(v):
    return float(np.float32(v))


def okw(h, **over):
    d = hyper_kwargs(h, **over)
    for k in ("alpha", "beta", "delta", "log_eps"):
        d[k] = f32(d[k])
    return d


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def workload(kind, B):
    """(workload, sparse path) of a launch path at B restarts."""
    if kind == "slab":
        return wl.config(2, B=B, n_scale=0.25), "slab"
    if kind == "stream":                                      # B <= 64: spmm_step_narrow, else spmm_step_warp
        return wl.config(3, B=B, n_scale=0.05), "stream"
    if kind == "maxsat":
        return wl.config(5, B=B, n_scale=0.05), None
    if kind == "maxsat_quadratic":
        w = wl.config(5, B=B, n_scale=0.03)
        w.hyper.gfun = 0
        return w, None
    if kind == "pdbo_s":
        return wl.pdbo_s_variant(wl.config(3, B=B, n_scale=0.05)), "stream"
    if kind == "pdbo_s_slab":
        return wl.pdbo_s_variant(wl.config(2, B=B, n_scale=0.25)), "slab"
    if kind == "pdbo_s_maxsat":
        return wl.pdbo_s_variant(wl.config(5, B=B, n_scale=0.05)), None
    if kind == "dense":
        return wl.config(4, B=B, n_scale=0.0625), None
    raise ValueError(kind)


CASES = [("slab", 1), ("slab", 10), ("slab", 13), ("stream", 1), ("stream", 10), ("stream", 70), ("stream", 131),
         ("maxsat", 3), ("maxsat", 10), ("maxsat", 130), ("maxsat_quadratic", 6), ("pdbo_s", 10), ("pdbo_s", 70), ("pdbo_s_slab", 10), ("pdbo_s_slab", 13),
         ("pdbo_s_maxsat", 10), ("dense", 10), ("dense", 1)]


@pytest.mark.parametrize("kind,B", CASES, ids=lambda v: str(v))
def test_run_at_any_B(api, oracle, kind, B):
    w, path = workload(kind, B)
    h, n = w.hyper, w.problem.n
    scalar = getattr(h, "dual", 0) == 1
    OP = oracle_problem(w.problem)
    P = create_problem(api, w, sparse_path=path)
    Bp = (B + 3) // 4 * 4
    X0p = np.zeros((n, Bp), dtype=np.float32)
    X0p[:, :B] = wl.x0_uniform(n, B, w.x0_seed)
    X0 = np.ascontiguousarray(X0p[:, :B])

    # one step against the oracle (teacher-forced, from x0)
    r1 = P.run(dev(X0), h.lambda0, api.params_from_hyper(h, iters=1, eval_every=1), want_final=True)
    assert r1["x"].shape == (n, B) and r1["x_bin"].shape == (n, B) and r1["obj"].shape == (B,)
    assert r1["lam"].shape == ((B,) if scalar else (n, B))
    ref = oracle.run(OP, X0, f32(h.lambda0), **okw(h, iters=1, eval_every=1))
    tol_x = TOL_STEP if kind != "dense" else 2e-3             # bf16 operand on the dense path (tests/test_gpu_dense.py)
    assert np.abs(r1["x"].cpu().numpy() - ref["x"]).max() <= tol_x
    ylam = r1["lam"].cpu().numpy()
    assert (np.abs(ylam - ref["y"]) <= TOL_STEP * np.maximum(1.0, np.abs(ref["y"])) + (1e-6 * f32(h.beta) * n if scalar else 0.0)).all()

    # a run of 230 iterations (ragged last chunk): exact objectives, arg-best and trace over the B real restarts only
    prm = api.params_from_hyper(h, iters=230, eval_every=50)
    r = P.run(dev(X0), h.lambda0, prm, want_final=True, trace_cap=16)
    obj, x_bin = r["obj"].cpu().numpy(), r["x_bin"].cpu().numpy()
    F = oracle.F_binary(OP, x_bin)
    if kind == "dense":
        assert np.allclose(obj, F, rtol=1e-5, atol=1e-2)
    else:
        assert np.array_equal(obj, F)
    best = int(r["best_restart"].item())
    assert 0 <= best < B and best == int(np.argmin(obj)) and float(r["best_obj"].item()) == obj.min()
    tb = r["trace_best"].cpu().numpy()[:5]
    assert np.all(np.diff(tb) <= 0) and tb[-1] == obj.min()

    # the same columns inside a run at the next multiple of 4: bit-identical (restarts are independent)
    if Bp != B:
        rp = P.run(dev(X0p), h.lambda0, prm, want_final=True)
        for k in ("x", "x_bin"):
            assert torch.equal(rp[k][:, :B], r[k]), k
        assert torch.equal(rp["obj"][:B], r["obj"])
        assert torch.equal(rp["lam"][..., :B], r["lam"])
        # and a resumed run keeps working at this B
        a = P.run(dev(X0), h.lambda0, api.params_from_hyper(h, iters=100, eval_every=50), want_final=True)
        a = P.resume(api.params_from_hyper(h, iters=130, eval_every=50), a)
        torch.cuda.synchronize()
        assert torch.equal(a["obj"], r["obj"]) and torch.equal(a["x_bin"], r["x_bin"])
    P.destroy()


@pytest.mark.parametrize("kind,B", [("slab", 10), ("stream", 70), ("maxsat", 10), ("dense", 10)], ids=lambda v: str(v))
def test_gradient_score_lagrangian_at_any_B(api, oracle, kind, B):
    w, path = workload(kind, B)
    n = w.problem.n
    OP = oracle_problem(w.problem)
    P = create_problem(api, w, sparse_path=path)
    rng = np.random.default_rng(9)
    X = rng.random((n, B), dtype=np.float32)
    X[:, 0] = X[:, 0] > 0.5
    G = P.grad(dev(X)).cpu().numpy()
    Gref = oracle.grad(OP, X.astype(np.float64))
    rel = (np.abs(G - Gref).max(axis=0) / np.maximum(np.abs(Gref).max(axis=0), 1.0)).max()
    assert G.shape == (n, B) and rel <= (TOL_STEP if kind != "dense" else 1e-2)
    obj = P.score(dev(X)).cpu().numpy()
    F = oracle.F_binary(OP, (X > 0.5).astype(np.uint8))
    assert obj.shape == (B,)
    assert np.array_equal(obj, F) if kind != "dense" else np.allclose(obj, F, rtol=1e-5, atol=1e-2)
    lam = rng.random((n, B), dtype=np.float32) * 3.0
    for gfun in (0, 1):
        L = P.lagrangian(dev(X), dev(lam), gfun=gfun, log_eps=1e-6).cpu().numpy()
        Lref = oracle.lagrangian(OP, X.astype(np.float64), lam.astype(np.float64), gfun)
        tol = 1e-5 * np.maximum(1.0, np.abs(Lref)) if kind != "dense" else 5e-3 * np.maximum(np.abs(Lref), n)   # dense: bf16 operand
        assert L.shape == (B,) and (np.abs(L - Lref) <= tol).all()
    P.destroy()


def test_maxkcut_at_any_B(api):
    kcut = pytest.importorskip("oracle.kcut")
    w = wl.maxkcut(300, 900, 3, B=10, seed=21, weights="pm1")
    Pw, h = w.problem, w.hyper
    n, k, B = Pw.n, Pw.k, w.B
    OK = kcut.Problem(n, k, Pw.rowptr, Pw.col, Pw.val.astype(np.float64))
    P = api.create_from_workload(Pw)
    Z0p = np.zeros((k, n, 12), dtype=np.float32)
    Z0p[:, :, :B] = wl.z0_uniform(k, n, B, w.x0_seed)
    Z0 = np.ascontiguousarray(Z0p[:, :, :B])
    kw = dict(alpha=f32(h.alpha), beta=f32(h.beta), gfun=h.gfun, log_eps=f32(h.log_eps))
    r1 = P.run(dev(Z0), h.lambda0, api.params_from_hyper(h, iters=1, eval_every=1), want_final=True)
    ref = kcut.run(OK, Z0, f32(h.lambda0), iters=1, eval_every=1, **kw)
    assert r1["x"].shape == (k, n, B)
    assert np.abs(r1["x"].cpu().numpy() - ref["z"]).max() <= TOL_STEP
    assert np.abs(r1["lam"].cpu().numpy() - ref["y"]).max() <= TOL_STEP * max(1.0, f32(h.lambda0))
    prm = api.params_from_hyper(h, iters=230, eval_every=50)
    r = P.run(dev(Z0), h.lambda0, prm, want_final=True)
    obj, lab = r["obj"].cpu().numpy(), r["x_bin"].cpu().numpy()
    assert np.array_equal(obj, kcut.objective(OK, lab))
    assert int(r["best_restart"].item()) == int(np.argmin(obj))
    rp = P.run(dev(Z0p), h.lambda0, prm, want_final=True)
    assert torch.equal(rp["x"][:, :, :B], r["x"]) and torch.equal(rp["obj"][:B], r["obj"]) and torch.equal(rp["x_bin"][:, :B], r["x_bin"])
    sc = P.score(dev(Z0)).cpu().numpy()                        # labels of given logits
    assert np.array_equal(sc, kcut.objective(OK, np.argmax(Z0, axis=0).astype(np.uint8)))
    P.destroy()


def test_mis_ones_and_host_run_at_B_10(api, oracle):
    """The paper's MIS setting (B = 10): |S| per restart (gda_extra.ones) and the host-buffer entry point."""
    w = wl.mis(600, 3, B=10)
    h, n, B = w.hyper, w.problem.n, w.B
    OP = oracle_problem(w.problem)
    P = create_problem(api, w)
    X0 = wl.x0_uniform(n, B, w.x0_seed)
    prm = api.params_from_hyper(h, iters=300)
    r = P.run(dev(X0), h.lambda0, prm, want_ones=True)
    obj, xb, ones = r["obj"].cpu().numpy(), r["x_bin"].cpu().numpy(), r["ones"].cpu().numpy()
    assert ones.shape == (B,) and np.array_equal(ones, xb.sum(axis=0)) and np.array_equal(obj, oracle.F_binary(OP, xb))
    rh = P.run_host(X0, h.lambda0, prm)
    assert np.array_equal(rh["obj"], obj) and np.array_equal(rh["x_bin"], xb) and rh["best_restart"] == int(np.argmin(obj))
    P.destroy()


@pytest.mark.parametrize("kind,B", [("slab", 20002), ("stream", 40003), ("maxsat", 30001)], ids=lambda v: str(v))
def test_large_odd_batches(api, oracle, kind, B):
    """Tens of thousands of restarts, not a multiple of anything: hundreds of 128-restart chunks, a ragged last one."""
    w, path = workload(kind, B)
    h, n = w.hyper, w.problem.n
    OP = oracle_problem(w.problem)
    P = create_problem(api, w, sparse_path=path)
    X0 = wl.x0_uniform(n, B, 3)
    sel = np.r_[0:40, B - 40:B]                                # the first and the last restarts through the oracle
    r1 = P.run(dev(X0), h.lambda0, api.params_from_hyper(h, iters=1, eval_every=1), want_final=True)
    ref = oracle.run(OP, np.ascontiguousarray(X0[:, sel]), f32(h.lambda0), **okw(h, iters=1, eval_every=1))
    assert np.abs(r1["x"].cpu().numpy()[:, sel] - ref["x"]).max() <= TOL_STEP
    r = P.run(dev(X0), h.lambda0, api.params_from_hyper(h, iters=120, eval_every=50))
    obj, xb = r["obj"].cpu().numpy(), r["x_bin"].cpu().numpy()
    assert np.array_equal(obj[sel], oracle.F_binary(OP, np.ascontiguousarray(xb[:, sel])))
    assert int(r["best_restart"].item()) == int(np.argmin(obj))
    P.destroy()


@pytest.mark.parametrize("B", [1, 10, 13])
@pytest.mark.parametrize("kind", ["slab", "stream", "maxsat", "dense"])
def test_outputs_stay_inside_the_callers_buffers(api, kind, B):
    """Every output of gda_run is documented as [B] or [n][B]: with B not a multiple of 4 the padding restarts must not be
    stored.  Each output is a slice in the middle of a larger buffer filled with a sentinel; the bytes on both sides must be
    untouched afterwards (torch rounds allocations up to 512 bytes, so an overrun of a tensor of its own goes unnoticed:
    count_ones_kernel once wrote ones[B .. 4 ceil(B/4))."""
    import ctypes as C
    if kind == "dense":
        w, path = wl.config(4, B=B, n_exact=300), None
    else:
        w, path = workload(kind, B)
    h, n = w.hyper, w.problem.n
    P = create_problem(api, w, sparse_path=path)
    x0 = dev(wl.x0_uniform(n, B, w.x0_seed))
    PAD = 64

    def guarded(numel, dtype, sentinel):
        buf = torch.full((numel + 2 * PAD,), sentinel, dtype=dtype, device="cuda")
        return buf, buf[PAD:PAD + numel]

    bufs = dict(x_bin=guarded(n * B, torch.uint8, 0xAB), obj=guarded(B, torch.float64, -7.25), best_restart=guarded(1, torch.int32, -77),
                x_final=guarded(n * B, torch.float32, -7.25), lambda_final=guarded(n * B, torch.float32, -7.25),
                best_obj=guarded(1, torch.float64, -7.25), ones=guarded(B, torch.int32, -77),
                trace_best=guarded(8, torch.float64, -7.25), trace_ns=guarded(8, torch.int64, -77))
    ex = api.Extra()
    ex.x_final, ex.lambda_final, ex.best_obj = (bufs[k][1].data_ptr() for k in ("x_final", "lambda_final", "best_obj"))
    ex.ones, ex.trace_best, ex.trace_ns, ex.trace_cap = bufs["ones"][1].data_ptr(), bufs["trace_best"][1].data_ptr(), bufs["trace_ns"][1].data_ptr(), 8
    prm = api.params_from_hyper(h, iters=30, eval_every=7)
    st = api.lib().gda_run(P._h, B, x0.data_ptr(), None, float(h.lambda0), C.byref(prm), bufs["x_bin"][1].data_ptr(),
                           bufs["obj"][1].data_ptr(), bufs["best_restart"][1].data_ptr(), C.byref(ex),
                           torch.cuda.current_stream().cuda_stream)
    assert st == 0, api.lib().gda_last_error()
    torch.cuda.synchronize()
    for name, (buf, view) in bufs.items():
        sentinel = buf[0].item()
        assert (buf[:PAD] == sentinel).all() and (buf[PAD + view.numel():] == sentinel).all(), name
    xb = bufs["x_bin"][1].view(n, B)
    assert (xb <= 1).all() and torch.equal(bufs["ones"][1], xb.sum(dim=0).to(torch.int32))
    rescored = P.score(xb.float())
    assert torch.equal(rescored, bufs["obj"][1]) if kind != "dense" else torch.allclose(rescored, bufs["obj"][1], rtol=1e-5, atol=1e-2)
    P.destroy()
