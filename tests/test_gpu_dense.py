"""GPU parity of the DENSE path (tcgen05 GEMM gradient + fused update, config 4) against the CPU oracle, on every
launch variant the library has: single CTAs (CG=1), CTA pairs (CG=2), clusters of two pairs with the A multicast and
clusters of four pairs (2 x 2) with the A and Q multicast -- the variant config 4 runs.

north_star requirements, as for every config: (b) teacher-forced single steps (gradient within 1e-2 on the bf16
path), here with the DEFAULT delta so that the perturbation branch of the epilogue is compared too; (c) free-running
trajectories within 1e-3 after 50 steps (delta = 0 and 1e-4); the exact-1/2 tie-break, bit for bit, which is the only
check of the (t, i, b) the epilogue feeds the hash (reading R3).  The oracle runs on sampled restart
columns (restarts are independent; `col_ids` hands it the true column index for the hash).
"""
import numpy as np
import pytest

from paper_2509_21064_b200 import workloads as wl
from tests.helpers import oracle_problem, hyper_kwargs

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

TOL_STEP = 1e-5
TOL_TRAJ = 1e-3
TOL_GRAD_BF16 = 1e-2
U_BF16 = 2.0 ** -8          # unit roundoff of bf16 (8 significant bits, round to nearest)


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


def variants():
    """(name, workload): one per launch variant of dense_gemm_kernel, plus a cluster shape with 4 units per cluster."""
    return [("single_cta", wl.config(4, B=128, n_scale=0.0625)),          # n=256,  B=128 : CG=1
            ("single_cta_3x", wl.config(4, B=384, n_scale=0.125)),        # n=512,  B=384 : CG=1, three restart blocks
            ("pair", wl.config(4, B=256, n_scale=0.1875)),                # n=768,  B=256 : CG=2, NP=1
            ("cluster", wl.config(4, B=256, n_scale=0.25)),               # n=1024, B=256 : CG=2, 1 x 2 pairs (cluster of 4), A multicast
            ("cluster8", wl.config(4, B=512, n_scale=0.25)),              # n=1024, B=512 : CG=2, 2 x 2 pairs (cluster of 8), A and Q multicast
            ("cluster8_10", wl.config(4, B=1024, n_scale=0.625)),         # n=2560, B=1024: ten clusters of 8
            ("cluster8_units", wl.config(4, B=2048, n_scale=0.5)),        # n=2048, B=2048: clusters of 8 with two units each (forced:
                                                                          # the library would pick clusters of 4 for this size)
            ("ragged", wl.config(4, B=200, n_exact=300)),                 # n=300,  B=200 : zero-padded to 512 x 256 (a CTA pair)
            ("ragged_small", wl.config(4, B=12, n_exact=70))]             # n=70,   B=12  : padded to 256 x 128 (one CTA)


VARIANTS = variants()
IDS = [v[0] for v in VARIANTS]


def create(api, name, problem):
    """gda_create_qubo_dense; GDA_OPT_DENSE_SHAPE = 3 forces the cluster-of-8 launch shape on this handle where asked."""
    P = api.create_from_workload(problem)
    if name == "cluster8_units":
        P.set_option(api.OPT_DENSE_SHAPE, 3)
    return P


def sample_columns(B, k=24):
    """The first and last columns of every 128-restart block edge plus a seeded sample: every epilogue warp position."""
    rng = np.random.default_rng(B)
    fixed = [0, 1, 31, 32, 127, B - 128, B - 97, B - 4, B - 1] + ([128, 255] if B > 256 else [])
    fixed = [c for c in fixed if 0 <= c < B]
    extra = rng.choice(B, size=min(k, B), replace=False).tolist()
    return np.array(sorted(set(fixed + extra)), dtype=np.int32)


def grad_sigma(Pw, X):
    """Standard deviation of the gradient error the bf16 operand causes: G = 2 Q_off zh + h with
    zh = bf16(z), z = x - 1/2; the rounding errors e_j = zh_j - z_j are independent, |e_j| <= u |z_j|, variance
    <= (u z_j)^2 / 3, so  sd(G_i - G_ref_i) <= 2 u / sqrt(3) * sqrt(sum_j Q_ij^2 z_j^2)."""
    Q = Pw.Q.astype(np.float64).copy()
    np.fill_diagonal(Q, 0.0)
    z = X.astype(np.float64) - 0.5
    return 2.0 * U_BF16 / np.sqrt(3.0) * np.sqrt((Q * Q) @ (z * z))


def assert_dense_step_close(xg, x_prev, y_prev, cols, OP, oracle, kw, tol):
    """|x+ - x+_ref| <= tol elementwise, except where rounding of the TENTATIVE iterate decides the discrete
    perturbation branch (reading R3; tests/test_gpu_parity.py::assert_x_step_close): an in-band x^t whose tentative
    x~ lies within tol of 1/2 (the side) or of the band edge (perturb or not) may take either branch."""
    ref = oracle.run(OP, x_prev, y_prev, col_ids=cols, nthreads=8, **kw)
    err = np.abs(xg - ref["x"])
    delta = kw["delta"]
    bad = err > tol
    if delta <= 0 or not bad.any():
        assert not bad.any(), (err.max(), float(tol.min()))
        return ref, 0.0
    tent = oracle.run(OP, x_prev, y_prev, col_ids=cols, nthreads=8, **dict(kw, delta=0.0))["x"]
    in_band = np.abs(x_prev.astype(np.float64) - 0.5) < delta
    d = np.abs(tent - 0.5)
    ambiguous = in_band & ((d < tol) | (np.abs(d - delta) < tol))
    assert not (bad & ~ambiguous).any(), float(err[bad & ~ambiguous].max())
    cand = np.stack([tent, np.full_like(tent, 0.5 - delta), np.full_like(tent, 0.5 + delta)])
    # one ulp of slack on the band edges: reading R3a steps one ulp away when 1/2 +- delta rounds inside the band
    assert (np.abs(cand - xg[None]).min(axis=0)[ambiguous] <= tol[ambiguous] + 1e-7).all()
    return ref, float(ambiguous.mean())


@pytest.mark.parametrize("name,w", VARIANTS, ids=IDS)
def test_dense_teacher_forced_steps_default_delta(api, oracle, name, w):
    """(b) on every variant, with the perturbation ON.  Gradient: within the north star's 1e-2 AND within 8 standard
    deviations of the bf16 rounding model; x+: alpha times that; y+: 1e-5 (no GEMM in the dual step)."""
    OP = oracle_problem(w.problem)
    P = create(api, name, w.problem)
    n, B, h = w.problem.n, w.B, w.hyper
    cols = sample_columns(B)
    ci = torch.from_numpy(cols).long().cuda()
    x = dev(wl.x0_uniform(n, B, w.x0_seed))
    lam = torch.full((n, B), h.lambda0, dtype=torch.float32, device="cuda")
    t = 0
    perturbed_seen = 0
    for hop in (0, 1, 60, 240, 400):
        if hop:
            r = P.run(x, lam, api.params_from_hyper(h, iters=hop, eval_every=50, t0=t), want_final=True)
            x, lam, t = r["x"], r["lam"], t + hop
        xp, lp = x[:, ci].cpu().numpy(), lam[:, ci].cpu().numpy()
        Gref = oracle.grad(OP, xp.astype(np.float64))
        G = P.grad(x)[:, ci].cpu().numpy().astype(np.float64)
        gmax = np.maximum(np.abs(Gref).max(axis=0, keepdims=True), 1.0)
        sig = grad_sigma(w.problem, xp)
        assert (np.abs(G - Gref) <= TOL_GRAD_BF16 * gmax).all()                                  # north star (b), bf16 path
        assert (np.abs(G - Gref) <= 8.0 * sig + TOL_STEP * gmax).all(), float((np.abs(G - Gref) / (8.0 * sig + TOL_STEP * gmax)).max())
        tol_x = f32(h.alpha) * (8.0 * sig + TOL_STEP * gmax) + TOL_STEP
        # the default delta = 1e-4, and a wide band (2e-2) that catches about a tenth of the entries once the iterates
        # have settled (the fixed point of the convex start sits near, not at, 1/2 when the linear term is non-zero)
        for delta in (h.delta, 2e-2):
            r1 = P.run(x, lam, api.params_from_hyper(h, iters=1, eval_every=1, t0=t, delta=delta), want_final=True)
            xg, yg = r1["x"][:, ci].cpu().numpy().astype(np.float64), r1["lam"][:, ci].cpu().numpy().astype(np.float64)
            ref, amb = assert_dense_step_close(xg, xp, lp, cols, OP, oracle, okw(h, iters=1, eval_every=1, t0=t, delta=delta), tol_x)
            assert (np.abs(yg - ref["y"]) / np.maximum(1.0, np.abs(ref["y"]))).max() <= TOL_STEP, (name, t)
            in_band = np.abs(xp.astype(np.float64) - 0.5) < f32(delta)
            perturbed_seen += int((in_band & (np.abs(np.abs(ref["x"] - 0.5) - f32(delta)) < 1e-6)).sum())
            assert amb < 0.05, (name, t, amb)
    assert perturbed_seen > 20, "too few perturbed entries were compared: the states do not reach the band"
    P.destroy()


@pytest.mark.parametrize("delta", [0.0, 1e-4])
@pytest.mark.parametrize("name,w", VARIANTS, ids=IDS)
def test_dense_free_running_50_steps(api, oracle, name, w, delta):
    """(c): 50 free-running steps from x0, max |x - x_ref| <= 1e-3 against the fp64 oracle on sampled columns."""
    OP = oracle_problem(w.problem)
    P = create(api, name, w.problem)
    n, B, h = w.problem.n, w.B, w.hyper
    cols = sample_columns(B)
    ci = torch.from_numpy(cols).long().cuda()
    X0 = wl.x0_uniform(n, B, w.x0_seed)
    r = P.run(dev(X0), h.lambda0, api.params_from_hyper(h, iters=50, eval_every=25, delta=delta), want_final=True)
    ref = oracle.run(OP, X0[:, cols], f32(h.lambda0), col_ids=cols, nthreads=8, **okw(h, iters=50, eval_every=25, delta=delta))
    ex = np.abs(r["x"][:, ci].cpu().numpy() - ref["x"])
    ey = np.abs(r["lam"][:, ci].cpu().numpy() - ref["y"])
    print(f"dense free-running 50 steps [{name}, delta={delta}]: max|dx| = {ex.max():.3e}, max|dy| = {ey.max():.3e}")
    assert ex.max() <= TOL_TRAJ
    # y+ = y + beta g(x), |g'| <= 1: the dual inherits at most beta * |dx| per step, plus half an ulp of y (fp32) per addition
    assert ey.max() <= 50 * (f32(h.beta) * TOL_TRAJ + 2.0 ** -24 * h.lambda0)
    # (a) on the way: the objective of the returned points, sampled columns, fp64 with the dense path's relative tolerance
    xb = r["x_bin"][:, ci].cpu().numpy()
    Fref = oracle.F_binary(OP, xb)
    tolF = 1e-5 * (xb.astype(np.float64).T @ np.abs(w.problem.Q.astype(np.float64)) @ xb.astype(np.float64)).diagonal() + 1e-3
    assert (np.abs(r["obj"].cpu().numpy()[cols] - Fref) <= tolF).all()
    P.destroy()


def integer_dense_qubo_with_zero_gradient_at_half(n, seed):
    """Integer Q (bf16-exact) and c = -(Q_off 1 + diag Q): grad f(1/2 * 1) = Q_off 1 + c + diag(Q) = 0 EXACTLY in
    fp32 and fp64, the dense analogue of the Max-Cut fixed point of PAPER.md:146."""
    rng = np.random.default_rng(seed)
    A = np.triu(rng.integers(-2, 3, size=(n, n)), 1).astype(np.float32)
    Q = A + A.T
    d = rng.integers(-3, 4, size=n).astype(np.float32)
    Q[np.arange(n), np.arange(n)] = d
    c = -(A + A.T).sum(axis=1) - d
    return wl.QuboDense(n=n, Q=Q, c=c.astype(np.float32))


@pytest.mark.parametrize("n,B", [(256, 128), (768, 256), (1024, 256), (1536, 512), (300, 200)], ids=["single_cta", "pair", "cluster", "cluster8_units", "ragged"])
def test_dense_tie_break_at_exact_half_matches_oracle(api, oracle, n, B):
    """x = 1/2 everywhere and a zero gradient: x~ = x = 1/2 exactly, so the side of the perturbation is the hash bit of
    (seed, t, i, b) for EVERY element (reading R3).  Bit-for-bit against the oracle's fp32 build."""
    Pw = integer_dense_qubo_with_zero_gradient_at_half(n, 17 + n)
    OP = oracle_problem(Pw)
    P = api.create_from_workload(Pw)
    X = np.full((n, B), 0.5, dtype=np.float32)
    assert np.abs(P.grad(dev(X)).cpu().numpy()).max() == 0.0
    seed = (9 << 32) | 1234567
    h = wl.Hyper(100.0, 1e-3, 0.5, 1e-3, 0, 1e-6, 1, 1, seed)
    for t0 in (0, 11, 70001):
        r = P.run(dev(X), 100.0, api.params_from_hyper(h, t0=t0), want_final=True)
        ref = oracle.run(OP, X, 100.0, precision="f32", nthreads=8, **okw(h, t0=t0))
        xg = r["x"].cpu().numpy()
        assert np.array_equal(xg, ref["x"]), (t0, float((xg != ref["x"]).mean()))
        vals, cnt = np.unique(xg, return_counts=True)
        assert len(vals) == 2 and cnt.min() > 0.4 * n * B               # both sides, about half each
    # t advances inside a chunk (t_off) and across chunks (the device counter): three steps, delta larger than any move
    h3 = wl.Hyper(100.0, 1e-3, 0.5, 1e-3, 0, 1e-6, 3, 2, seed)
    r = P.run(dev(X), 100.0, api.params_from_hyper(h3, t0=5), want_final=True)
    ref = oracle.run(OP, X, 100.0, precision="f64", nthreads=8, **okw(h3, t0=5))
    assert np.abs(r["x"].cpu().numpy() - ref["x"]).max() <= 1e-3 * 1e-2 * 2 * n + 1e-5
    P.destroy()


@pytest.mark.parametrize("name,w", [VARIANTS[0], VARIANTS[3], VARIANTS[7], VARIANTS[8]], ids=[IDS[0], IDS[3], IDS[7], IDS[8]])
def test_dense_lagrangian_and_dual_bound(api, oracle, name, w):
    """gda_lagrangian on the dense path: L(x, y) = f(x) + sum_i y_i g(x_i) with f from the tcgen05
    gradient, f = sum_i x_i (G_i + c'_i) / 2.  Tolerance: the bf16 operand's effect on f, |x|^T sigma(G) / 2 by the
    rounding model of grad_sigma (8 standard deviations of a sum of independent terms), plus fp32 products."""
    OP = oracle_problem(w.problem)
    P = create(api, name, w.problem)
    n, B = w.problem.n, w.B
    rng = np.random.default_rng(31)
    X = rng.random((n, B), dtype=np.float32)
    X[:, 0] = X[:, 0] > 0.5                                     # a binary column: z = +-1/2 is exact in bf16 and L = F
    Y = rng.normal(size=(n, B)).astype(np.float32)
    cols = sample_columns(B, 12)
    sig = grad_sigma(w.problem, X[:, cols])
    tol_f = 8.0 * 0.5 * np.sqrt(((X[:, cols].astype(np.float64) * sig) ** 2).sum(axis=0))
    for lam, lam_ref in ((dev(Y), Y[:, cols].astype(np.float64)), (1.5, 1.5)):
        got = P.lagrangian(dev(X), lam).cpu().numpy()[cols]
        ref = oracle.lagrangian(OP, X[:, cols].astype(np.float64), lam_ref, 0)
        scale = np.abs(oracle.f_ext(OP, X[:, cols].astype(np.float64))) + np.abs(ref) + n
        assert (np.abs(got - ref) <= tol_f + 1e-5 * scale).all(), float((np.abs(got - ref) / (tol_f + 1e-5 * scale)).max())
    F0 = oracle.F_binary(OP, X[:, :1].astype(np.uint8))[0]
    assert abs(P.lagrangian(dev(X), dev(Y))[0].item() - F0) <= 1e-5 * (np.abs(w.problem.Q).sum() + n)
    P.destroy()
