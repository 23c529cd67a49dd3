"""gda_score_qubo_csr_static against gda_score: the scoring entry point for callers that cannot allocate device memory.

Some hosts of this library must not call cudaMalloc: a process whose own pool was given all of the HBM at start-up, a
loop with a latency bound (cudaMalloc / cudaFree may synchronise the whole device), a plug-in that may only touch the
buffers it was handed.  For them `gda_score_qubo_csr_static` scores rounded points of a QUBO from the CSR the caller
already keeps on the device, with its partial sums in a fixed 4 MiB `__device__` array inside the library instead of a
workspace (limit: B <= 4096 restarts; one array per GPU, shared by all calls -- overlapping calls race, calls on one
stream are ordered; the array keeps the last call's contents).

What is checked here: the objectives equal those of the existing path (`gda_create_qubo_csr` + `gda_score`, which the
parity tests pin to the oracle) on TWO CALLS IN A ROW -- the second with another problem and a smaller shape, so it runs
over whatever the first left in the array -- with the tolerance the parity tests use for scoring: bit-equal for integer
coefficients, rtol 1e-6 / atol 1e-5 otherwise (tests/test_gpu_parity.py).  This file sorts last on purpose: `pytest -x`
stops at the first failure, and a failure here must not hide any other test.  It passes alone in a fresh process (the
first call on the GPU then does the one-time address look-up) and after the other tests.
"""
import numpy as np
import pytest

from paper_2509_21064_b200 import api, build, workloads as wl


def float_qubo_csr(n, seed):
    """Symmetric Q with non-integer values, a non-zero diagonal and a linear term, both directions stored."""
    rng = np.random.default_rng(seed)
    m = 3 * n
    i, j = rng.integers(0, n, size=m), rng.integers(0, n, size=m)
    keep = i != j
    pairs = np.unique(np.stack([np.minimum(i, j)[keep], np.maximum(i, j)[keep]], axis=1), axis=0)
    v = rng.normal(size=len(pairs)).astype(np.float32)
    diag = rng.normal(size=n).astype(np.float32)
    rows = np.concatenate([pairs[:, 0], pairs[:, 1], np.arange(n)])
    cols = np.concatenate([pairs[:, 1], pairs[:, 0], np.arange(n)])
    vals = np.concatenate([v, v, diag])
    order = np.lexsort((cols, rows))
    rows, cols, vals = rows[order], cols[order], vals[order]
    rowptr = np.zeros(n + 1, dtype=np.int32)
    np.add.at(rowptr, rows + 1, 1)
    return wl.QuboCSR(n=n, rowptr=np.cumsum(rowptr).astype(np.int32), col=cols.astype(np.int32), val=vals.astype(np.float32),
                      c=rng.normal(size=n).astype(np.float32))


def points(n, B, seed):
    X = np.random.default_rng(seed).random((n, B), dtype=np.float32)
    X[:, 0] = X[:, 0] > 0.5                      # an exactly binary column
    if B > 1:
        X[:, 1] = 0.5                            # exactly 1/2 rounds to 0 (reading R5)
    return X


@pytest.mark.gpu
def test_static_scratch_score_matches_gda_score_on_two_calls_in_a_row():
    import torch
    build.build()
    dev = torch.device("cuda:0")
    torch.cuda.set_device(dev)
    up = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)

    # call 1: Max-Cut shaped like config 3 (integer weights, n = 12 001 and B = 333: ragged in both directions);
    # call 2: a smaller float-valued QUBO with a diagonal at B = 13, scored over the leftovers of call 1
    cases = [(wl.config(3, B=333, n_scale=12001 / 20000).problem, 333, True),
             (float_qubo_csr(257, seed=9), 13, False)]
    staged = []
    for k, (Q, B, integral) in enumerate(cases):                 # every tensor exists before the calls under test
        X = points(Q.n, B, seed=20 + k)
        staged.append((Q, integral, up(Q.rowptr), up(Q.col), up(Q.val), up(Q.c), up(X),
                       torch.full((B,), float("nan"), dtype=torch.float64, device=dev)))
    ref = []
    for Q, integral, *_rest, x, _obj in staged:                  # the existing path: handle + workspace + gda_score
        P = api.Problem.create_qubo_csr(Q.n, Q.rowptr, Q.col, Q.val, Q.c)
        assert P.info().integral == int(integral)
        ref.append(P.score(x).cpu().numpy())
        P.destroy()

    def both_calls():
        for Q, _i, rowptr, col, val, c, x, obj in staged:        # back to back on one stream, no synchronisation between
            obj.fill_(float("nan"))
            api.score_qubo_csr_static(Q.n, rowptr, col, val, c, x, obj)
        torch.cuda.synchronize()
        return [s[-1].cpu().numpy() for s in staged]

    def check(got):
        for (Q, integral, *_), g, r in zip(staged, got, ref):
            assert np.isfinite(g).all()
            if integral:
                assert np.array_equal(g, r)
            else:
                assert np.allclose(g, r, rtol=1e-6, atol=1e-5)

    check(both_calls())                                          # includes the first call on this GPU (address look-up)
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info(dev)[0]
    check(both_calls())                                          # and again over the array as the pair above left it
    free_after = torch.cuda.mem_get_info(dev)[0]
    assert free_before - free_after < (1 << 20)                  # no device memory was taken by the calls themselves

    # c = NULL means a zero linear term
    Q, _i, rowptr, col, val, c, x, obj = staged[1]
    api.score_qubo_csr_static(Q.n, rowptr, col, val, None, x, obj)
    lin = ((x > 0.5).double() * c.double()[:, None]).sum(dim=0)  # c^T x_hat, to take the linear term off the reference
    assert np.allclose(obj.cpu().numpy(), ref[1] - lin.cpu().numpy(), rtol=1e-6, atol=1e-4)


@pytest.mark.gpu
def test_static_scratch_score_rejects_what_it_cannot_serve():
    import torch
    build.build()
    dev = torch.device("cuda:0")
    torch.cuda.set_device(dev)
    Q = wl.config(1).problem
    up = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)
    rowptr, col, val, c = up(Q.rowptr), up(Q.col), up(Q.val), up(Q.c)
    B = api.STATIC_SCORE_MAX_B + 1
    x = torch.rand((Q.n, B), dtype=torch.float32, device=dev)
    obj = torch.zeros(B, dtype=torch.float64, device=dev)
    with pytest.raises(api.GdaError) as e:                       # beyond the fixed array: a clear refusal, not a wrong answer
        api.score_qubo_csr_static(Q.n, rowptr, col, val, c, x, obj)
    assert e.value.status == 4 and "GDA_STATIC_SCORE_MAX_B" in str(e.value)
    host = np.zeros(4, dtype=np.float64)                         # a host pointer where device memory is required
    st = api.lib().gda_score_qubo_csr_static(Q.n, rowptr.data_ptr(), col.data_ptr(), val.data_ptr(), c.data_ptr(), 4,
                                             x.data_ptr(), host.ctypes.data, None)
    assert st == 1 and b"DEVICE" in api.lib().gda_last_error()
    # the largest B it serves, against the existing path
    B = api.STATIC_SCORE_MAX_B
    x = torch.rand((Q.n, B), dtype=torch.float32, device=dev)
    obj = torch.zeros(B, dtype=torch.float64, device=dev)
    api.score_qubo_csr_static(Q.n, rowptr, col, val, c, x, obj)
    P = api.Problem.create_qubo_csr(Q.n, Q.rowptr, Q.col, Q.val, Q.c)
    assert torch.equal(obj, P.score(x))
    P.destroy()
