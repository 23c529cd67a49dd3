"""Glue used by tests only: turn a workloads.* problem into an oracle Problem."""
import numpy as np

from oracle import pdbo
from paper_2509_21064_b200 import workloads as wl


def oracle_problem(P):
    if isinstance(P, wl.QuboCSR):
        return pdbo.Problem.qubo_csr(P.n, P.rowptr, P.col, P.val, P.c)
    if isinstance(P, wl.QuboDense):
        return pdbo.Problem.qubo_dense(P.n, P.Q, P.c)
    if isinstance(P, wl.MaxSat):
        return pdbo.Problem.maxsat(P.n, P.m, P.cptr, P.lit, P.w)
    raise TypeError(type(P))


def hyper_kwargs(h, **over):
    d = dict(alpha=h.alpha, beta=h.beta, delta=h.delta, gfun=h.gfun, log_eps=h.log_eps,
             iters=h.iters, eval_every=h.eval_every, seed=h.seed)
    if getattr(h, "dual", 0):
        d["dual"] = h.dual
    d.update(over)
    return d


def create_problem(api, w_or_problem, sparse_path=None):
    """gda_create_* for a workload (or a bare problem container).  `sparse_path` = "slab" | "stream" (or
    workload.extra["sparse_path"]) forces the sparse launch path of THIS handle (gda_set_option, GDA_OPT_SPARSE_PATH);
    None leaves the choice to the library's cost model."""
    problem = getattr(w_or_problem, "problem", w_or_problem)
    path = sparse_path or getattr(w_or_problem, "extra", {}).get("sparse_path")
    P = api.create_from_workload(problem)
    if path:
        P.set_option(api.OPT_SPARSE_PATH, api.SPARSE_PATH[path])
    return P
