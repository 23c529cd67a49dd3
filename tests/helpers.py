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
    workload.extra["sparse_path"]) forces the sparse launch path through GDA_SPARSE_PATH, which the library reads at
    create; None leaves the choice to its cost model."""
    import os
    problem = getattr(w_or_problem, "problem", w_or_problem)
    path = sparse_path or getattr(w_or_problem, "extra", {}).get("sparse_path")
    if path:
        os.environ["GDA_SPARSE_PATH"] = path
    try:
        return api.create_from_workload(problem)
    finally:
        os.environ.pop("GDA_SPARSE_PATH", None)
