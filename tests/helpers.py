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
