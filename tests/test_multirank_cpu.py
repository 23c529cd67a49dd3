"""World-size-2 gloo test (CPU) of the multi-rank host logic used by bench.py --gpus N."""
import os
import socket

import numpy as np
import pytest

torch = pytest.importorskip("torch")
import torch.distributed as dist           # noqa: E402
import torch.multiprocessing as mp         # noqa: E402

from paper_2509_21064_b200 import multirank, workloads as wl   # noqa: E402


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, case, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    objs = {"distinct": [(-10.0, 3), (-12.0, 5)], "tie": [(-7.0, 9), (-7.0, 2)]}[case]
    g = multirank.combine_best(objs[rank][0], objs[rank][1], rank, world)
    t = multirank.max_over_ranks(1.0 + rank, world)
    x0 = wl.x0_uniform(5, 4, multirank.rank_x0_seed(11, rank))
    out[rank] = (g, t, float(x0.sum()))
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("case", ["distinct", "tie"])
def test_combine_best_across_two_ranks(case):
    port = _free_port()
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(2, port, case, out), nprocs=2, join=True)
    exp = (-12.0, 1, 5) if case == "distinct" else (-7.0, 0, 9)       # tie -> lowest rank
    assert out[0][0] == exp and out[1][0] == exp
    assert out[0][1] == 2.0 and out[1][1] == 2.0                      # max over ranks
    assert out[0][2] != out[1][2]                                     # ranks start from different points


def test_single_rank_issues_no_collective():
    assert multirank.combine_best(-3.0, 4, 0, 1) == (-3.0, 0, 4)
    assert multirank.max_over_ranks(2.5, 1) == 2.5
    assert multirank.rank_x0_seed(100, 0) == 100
