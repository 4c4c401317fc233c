"""world_size-2 gloo test of the multi-GPU arm's host logic (paper_1305_0036_b200/replicas.py): per-rank seeds give
different ensemble members, timing is the max over ranks, throughput is the whole-job aggregate."""
import os
import socket
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from paper_1305_0036_b200 import replicas as R
    from paper_1305_0036_b200 import workloads as W
    w = W.grid_like(10, seed=8, state_seed=9)
    w.state_seed = R.replica_state_seed(w.state_seed, rank)
    psi = w.state()
    ms_local = 100.0 + 50.0 * rank                 # rank 1 is the slow one
    ms = R.max_over_ranks(ms_local)
    norms = R.gather_scalars(float(np.vdot(psi, psi).real))
    firsts = R.gather_scalars(float(psi[0].real))
    q.put((rank, ms, R.whole_job_steps_per_s(5, world, ms), norms, firsts, w.state_seed))
    dist.barrier()
    dist.destroy_process_group()


def test_two_replicas_gloo():
    world = 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ms, value, norms, firsts, seed in res:
        assert ms == 150.0                          # max over ranks, seen by every rank
        assert abs(value - 2 * 5 / 0.150) < 1e-9    # whole-job aggregate
        assert all(abs(n - 1.0) < 1e-12 for n in norms)
        assert firsts[0] != firsts[1]               # different ensemble members
        assert seed == 9 + 1000 * rank


def test_single_process_paths():
    from paper_1305_0036_b200 import replicas as R
    assert R.max_over_ranks(3.5) == 3.5
    assert R.gather_scalars(2.0) == [2.0]
    assert R.replica_state_seed(None, 3) == 3000
    assert R.whole_job_steps_per_s(4, 1, 2000.0) == 2.0
