"""Host side of the sharded path (paper_1305_0036_b200/sharded.py) on CPU with gloo, world_size 2 and 4: the all-to-all
IS the index-bit swap the library's spin layouts assume (rank bits <-> top local bits), and the per-rank contributions to
<S^z_j> add up to the definition.  (The kernels of the sharded path are covered on the GPU by tests/test_gpu_sharded.py.)"""
import os
import socket
import sys

import numpy as np
import pytest
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
    from paper_1305_0036_b200 import sharded as S
    g = S.log2_exact(world)
    n = 6                                              # local bits
    N = n + g
    # amplitude value = its GLOBAL index (rank bits on top), so that positions can be read back after the swap
    glob = (rank << n) + np.arange(1 << n)
    src = torch.tensor(glob.astype(np.float64) + 1j * (glob.astype(np.float64) + 0.5), dtype=torch.complex128)
    dst = torch.zeros_like(src)
    S.alltoall_exchange(src, dst)
    got = dst.numpy().real.astype(np.int64)
    # after the swap, local index (top, low) on rank r holds what rank `top` had at local index (r, low)
    low = np.arange(1 << n) & ((1 << (n - g)) - 1)
    top = np.arange(1 << n) >> (n - g)
    expect = (top << n) + (rank << (n - g)) + low
    ok_swap = bool(np.array_equal(got, expect)) and bool(np.allclose(dst.numpy().imag, expect + 0.5))
    back = torch.zeros_like(src)
    S.alltoall_exchange(dst, back)                    # the swap is an involution
    ok_inv = bool(torch.equal(back, src))

    # <S^z_j> assembled from per-rank pieces = the definition on the full vector (layout 0)
    rng = np.random.Generator(np.random.PCG64(5))
    full = rng.standard_normal(1 << N) + 1j * rng.standard_normal(1 << N)
    loc = full[S.shard_slice(N, world, rank)]
    p = np.abs(loc) ** 2
    local_sz = np.array([np.sum((((np.arange(1 << n) >> b) & 1) - 0.5) * p) for b in range(n)])
    contrib = torch.tensor(S.assemble_sz(local_sz, float(p.sum()), np.arange(N), n, rank))
    dist.all_reduce(contrib)
    pf = np.abs(full) ** 2
    ref = np.array([np.sum((((np.arange(1 << N) >> j) & 1) - 0.5) * pf) for j in range(N)])
    ok_sz = bool(np.allclose(contrib.numpy(), ref, rtol=0, atol=1e-9))
    q.put((rank, ok_swap, ok_inv, ok_sz))
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("world", [2, 4])
def test_index_bit_swap_and_observable_assembly_gloo(world):
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=180) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert [r[0] for r in res] == list(range(world))
    assert all(r[1] for r in res), "all-to-all is not the rank-bit <-> top-local-bit swap"
    assert all(r[2] for r in res), "swap is not an involution"
    assert all(r[3] for r in res), "<S^z_j> pieces do not add up"


def test_shard_slices_and_rank_count():
    from paper_1305_0036_b200 import sharded as S
    assert S.log2_exact(1) == 0 and S.log2_exact(8) == 3
    with pytest.raises(ValueError):
        S.log2_exact(6)
    assert S.shard_slice(10, 4, 3) == slice(3 << 8, 4 << 8)
    parts = [S.shard_slice(7, 8, r) for r in range(8)]
    assert parts[0].start == 0 and parts[-1].stop == 1 << 7 and all(a.stop == b.start for a, b in zip(parts, parts[1:]))
