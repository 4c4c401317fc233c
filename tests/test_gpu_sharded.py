"""GPU parity of the sharded path (SURVEY 8 e / 8 f NEXT-5; csrc/ts_shard.cu, paper_1305_0036_b200/sharded.py): one state
vector split over 2^g "ranks" -- here all on ONE GPU (LocalCluster: one thread per rank, the all-to-all index-bit swap done
by device copies) -- against the CPU oracle run on the FULL state.  Every rotation, diagonal and the sequence run in the
library's kernels; what the test exercises beyond the single-GPU path is the effective Hamiltonian of a shard (fields of
the frozen rank-bit spins, the rank-dependent energy offset), the two spin layouts and the exchange pattern.  Gates as
everywhere: amplitudes max-abs and 2-norm <= 1e-11, <S^z_j> <= 1e-10."""
import numpy as np
import pytest

from oracle import ts_oracle as O
from paper_1305_0036_b200 import workloads as W

pytestmark = pytest.mark.gpu

AMP_TOL = 1e-11
OBS_TOL = 1e-10


@pytest.fixture(scope="module")
def S():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    from paper_1305_0036_b200 import binding, sharded
    binding.load()
    return sharded


def run_case(S, N, world, order, steps, seed, symmetric_fill=False, peer_memory=False):
    w = W.generic(N, seed=seed, tau=0.02, n_steps=steps, symmetric_fill=symmetric_fill)
    ref = w.state()
    O.evolve(ref, N, w.h, w.J, w.tau, steps, order, True)
    cl = S.LocalCluster(N, w.h, w.J, world, peer_memory=peer_memory)
    cl.set_state(w.state())
    cl.evolve(w.tau, steps, order)
    got = cl.get_state()
    d = got - ref
    assert np.max(np.abs(d)) <= AMP_TOL, f"max-abs {np.max(np.abs(d)):.3e}"
    assert np.linalg.norm(d) <= AMP_TOL, f"2-norm {np.linalg.norm(d):.3e}"
    assert np.max(np.abs(cl.expect_z_all() - O.expect_all(ref, N, O.Z))) <= OBS_TOL
    assert abs(cl.norm2() - O.norm2(ref, N)) <= OBS_TOL
    for s in cl.shards:
        assert s.info() == (N - S.log2_exact(world), 0, 0)      # whole steps end in layout 0, in the first buffer
    cl.close()


# (N, ranks): local shards of 12..15 spins run the tiled plan, smaller ones one launch per spin
@pytest.mark.parametrize("N,world", [(14, 2), (15, 4), (16, 4), (17, 8), (13, 2), (10, 4), (7, 2), (6, 8)])
@pytest.mark.parametrize("order", [4, 2])
def test_sharded_matches_full_oracle(S, N, world, order):
    run_case(S, N, world, order, steps=2, seed=4000 + 10 * N + world)


@pytest.mark.parametrize("N,world", [(22, 8), (21, 2)])
def test_sharded_with_multi_group_shards(S, N, world):
    """Shards of 19 / 20 spins: several bit groups per shard, a two-stage top group, and the arriving spins rotated by
    the top group's tile pass restricted to its top g bits (fused with the diagonal)."""
    run_case(S, N, world, 4, steps=1, seed=4700 + N)


# shards of >= 13 spins (the arrival pass is the top bit group's tile pass); single- and two-stage top groups, g = 1, 2, 3
@pytest.mark.parametrize("N,world", [(14, 2), (15, 2), (16, 4), (17, 4), (19, 8), (20, 4), (22, 8)])
@pytest.mark.parametrize("order", [4, 2])
def test_peer_memory_mode_matches_full_oracle(S, N, world, order):
    """Peer-memory mode: no exchange; the arrival pass gathers its tiles from the other shards' buffers (here: plain
    pointers on the same GPU; across GPUs: peer-mapped pointers) and writes into the shard's other buffer."""
    run_case(S, N, world, order, steps=2 if N <= 20 else 1, seed=4800 + 10 * N + world, peer_memory=True)


def test_peer_memory_mode_needs_a_top_group(S):
    from paper_1305_0036_b200 import binding as B
    w = W.generic(10, seed=3, tau=0.01, n_steps=1)
    with pytest.raises(B.TSError):
        S.LocalCluster(10, w.h, w.J, 4, peer_memory=True)        # shards of 8 spins have no tile groups


def test_one_rank_is_the_unsharded_path(S):
    run_case(S, 13, 1, 4, steps=1, seed=4500)


def test_sharded_with_lower_triangle_and_diagonal_of_J_filled(S):
    run_case(S, 14, 4, 4, steps=1, seed=4600, symmetric_fill=True)          # reading A1 through the effective fields


def test_spin_maps_are_the_two_layouts_of_the_index_bit_swap(S):
    N, world = 9, 4
    w = W.generic(N, seed=1, tau=0.01, n_steps=1)
    s = S.ShardedTrotterSuzuki(N, w.h, w.J, rank=3, world=world, exchange=lambda a, b: None)
    assert list(s.spin_map(0)) == [0, 1, 2, 3, 4, 5, 6, 7, 8]
    assert list(s.spin_map(1)) == [0, 1, 2, 3, 4, 7, 8, 5, 6]    # top two local bits <-> the two rank bits
    s.close()


def test_argument_errors(S):
    from paper_1305_0036_b200 import binding as B
    w = W.generic(6, seed=2, tau=0.01, n_steps=1)
    with pytest.raises(ValueError):
        S.ShardedTrotterSuzuki(6, w.h, w.J, rank=0, world=3)
    with pytest.raises(B.TSError):
        S.ShardedTrotterSuzuki(6, w.h, w.J, rank=2, world=2)
    with pytest.raises(B.TSError):
        S.ShardedTrotterSuzuki(3, w.h[:, :3], w.J[:, :3, :3], rank=0, world=4)      # 2 g > N
