"""Host-side checks of the seeded input recipes; CPU only."""
import numpy as np

from paper_1305_0036_b200 import workloads as W


def _nbonds(J):
    return int(np.count_nonzero(J[W.Z]))


def test_config_shapes_and_bond_counts():
    c1, c2, c3, c4, c5, cm = (W.config(i) for i in (1, 2, 3, 4, 5, "M"))
    assert (c1.N, _nbonds(c1.J)) == (10, 9)
    assert (c2.N, _nbonds(c2.J)) == (16, 16)
    assert (c3.N, _nbonds(c3.J)) == (22, 231)
    assert (c4.N, _nbonds(c4.J)) == (27, 43)          # 4x7 grid minus last site (reading A16)
    assert (c5.N, _nbonds(c5.J)) == (32, 52)
    assert (cm.N, _nbonds(cm.J)) == (30, 49)
    for c in (c1, c2, c3, c4, c5, cm):
        assert c.h.shape == (3, c.N) and c.J.shape == (3, c.N, c.N)
        assert np.all(np.tril(c.J) == 0)              # stored once, j < k
    assert c2.basis_index == 0xAAAA
    assert abs(np.abs(c3.J[W.Z]).max() - 2.0) < 1e-15 and np.allclose(c3.J[W.X], -0.5 * c3.J[W.Z])
    assert np.all(c2.h[W.X] == 0.3) and np.all(c1.h[W.X] == 0)


def test_checkerboard_neel():
    k = W.checkerboard_index(4, 8)
    for j in range(32):
        r, c = divmod(j, 8)
        assert (k >> j) & 1 == (r + c) & 1
    # nearest neighbours always differ
    for (a, b) in W.grid_bonds(4, 8):
        assert ((k >> a) ^ (k >> b)) & 1 == 1


def test_states_are_normalised_and_chunking_is_consistent():
    for w in (W.config(1), W.config(2), W.dipolar_like(12, 5), W.generic(11, 3)):
        psi = w.state()
        assert abs(np.vdot(psi, psi).real - 1.0) < 1e-12
        parts = np.concatenate([c for _, c in w.state_chunks(chunk_log2=6)])
        if w.state_kind != "gaussian":
            assert np.allclose(parts, psi, atol=1e-15)
    # gaussian: the chunked stream equals one big draw of the same generator
    w = W.generic(10, 3)
    big = np.random.Generator(np.random.PCG64(w.state_seed)).standard_normal(2 << 10)
    big = (big / np.sqrt(np.dot(big, big))).view(np.complex128)
    assert np.allclose(np.concatenate([c for _, c in w.state_chunks(6)]), big, atol=1e-15)


def test_product_state_is_kron_of_spins():
    w = W.dipolar_like(5, 9)
    psi = w.state()
    for k in (0, 7, 21, 31):
        ref = np.prod([w.spin_states[j][(k >> j) & 1] for j in range(5)])
        assert abs(psi[k] - ref) < 1e-15


def test_clustered_workload_structure():
    cl = W.interleaved_clusters(9, 3)
    assert cl == [[0, 3, 6], [1, 4, 7], [2, 5, 8]]
    w = W.clustered(9, cl, seed=4)
    for a in range(3):
        for j in range(9):
            for k in range(9):
                if w.J[a, j, k] != 0:
                    assert j < k and (j % 3) == (k % 3)
    psi = w.state()
    k = 0b101100110
    ref = 1.0
    for bits, st in zip(w.clusters, w.cluster_states):
        ref = ref * st[sum(((k >> b) & 1) << i for i, b in enumerate(bits))]
    assert abs(psi[k] - ref) < 1e-15
    sub = W.sub_workload(w, 1)
    assert sub.N == 3 and sub.J[W.X, 0, 2] == w.J[W.X, 1, 7] and sub.h[W.Y, 2] == w.h[W.Y, 7]
