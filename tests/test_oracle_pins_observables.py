"""Pins of the oracle's NEXT-1 / NEXT-2 functions (SURVEY 8 f): two-site correlators, total magnetisation, <H>, and the
random-phase state of eq. A.1 -- written BEFORE the CUDA kernels that are compared with them.

Each pin is something other than the oracle's own formula: Kronecker-built dense operators (tests/dense_ref.py,
separate code), closed forms on product / singlet states, the published first outputs of SplitMix64, energy
conservation of the exact dynamics, and exact statistical properties of the eq. A.1 state.
"""
import numpy as np
import pytest

import dense_ref as D
from oracle import ts_oracle as O
from paper_1305_0036_b200 import workloads as W


def rand_state(N, seed, normalise=False):
    rng = np.random.Generator(np.random.PCG64(seed))
    v = rng.standard_normal(2 << N).view(np.complex128).copy()
    if normalise:
        v /= np.linalg.norm(v)
    return v


# --------------------------------------------------------------------------------------------- two-site correlators
@pytest.mark.parametrize("N", [2, 3, 5])
def test_correlators_match_dense_operators_on_unnormalised_states(N):
    psi = rand_state(N, 10 + N)          # NOT normalised: pins "un-normalised" (A15) as well
    for a in range(3):
        for j in range(N):
            for k in range(N):
                if j == k:
                    continue
                op = D.site_op(D.SPIN[a], j, N) @ D.site_op(D.SPIN[a], k, N)
                exp = np.vdot(psi, op @ psi)
                assert abs(exp.imag) < 1e-12
                assert abs(O.correlate(psi, N, a, j, k) - exp.real) < 1e-12, (a, j, k)


def test_correlators_closed_forms():
    """Singlet (|up,down> - |down,up>)/sqrt 2 on spins (0, 1): <S^a_0 S^a_1> = -1/4 for every axis (S_0 . S_1 = -3/4).
    Triplet |up,up>: zz = +1/4, xx = yy = 0.  Product state with a third, uncorrelated spin: unchanged."""
    s = np.zeros(8, dtype=np.complex128)
    # spin 2 down (bit 2 = 0); index = bit0 + 2 bit1: |up_0 down_1> = 1, |down_0 up_1> = 2
    s[1] = 1 / np.sqrt(2)
    s[2] = -1 / np.sqrt(2)
    for a in range(3):
        assert abs(O.correlate(s, 3, a, 0, 1) + 0.25) < 1e-15
        assert abs(O.correlate(s, 3, a, 1, 0) + 0.25) < 1e-15
    t = np.zeros(8, dtype=np.complex128)
    t[3] = 1.0
    assert abs(O.correlate(t, 3, O.Z, 0, 1) - 0.25) < 1e-15
    assert abs(O.correlate(t, 3, O.X, 0, 1)) < 1e-15
    assert abs(O.correlate(t, 3, O.Y, 0, 1)) < 1e-15
    # zz against the uncorrelated spin 2 (down): <S^z_0 S^z_2> = (+1/2)(-1/2)
    assert abs(O.correlate(t, 3, O.Z, 0, 2) + 0.25) < 1e-15


def test_correlator_of_a_product_state_factorises():
    w = W.config(3)                      # random product state recipe (A19), N = 22 is too big: rebuild at N = 6
    spins = W.random_product_spins(6, 77)
    psi = np.ones(1, dtype=np.complex128)
    for j in range(6):
        psi = np.kron(spins[j], psi)
    for a in range(3):
        one = [O.expect(psi, 6, a, j) for j in range(6)]
        for j, k in ((0, 5), (2, 3), (4, 1)):
            assert abs(O.correlate(psi, 6, a, j, k) - one[j] * one[k]) < 1e-13
    assert w.N == 22


def test_total_sz_is_sum_of_site_values_and_dense_operator():
    N = 5
    psi = rand_state(N, 3)
    Sz = sum(D.site_op(D.SZ, j, N) for j in range(N))
    assert abs(O.total_sz(psi, N) - np.vdot(psi, Sz @ psi).real) < 1e-12
    assert abs(O.total_sz(psi, N) - sum(O.expect(psi, N, O.Z, j) for j in range(N))) < 1e-13


# --------------------------------------------------------------------------------------------- <H>
@pytest.mark.parametrize("sym", [False, True])
def test_energy_expect_matches_dense_hamiltonian(sym):
    N = 6
    w = W.generic(N, seed=61 + sym, symmetric_fill=sym)     # symmetric_fill also sets a diagonal, which must be ignored
    psi = rand_state(N, 9)
    H = D.hamiltonian(N, w.h, w.J)
    exp = np.vdot(psi, H @ psi)
    assert abs(exp.imag) < 1e-11
    assert abs(O.energy_expect(psi, N, w.h, w.J) - exp.real) < 1e-11


def test_energy_is_conserved_by_the_trotter_dynamics_to_order_tau4():
    """<H> is a constant of the exact motion; under U_4(tau) it drifts by O(tau^4): halving tau cuts the drift ~16x."""
    N = 8
    w = W.generic(N, seed=88)
    psi0 = rand_state(N, 5, normalise=True)
    E0 = O.energy_expect(psi0, N, w.h, w.J)
    drifts = []
    for tau, n in ((0.08, 5), (0.04, 10)):
        psi = psi0.copy()
        O.evolve(psi, N, w.h, w.J, tau, n, 4, True)
        drifts.append(abs(O.energy_expect(psi, N, w.h, w.J) - E0))
    assert drifts[0] < 1e-4 and drifts[1] < drifts[0]
    assert 8.0 < drifts[0] / drifts[1] < 32.0, drifts


# --------------------------------------------------------------------------------------------- eq. A.1
def test_splitmix64_published_outputs():
    """SplitMix64 seeded with 0: the first outputs of the reference implementation (Steele, Lea, Flood 2014; the
    values quoted by every implementation's self-test)."""
    exp = [0xE220A8397B1DCDAF, 0x6E789E6AA1B965F4, 0x06C45D188009454F, 0xF88BB8A8724C81EC]
    got = [O.splitmix64(0, j) for j in range(4)]
    assert got == exp, [hex(x) for x in got]


def test_splitmix64_independent_python_restatement():
    M = (1 << 64) - 1

    def sm(seed, j):
        z = (seed + (j + 1) * 0x9E3779B97F4A7C15) & M
        z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & M
        z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & M
        return z ^ (z >> 31)
    for seed in (0, 1, 12345678901234567):
        for j in (0, 1, 2, 1000, (1 << 40) + 3):
            assert O.splitmix64(seed, j) == sm(seed, j)


@pytest.mark.parametrize("N,up", [(1, 0), (4, 0), (6, 3), (10, 9), (12, 5)])
def test_random_phase_state_structure(N, up):
    """Eq. A.1: amplitude 0 wherever spin `up` is down; modulus exactly 2^-(N-1)/2 elsewhere; norm 1; <S^z_up> = +1/2
    and <S^z_j> = 0 for every other spin (all Ising states of the rest equally weighted)."""
    psi = O.random_phase_state(N, up, seed=42)
    k = np.arange(1 << N)
    upmask = ((k >> up) & 1) == 1
    assert np.all(psi[~upmask] == 0)
    assert np.max(np.abs(np.abs(psi[upmask]) - 2.0 ** (-(N - 1) / 2))) < 1e-16 * 4
    assert abs(O.norm2(psi, N) - 1.0) < 1e-13
    sz = O.expect_all(psi, N, O.Z)
    assert abs(sz[up] - 0.5) < 1e-13
    for j in range(N):
        if j != up:
            assert abs(sz[j]) < 1e-13


def test_random_phase_state_phases_follow_the_generator_and_are_uniform():
    N, up, seed = 13, 4, 7
    psi = O.random_phase_state(N, up, seed)
    k = np.arange(1 << N)
    sel = k[((k >> up) & 1) == 1]
    j = ((sel >> (up + 1)) << up) | (sel & ((1 << up) - 1))          # index with bit `up` removed: beta_j of eq. A.1
    u = np.array([O.splitmix64(seed, int(x)) >> 11 for x in j], dtype=np.float64) * 2.0 ** -53
    exp = np.exp(2j * np.pi * u) * 2.0 ** (-(N - 1) / 2)
    assert np.max(np.abs(psi[sel] - exp)) < 1e-15
    # uniform phases: the mean of e^{i phi} over M samples is O(1/sqrt M); 16 bins within 5 sigma
    M = sel.size
    assert abs(np.mean(psi[sel]) * 2.0 ** ((N - 1) / 2)) < 5.0 / np.sqrt(M)
    hist, _ = np.histogram(u, bins=16, range=(0, 1))
    assert np.max(np.abs(hist - M / 16)) < 5.0 * np.sqrt(M / 16)
    # different seeds and different spins give different states
    assert np.max(np.abs(psi - O.random_phase_state(N, up, seed + 1))) > 1e-3
    # local observable of the infinite-temperature ensemble: <S^x_j> ~ O(2^-N/2) for the thermal spins
    for jj in (0, 7):
        assert abs(O.expect(psi, N, O.X, jj)) < 5.0 * 2.0 ** (-(N - 1) / 2)
