"""Pins of the CPU oracle (oracle/ts_oracle.c) to things OTHER than itself: the paper's printed examples and
identities, closed forms, dense linear algebra built separately in tests/dense_ref.py.  CPU only."""
import os

import numpy as np
import pytest

import dense_ref as D
from oracle import ts_oracle as O
from paper_1305_0036_b200 import workloads as W

GOLD = os.path.join(os.path.dirname(__file__), "golden")
A_SUZUKI = 1.0 / (4.0 - 4.0 ** (1.0 / 3.0))


def basis(N, k):
    v = np.zeros(1 << N, dtype=np.complex128)
    v[k] = 1.0
    return v


def sweep_matrix(N, kind):
    """Matrix of an oracle sweep (normalised by 2^{-N/2}), column by column."""
    M = np.zeros((1 << N, 1 << N), dtype=complex)
    for k in range(1 << N):
        v = basis(N, k)
        O.apply_sweep(v, N, kind)
        M[:, k] = v
    return M * 2.0 ** (-N / 2)


def rand_state(N, seed):
    rng = np.random.Generator(np.random.PCG64(seed))
    v = rng.standard_normal(2 << N).view(np.complex128).copy()
    return v / np.linalg.norm(v)


# ---------------------------------------------------------------------------- eq. 5 and the identities P:69-71
def test_eq5_identities_as_printed():
    """(R^y)^dag S^x R^y = S^z and (R^x)^dag S^y R^x = S^z hold for the printed matrices in (up, down) order."""
    Ry = np.array([[1, -1], [1, 1]], dtype=complex) / np.sqrt(2)
    Rx = np.array([[1, 1j], [1j, 1]], dtype=complex) / np.sqrt(2)
    sx = np.array([[0, 1], [1, 0]], dtype=complex) / 2       # (up, down) order
    sy = np.array([[0, -1j], [1j, 0]], dtype=complex) / 2
    sz = np.array([[1, 0], [0, -1]], dtype=complex) / 2
    assert np.allclose(Ry.conj().T @ sx @ Ry, sz, atol=1e-15)
    assert np.allclose(Rx.conj().T @ sy @ Rx, sz, atol=1e-15)


def test_oracle_sweeps_are_eq5_reindexed():
    """The oracle's four sweeps at N=1 are eq. 5's matrices (and their adjoints) with rows/columns flipped from the
    printed (up, down) order to bit order (down, up)  (reading A7)."""
    Ry = np.array([[1, -1], [1, 1]], dtype=complex) / np.sqrt(2)
    Rx = np.array([[1, 1j], [1j, 1]], dtype=complex) / np.sqrt(2)
    P = np.array([[0, 1], [1, 0]], dtype=complex)
    assert np.allclose(sweep_matrix(1, O.SWEEP_Y), P @ Ry @ P, atol=1e-15)
    assert np.allclose(sweep_matrix(1, O.SWEEP_YDAG), P @ Ry.conj().T @ P, atol=1e-15)
    assert np.allclose(sweep_matrix(1, O.SWEEP_X), P @ Rx @ P, atol=1e-15)
    assert np.allclose(sweep_matrix(1, O.SWEEP_XDAG), P @ Rx.conj().T @ P, atol=1e-15)


@pytest.mark.parametrize("N", [1, 2, 3])
def test_sweeps_rotate_spin_operators(N):
    """Y^dag S^x_j Y = S^z_j and X^dag S^y_j X = S^z_j for every spin, in bit order, with dense_ref's operators."""
    Ym, Xm = sweep_matrix(N, O.SWEEP_Y), sweep_matrix(N, O.SWEEP_X)
    assert np.allclose(sweep_matrix(N, O.SWEEP_YDAG), Ym.conj().T, atol=1e-15)
    assert np.allclose(sweep_matrix(N, O.SWEEP_XDAG), Xm.conj().T, atol=1e-15)
    assert np.allclose(Ym.conj().T @ Ym, np.eye(1 << N), atol=1e-14)
    for j in range(N):
        assert np.allclose(Ym.conj().T @ D.site_op(D.SX, j, N) @ Ym, D.site_op(D.SZ, j, N), atol=1e-14)
        assert np.allclose(Xm.conj().T @ D.site_op(D.SY, j, N) @ Xm, D.site_op(D.SZ, j, N), atol=1e-14)


# ------------------------------------------------------------------------------ pairing and tiles
def _read_rows(name):
    rows = []
    with open(os.path.join(GOLD, name)) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            rows.append(line.split())
    return rows


def test_pairing_spin2_of_4_golden():
    pairs = {(int(a), int(b)) for a, b in _read_rows("pairs_spin2_of_4.txt")}
    assert len(pairs) == 8
    got = set()
    for k in range(16):
        v = basis(4, k)
        O.rotate_bit(v, 4, 1, O.SWEEP_Y)                     # paper spin 2 <-> bit 1
        nz = tuple(sorted(np.nonzero(v)[0]))
        assert len(nz) == 2
        got.add(nz)
    assert got == pairs


def test_closed_set_P141_golden():
    states = sorted(int(r[0], 2) for r in _read_rows("closed_set_P141.txt"))
    # spin 3 up <-> bit 2 = 1, spin 1 down <-> bit 0 = 0 (pins spin j <-> bit j-1 and up <-> 1)
    assert states == sorted(k for k in range(16) if (k >> 2) & 1 == 1 and (k & 1) == 0)
    # closed under rotating spins 2 and 4 (bits 1 and 3) in the oracle
    for k in states:
        for bit in (1, 3):
            v = basis(4, k)
            O.rotate_bit(v, 4, bit, O.SWEEP_X)
            assert set(np.nonzero(v)[0]) <= set(states)


@pytest.mark.parametrize("name,bits", [("tiles_low_P149.txt", (0, 1)), ("tiles_high_P156.txt", (2, 3))])
def test_tile_tables_golden(name, bits):
    """A thread block's states are closed under the rotations of the table's two spins, and the tables partition
    the 16 states."""
    seen = set()
    for row in _read_rows(name):
        states = {int(x) for x in row[1:]}
        seen |= states
        for k in states:
            for bit in bits:
                v = basis(4, k)
                O.rotate_bit(v, 4, bit, O.SWEEP_YDAG)
                assert set(np.nonzero(v)[0]) <= states
    assert seen == set(range(16))


def test_eq9_phase_pattern_golden():
    """eq. 9 with the evolution sign of P:44: aligned pair exp(-itJ/4), anti-aligned exp(+itJ/4)."""
    t, Jz = 0.37, 1.3
    h = np.zeros((3, 2))
    J = np.zeros((3, 2, 2))
    J[W.Z, 0, 1] = Jz
    idx = {"uu": 3, "ud": 2, "du": 1, "dd": 0}               # (spin 2, spin 1) -> bits (1, 0)
    for name, coef in _read_rows("eq9_phases.txt"):
        v = basis(2, idx[name])
        O.apply_diag(v, 2, h[W.Z], J[W.Z], t)
        assert abs(v[idx[name]] - np.exp(1j * float(coef) * t * Jz)) < 1e-15


# ------------------------------------------------------------------------------------------- diagonal energies
@pytest.mark.parametrize("N,seed", [(1, 11), (2, 12), (3, 13), (5, 14), (7, 15)])
def test_energy_is_diagonal_of_dense_Hz(N, seed):
    w = W.generic(N, seed, symmetric_fill=True)
    for a in range(3):
        # put alpha's couplings on the z axis of a dense Hamiltonian: its diagonal must equal E_alpha(k)
        h = np.zeros((3, N)); J = np.zeros((3, N, N))
        h[W.Z] = w.h[a]; J[W.Z] = w.J[a]
        Hz = D.hamiltonian_alpha(N, h, J, W.Z)
        assert np.allclose(Hz, np.diag(np.diag(Hz)))
        E = O.energy_table(N, w.h[a], w.J[a])
        assert np.allclose(E, np.real(np.diag(Hz)), atol=1e-14)
        assert E[5 % (1 << N)] == O.energy(N, w.h[a], w.J[a], 5 % (1 << N))


def test_energy_reading_A1_conventions():
    """Ordered-pair sum: J stored once gives coupling J; stored in both triangles gives 2J; diagonal ignored."""
    N = 4
    w = W.generic(N, 21)
    Ju = w.J[W.Z]
    Js = 0.5 * (Ju + Ju.T)
    Jd = Ju + np.diag([3.0, -1.0, 2.0, 0.5])
    for k in range(16):
        e = O.energy(N, w.h[W.Z], Ju, k)
        assert abs(O.energy(N, w.h[W.Z], Js, k) - e) < 1e-14
        assert O.energy(N, w.h[W.Z], Jd, k) == e
        # by hand: sum_j h_j s_j + sum_{j<m} J_jm s_j s_m
        s = [((k >> j) & 1) - 0.5 for j in range(N)]
        ref = sum(w.h[W.Z][j] * s[j] for j in range(N)) + sum(
            Ju[j, m] * s[j] * s[m] for j in range(N) for m in range(j + 1, N))
        assert abs(e - ref) < 1e-14


def test_pure_Z_hamiltonian_is_exact_phase():
    N = 6
    w = W.generic(N, 31)
    h = np.zeros((3, N)); J = np.zeros((3, N, N))
    h[W.Z] = w.h[W.Z]; J[W.Z] = w.J[W.Z]
    psi0 = w.state()
    psi = psi0.copy()
    O.evolve(psi, N, h, J, 0.05, 7, order=4)
    # sum of all sub-step times of U4 is tau, so the total phase is exp(-i 7 tau E_z(k)); the X and Y factors are
    # identity up to the sweeps' forward/backward cancellation.
    Hz = np.real(np.diag(D.hamiltonian_alpha(N, h, J, W.Z)))
    assert np.max(np.abs(psi - psi0 * np.exp(-1j * 7 * 0.05 * Hz))) < 1e-13


def test_diag_table_equals_direct_bitwise():
    N = 9
    w = W.generic(N, 41)
    a = rand_state(N, 42); b = a.copy()
    O.apply_diag(a, N, w.h[1], w.J[1], 0.3)
    O.apply_diag(b, N, w.h[1], w.J[1], 0.3, table=O.energy_table(N, w.h[1], w.J[1]))
    assert np.array_equal(a, b)
    c = rand_state(N, 43); d = c.copy()
    O.evolve(c, N, w.h, w.J, 0.02, 2, order=4, use_tables=True)
    O.evolve(d, N, w.h, w.J, 0.02, 2, order=4, use_tables=False)
    assert np.array_equal(c, d)


# ------------------------------------------------------------------------- single factors vs dense exponentials
@pytest.mark.parametrize("N,seed", [(1, 51), (2, 52), (4, 53), (6, 54), (8, 55)])
def test_each_factor_is_exact(N, seed):
    """Y D_x Y^dag = exp(-itH_x), X D_y X^dag = exp(-itH_y), D_z = exp(-itH_z)  (eq. 7, 9, 10)."""
    w = W.generic(N, seed)
    t = 0.23
    for a in range(3):
        psi0 = rand_state(N, seed + 100 + a)
        psi = psi0.copy()
        O.apply_H_alpha(psi, N, w.h, w.J, a, t)
        ref = D.expm_herm(D.hamiltonian_alpha(N, w.h, w.J, a), t) @ psi0
        assert np.max(np.abs(psi - ref)) < 1e-13, (a, np.max(np.abs(psi - ref)))


# ---------------------------------------------------------------------------------- closed forms: Larmor (N=1)
@pytest.mark.parametrize("order", [1, 2, 4])
def test_larmor_closed_forms(order):
    """Single spin in a single-axis field: every product formula is exact for any tau; signs of the precession
    pin the rotation matrices and the observables."""
    om, tau, n = 1.7, 0.13, 9
    t = tau * n
    J = np.zeros((3, 1, 1))
    up = np.array([0, 1], dtype=np.complex128)
    plusx = np.array([1, 1], dtype=np.complex128) / np.sqrt(2)
    # H = om S^x from up: <S^z> = cos/2, <S^y> = -sin/2, <S^x> = 0
    h = np.zeros((3, 1)); h[W.X, 0] = om
    psi = up.copy(); O.evolve(psi, 1, h, J, tau, n, order)
    assert abs(O.expect(psi, 1, W.Z, 0) - 0.5 * np.cos(om * t)) < 1e-13
    assert abs(O.expect(psi, 1, W.Y, 0) + 0.5 * np.sin(om * t)) < 1e-13
    assert abs(O.expect(psi, 1, W.X, 0)) < 1e-13
    # H = om S^y from up: <S^z> = cos/2, <S^x> = +sin/2
    h = np.zeros((3, 1)); h[W.Y, 0] = om
    psi = up.copy(); O.evolve(psi, 1, h, J, tau, n, order)
    assert abs(O.expect(psi, 1, W.Z, 0) - 0.5 * np.cos(om * t)) < 1e-13
    assert abs(O.expect(psi, 1, W.X, 0) - 0.5 * np.sin(om * t)) < 1e-13
    # H = om S^z from +x: <S^x> = cos/2, <S^y> = +sin/2
    h = np.zeros((3, 1)); h[W.Z, 0] = om
    psi = plusx.copy(); O.evolve(psi, 1, h, J, tau, n, order)
    assert abs(O.expect(psi, 1, W.X, 0) - 0.5 * np.cos(om * t)) < 1e-13
    assert abs(O.expect(psi, 1, W.Y, 0) - 0.5 * np.sin(om * t)) < 1e-13


def test_larmor_tilted_field_rodrigues():
    """Tilted field: <S>(t) is the Rodrigues rotation of <S>(0) about h by |h| t; 4th-order error ~ tau^4."""
    hv = np.array([0.7, -0.4, 1.1])
    T = 1.0
    s0 = np.array([0.0, 0.0, 0.5])
    n_hat = hv / np.linalg.norm(hv)
    ang = np.linalg.norm(hv) * T
    ref = (s0 * np.cos(ang) + np.cross(n_hat, s0) * np.sin(ang) + n_hat * np.dot(n_hat, s0) * (1 - np.cos(ang)))
    errs = []
    for n in (10, 20, 40):
        psi = np.array([0, 1], dtype=np.complex128)
        O.evolve(psi, 1, hv.reshape(3, 1), np.zeros((3, 1, 1)), T / n, n, 4)
        got = np.array([O.expect(psi, 1, a, 0) for a in range(3)])
        errs.append(np.max(np.abs(got - ref)))
    assert errs[0] < 1e-5
    assert 12 < errs[0] / errs[1] < 20 and 12 < errs[1] / errs[2] < 20, errs


# ------------------------------------------------------------------------ closed forms: two-spin exchange (N=2)
@pytest.mark.parametrize("order", [1, 2, 4])
def test_two_spin_exchange_closed_forms(order):
    """No fields: XX, YY, ZZ commute, so every formula is exact.  J stored once (j<k):
    from |up down>: <S^z_1> = cos((Jx+Jy) t/2)/2; from |up up>: <S^z_1> = cos((Jx-Jy) t/2)/2."""
    Jx, Jy, Jz = 0.9, 0.4, -1.3
    tau, n = 0.11, 13
    t = tau * n
    h = np.zeros((3, 2))
    J = np.zeros((3, 2, 2)); J[0, 0, 1] = Jx; J[1, 0, 1] = Jy; J[2, 0, 1] = Jz
    psi = basis(2, 0b01); O.evolve(psi, 2, h, J, tau, n, order)      # spin 1 (bit 0) up, spin 2 down
    assert abs(O.expect(psi, 2, W.Z, 0) - 0.5 * np.cos((Jx + Jy) * t / 2)) < 1e-13
    assert abs(O.expect(psi, 2, W.Z, 1) + 0.5 * np.cos((Jx + Jy) * t / 2)) < 1e-13
    psi = basis(2, 0b11); O.evolve(psi, 2, h, J, tau, n, order)
    assert abs(O.expect(psi, 2, W.Z, 0) - 0.5 * np.cos((Jx - Jy) * t / 2)) < 1e-13
    # symmetric fill doubles the effective coupling (reading A1)
    J2 = J + np.transpose(J, (0, 2, 1))
    psi = basis(2, 0b01); O.evolve(psi, 2, h, J2, tau, n, order)
    assert abs(O.expect(psi, 2, W.Z, 0) - 0.5 * np.cos((Jx + Jy) * t)) < 1e-13


# -------------------------------------------------------------------- composition order: U1, U2, U4
@pytest.mark.parametrize("N,order,seed", [(2, 1, 61), (3, 2, 62), (3, 4, 63), (5, 1, 64), (6, 2, 65), (8, 4, 66)])
def test_product_formulas_vs_dense_products(N, order, seed):
    w = W.generic(N, seed)
    tau = 0.07
    psi0 = rand_state(N, seed + 1)
    psi = psi0.copy()
    O.evolve(psi, N, w.h, w.J, tau, 1, order)
    ref = D.trotter_dense(N, w.h, w.J, tau, order) @ psi0
    assert np.max(np.abs(psi - ref)) < 1e-12
    # the order of the factors matters at this tolerance: the reversed U1 is a different operator
    if order == 1:
        Hs = [D.hamiltonian_alpha(N, w.h, w.J, a) for a in range(3)]
        wrong = D.expm_herm(Hs[2], tau) @ D.expm_herm(Hs[1], tau) @ D.expm_herm(Hs[0], tau) @ psi0
        assert np.max(np.abs(psi - wrong)) > 1e-6


def test_suzuki_constant():
    assert abs(A_SUZUKI - 0.41449077179437571) < 1e-16
    assert abs((1 - 4 * A_SUZUKI) + 0.65796308717750285) < 1e-15


# --------------------------------------------------------------------------- whole method vs exact exp(-iHt)
def test_fourth_order_error_law():
    N = 6
    w = W.generic(N, 71)
    T = 0.4
    H = D.hamiltonian(N, w.h, w.J)
    psi0 = rand_state(N, 72)
    exact = D.expm_herm(H, T) @ psi0
    errs = []
    for n in (10, 20, 40, 80):
        psi = psi0.copy()
        O.evolve(psi, N, w.h, w.J, T / n, n, 4)
        errs.append(np.max(np.abs(psi - exact)))
    r = [errs[i] / errs[i + 1] for i in range(3)]
    assert all(14.0 < x < 18.0 for x in r), (errs, r)
    # second order: ratio 4
    e2 = []
    for n in (20, 40):
        psi = psi0.copy()
        O.evolve(psi, N, w.h, w.J, T / n, n, 2)
        e2.append(np.max(np.abs(psi - exact)))
    assert 3.5 < e2[0] / e2[1] < 4.5, e2


def test_config1_against_exact_dynamics():
    """BASELINE config 1 (N=10 chain, tau=0.01, 100 steps): the TS error itself is ~4e-12, so the oracle can be
    compared with exact diagonalisation directly."""
    w = W.config(1)
    psi0 = w.state()
    psi = psi0.copy()
    O.evolve(psi, w.N, w.h, w.J, w.tau, w.n_steps, 4)
    exact = D.expm_herm(D.hamiltonian(w.N, w.h, w.J), w.tau * w.n_steps) @ psi0
    gap = np.max(np.abs(psi - exact))
    assert gap < 2e-11, gap
    assert abs(O.norm2(psi, w.N) - 1.0) < 1e-13


# -------------------------------------------------------------------------------- unitarity and reversibility
@pytest.mark.parametrize("N,seed", [(5, 81), (9, 82), (12, 83)])
def test_norm_conservation(N, seed):
    w = W.generic(N, seed)
    psi = w.state()
    O.evolve(psi, N, w.h, w.J, 0.02, 200 if N <= 9 else 20, 4)
    assert abs(O.norm2(psi, N) - 1.0) < 1e-13


def test_loschmidt_echo_sigma_zero():
    """eq. 11 with Sigma = 0: n steps with +tau then n steps with -tau returns psi_0."""
    N = 8
    w = W.generic(N, 91)
    psi0 = w.state()
    psi = psi0.copy()
    O.evolve(psi, N, w.h, w.J, 0.03, 50, 4)
    assert np.max(np.abs(psi - psi0)) > 1e-2
    O.evolve(psi, N, w.h, w.J, -0.03, 50, 4)
    M = abs(O.overlap(psi0, psi, N)) ** 2
    assert abs(1 - M) < 1e-12
    assert np.max(np.abs(psi - psi0)) < 1e-12


def test_magnetisation_conserved_by_polarisation_conserving_H():
    """for J^x = J^y and h^x = h^y = 0 total S^z is conserved by H; the TS drift is O(tau^4)."""
    w = W.config(1)
    psi = w.state()
    m0 = sum(O.expect_all(psi, w.N, W.Z))
    O.evolve(psi, w.N, w.h, w.J, w.tau, 50, 4)
    m1 = sum(O.expect_all(psi, w.N, W.Z))
    assert abs(m1 - m0) < 1e-9


# ------------------------------------------------------------------------------------------------ observables
@pytest.mark.parametrize("N", [1, 3, 6])
def test_observables_vs_dense_operators(N):
    psi = rand_state(N, 100 + N) * 1.3      # un-normalised on purpose: no division by the norm
    for a in range(3):
        for j in range(N):
            assert abs(O.expect(psi, N, a, j) - D.expect_dense(psi, N, a, j)) < 1e-14
    assert abs(O.norm2(psi, N) - 1.69) < 1e-14
    phi = rand_state(N, 200 + N)
    assert abs(O.overlap(phi, psi, N) - np.vdot(phi, psi)) < 1e-14


# ------------------------------------------------------------------------- brute force on tiny hand-built cases
def test_two_spin_full_matrix_by_hand():
    """N=2, H = Jz S^z_1 S^z_2 + hx S^x_1: 4x4 matrix written out by hand in index order (bits: spin2 spin1)."""
    Jz, hx, t = 0.8, 0.6, 0.5
    H = np.array([[Jz / 4, hx / 2, 0, 0],
                  [hx / 2, -Jz / 4, 0, 0],
                  [0, 0, -Jz / 4, hx / 2],
                  [0, 0, hx / 2, Jz / 4]], dtype=complex)
    h = np.zeros((3, 2)); h[W.X, 0] = hx
    J = np.zeros((3, 2, 2)); J[W.Z, 0, 1] = Jz
    assert np.allclose(D.hamiltonian(2, h, J), H)
    psi0 = rand_state(2, 7)
    n = 64
    psi = psi0.copy()
    O.evolve(psi, 2, h, J, t / n, n, 4)
    assert np.max(np.abs(psi - D.expm_herm(H, t) @ psi0)) < 1e-9


# ------------------------------------------------------- cluster factorisation (used for N >= 27 parity checks)
@pytest.mark.parametrize("order", [2, 4])
def test_cluster_factorisation_of_the_product_formulas(order):
    """If J couples only inside disjoint clusters and psi_0 is a product over clusters, every TS factor is a tensor
    product over clusters, so U_2 and U_4 factorise: amplitude(k) = prod_c amplitude_c(k restricted to c)."""
    N = 9
    w = W.clustered(N, W.interleaved_clusters(N, 3), seed=17, tau=0.05, n_steps=6, order=order)
    psi = w.state()
    O.evolve(psi, N, w.h, w.J, w.tau, w.n_steps, order)
    parts = []
    for ci in range(3):
        s = W.sub_workload(w, ci)
        v = s.state()
        O.evolve(v, s.N, s.h, s.J, s.tau, s.n_steps, order)
        parts.append(v)
    k = np.arange(1 << N, dtype=np.int64)
    ref = np.ones(1 << N, dtype=np.complex128)
    for bits, v in zip(w.clusters, parts):
        ref *= v[W.extract_bits(k, bits)]
    assert np.max(np.abs(psi - ref)) < 1e-14
