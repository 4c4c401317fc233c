"""Dense-matrix reference used ONLY to pin the oracle (tests, N <= 10).

Written independently of oracle/ts_oracle.c: operators are built as Kronecker products of 2x2 matrices and the
Hamiltonian of eq. 1 is exponentiated by diagonalisation.  Nothing here is used by the CUDA path.

Basis order of each 2x2 factor: index 0 = bit 0 = down, index 1 = bit 1 = up, so
S^z = diag(-1/2, +1/2), S^x = [[0, 1/2], [1/2, 0]], S^y = [[0, +i/2], [-i/2, 0]]  (<down|S^y|up> = +i/2).
Spin j <-> bit j: in a Kronecker product the LAST factor is the fastest (bit 0), so spin j is factor N-1-j.
"""
import numpy as np

SZ = np.array([[-0.5, 0.0], [0.0, 0.5]], dtype=complex)
SX = np.array([[0.0, 0.5], [0.5, 0.0]], dtype=complex)
SY = np.array([[0.0, 0.5j], [-0.5j, 0.0]], dtype=complex)
SPIN = (SX, SY, SZ)
I2 = np.eye(2, dtype=complex)


def site_op(op2, j, N):
    out = np.ones((1, 1), dtype=complex)
    for f in range(N):             # factor f <-> spin N-1-f
        out = np.kron(out, op2 if (N - 1 - f) == j else I2)
    return out


def hamiltonian_alpha(N, h, J, a):
    """H_alpha = sum_j h^a_j S^a_j + sum_{j != k} J^a_{jk} S^a_j S^a_k  (eq. 1; reading A1)."""
    dim = 1 << N
    H = np.zeros((dim, dim), dtype=complex)
    ops = [site_op(SPIN[a], j, N) for j in range(N)]
    for j in range(N):
        H += h[a][j] * ops[j]
    for j in range(N):
        for k in range(N):
            if j != k and J[a][j][k] != 0.0:
                H += J[a][j][k] * (ops[j] @ ops[k])
    return H


def hamiltonian(N, h, J):
    return sum(hamiltonian_alpha(N, h, J, a) for a in range(3))


def expm_herm(H, t):
    """exp(-i t H) for Hermitian H by diagonalisation."""
    w, V = np.linalg.eigh(H)
    return (V * np.exp(-1j * t * w)) @ V.conj().T


def trotter_dense(N, h, J, tau, order):
    """The product formulas of P:52-58 as dense matrices, built from dense exponentials of H_x, H_y, H_z:
    U1(t) = e^{-itHx} e^{-itHy} e^{-itHz};  U2(t) = U1^dag(-t/2) U1(t/2);  U4 = U2(at)^2 U2((1-4a)t) U2(at)^2."""
    Hx, Hy, Hz = (hamiltonian_alpha(N, h, J, a) for a in range(3))

    def U1(t):
        return expm_herm(Hx, t) @ expm_herm(Hy, t) @ expm_herm(Hz, t)

    def U2(t):
        return U1(-t / 2).conj().T @ U1(t / 2)

    if order == 1:
        return U1(tau)
    if order == 2:
        return U2(tau)
    a = 1.0 / (4.0 - 4.0 ** (1.0 / 3.0))
    A = U2(a * tau)
    B = U2((1 - 4 * a) * tau)
    return A @ A @ B @ A @ A


def expect_dense(psi, N, a, j):
    return float(np.real(np.vdot(psi, site_op(SPIN[a], j, N) @ psi)))
