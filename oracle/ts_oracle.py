"""ctypes wrapper of the CPU oracle (oracle/ts_oracle.c).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this.
It imports nothing from paper_1305_0036_b200 (the CUDA path), and that package imports nothing from here.
All arithmetic is in ts_oracle.c; this file only marshals numpy arrays.
"""
import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_lib = None

SWEEP_YDAG, SWEEP_Y, SWEEP_XDAG, SWEEP_X = 0, 1, 2, 3
X, Y, Z = 0, 1, 2

_dp = ctypes.POINTER(ctypes.c_double)


def _load():
    global _lib
    if _lib is not None:
        return _lib
    import importlib.util
    spec = importlib.util.spec_from_file_location("_ts_oracle_build", os.path.join(_HERE, "build.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    path = mod.build()
    lib = ctypes.CDLL(path)
    lib.tso_num_threads.restype = ctypes.c_int
    lib.tso_energy.restype = ctypes.c_double
    lib.tso_energy.argtypes = [ctypes.c_int, _dp, _dp, ctypes.c_uint64]
    lib.tso_energy_table.restype = None
    lib.tso_energy_table.argtypes = [ctypes.c_int, _dp, _dp, _dp]
    lib.tso_apply_diag.restype = None
    lib.tso_apply_diag.argtypes = [_dp, ctypes.c_int, _dp, _dp, _dp, ctypes.c_double]
    lib.tso_rotate_bit.restype = None
    lib.tso_rotate_bit.argtypes = [_dp, ctypes.c_int, ctypes.c_int, ctypes.c_int]
    lib.tso_apply_sweep.restype = None
    lib.tso_apply_sweep.argtypes = [_dp, ctypes.c_int, ctypes.c_int]
    lib.tso_scale.restype = None
    lib.tso_scale.argtypes = [_dp, ctypes.c_int, ctypes.c_double]
    lib.tso_evolve.restype = ctypes.c_int
    lib.tso_evolve.argtypes = [_dp, ctypes.c_int, _dp, _dp, ctypes.c_double, ctypes.c_int64, ctypes.c_int,
                               ctypes.c_int]
    lib.tso_apply_H_alpha.restype = ctypes.c_int
    lib.tso_apply_H_alpha.argtypes = [_dp, ctypes.c_int, _dp, _dp, ctypes.c_int, ctypes.c_double]
    lib.tso_expect.restype = ctypes.c_double
    lib.tso_expect.argtypes = [_dp, ctypes.c_int, ctypes.c_int, ctypes.c_int]
    lib.tso_norm2.restype = ctypes.c_double
    lib.tso_norm2.argtypes = [_dp, ctypes.c_int]
    lib.tso_overlap.restype = None
    lib.tso_overlap.argtypes = [_dp, _dp, ctypes.c_int, _dp]
    lib.tso_correlate.restype = ctypes.c_double
    lib.tso_correlate.argtypes = [_dp, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int]
    lib.tso_total_sz.restype = ctypes.c_double
    lib.tso_total_sz.argtypes = [_dp, ctypes.c_int]
    lib.tso_energy_expect.restype = ctypes.c_double
    lib.tso_energy_expect.argtypes = [_dp, ctypes.c_int, _dp, _dp]
    lib.tso_splitmix64.restype = ctypes.c_uint64
    lib.tso_splitmix64.argtypes = [ctypes.c_uint64, ctypes.c_uint64]
    lib.tso_random_phase_state.restype = None
    lib.tso_random_phase_state.argtypes = [_dp, ctypes.c_int, ctypes.c_int, ctypes.c_uint64]
    _lib = lib
    return lib


def _psi_ptr(psi, N):
    assert isinstance(psi, np.ndarray) and psi.dtype == np.complex128 and psi.flags.c_contiguous
    assert psi.size == (1 << N), (psi.size, N)
    return psi.ctypes.data_as(_dp)


def _f64(a, shape):
    a = np.ascontiguousarray(a, dtype=np.float64)
    assert a.shape == shape, (a.shape, shape)
    return a


def num_threads() -> int:
    return int(_load().tso_num_threads())


def energy(N, h_a, J_a, k) -> float:
    """E_alpha(k) of eq. 1 for one alpha: h_a [N], J_a [N][N]."""
    h_a = _f64(h_a, (N,)); J_a = _f64(J_a, (N, N))
    return float(_load().tso_energy(N, h_a.ctypes.data_as(_dp), J_a.ctypes.data_as(_dp), int(k)))


def energy_table(N, h_a, J_a) -> np.ndarray:
    h_a = _f64(h_a, (N,)); J_a = _f64(J_a, (N, N))
    E = np.empty(1 << N, dtype=np.float64)
    _load().tso_energy_table(N, h_a.ctypes.data_as(_dp), J_a.ctypes.data_as(_dp), E.ctypes.data_as(_dp))
    return E


def apply_diag(psi, N, h_a, J_a, t, table=None):
    """In place: c_k <- c_k exp(-i t E(k))."""
    h_a = _f64(h_a, (N,)); J_a = _f64(J_a, (N, N))
    tp = None
    if table is not None:
        table = _f64(table, (1 << N,))
        tp = table.ctypes.data_as(_dp)
    _load().tso_apply_diag(_psi_ptr(psi, N), N, h_a.ctypes.data_as(_dp), J_a.ctypes.data_as(_dp), tp, float(t))


def rotate_bit(psi, N, j, kind):
    assert 0 <= j < N
    _load().tso_rotate_bit(_psi_ptr(psi, N), N, int(j), int(kind))


def apply_sweep(psi, N, kind):
    _load().tso_apply_sweep(_psi_ptr(psi, N), N, int(kind))


def scale(psi, N, f):
    _load().tso_scale(_psi_ptr(psi, N), N, float(f))


def evolve(psi, N, h, J, tau, n_steps, order=4, use_tables=True):
    """In place: psi <- U_order(tau)^n_steps psi.  h [3][N], J [3][N][N]."""
    h = _f64(h, (3, N)); J = _f64(J, (3, N, N))
    rc = _load().tso_evolve(_psi_ptr(psi, N), N, h.ctypes.data_as(_dp), J.ctypes.data_as(_dp), float(tau),
                            int(n_steps), int(order), 1 if use_tables else 0)
    if rc != 0:
        raise ValueError("tso_evolve: bad arguments or out of memory")


def apply_H_alpha(psi, N, h, J, alpha, t):
    """In place: psi <- exp(-i t H_alpha) psi (one factor of eq. 3)."""
    h = _f64(h, (3, N)); J = _f64(J, (3, N, N))
    rc = _load().tso_apply_H_alpha(_psi_ptr(psi, N), N, h.ctypes.data_as(_dp), J.ctypes.data_as(_dp),
                                   int(alpha), float(t))
    if rc != 0:
        raise ValueError("tso_apply_H_alpha: bad arguments")


def expect(psi, N, alpha, j) -> float:
    assert 0 <= j < N and alpha in (0, 1, 2)
    return float(_load().tso_expect(_psi_ptr(psi, N), N, int(alpha), int(j)))


def expect_all(psi, N, alpha) -> np.ndarray:
    return np.array([expect(psi, N, alpha, j) for j in range(N)])


def norm2(psi, N) -> float:
    return float(_load().tso_norm2(_psi_ptr(psi, N), N))


def overlap(phi, psi, N) -> complex:
    out = np.zeros(2)
    _load().tso_overlap(_psi_ptr(phi, N), _psi_ptr(psi, N), N, out.ctypes.data_as(_dp))
    return complex(out[0], out[1])


def correlate(psi, N, alpha, j, k) -> float:
    """<psi| S^alpha_j S^alpha_k |psi>, j != k."""
    assert j != k
    return float(_load().tso_correlate(_psi_ptr(psi, N), N, alpha, j, k))


def total_sz(psi, N) -> float:
    return float(_load().tso_total_sz(_psi_ptr(psi, N), N))


def energy_expect(psi, N, h, J) -> float:
    """<psi|H|psi> for eq. 1, from one- and two-site expectation values."""
    h = _f64(h, (3, N))
    J = _f64(J, (3, N, N))
    return float(_load().tso_energy_expect(_psi_ptr(psi, N), N, h.ctypes.data_as(_dp), J.ctypes.data_as(_dp)))


def splitmix64(seed, j) -> int:
    return int(_load().tso_splitmix64(ctypes.c_uint64(seed), ctypes.c_uint64(j)))


def random_phase_state(N, up_spin, seed) -> np.ndarray:
    """Eq. A.1: spin `up_spin` up, the other N-1 spins in an equal-weight random-phase superposition."""
    psi = np.empty(1 << N, dtype=np.complex128)
    _load().tso_random_phase_state(_psi_ptr(psi, N), N, up_spin, ctypes.c_uint64(seed))
    return psi
