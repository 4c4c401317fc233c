"""GPU parity: the CUDA path (through the C ABI, via paper_1305_0036_b200.binding) against the CPU oracle on the
same seeded inputs, element by element.  Gates (BASELINE.json north_star): amplitudes max-abs <= 1e-11, observables
<= 1e-10; plus ||psi_gpu - psi_oracle||_2 <= 1e-11 (SURVEY 8 c)."""
import os

import numpy as np
import pytest

from oracle import ts_oracle as O
from paper_1305_0036_b200 import workloads as W

pytestmark = pytest.mark.gpu

AMP_TOL = 1e-11
OBS_TOL = 1e-10
FULL = os.environ.get("TS_PARITY_FULL", "0") == "1"


@pytest.fixture(scope="module")
def B():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    from paper_1305_0036_b200 import binding
    binding.load()
    return binding


def run_gpu(B, w, n_steps=None, order=None, plan=None, tau=None, kernel=None):
    ts = B.TrotterSuzuki(w.N, w.h, w.J)
    if kernel is not None:
        ts.set_option(B.OPT_KERNEL, kernel)
    if plan is not None:
        ts.set_plan(*plan)
    ts.set_state(w.state())
    ts.evolve(w.tau if tau is None else tau, w.n_steps if n_steps is None else n_steps,
              w.order if order is None else order)
    return ts


def run_oracle(w, n_steps=None, order=None, tau=None):
    psi = w.state()
    O.evolve(psi, w.N, w.h, w.J, w.tau if tau is None else tau, w.n_steps if n_steps is None else n_steps,
             w.order if order is None else order, use_tables=True)
    return psi


def check_amps(got, ref, tol=AMP_TOL):
    d = got - ref
    assert np.max(np.abs(d)) <= tol, f"max-abs {np.max(np.abs(d)):.3e}"
    assert np.linalg.norm(d) <= tol, f"2-norm {np.linalg.norm(d):.3e}"


def check_obs(ts, psi_ref, N):
    for a in (0, 1, 2):
        got = ts.expect_all(a)
        ref = O.expect_all(psi_ref, N, a)
        assert np.max(np.abs(got - ref)) <= OBS_TOL, (a, got, ref)
    assert abs(ts.norm2() - O.norm2(psi_ref, N)) <= OBS_TOL


# --------------------------------------------------------------------------------------------- small N (N < 12)
@pytest.mark.parametrize("N", [1, 2, 3, 5, 8, 11])
@pytest.mark.parametrize("order", [2, 4])
@pytest.mark.parametrize("plan", ["auto", "naive"])
def test_small_N_generic(B, N, order, plan):
    """plan = auto: the single-CTA path (ts_small.cu); plan = naive: the paper's launch-per-spin scheme (ts_naive.cu)."""
    w = W.generic(N, seed=100 + N, tau=0.02, n_steps=3, order=order, symmetric_fill=(N % 2 == 1))
    ts = run_gpu(B, w, plan=(B.PLAN_NAIVE, 0, 0) if plan == "naive" else None)
    assert ("naive" if plan == "naive" else "small") in ts.describe_plan()
    ref = run_oracle(w)
    check_amps(ts.get_state(), ref)
    check_obs(ts, ref, N)


def test_naive_matches_tiled_path_forced(B):
    """The same workload through both plans at N = 13 (the two CUDA paths share only the sequencer)."""
    w = W.generic(13, seed=7, tau=0.02, n_steps=2)
    a = run_gpu(B, w, plan=(B.PLAN_NAIVE, 0, 0)).get_state()
    b = run_gpu(B, w, plan=(B.PLAN_TILED, 0, 0)).get_state()
    ref = run_oracle(w)
    check_amps(a, ref)
    check_amps(b, ref)


# --------------------------------------------------------------------------------------------- tiled path
# (N, run_bits, max_group_bits): default plans and forced multi-group plans (ragged last group, single- and
# two-stage high groups, 2/3/4+ groups)
TILED_CASES = [
    (12, 0, 0),      # one group: the low tile only
    (13, 0, 0),      # A + 1-bit high group (run 2^11)
    (15, 0, 1),      # A + three 1-bit groups
    (16, 0, 0),      # A + 4-bit group, single stage
    (16, 0, 2),      # A + 2 + 2
    (17, 0, 0),      # A + 5-bit group (full single stage)
    (18, 0, 0),      # A + 6-bit group: two-stage high group, run 2^6
    (19, 0, 3),      # A + 3 + 2 + 2
    (20, 2, 0),      # A + 8-bit group
    (21, 0, 0),      # A + 9-bit group, run 2^3 (the N = 30 geometry)
    (22, 2, 0),      # A + 10-bit group, run 2^2
    (22, 3, 0),      # A + 5 + 5
]


# kernel 1: the TMA kernels at every size; 2: the library's own choice (one CTA per tile up to two tiles per SM)
@pytest.mark.parametrize("kernel", [1, 2])
@pytest.mark.parametrize("N,rb,mg", TILED_CASES)
def test_tiled_generic(B, N, rb, mg, kernel):
    w = W.generic(N, seed=200 + N, tau=0.02, n_steps=2 if N < 20 else 1, order=4, symmetric_fill=(N == 16))
    ts = run_gpu(B, w, plan=(B.PLAN_TILED, rb, mg), kernel=kernel)
    if N >= 13:
        assert ("kernels=v2" in ts.describe_plan()) == (kernel == 1 or N >= 21)
    ref = run_oracle(w)
    check_amps(ts.get_state(), ref)
    if N <= 18:
        check_obs(ts, ref, N)


@pytest.mark.parametrize("N", [12, 14, 18])
def test_tiled_order2_and_negative_tau(B, N):
    w = W.generic(N, seed=300 + N, tau=0.03, n_steps=3, order=2)
    ts = run_gpu(B, w, kernel=1)
    ref = run_oracle(w)
    check_amps(ts.get_state(), ref)
    # echo: evolving back with -tau returns the initial state (U_2, U_4 are palindromic)
    ts.evolve(-w.tau, w.n_steps, 2)
    check_amps(ts.get_state(), w.state(), tol=1e-12)
    O.evolve(ref, N, w.h, w.J, -w.tau, w.n_steps, 2, True)
    check_amps(ref, w.state(), tol=1e-12)


def test_split_evolve_equals_single_call(B):
    """n steps in one call == n calls of one step (merging across step boundaries only changes round-off)."""
    w = W.generic(14, seed=11, tau=0.02, n_steps=4)
    a = run_gpu(B, w).get_state()
    ts = run_gpu(B, w, n_steps=1)
    for _ in range(3):
        ts.evolve(w.tau, 1, 4)
    check_amps(ts.get_state(), a, tol=1e-13)


# --------------------------------------------------------------------------------------------- BASELINE configs
def test_config1_chain10(B):
    w = W.config(1)
    ts = run_gpu(B, w)
    ref = run_oracle(w)
    check_amps(ts.get_state(), ref)
    check_obs(ts, ref, w.N)
    assert abs(ts.norm2() - 1.0) <= 1e-13


def test_config2_ring16_trace(B):
    """<S^z_1>(t) after every step (paper spin 1 = bit 0), 200 steps."""
    w = W.config(2)
    ts = B.TrotterSuzuki(w.N, w.h, w.J)
    ts.set_basis_state(w.basis_index)
    psi = w.state()
    assert ts.expect(2, 0) == -0.5
    got, ref = [], []
    for _ in range(w.n_steps):
        ts.evolve(w.tau, 1, 4)
        got.append(ts.expect(2, 0))
        O.evolve(psi, w.N, w.h, w.J, w.tau, 1, 4, True)
        ref.append(O.expect(psi, w.N, 2, 0))
    assert np.max(np.abs(np.array(got) - np.array(ref))) <= OBS_TOL
    check_amps(ts.get_state(), psi)
    # 200 separate steps = 8 000 diagonals; each multiplies an amplitude by a table product whose modulus is 1 up to a few
    # ulp that are FIXED per (tile, thread, register): starting from a basis state nothing averages them out at first.
    # Bound: 8 000 x 2 x 3e-17 = 5e-13; the oracle's own norm is held to 1e-13 by tests/test_oracle_pins.py.
    assert abs(ts.norm2() - 1.0) <= 5e-13


def test_config3_dipolar22_all_100_steps(B):
    """BASELINE config 3 at its configured 100 steps (the oracle needs ~1 s per step at N = 22 on the box's 16 cores)."""
    w = W.config(3)
    n = w.n_steps
    assert n == 100
    ts = run_gpu(B, w, n_steps=n)
    ref = run_oracle(w, n_steps=n)
    check_amps(ts.get_state(), ref)
    got = ts.expect_all(2)
    assert np.max(np.abs(got - O.expect_all(ref, w.N, 2))) <= OBS_TOL


def test_config2_trace_without_host_round_trips(B):
    """ts_evolve_observe: the same <S^z_1>(t) trace as above from one call (device-side trace, one copy at the end),
    plus all-site and x / y traces of a few steps against the oracle."""
    w = W.config(2)
    ts = B.TrotterSuzuki(w.N, w.h, w.J)
    ts.set_basis_state(w.basis_index)
    got = ts.evolve_observe(w.tau, w.n_steps, 4, B.Z, 0)
    psi = w.state()
    ref = []
    for _ in range(w.n_steps):
        O.evolve(psi, w.N, w.h, w.J, w.tau, 1, 4, True)
        ref.append(O.expect(psi, w.N, 2, 0))
    assert got.shape == (w.n_steps,)
    assert np.max(np.abs(got - np.array(ref))) <= OBS_TOL
    check_amps(ts.get_state(), psi)
    ts.set_basis_state(w.basis_index)
    allz = ts.evolve_observe(w.tau, 3, 4, B.Z, -1)
    ts.set_basis_state(w.basis_index)
    sx = ts.evolve_observe(w.tau, 3, 4, B.X, 5)
    ts.set_basis_state(w.basis_index)
    sy = ts.evolve_observe(w.tau, 3, 4, B.Y, 5)
    psi = w.state()
    for k in range(3):
        O.evolve(psi, w.N, w.h, w.J, w.tau, 1, 4, True)
        assert np.max(np.abs(allz[k] - O.expect_all(psi, w.N, 2))) <= OBS_TOL
        assert abs(sx[k] - O.expect(psi, w.N, 0, 5)) <= OBS_TOL
        assert abs(sy[k] - O.expect(psi, w.N, 1, 5)) <= OBS_TOL
