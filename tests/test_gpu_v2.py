"""GPU parity of the production kernels (ts_tile_v2.cuh: warp-specialised TMA tile passes and the L2-blocked triple launch)
against the CPU oracle, through the C ABI.

The triple launch is the dominant kernel of the N = 30 benchmark; here it is forced at sizes the FULL oracle reaches
(N = 16 .. 24) with every h and J entry non-zero, over several steps, orders 2 and 4, with chunks from 2^13 to 2^21
amplitudes (tiny chunks = many dependency hand-overs between CTAs per launch), and each test asserts from the library's
own launch counters that the triple launch really ran.  Gates as everywhere: amplitudes max-abs and 2-norm <= 1e-11,
observables <= 1e-10 (BASELINE.json north_star, SURVEY 8 c).
"""
import numpy as np
import pytest

from oracle import ts_oracle as O
from paper_1305_0036_b200 import workloads as W

pytestmark = pytest.mark.gpu

AMP_TOL = 1e-11
OBS_TOL = 1e-10


@pytest.fixture(scope="module")
def B():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    from paper_1305_0036_b200 import binding
    binding.load()
    return binding


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


def oracle_run(w, n_steps, order):
    psi = w.state()
    O.evolve(psi, w.N, w.h, w.J, w.tau, n_steps, order, True)
    return psi


# (N, high groups bottom to top): the first high group + A form the chunk of the triple launch
TRIPLE_CASES = [
    (16, [1, 3]),        # chunk 2^13: 2 tiles per chunk, 8 chunks
    (17, [2, 3]),        # chunk 2^14
    (18, [3, 3]),        # chunk 2^15, single-stage high groups
    (19, [5, 2]),        # chunk 2^17, full single stage
    (20, [6, 2]),        # chunk 2^18: two-stage high group (run 2^6)
    (21, [7, 1, 1]),     # chunk 2^19, four groups
    (22, [8, 2]),        # chunk 2^20, run 2^4
    (22, [9, 1]),        # the default plan at N = 22: chunk 2^21 = the N = 30 geometry, 2 chunks
    (23, [9, 2]),        # default plan, 4 chunks
]


FAMILIES = [1]         # TS_OPT_KERNEL: the warp-specialised TMA kernels (ts_tile_v2.cuh)


@pytest.mark.parametrize("N,groups", TRIPLE_CASES)
@pytest.mark.parametrize("order", [4, 2])
@pytest.mark.parametrize("family", FAMILIES)
def test_triple_launch_generic_J_full_oracle(B, N, groups, order, family):
    steps = 3 if N <= 22 else 2
    w = W.generic(N, seed=500 + 7 * N + len(groups) + order, tau=0.02, n_steps=steps, order=order, symmetric_fill=(N % 3 == 0))
    ts = B.TrotterSuzuki(N, w.h, w.J)
    ts.set_option(B.OPT_KERNEL, family)
    ts.set_option(B.OPT_CHUNK_MIN_LOG2, 13)        # small chunks on purpose: many hand-overs between CTAs per launch
    ts.set_plan_groups(groups)
    ts.set_state(w.state())
    ts.reset_profile()
    ts.evolve(w.tau, steps, order)
    prof = ts.get_profile()
    assert prof["tile_chunk3"]["launches"] > 0, (ts.describe_plan(), prof)
    ref = oracle_run(w, steps, order)
    check_amps(ts.get_state(), ref)
    check_obs(ts, ref, N)
    ts.close()


@pytest.mark.parametrize("family", FAMILIES)
def test_default_plan_N24_triple_launch_three_steps(B, family):
    """The default plan (A + 9 + rest) at N = 24 against the full oracle: the bench plan's geometry with 8 chunks."""
    N = 24
    w = W.generic(N, seed=2424, tau=0.02, n_steps=3)
    ts = B.TrotterSuzuki(N, w.h, w.J)
    ts.set_option(B.OPT_KERNEL, family)
    ts.set_state(w.state())
    ts.reset_profile()
    ts.evolve(w.tau, 3, 4)
    prof = ts.get_profile()
    assert "L2-blocked" in ts.describe_plan()
    assert prof["tile_chunk3"]["launches"] == 3 * 10 - 1, prof    # one per sweep pair meeting at group A: 10 per step, minus the call's first
    ref = oracle_run(w, 3, 4)
    check_amps(ts.get_state(), ref)
    assert np.max(np.abs(ts.expect_all(B.Z) - O.expect_all(ref, N, 2))) <= OBS_TOL
    ts.close()


@pytest.mark.parametrize("N,groups", [(18, [3, 3]), (22, [9, 1]), (21, [9]), (19, [4, 3]), (22, [5, 5]), (23, [10, 1])])
def test_kernel_families_agree_and_match_oracle(B, N, groups):
    """The same plan through (a) the v2 kernels with the triple launch, (b) v2 without it, (c) the one-CTA-per-tile
    kernels: each against the oracle."""
    w = W.generic(N, seed=900 + N, tau=0.02, n_steps=2)
    ref = oracle_run(w, 2, 4)
    for kernel, chunk in ((1, 1), (1, 0), (0, 0)):
        ts = B.TrotterSuzuki(N, w.h, w.J)
        ts.set_plan_groups(groups)
        ts.set_option(B.OPT_KERNEL, kernel)
        ts.set_option(B.OPT_CHUNK, chunk)
        ts.set_option(B.OPT_CHUNK_MIN_LOG2, 13)
        assert ts.get_option(B.OPT_KERNEL) == kernel
        ts.set_state(w.state())
        ts.reset_profile()
        ts.evolve(w.tau, 2, 4)
        prof = ts.get_profile()
        if not (kernel and chunk and len(groups) >= 2):
            assert prof["tile_chunk3"]["launches"] == 0
        check_amps(ts.get_state(), ref)
        ts.close()


@pytest.mark.parametrize("max_ctas", [1, 2, 3, 5, 148])
@pytest.mark.parametrize("N,groups", [(16, [4]), (17, [2, 3]), (19, [7]), (18, [3, 3])])
@pytest.mark.parametrize("family", FAMILIES)
def test_few_ctas_walk_many_tiles(B, N, groups, max_ctas, family):
    """Persistent kernels with 1..5 CTAs: every CTA runs tens of jobs through its three tile buffers (buffer reuse, the
    loader / storer / compute hand-over at every phase parity, ragged job counts per CTA), with and without the triple
    launch.  Full oracle."""
    w = W.generic(N, seed=800 + N + max_ctas, tau=0.02, n_steps=2)
    ts = B.TrotterSuzuki(N, w.h, w.J)
    ts.set_plan_groups(groups)
    ts.set_option(B.OPT_KERNEL, family)
    ts.set_option(B.OPT_MAX_CTAS, max_ctas)
    ts.set_option(B.OPT_CHUNK_MIN_LOG2, 13)
    ts.set_state(w.state())
    ts.evolve(w.tau, 2, 4)
    check_amps(ts.get_state(), oracle_run(w, 2, 4))
    ts.close()


def test_triple_launch_repeated_in_one_process(B):
    """Races are what a multi-CTA hand-over can hide: the same small-chunk launch 30 times over, fresh inputs each."""
    N = 18
    for rep in range(30):
        w = W.generic(N, seed=7000 + rep, tau=0.02, n_steps=4)
        ts = B.TrotterSuzuki(N, w.h, w.J)
        ts.set_option(B.OPT_KERNEL, 1)
        ts.set_option(B.OPT_MAX_CTAS, (0, 37, 100)[rep % 3])
        ts.set_option(B.OPT_CHUNK_MIN_LOG2, 13)
        ts.set_plan_groups([2, 4] if rep % 2 else [3, 3])
        ts.set_state(w.state())
        ts.reset_profile()
        ts.evolve(w.tau, 4, 4)
        assert ts.get_profile()["tile_chunk3"]["launches"] > 0
        check_amps(ts.get_state(), oracle_run(w, 4, 4))
        ts.close()


# --------------------------------------------------------------------------------------------- exported calls
def test_overlap_and_loschmidt_echo(B):
    """ts_overlap against the oracle's overlap, and M_LE = |<psi_0| U(-tau)^n U(tau)^n |psi_0>|^2 = 1 (eq. 11 with
    Sigma = 0) through it."""
    import torch
    N = 16
    w = W.generic(N, seed=1616, tau=0.02, n_steps=5)
    ts = B.TrotterSuzuki(N, w.h, w.J)
    psi0 = w.state()
    phi = torch.from_numpy(psi0).to(ts.device)
    ts.set_state(psi0)
    ts.evolve(w.tau, 5, 4)
    ref = oracle_run(w, 5, 4)
    got = ts.overlap(phi)
    exp = O.overlap(psi0, ref, N)
    assert abs(got - exp) <= OBS_TOL
    ts.evolve(-w.tau, 5, 4)
    back = ts.overlap(phi)
    assert abs(1.0 - abs(back) ** 2) <= 1e-12
    assert abs(back.imag) <= 1e-12
    ts.close()


def test_non_default_stream_and_device_readback(B):
    import torch
    N = 15
    w = W.generic(N, seed=1515, tau=0.02, n_steps=2)
    ts = B.TrotterSuzuki(N, w.h, w.J)
    s = torch.cuda.Stream()
    ts.use_stream(s)
    with torch.cuda.stream(s):
        ts.set_state(w.state())
        ts.evolve(w.tau, 2, 4)
        dst = torch.empty(1 << N, dtype=torch.complex128, device=ts.device)
        B._check(ts._lib.ts_get_state(ts._ctx, B._vp(dst.data_ptr()), 0, 1 << N, B.DEVICE), "ts_get_state")
    s.synchronize()
    ref = oracle_run(w, 2, 4)
    check_amps(dst.cpu().numpy(), ref)
    # a window read back to the device, then to the host
    part = torch.empty(1000, dtype=torch.complex128, device=ts.device)
    B._check(ts._lib.ts_get_state(ts._ctx, B._vp(part.data_ptr()), 12345, 1000, B.DEVICE), "ts_get_state")
    s.synchronize()
    check_amps(part.cpu().numpy(), ref[12345:13345])
    ts.close()


def test_evolve_observe_order2(B):
    N = 14
    w = W.generic(N, seed=1414, tau=0.03, n_steps=4, order=2)
    ts = B.TrotterSuzuki(N, w.h, w.J)
    ts.set_state(w.state())
    got = ts.evolve_observe(w.tau, 4, 2, B.Z, -1)
    psi = w.state()
    for k in range(4):
        O.evolve(psi, N, w.h, w.J, w.tau, 1, 2, True)
        assert np.max(np.abs(got[k] - O.expect_all(psi, N, 2))) <= OBS_TOL
    check_amps(ts.get_state(), psi)
    ts.close()


def test_config5_recipe_at_N24_against_full_oracle(B):
    """BASELINE config 5 (4x8 lattice, checkerboard Neel, N = 32) cannot meet the full oracle (reading A23); the SAME
    recipe -- same couplings, same field distributions and seed, checkerboard Neel -- on a 4x6 lattice (N = 24) can:
    2 steps, all amplitudes and all <S^z_j>."""
    w = W.config5_like(24)
    assert w.N == 24 and w.state_kind == "basis"
    ts = B.TrotterSuzuki(w.N, w.h, w.J)
    ts.set_basis_state(w.basis_index)
    ts.evolve(w.tau, 2, 4)
    ref = oracle_run(w, 2, 4)
    check_amps(ts.get_state(), ref)
    assert np.max(np.abs(ts.expect_all(B.Z) - O.expect_all(ref, w.N, 2))) <= OBS_TOL
    assert abs(ts.norm2() - 1.0) <= 1e-13
    ts.close()


# --------------------------------------------------------------------------------------------- small-N path
@pytest.mark.parametrize("N", [1, 2, 5, 10, 12])
@pytest.mark.parametrize("order", [2, 4])
def test_small_path_single_launch(B, N, order):
    """N <= 12: the whole ts_evolve call is ONE launch of one CTA (small systems are latency-bound)."""
    w = W.generic(N, seed=40 + N, tau=0.02, n_steps=7, order=order, symmetric_fill=(N % 2 == 0))
    ts = B.TrotterSuzuki(N, w.h, w.J)
    assert "small" in ts.describe_plan()
    ts.set_state(w.state())
    ts.reset_profile()
    ts.evolve(w.tau, 7, order)
    prof = ts.get_profile()
    assert prof["small"]["launches"] == 1 and sum(v["launches"] for v in prof.values()) == 1
    ref = oracle_run(w, 7, order)
    check_amps(ts.get_state(), ref)
    check_obs(ts, ref, N)
    ts.evolve(-w.tau, 7, order)                    # echo
    check_amps(ts.get_state(), w.state(), tol=1e-12)
    ts.close()


def test_small_path_off_gives_the_launch_per_spin_scheme(B):
    w = W.generic(9, seed=99, tau=0.02, n_steps=2)
    ts = B.TrotterSuzuki(9, w.h, w.J)
    ts.set_option(B.OPT_SMALL, 0)
    assert "naive" in ts.describe_plan()
    ts.set_state(w.state())
    ts.evolve(w.tau, 2, 4)
    check_amps(ts.get_state(), oracle_run(w, 2, 4))
    ts.close()


# --------------------------------------------------------------------------------------------- NEXT-1 / NEXT-2
@pytest.mark.parametrize("N", [4, 13, 16])
def test_correlators_total_sz_energy(B, N):
    w = W.generic(N, seed=60 + N, tau=0.02, n_steps=2, symmetric_fill=(N == 13))
    ts = B.TrotterSuzuki(N, w.h, w.J)
    ts.set_state(w.state())
    ts.evolve(w.tau, 2, 4)
    ref = oracle_run(w, 2, 4)
    pairs = [(0, 1), (1, 0), (0, N - 1), (N - 2, 1), (N // 2, N // 2 + 1)]
    for a in (B.X, B.Y, B.Z):
        for j, k in pairs:
            assert abs(ts.correlate(a, j, k) - O.correlate(ref, N, a, j, k)) <= OBS_TOL, (a, j, k)
    assert abs(ts.total_sz() - O.total_sz(ref, N)) <= OBS_TOL
    before = ts.get_state()
    E = ts.energy()
    assert abs(E - O.energy_expect(ref, N, w.h, w.J)) <= 1e-9 * max(1.0, abs(E))
    # ts_energy rotates the state into the x and y frames and back: only round-off may remain
    assert np.linalg.norm(ts.get_state() - before) <= 1e-13
    ts.close()


def test_energy_at_N22_default_plan(B):
    """<H> through the tiled path (sweeps via tile passes of every group, exact 2^-N on the way back)."""
    N = 22
    w = W.dipolar_like(N, seed=3)
    ts = B.TrotterSuzuki(N, w.h, w.J)
    psi = w.state()
    ts.set_state(psi)
    E = ts.energy()
    # product state: <H> = sum_a sum_{j<k} Jeff^a_jk <S^a_j><S^a_k>  (h = 0), from the oracle's one-site values at N = 22
    one = np.array([O.expect_all(psi, N, a) for a in range(3)])
    exp = sum(w.J[a, j, k] * one[a, j] * one[a, k] for a in range(3) for j in range(N) for k in range(j + 1, N))
    assert abs(E - exp) <= 1e-10
    assert np.linalg.norm(ts.get_state() - psi) <= 1e-13
    ts.close()


@pytest.mark.parametrize("N,up", [(8, 3), (14, 0), (20, 19)])
def test_random_phase_state_eq_A1(B, N, up):
    ts = B.TrotterSuzuki(N, np.zeros((3, N)), np.zeros((3, N, N)))
    ts.set_random_phase_state(up, seed=1234 + N)
    ref = O.random_phase_state(N, up, 1234 + N)
    got = ts.get_state()
    assert np.max(np.abs(got - ref)) <= 1e-15
    assert np.all(got[((np.arange(1 << N) >> up) & 1) == 0] == 0)
    sz = ts.expect_all(B.Z)
    assert abs(sz[up] - 0.5) <= 1e-12 and np.max(np.abs(np.delete(sz, up))) <= 1e-12
    ts.close()


def test_loschmidt_echo_heisenberg_ring_N16(B):
    """The paper's echo experiment (N = 16 ring, nearest-neighbour Heisenberg, random superposition of Ising
    states, Sigma = 0) at a reduced step count: M_LE = 1 up to round-off, |1 - M_LE| <= 1e-12 (the digits printed at
    P:217 measure Fermi fast-math round-off and are not targets), and the state itself comes back."""
    N = 16
    w = W.chain_like(N, seed=16, tau=0.02, periodic=True)
    w.h[:] = 0.0
    ts = B.TrotterSuzuki(N, w.h, w.J)
    ts.set_random_phase_state(0, seed=5)
    psi0 = ts.get_state()
    m_le, ov = ts.loschmidt_echo(0.02, 500, 4)
    assert abs(1.0 - m_le) <= 1e-12, m_le
    assert np.max(np.abs(ts.get_state() - psi0)) <= 1e-12
    # forward only: the overlap moves away from 1 (the echo is not trivial)
    ts.evolve(0.02, 50, 4)
    import torch
    assert abs(ts.overlap(torch.from_numpy(psi0).to(ts.device))) < 0.99
    ts.close()


def test_total_magnetisation_drift_heisenberg_ring(B):
    """under a polarisation-conserving Hamiltonian the total magnetisation of the evolved state must stay what it
    was; the TS error makes it drift -- "a linear increase ... consistent with ... the TS error".  Heisenberg ring with
    random z fields ([H, S^z_tot] = 0), Gaussian state, N = 20, reduced step counts: the drift at fixed total time
    follows the tau^4 law of the 4th-order scheme (x16 per doubling of tau), matches the oracle's, and is tiny."""
    N = 20
    w = W.chain_like(N, seed=22, tau=0.04, periodic=True)
    ts = B.TrotterSuzuki(N, w.h, w.J)
    drift = {}
    for tau, n in ((0.04, 25), (0.02, 50)):
        ts.set_state(w.state())
        m0 = ts.total_sz()
        ts.evolve(tau, n, 4)
        drift[tau] = ts.total_sz() - m0
        assert abs(ts.norm2() - 1.0) <= 1e-12
    assert 1e-13 < abs(drift[0.04]) < 1e-8, drift
    assert 10.0 < drift[0.04] / drift[0.02] < 24.0, drift
    psi = w.state()
    m0 = O.total_sz(psi, N)
    O.evolve(psi, N, w.h, w.J, 0.04, 25, 4, True)
    assert abs((O.total_sz(psi, N) - m0) - drift[0.04]) <= 1e-12
    ts.close()


# --------------------------------------------------------------------------------------------- NEXT-3: the paper's variants
@pytest.mark.parametrize("N", [9, 13, 18])
def test_naive_plan_with_stored_energy_vectors(B, N):
    """The paper's pre-computed phase-correction variant (three 2^N-element vectors) against the oracle, and
    against the on-the-fly variant of the same plan."""
    w = W.generic(N, seed=300 + N, tau=0.02, n_steps=2)
    ref = oracle_run(w, 2, 4)
    out = []
    for src in (0, 1):
        ts = B.TrotterSuzuki(N, w.h, w.J)
        ts.set_plan(B.PLAN_NAIVE, 0, 0)
        ts.set_option(B.OPT_DIAG_SOURCE, src)
        ts.set_state(w.state())
        ts.evolve(w.tau, 2, 4)
        out.append(ts.get_state())
        check_amps(out[-1], ref)
        assert ts.get_profile()["naive_rot"]["launches"] == 2 * 20 * N
        ts.close()
    assert np.max(np.abs(out[0] - out[1])) <= 1e-13


# --------------------------------------------------------------------------------------------- CUDA-graph replay (small states)
@pytest.mark.parametrize("N,kernel", [(13, 2), (16, 2), (16, 1), (19, 2), (21, 2)])
@pytest.mark.parametrize("order", [4, 2])
def test_graph_replay_of_small_states(B, N, kernel, order):
    """N <= 21: a call of >= 4 steps replays one step's launches from a CUDA graph (head + unit x (n - 2) + tail).  Same
    amplitudes, bit for bit, as the launch-by-launch path, and both against the oracle; the launch counters count the
    replayed launches."""
    steps = 6
    w = W.generic(N, seed=9000 + N + order, tau=0.02, n_steps=steps, order=order)
    out = []
    for graph in (1, 0):
        ts = B.TrotterSuzuki(N, w.h, w.J)
        ts.set_option(B.OPT_KERNEL, kernel)
        ts.set_option(B.OPT_GRAPH, graph)
        ts.set_state(w.state())
        ts.reset_profile()
        ts.evolve(w.tau, steps, order)
        prof = ts.get_profile()
        assert ts.get_option(B.OPT_GRAPH_REPLAYS) == (steps - 2 if graph else 0)
        out.append((ts.get_state(), sum(v["launches"] for v in prof.values())))
        ts.evolve(w.tau, 1, order)                 # a later call on the same context (the graph is released lazily)
        ts.close()
    assert out[0][1] == out[1][1]                  # same number of kernel launches accounted
    assert np.array_equal(out[0][0], out[1][0])
    check_amps(out[0][0], oracle_run(w, steps, order))


def test_evolve_observe_graph_replay_matches_launch_by_launch(B):
    """ts_evolve_observe on a small state replays [one step + the row's reduction] from a CUDA graph, the row index
    advancing on the device: same trace, bit for bit, as the launch-by-launch path, and against the oracle."""
    N, steps = 15, 12
    w = W.generic(N, seed=9100, tau=0.02, n_steps=steps)
    traces = []
    for graph in (1, 0):
        ts = B.TrotterSuzuki(N, w.h, w.J)
        ts.set_option(B.OPT_GRAPH, graph)
        ts.set_state(w.state())
        traces.append(ts.evolve_observe(w.tau, steps, 4, B.Z, -1))          # all sites, every step
        assert ts.get_option(B.OPT_GRAPH_REPLAYS) == (steps - 1 if graph else 0)
        ts.close()
    assert np.array_equal(traces[0], traces[1])
    psi = w.state()
    for k in range(steps):
        O.evolve(psi, N, w.h, w.J, w.tau, 1, 4, True)
        assert np.max(np.abs(traces[0][k] - O.expect_all(psi, N, O.Z))) <= OBS_TOL


def test_effective_clock_probe(B):
    """TS_OPT_LAST_LAUNCH_KHZ: SM cycles per wall nanosecond as seen by CTA 0's loader of the last persistent launch."""
    N = 24
    w = W.generic(N, seed=77, tau=0.01, n_steps=1)
    ts = B.TrotterSuzuki(N, w.h, w.J)
    ts.set_random_phase_state(0, seed=1)
    ts.evolve(w.tau, 2, 4)
    khz = ts.get_option(B.OPT_LAST_LAUNCH_KHZ)
    assert 300_000 < khz < 3_000_000, khz
    ts.close()
