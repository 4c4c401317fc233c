"""Seeded synthetic workloads (Hamiltonians and initial states) shared by the oracle tests, the GPU parity tests,
`__graft_entry__.smoke()` and `bench.py`.

This module holds NONE of the method's arithmetic (no rotations, phases, energies, Trotter formulas): it only
draws numbers and fills the inputs of eq. 1-2 of the paper (h[3][N], J[3][N][N], psi_0).  It is the only
code that serves both the CPU oracle and the CUDA path; it imports neither.

One generator everywhere: numpy `Generator(PCG64(seed))` (reading A21).  Draw orders are stated
next to each recipe.  Couplings are stored ONCE per unordered pair, at J[alpha][j][k] with j < k (reading A1).
Axis index: alpha = 0, 1, 2 for x, y, z.  Spin j <-> bit j of the amplitude index; bit 1 = up.

The five BASELINE.json configs are `config(1..5)`; the metric workload (N = 30) is `config("M")`.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Callable, List, Optional, Sequence, Tuple

import numpy as np

X, Y, Z = 0, 1, 2


def _rng(seed: int) -> np.random.Generator:
    return np.random.Generator(np.random.PCG64(seed))


@dataclass
class Workload:
    name: str
    N: int
    h: np.ndarray                 # [3][N]
    J: np.ndarray                 # [3][N][N], filled for j < k only
    tau: float
    n_steps: int
    order: int = 4
    state_kind: str = "gaussian"  # "gaussian" | "basis" | "product" | "cluster_product"
    state_seed: Optional[int] = None
    basis_index: Optional[int] = None
    spin_states: Optional[np.ndarray] = None          # [N][2] = (amp of bit 0 (down), amp of bit 1 (up))
    clusters: Optional[List[List[int]]] = None        # bit lists, for cluster-factorised workloads
    cluster_states: Optional[List[np.ndarray]] = None
    note: str = ""
    n_bonds: int = 0

    @property
    def dim(self) -> int:
        return 1 << self.N

    def state(self) -> np.ndarray:
        """The full initial state as a complex128 numpy array (host).  Use `state_chunks` for N >= 28."""
        out = np.empty(self.dim, dtype=np.complex128)
        for first, chunk in self.state_chunks(chunk_log2=min(self.N, 24)):
            out[first:first + chunk.size] = chunk
        return out

    def state_chunks(self, chunk_log2: int = 24):
        """Yield (first_index, complex128 chunk) in index order; chunks have 2^chunk_log2 amplitudes."""
        dim = self.dim
        csz = 1 << min(chunk_log2, self.N)
        if self.state_kind == "basis":
            for first in range(0, dim, csz):
                c = np.zeros(csz, dtype=np.complex128)
                if first <= self.basis_index < first + csz:
                    c[self.basis_index - first] = 1.0
                yield first, c
        elif self.state_kind == "gaussian":
            # interleaved (re, im) standard normals in index order; normalised by the exact 2-norm.
            # Two passes over the same stream: one for the norm, one to emit.
            rng = _rng(self.state_seed)
            nrm2 = 0.0
            for first in range(0, dim, csz):
                v = rng.standard_normal(2 * csz)
                nrm2 += float(np.dot(v, v))
            inv = 1.0 / np.sqrt(nrm2)
            rng = _rng(self.state_seed)
            for first in range(0, dim, csz):
                v = rng.standard_normal(2 * csz)
                yield first, (v * inv).view(np.complex128)
        elif self.state_kind == "product":
            for first in range(0, dim, csz):
                yield first, _product_chunk(self.spin_states, self.N, first, csz)
        elif self.state_kind == "cluster_product":
            for first in range(0, dim, csz):
                k = np.arange(first, first + csz, dtype=np.int64)
                c = np.ones(csz, dtype=np.complex128)
                for bits, st in zip(self.clusters, self.cluster_states):
                    c *= st[extract_bits(k, bits)]
                yield first, c
        else:
            raise ValueError(self.state_kind)


def extract_bits(k: np.ndarray, bits: Sequence[int]) -> np.ndarray:
    """Gather bits `bits` of each index in k into a compact index (bits[i] -> bit i)."""
    out = np.zeros_like(k)
    for i, b in enumerate(bits):
        out |= ((k >> b) & 1) << i
    return out


def _product_chunk(spin_states: np.ndarray, N: int, first: int, csz: int) -> np.ndarray:
    """Amplitudes first..first+csz-1 of the product state  (x)_j (s[j][0]|down> + s[j][1]|up>)."""
    nlow = int(np.log2(csz))
    low = np.ones(1, dtype=np.complex128)
    for j in range(nlow):            # bit j varies slower than bits < j  ->  kron(new, low)
        low = np.kron(spin_states[j], low)
    pref = 1.0 + 0.0j
    for j in range(nlow, N):
        pref *= spin_states[j][(first >> j) & 1]
    return low * pref


# ------------------------------------------------------------------------------------------------ lattices
def chain_bonds(N: int, periodic: bool) -> List[Tuple[int, int]]:
    b = [(j, j + 1) for j in range(N - 1)]
    if periodic and N > 2:
        b.append((0, N - 1))
    return b


def grid_bonds(rows: int, cols: int, n_sites: Optional[int] = None) -> List[Tuple[int, int]]:
    """Open rows x cols grid, site j at (j // cols, j % cols); sites >= n_sites removed (reading A16)."""
    n = rows * cols if n_sites is None else n_sites
    b = []
    for j in range(n):
        r, c = divmod(j, cols)
        if c + 1 < cols and j + 1 < n:
            b.append((j, j + 1))
        if r + 1 < rows and j + cols < n:
            b.append((j, j + cols))
    return b


def _fill_bonds(N: int, bonds, Jxyz) -> np.ndarray:
    J = np.zeros((3, N, N))
    for (j, k) in bonds:
        j, k = min(j, k), max(j, k)
        for a in range(3):
            J[a, j, k] = Jxyz[a]
    return J


def checkerboard_index(rows: int, cols: int) -> int:
    """Neel state on a grid: bit j = (row + col) mod 2 (reading A17)."""
    k = 0
    for j in range(rows * cols):
        r, c = divmod(j, cols)
        if (r + c) & 1:
            k |= 1 << j
    return k


def _grid_workload(name, rows, cols, n_sites, seed_fields, tau, n_steps, **state) -> Workload:
    """Anisotropic XYZ nearest-neighbour grid: J = (0.8, 1.0, 1.2); h^z ~ N(0, 0.5), h^x ~ N(0, 0.2), drawn z
    first then x (standard deviations, reading A18)."""
    N = n_sites
    bonds = grid_bonds(rows, cols, n_sites)
    rng = _rng(seed_fields)
    h = np.zeros((3, N))
    h[Z] = rng.normal(0.0, 0.5, N)
    h[X] = rng.normal(0.0, 0.2, N)
    return Workload(name=name, N=N, h=h, J=_fill_bonds(N, bonds, (0.8, 1.0, 1.2)), tau=tau, n_steps=n_steps,
                    n_bonds=len(bonds), **state)


def dipolar_couplings(N: int, seed: int) -> np.ndarray:
    """All-to-all dipolar network (reading A20): r_j ~ U[0,1)^3 drawn row-major, d_jk = r_jk^-3 / max d;
    J^z = 2 d, J^x = J^y = -d, stored for j < k."""
    rng = _rng(seed)
    pos = rng.random((N, 3))
    J = np.zeros((3, N, N))
    d = np.zeros((N, N))
    for j in range(N):
        for k in range(j + 1, N):
            d[j, k] = np.linalg.norm(pos[j] - pos[k]) ** -3
    d /= d.max()
    J[Z] = 2.0 * d
    J[X] = -d
    J[Y] = -d
    return J


def random_product_spins(N: int, seed: int) -> np.ndarray:
    """Per spin cos(theta) ~ U[-1,1], phi ~ U[0, 2 pi) (drawn theta, phi per spin in order); spin state
    cos(theta/2)|up> + e^{i phi} sin(theta/2)|down>  (reading A19).  Returns [N][2] = (down amp, up amp)."""
    rng = _rng(seed)
    s = np.zeros((N, 2), dtype=np.complex128)
    for j in range(N):
        ct = rng.uniform(-1.0, 1.0)
        phi = rng.uniform(0.0, 2.0 * np.pi)
        th = np.arccos(ct)
        s[j, 1] = np.cos(th / 2)
        s[j, 0] = np.exp(1j * phi) * np.sin(th / 2)
    return s


# ----------------------------------------------------------------------------------------- BASELINE configs
def config(which) -> Workload:
    if which == 1:
        # N=10 open Heisenberg chain, J^x=J^y=J^z=1 nn; h^z ~ U[-0.5,0.5] seed 0; Gaussian state seed 1.
        N = 10
        bonds = chain_bonds(N, periodic=False)
        h = np.zeros((3, N))
        h[Z] = _rng(0).uniform(-0.5, 0.5, N)
        return Workload("config1_chain10", N, h, _fill_bonds(N, bonds, (1.0, 1.0, 1.0)), tau=0.01, n_steps=100,
                        state_kind="gaussian", state_seed=1, n_bonds=len(bonds))
    if which == 2:
        # N=16 periodic XXZ ring, J^x=J^y=1, J^z=0.5; h^x=0.3; h^z ~ U[-1,1] seed 2; Neel bit j = j mod 2.
        N = 16
        bonds = chain_bonds(N, periodic=True)
        h = np.zeros((3, N))
        h[X] = 0.3
        h[Z] = _rng(2).uniform(-1.0, 1.0, N)
        return Workload("config2_ring16", N, h, _fill_bonds(N, bonds, (1.0, 1.0, 0.5)), tau=0.02, n_steps=200,
                        state_kind="basis", basis_index=0xAAAA, n_bonds=len(bonds))
    if which == 3:
        # N=22 all-to-all dipolar, seed 3; h=0; random product state seed 4.
        N = 22
        return Workload("config3_dipolar22", N, np.zeros((3, N)), dipolar_couplings(N, 3), tau=0.005,
                        n_steps=100, state_kind="product", spin_states=random_product_spins(N, 4),
                        n_bonds=N * (N - 1) // 2)
    if which == 4:
        # N=27: 4x7 open grid minus its last site (reading A16): 27 sites, 43 bonds.
        return _grid_workload("config4_grid27", 4, 7, 27, 5, tau=0.01, n_steps=50,
                              state_kind="gaussian", state_seed=6)
    if which == 5:
        # N=32: 4x8 open grid, 52 bonds; checkerboard Neel.
        return _grid_workload("config5_grid32", 4, 8, 32, 7, tau=0.01, n_steps=10,
                              state_kind="basis", basis_index=checkerboard_index(4, 8))
    if which == "M":
        # metric workload: N=30, 5x6 open grid, 49 bonds, seed 8; Gaussian state seed 9.
        return _grid_workload("metric_grid30", 5, 6, 30, 8, tau=0.01, n_steps=5,
                              state_kind="gaussian", state_seed=9)
    raise KeyError(which)


def config5_like(N: int) -> Workload:
    """BASELINE config 5's recipe (4-row open XYZ lattice, fields from seed 7, checkerboard Neel state, tau = 0.01) on
    a 4 x (N/4) lattice: the size at which that Hamiltonian family can meet the full oracle (reading A23)."""
    assert N % 4 == 0 and N >= 8
    cols = N // 4
    return _grid_workload(f"config5_like_grid{N}", 4, cols, N, 7, tau=0.01, n_steps=10,
                          state_kind="basis", basis_index=checkerboard_index(4, cols))


def grid_like(N: int, seed: int, tau: float = 0.01, n_steps: int = 2, state_seed: Optional[int] = None,
              cols: Optional[int] = None) -> Workload:
    """Same recipe as configs 4/5/M on a ceil(N/cols) x cols open grid truncated to N sites."""
    if cols is None:
        cols = max(1, int(np.floor(np.sqrt(N))))
        while cols > 1 and cols * cols > N:
            cols -= 1
        cols = max(cols, 1) if N < 4 else max(cols, 2)
    rows = (N + cols - 1) // cols
    return _grid_workload(f"grid{N}", rows, cols, N, seed, tau=tau, n_steps=n_steps,
                          state_kind="gaussian", state_seed=seed + 1000 if state_seed is None else state_seed)


def chain_like(N: int, seed: int, tau: float = 0.01, n_steps: int = 2, periodic: bool = False) -> Workload:
    """Heisenberg chain/ring with random z fields, Gaussian state (config-1 recipe at any N)."""
    bonds = chain_bonds(N, periodic)
    h = np.zeros((3, N))
    h[Z] = _rng(seed).uniform(-0.5, 0.5, N)
    return Workload(f"chain{N}", N, h, _fill_bonds(N, bonds, (1.0, 1.0, 1.0)), tau=tau, n_steps=n_steps,
                    state_kind="gaussian", state_seed=seed + 1000, n_bonds=len(bonds))


def dipolar_like(N: int, seed: int, tau: float = 0.005, n_steps: int = 2) -> Workload:
    """Config-3 recipe at any N: all-to-all dipolar couplings, random product state."""
    return Workload(f"dipolar{N}", N, np.zeros((3, N)), dipolar_couplings(N, seed), tau=tau, n_steps=n_steps,
                    state_kind="product", spin_states=random_product_spins(N, seed + 1000),
                    n_bonds=N * (N - 1) // 2)


def generic(N: int, seed: int, tau: float = 0.01, n_steps: int = 2, order: int = 4,
            symmetric_fill: bool = False) -> Workload:
    """Every parameter of eq. 1 non-zero: h[3][N] ~ N(0, 0.5), J[3][j<k] ~ N(0, 1/sqrt(N)); Gaussian state.
    With symmetric_fill the lower triangle and the diagonal are filled too (exercises reading A1)."""
    rng = _rng(seed)
    h = rng.normal(0.0, 0.5, (3, N))
    J = np.zeros((3, N, N))
    sc = 1.0 / np.sqrt(max(N, 1))
    for a in range(3):
        for j in range(N):
            for k in range(j + 1, N):
                J[a, j, k] = rng.normal(0.0, sc)
    if symmetric_fill:
        for a in range(3):
            for j in range(N):
                for k in range(j):
                    J[a, j, k] = rng.normal(0.0, sc)
                J[a, j, j] = rng.normal(0.0, 1.0)
    return Workload(f"generic{N}", N, h, J, tau=tau, n_steps=n_steps, order=order, state_kind="gaussian",
                    state_seed=seed + 1000, n_bonds=N * (N - 1) // 2)


def clustered(N: int, cluster_bits: List[List[int]], seed: int, tau: float = 0.01, n_steps: int = 2,
              order: int = 4) -> Workload:
    """Cluster-factorised workload: couplings only inside the given disjoint
    bit sets, all-to-all inside each with J ~ N(0, 0.5), fields h ~ N(0, 0.5) on every spin; the initial state is
    the tensor product of one normalised complex-Gaussian state per cluster.  Draw order: per cluster in list
    order: fields (3 x n), couplings (alpha, then pairs j<k in cluster order), state (interleaved re, im)."""
    seen = sorted(b for c in cluster_bits for b in c)
    assert seen == list(range(N)), "clusters must partition the bits"
    rng = _rng(seed)
    h = np.zeros((3, N))
    J = np.zeros((3, N, N))
    states = []
    for bits in cluster_bits:
        n = len(bits)
        hc = rng.normal(0.0, 0.5, (3, n))
        for a in range(3):
            for i, b in enumerate(bits):
                h[a, b] = hc[a, i]
        for a in range(3):
            for i in range(n):
                for m in range(i + 1, n):
                    v = rng.normal(0.0, 0.5)
                    j, k = min(bits[i], bits[m]), max(bits[i], bits[m])
                    J[a, j, k] = v
        v = rng.standard_normal(2 << n)
        v /= np.sqrt(np.dot(v, v))
        states.append(v.view(np.complex128).copy())
    nb = sum(len(c) * (len(c) - 1) // 2 for c in cluster_bits)
    return Workload(f"clustered{N}", N, h, J, tau=tau, n_steps=n_steps, order=order,
                    state_kind="cluster_product", clusters=[list(c) for c in cluster_bits],
                    cluster_states=states, n_bonds=nb)


def sub_workload(w: Workload, ci: int) -> Workload:
    """The ci-th cluster of a clustered workload as a stand-alone small problem (cluster bit i -> bit i)."""
    bits = w.clusters[ci]
    n = len(bits)
    h = np.zeros((3, n))
    J = np.zeros((3, n, n))
    for a in range(3):
        for i, b in enumerate(bits):
            h[a, i] = w.h[a, b]
            for m, b2 in enumerate(bits):
                if i < m:
                    J[a, i, m] = w.J[a, min(b, b2), max(b, b2)]
    st = w.cluster_states[ci]
    sub = Workload(f"{w.name}_c{ci}", n, h, J, tau=w.tau, n_steps=w.n_steps, order=w.order, state_kind="custom")
    sub._custom = st
    sub.state = lambda st=st: st.copy()
    return sub


def interleaved_clusters(N: int, n_clusters: int) -> List[List[int]]:
    """Cluster c holds bits c, c + n_clusters, c + 2 n_clusters, ...: every cluster spans low, middle and high
    index bits, so its couplings cross every tile boundary of the CUDA path."""
    return [list(range(c, N, n_clusters)) for c in range(n_clusters)]
