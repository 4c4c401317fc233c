"""Thin ctypes binding of libts_b200.so (include/ts_b200.h).  Argument marshalling only: every step of the hot path
runs in the library's CUDA kernels.  PyTorch supplies device memory and the stream, nothing else.

There is NO fallback: if the library is missing or no CUDA device is usable, calls raise.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libts_b200.so")

TS_OK, TS_ERR_ARG, TS_ERR_NOMEM, TS_ERR_CUDA, TS_ERR_NOSTATE = 0, -1, -2, -3, -4
X, Y, Z = 0, 1, 2
HOST, DEVICE = 0, 1
PLAN_AUTO, PLAN_NAIVE, PLAN_TILED = 0, 1, 2
OPT_KERNEL, OPT_CHUNK, OPT_CHUNK_MAX_LOG2, OPT_L2_PROMOTION, OPT_SMALL, OPT_DIAG_SOURCE, OPT_MAX_CTAS, OPT_L2_HINTS, OPT_PAIR, OPT_PROBE, OPT_CHUNK_MIN_LOG2, OPT_GRAPH, OPT_GRAPH_MAX_N, OPT_GRAPH_REPLAYS, OPT_LAST_LAUNCH_KHZ = 0, 1, 2, 3, 4, 5, 6, 7, 8, 9, 10, 11, 12, 13, 14
KC_NAMES = ("tile_fused", "tile_single", "naive_rot", "naive_diag", "reduce", "setup", "tile_chunk3", "small")
KC_COUNT = len(KC_NAMES)

# every symbol include/ts_b200.h declares (tests check that the library exports all of them)
SYMBOLS = ("ts_create", "ts_destroy", "ts_set_stream", "ts_bind_state", "ts_set_state", "ts_set_basis_state",
           "ts_set_state_range", "ts_get_state", "ts_evolve", "ts_evolve_observe", "ts_expect", "ts_expect_all", "ts_norm2", "ts_overlap", "ts_set_plan",
           "ts_describe_plan", "ts_set_profiling", "ts_get_profile", "ts_reset_profile", "ts_strerror", "ts_version",
           "ts_set_plan_groups", "ts_set_option", "ts_get_option", "ts_get_profile_passes", "ts_correlate", "ts_total_sz",
           "ts_energy", "ts_set_random_phase_state", "ts_loschmidt_echo", "ts_load_plan_file",
           "ts_shard_create", "ts_shard_destroy", "ts_shard_bind", "ts_shard_bind_peers", "ts_shard_set_stream", "ts_shard_evolve", "ts_shard_info",
           "ts_shard_spin_map", "ts_shard_ctx")

_lib = None
_vp, _dp, _i64p = ctypes.c_void_p, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_int64)
EXCHANGE_FN = ctypes.CFUNCTYPE(ctypes.c_int, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p)   # ts_exchange_fn


class TSError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        super().__init__(f"{where}: {strerror(status)} (status {status})")


def load() -> ctypes.CDLL:
    """Load libts_b200.so (built by `python -m paper_1305_0036_b200.build`); raises if it is missing."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise FileNotFoundError(f"{LIB_PATH} not found: build it with `python -m paper_1305_0036_b200.build` "
                                "(there is no CPU fallback)")
    lib = ctypes.CDLL(LIB_PATH)
    I, D, U64, I64 = ctypes.c_int, ctypes.c_double, ctypes.c_uint64, ctypes.c_int64
    sig = {
        "ts_create": (I, [ctypes.POINTER(_vp), I, _dp, _dp]),
        "ts_destroy": (I, [_vp]),
        "ts_set_stream": (I, [_vp, _vp]),
        "ts_bind_state": (I, [_vp, _vp]),
        "ts_set_state": (I, [_vp, _vp, I]),
        "ts_set_state_range": (I, [_vp, _vp, U64, U64, I]),
        "ts_set_basis_state": (I, [_vp, U64]),
        "ts_get_state": (I, [_vp, _vp, U64, U64, I]),
        "ts_evolve": (I, [_vp, D, I64, I]),
        "ts_evolve_observe": (I, [_vp, D, I64, I, I, I, _dp]),
        "ts_expect": (I, [_vp, I, I, _dp]),
        "ts_expect_all": (I, [_vp, I, _dp]),
        "ts_norm2": (I, [_vp, _dp]),
        "ts_overlap": (I, [_vp, _vp, _dp]),
        "ts_set_plan": (I, [_vp, I, I, I]),
        "ts_describe_plan": (I, [_vp, ctypes.c_char_p, I]),
        "ts_set_plan_groups": (I, [_vp, I, ctypes.POINTER(I)]),
        "ts_set_option": (I, [_vp, I, I]),
        "ts_load_plan_file": (I, [_vp, ctypes.c_char_p]),
        "ts_get_option": (I, [_vp, I, ctypes.POINTER(I)]),
        "ts_get_profile_passes": (I, [_vp, _dp]),
        "ts_correlate": (I, [_vp, I, I, I, _dp]),
        "ts_total_sz": (I, [_vp, _dp]),
        "ts_energy": (I, [_vp, _dp]),
        "ts_set_random_phase_state": (I, [_vp, I, U64]),
        "ts_loschmidt_echo": (I, [_vp, D, I64, I, _dp]),
        "ts_set_profiling": (I, [_vp, I]),
        "ts_get_profile": (I, [_vp, _i64p, _dp]),
        "ts_reset_profile": (I, [_vp]),
        "ts_shard_create": (I, [ctypes.POINTER(_vp), I, _dp, _dp, I, I]),
        "ts_shard_destroy": (I, [_vp]),
        "ts_shard_bind": (I, [_vp, _vp, _vp]),
        "ts_shard_bind_peers": (I, [_vp, ctypes.POINTER(_vp), ctypes.POINTER(_vp)]),
        "ts_shard_set_stream": (I, [_vp, _vp]),
        "ts_shard_evolve": (I, [_vp, D, I64, I, EXCHANGE_FN, _vp]),
        "ts_shard_info": (I, [_vp, ctypes.POINTER(I), ctypes.POINTER(I), ctypes.POINTER(I)]),
        "ts_shard_spin_map": (I, [_vp, I, ctypes.POINTER(I)]),
        "ts_shard_ctx": (_vp, [_vp, I]),
        "ts_strerror": (ctypes.c_char_p, [I]),
        "ts_version": (ctypes.c_char_p, []),
    }
    for name, (res, args) in sig.items():
        fn = getattr(lib, name)
        fn.restype, fn.argtypes = res, args
    _lib = lib
    return lib


def strerror(status: int) -> str:
    return load().ts_strerror(int(status)).decode()


def version() -> str:
    return load().ts_version().decode()


def _check(status: int, where: str):
    if status != TS_OK:
        raise TSError(status, where)


class TrotterSuzuki:
    """ts_create(N, h[3][N], J[3][N][N]) + a complex128 torch tensor on `device` bound as the state vector."""

    def __init__(self, N: int, h, J, device: str = "cuda:0", allocate: bool = True):
        import torch
        self._torch = torch
        if not torch.cuda.is_available():
            raise RuntimeError("no CUDA device: the Trotter-Suzuki path has no CPU fallback")
        self.N = int(N)
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        self._lib = load()
        h = np.ascontiguousarray(h, dtype=np.float64)
        J = np.ascontiguousarray(J, dtype=np.float64)
        if h.shape != (3, N) or J.shape != (3, N, N):
            raise ValueError(f"h must be [3][{N}] and J [3][{N}][{N}]")
        self._ctx = _vp()
        _check(self._lib.ts_create(ctypes.byref(self._ctx), N, h.ctypes.data_as(_dp), J.ctypes.data_as(_dp)),
               "ts_create")
        self.psi = None
        self.use_stream(torch.cuda.current_stream(self.device))
        if allocate:
            self.psi = torch.empty(1 << N, dtype=torch.complex128, device=self.device)
            _check(self._lib.ts_bind_state(self._ctx, _vp(self.psi.data_ptr())), "ts_bind_state")

    # ------------------------------------------------------------------ plumbing
    def use_stream(self, stream):
        self._stream = stream
        _check(self._lib.ts_set_stream(self._ctx, _vp(stream.cuda_stream)), "ts_set_stream")

    def close(self):
        if getattr(self, "_ctx", None):
            self._lib.ts_destroy(self._ctx)
            self._ctx = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_plan(self, mode: int = PLAN_AUTO, run_bits: int = 0, max_group_bits: int = 0):
        _check(self._lib.ts_set_plan(self._ctx, mode, run_bits, max_group_bits), "ts_set_plan")

    def set_plan_groups(self, high_bits):
        """Explicit bits of every high group, bottom to top (sum = N - 12)."""
        arr = (ctypes.c_int * len(high_bits))(*[int(b) for b in high_bits])
        _check(self._lib.ts_set_plan_groups(self._ctx, len(high_bits), arr), "ts_set_plan_groups")

    def load_plan_file(self, path: str):
        """Apply the tuned plan stored for this N in a plan file (paper_1305_0036_b200/tuner.py writes them)."""
        _check(self._lib.ts_load_plan_file(self._ctx, str(path).encode()), "ts_load_plan_file")

    def set_option(self, key: int, value: int):
        _check(self._lib.ts_set_option(self._ctx, int(key), int(value)), "ts_set_option")

    def get_option(self, key: int) -> int:
        out = ctypes.c_int()
        _check(self._lib.ts_get_option(self._ctx, int(key), ctypes.byref(out)), "ts_get_option")
        return out.value

    def describe_plan(self) -> str:
        buf = ctypes.create_string_buffer(512)
        _check(self._lib.ts_describe_plan(self._ctx, buf, 512), "ts_describe_plan")
        return buf.value.decode()

    # ------------------------------------------------------------------ state
    def set_state(self, amps):
        """amps: numpy complex128 array (host; copied) or a torch complex128 tensor (host pinned / device)."""
        torch = self._torch
        n = 1 << self.N
        if isinstance(amps, np.ndarray):
            a = np.ascontiguousarray(amps, dtype=np.complex128)
            if a.size != n:
                raise ValueError("state must have 2^N amplitudes")
            _check(self._lib.ts_set_state(self._ctx, _vp(a.ctypes.data), HOST), "ts_set_state")
            self._stream.synchronize()      # `a` may be a temporary
        else:
            if amps.dtype != torch.complex128 or amps.numel() != n or not amps.is_contiguous():
                raise ValueError("state must be a contiguous complex128 tensor with 2^N elements")
            where = DEVICE if amps.is_cuda else HOST
            _check(self._lib.ts_set_state(self._ctx, _vp(amps.data_ptr()), where), "ts_set_state")

    def set_state_range(self, amps, first: int):
        """Chunked upload: amps (numpy complex128, or a torch complex128 tensor on host/device) -> state[first:]."""
        if isinstance(amps, np.ndarray):
            a = np.ascontiguousarray(amps, dtype=np.complex128)
            _check(self._lib.ts_set_state_range(self._ctx, _vp(a.ctypes.data), int(first), a.size, HOST),
                   "ts_set_state_range")
            self._stream.synchronize()      # `a` may be a temporary
        else:
            if amps.dtype != self._torch.complex128 or not amps.is_contiguous():
                raise ValueError("chunk must be a contiguous complex128 tensor")
            _check(self._lib.ts_set_state_range(self._ctx, _vp(amps.data_ptr()), int(first), amps.numel(),
                                                DEVICE if amps.is_cuda else HOST), "ts_set_state_range")

    def set_state_chunks(self, chunks):
        """chunks: iterable of (first_index, numpy complex128 chunk), e.g. Workload.state_chunks()."""
        for first, chunk in chunks:
            self.set_state_range(chunk, first)

    def set_basis_state(self, k: int):
        _check(self._lib.ts_set_basis_state(self._ctx, int(k)), "ts_set_basis_state")

    def get_state(self, first: int = 0, count: Optional[int] = None) -> np.ndarray:
        n = 1 << self.N
        count = n - first if count is None else count
        out = np.empty(count, dtype=np.complex128)
        _check(self._lib.ts_get_state(self._ctx, _vp(out.ctypes.data), first, count, HOST), "ts_get_state")
        return out

    def get_state_into(self, host_tensor, first: int = 0):
        """Copy into a (pinned) host torch tensor; synchronises."""
        _check(self._lib.ts_get_state(self._ctx, _vp(host_tensor.data_ptr()), first, host_tensor.numel(), HOST),
               "ts_get_state")

    # ------------------------------------------------------------------ the hot path
    def evolve(self, tau: float, n_steps: int, order: int = 4):
        _check(self._lib.ts_evolve(self._ctx, float(tau), int(n_steps), int(order)), "ts_evolve")

    def evolve_observe(self, tau: float, n_steps: int, order: int = 4, alpha: int = Z, j: int = -1) -> np.ndarray:
        """n_steps steps, the observable after every step: [n_steps][N] for alpha = Z, j = -1, else [n_steps]."""
        shape = (n_steps, self.N) if (alpha == Z and j < 0) else (n_steps,)
        out = np.zeros(shape)
        _check(self._lib.ts_evolve_observe(self._ctx, float(tau), int(n_steps), int(order), int(alpha), int(j),
                                           out.ctypes.data_as(_dp)), "ts_evolve_observe")
        return out

    def expect(self, alpha: int, j: int) -> float:
        out = ctypes.c_double()
        _check(self._lib.ts_expect(self._ctx, alpha, j, ctypes.byref(out)), "ts_expect")
        return out.value

    def expect_all(self, alpha: int) -> np.ndarray:
        out = np.zeros(self.N)
        _check(self._lib.ts_expect_all(self._ctx, alpha, out.ctypes.data_as(_dp)), "ts_expect_all")
        return out

    def norm2(self) -> float:
        out = ctypes.c_double()
        _check(self._lib.ts_norm2(self._ctx, ctypes.byref(out)), "ts_norm2")
        return out.value

    def overlap(self, phi) -> complex:
        """<phi|psi> with phi a device complex128 tensor."""
        out = (ctypes.c_double * 2)()
        _check(self._lib.ts_overlap(self._ctx, _vp(phi.data_ptr()), out), "ts_overlap")
        return complex(out[0], out[1])

    def correlate(self, alpha: int, j: int, k: int) -> float:
        out = ctypes.c_double()
        _check(self._lib.ts_correlate(self._ctx, alpha, j, k, ctypes.byref(out)), "ts_correlate")
        return out.value

    def total_sz(self) -> float:
        out = ctypes.c_double()
        _check(self._lib.ts_total_sz(self._ctx, ctypes.byref(out)), "ts_total_sz")
        return out.value

    def energy(self) -> float:
        out = ctypes.c_double()
        _check(self._lib.ts_energy(self._ctx, ctypes.byref(out)), "ts_energy")
        return out.value

    def set_random_phase_state(self, up_spin: int, seed: int):
        _check(self._lib.ts_set_random_phase_state(self._ctx, int(up_spin), int(seed)), "ts_set_random_phase_state")

    def loschmidt_echo(self, tau: float, n_steps: int, order: int = 4):
        """(M_LE, <psi_0|psi>) after n steps forward and n steps back (eq. 11 with Sigma = 0)."""
        out = (ctypes.c_double * 3)()
        _check(self._lib.ts_loschmidt_echo(self._ctx, float(tau), int(n_steps), int(order), out), "ts_loschmidt_echo")
        return out[0], complex(out[1], out[2])

    # ------------------------------------------------------------------ profiling
    def set_profiling(self, enable: bool):
        _check(self._lib.ts_set_profiling(self._ctx, 1 if enable else 0), "ts_set_profiling")

    def reset_profile(self):
        _check(self._lib.ts_reset_profile(self._ctx), "ts_reset_profile")

    def get_profile(self) -> dict:
        l = (ctypes.c_int64 * KC_COUNT)()
        m = (ctypes.c_double * KC_COUNT)()
        _check(self._lib.ts_get_profile(self._ctx, l, m), "ts_get_profile")
        sp = (ctypes.c_double * KC_COUNT)()
        _check(self._lib.ts_get_profile_passes(self._ctx, sp), "ts_get_profile_passes")
        return {KC_NAMES[i]: {"launches": int(l[i]), "ms": float(m[i]), "state_passes": float(sp[i])}
                for i in range(KC_COUNT)}
