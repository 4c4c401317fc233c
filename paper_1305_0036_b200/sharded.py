"""One state vector sharded over G = 2^g GPUs (SURVEY 8 e, 8 f NEXT-5): binding of the ts_shard_* calls plus the collective.

The method's arithmetic (rotations, diagonals, their sequence, the effective Hamiltonian of a shard) is the library's
(csrc/ts_shard.cu).  This module supplies what joins the ranks:

  * `alltoall_exchange`: the once-per-sweep index-bit swap as `torch.distributed.all_to_all_single` (NCCL over NVLink /
    NVSwitch on GPUs; gloo in the CPU test): block rho' of a rank's shard goes to rank rho', block rho' of the result comes
    from rank rho';
  * `ShardedTrotterSuzuki`: one rank's shard (two device buffers, the ts_shard object, the exchange callback); with
    `bind_peers` (or `share_buffers_over_ipc` under torch.distributed) it runs in PEER-MEMORY MODE: the library's arrival
    pass gathers its tiles straight from the peers' shards over NVLink and the callback shrinks to a barrier;
  * `LocalCluster`: all G shards of a small system on ONE GPU, one Python thread per rank, the exchange done by plain
    device copies between the shards -- how the sharded path is checked against the oracle on a single-GPU box;
  * index bookkeeping to scatter / gather a full state and to assemble <S^z_j> over ranks.
"""
from __future__ import annotations

import ctypes
import threading
from typing import Callable, List, Optional

import numpy as np

from . import binding as B


def log2_exact(world: int) -> int:
    g = int(world).bit_length() - 1
    if world < 1 or (1 << g) != world:
        raise ValueError(f"the number of ranks must be a power of two, got {world}")
    return g


def shard_slice(N: int, world: int, rank: int) -> slice:
    """Layout 0: rank rho holds the amplitudes whose top g index bits equal rho, i.e. a contiguous slice."""
    n = N - log2_exact(world)
    return slice(rank << n, (rank + 1) << n)


def alltoall_exchange(src, dst, group=None) -> None:
    """Index-bit swap of the g rank bits with the top g local bits: equal-split all-to-all of the shard."""
    import torch
    import torch.distributed as dist
    if src.is_complex():
        src, dst = torch.view_as_real(src), torch.view_as_real(dst)
    dist.all_to_all_single(dst, src, group=group)


def assemble_sz(local_sz: np.ndarray, local_norm2: float, spin_of_bit: np.ndarray, n_local: int, rank: int) -> np.ndarray:
    """This rank's contribution to <S^z_j> of every spin j of the full system: local bits carry what ts_expect_all(z)
    summed over the shard; a spin on rank bit r has the fixed value bit_r(rank) - 1/2 on all of the shard's amplitudes."""
    N = spin_of_bit.size
    out = np.zeros(N)
    for b in range(n_local):
        out[spin_of_bit[b]] = local_sz[b]
    for r in range(N - n_local):
        out[spin_of_bit[n_local + r]] = (((rank >> r) & 1) - 0.5) * local_norm2
    return out


class ShardedTrotterSuzuki:
    """Rank `rank` of `world` = 2^g: 2^(N-g) amplitudes on `device`.  `exchange(src, dst)` defaults to the NCCL all-to-all."""

    def __init__(self, N: int, h, J, rank: int, world: int, device: str = "cuda:0",
                 exchange: Optional[Callable] = None, group=None):
        import torch
        self._torch = torch
        if not torch.cuda.is_available():
            raise RuntimeError("no CUDA device: the Trotter-Suzuki path has no CPU fallback")
        self.N, self.rank, self.world, self.g = int(N), int(rank), int(world), log2_exact(world)
        self.n = self.N - self.g
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        self._lib = B.load()
        h = np.ascontiguousarray(h, dtype=np.float64)
        J = np.ascontiguousarray(J, dtype=np.float64)
        if h.shape != (3, N) or J.shape != (3, N, N):
            raise ValueError(f"h must be [3][{N}] and J [3][{N}][{N}]")
        self._s = ctypes.c_void_p()
        B._check(self._lib.ts_shard_create(ctypes.byref(self._s), N, h.ctypes.data_as(B._dp), J.ctypes.data_as(B._dp),
                                           self.g, self.rank), "ts_shard_create")
        self.buf = [torch.zeros(1 << self.n, dtype=torch.complex128, device=self.device) for _ in range(2)]
        B._check(self._lib.ts_shard_bind(self._s, B._vp(self.buf[0].data_ptr()), B._vp(self.buf[1].data_ptr())), "ts_shard_bind")
        B._check(self._lib.ts_shard_set_stream(self._s, B._vp(torch.cuda.current_stream(self.device).cuda_stream)),
                 "ts_shard_set_stream")
        self._exchange = exchange if exchange is not None else (lambda s, d: alltoall_exchange(s, d, group))
        self._barrier = lambda: None
        self._error = None
        self._cb = B.EXCHANGE_FN(self._callback)       # keep the thunk alive as long as the shard

    def _callback(self, user, src, dst) -> int:
        try:
            if not src:                                # peer-memory mode: only a barrier is asked for
                self._barrier()
                return 0
            k = 0 if src == self.buf[0].data_ptr() else 1
            self._exchange(self.buf[k], self.buf[k ^ 1])
            return 0
        except BaseException as exc:                   # never let an exception cross the C frame
            self._error = exc
            return 1

    # ------------------------------------------------------------------ peer-memory mode
    def bind_peers(self, ptrs0, ptrs1, barrier: Callable[[], None]) -> None:
        """ptrs0[r], ptrs1[r]: device pointers (valid on this device) of rank r's two buffers; `barrier()` must order every
        rank's queued work before what this rank queues next."""
        a0 = (B._vp * self.world)(*[B._vp(int(p)) for p in ptrs0])
        a1 = (B._vp * self.world)(*[B._vp(int(p)) for p in ptrs1])
        B._check(self._lib.ts_shard_bind_peers(self._s, a0, a1), "ts_shard_bind_peers")
        self._barrier = barrier

    def share_buffers_over_ipc(self, group=None) -> None:
        """Peer-memory mode under torch.distributed, one process per GPU of one node: every rank exports its two buffers as
        CUDA IPC handles (torch's storage sharing), all-gathers them, maps the peers' buffers into its own address space and
        hands the pointers to the library; the barrier is a one-element all-reduce on the stream.  (Written against the
        torch 2.11 storage-sharing calls; no multi-GPU box was available to this build to run it on.)"""
        import torch
        import torch.distributed as dist
        mine = [b.untyped_storage()._share_cuda_() for b in self.buf]
        everyone = [None] * self.world
        dist.all_gather_object(everyone, mine, group=group)
        self._peer_keepalive = []
        ptrs = [[], []]
        for r, handles in enumerate(everyone):
            for k in range(2):
                if r == self.rank:
                    ptrs[k].append(self.buf[k].data_ptr())
                    continue
                h = list(handles[k])
                h[0] = self.device.index if self.device.index is not None else torch.cuda.current_device()
                st = torch.UntypedStorage._new_shared_cuda(*h)
                t = torch.empty(0, dtype=torch.complex128, device=self.device).set_(st)
                self._peer_keepalive.append(t)
                ptrs[k].append(t.data_ptr())
        token = torch.zeros(1, device=self.device)

        def barrier():
            dist.all_reduce(token, group=group)
        self.bind_peers(ptrs[0], ptrs[1], barrier)

    # ------------------------------------------------------------------ state
    def info(self):
        n, c, b = ctypes.c_int(), ctypes.c_int(), ctypes.c_int()
        B._check(self._lib.ts_shard_info(self._s, ctypes.byref(n), ctypes.byref(c), ctypes.byref(b)), "ts_shard_info")
        return n.value, c.value, b.value

    def spin_map(self, config: int) -> np.ndarray:
        out = (ctypes.c_int * self.N)()
        B._check(self._lib.ts_shard_spin_map(self._s, config, out), "ts_shard_spin_map")
        return np.array(list(out), dtype=np.int64)

    def set_local_state(self, amps) -> None:
        """`amps`: this rank's 2^(N-g) amplitudes in layout 0 (`full_state[shard_slice(N, world, rank)]`)."""
        torch = self._torch
        t = torch.as_tensor(np.ascontiguousarray(amps, dtype=np.complex128)) if not torch.is_tensor(amps) else amps
        B._check(self._lib.ts_shard_bind(self._s, B._vp(self.buf[0].data_ptr()), B._vp(self.buf[1].data_ptr())), "ts_shard_bind")
        self.buf[0].copy_(t.reshape(-1), non_blocking=False)

    def local_state(self) -> np.ndarray:
        _, cfg, b = self.info()
        if cfg != 0:
            raise RuntimeError("the shard is in layout 1 (mid-step); whole steps end in layout 0")
        self._torch.cuda.synchronize(self.device)
        return self.buf[b].cpu().numpy()

    # ------------------------------------------------------------------ the hot path
    def evolve(self, tau: float, n_steps: int, order: int = 4) -> None:
        self._torch.cuda.set_device(self.device)       # (the current device is per thread)
        self._error = None
        st = self._lib.ts_shard_evolve(self._s, float(tau), int(n_steps), int(order), self._cb, None)
        if self._error is not None:
            raise self._error
        B._check(st, "ts_shard_evolve")

    # ------------------------------------------------------------------ observables (this rank's part; sums are all-reduces)
    def local_sz_contribution(self) -> np.ndarray:
        n, cfg, _ = self.info()
        ctx = B._vp(self._lib.ts_shard_ctx(self._s, cfg))
        sz = np.zeros(n)
        B._check(self._lib.ts_expect_all(ctx, B.Z, sz.ctypes.data_as(B._dp)), "ts_expect_all")
        nrm = ctypes.c_double()
        B._check(self._lib.ts_norm2(ctx, ctypes.byref(nrm)), "ts_norm2")
        return assemble_sz(sz, nrm.value, self.spin_map(cfg), n, self.rank)

    def local_norm2(self) -> float:
        _, cfg, _ = self.info()
        nrm = ctypes.c_double()
        B._check(self._lib.ts_norm2(B._vp(self._lib.ts_shard_ctx(self._s, cfg)), ctypes.byref(nrm)), "ts_norm2")
        return nrm.value

    def expect_z_all(self, group=None) -> np.ndarray:
        """<S^z_j> of all N spins of the full system (an all-reduce over the ranks of `group`)."""
        import torch.distributed as dist
        t = self._torch.as_tensor(self.local_sz_contribution(), device=self.device)
        dist.all_reduce(t, group=group)
        return t.cpu().numpy()

    def close(self) -> None:
        if self._s:
            self._lib.ts_shard_destroy(self._s)
            self._s = ctypes.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class LocalCluster:
    """All 2^g shards of a small system on one GPU, one thread per rank; the exchange is done by device copies between
    the shards (all on the same stream, so stream order is the only synchronisation the data needs; the thread barrier
    makes sure every rank has issued its part of the sweep before anybody copies)."""

    def __init__(self, N: int, h, J, world: int, device: str = "cuda:0", peer_memory: bool = False):
        import torch
        self._torch = torch
        self.N, self.world = int(N), int(world)
        self.device = torch.device(device)
        self._barrier = threading.Barrier(world)
        self._src: List = [None] * world
        self.shards = [ShardedTrotterSuzuki(N, h, J, r, world, device, exchange=self._make_exchange(r)) for r in range(world)]
        if peer_memory:
            # every "peer" buffer lives on this GPU: plain pointers.  All ranks launch into the same stream, so the thread
            # barrier (everybody has QUEUED its local sweep) is all the ordering the gather needs.
            p0 = [s.buf[0].data_ptr() for s in self.shards]
            p1 = [s.buf[1].data_ptr() for s in self.shards]
            for s in self.shards:
                s.bind_peers(p0, p1, lambda: self._barrier.wait(timeout=120))

    def _make_exchange(self, r: int):
        def exchange(src, dst):
            self._src[r] = src
            self._barrier.wait(timeout=120)
            blk = src.numel() // self.world
            for rp in range(self.world):
                dst[rp * blk:(rp + 1) * blk].copy_(self._src[rp][r * blk:(r + 1) * blk])
            self._barrier.wait(timeout=120)
        return exchange

    def set_state(self, full: np.ndarray) -> None:
        for r, s in enumerate(self.shards):
            s.set_local_state(full[shard_slice(self.N, self.world, r)])

    def get_state(self) -> np.ndarray:
        return np.concatenate([s.local_state() for s in self.shards])

    def evolve(self, tau: float, n_steps: int, order: int = 4) -> None:
        errors: List = []

        def run(s):
            try:
                s.evolve(tau, n_steps, order)
            except BaseException as exc:
                errors.append(exc)
                self._barrier.abort()
        threads = [threading.Thread(target=run, args=(s,)) for s in self.shards]
        for t in threads:
            t.start()
        for t in threads:
            t.join()
        self._torch.cuda.synchronize(self.device)
        if errors:
            raise errors[0]

    def expect_z_all(self) -> np.ndarray:
        return np.sum([s.local_sz_contribution() for s in self.shards], axis=0)

    def norm2(self) -> float:
        return float(sum(s.local_norm2() for s in self.shards))

    def close(self) -> None:
        for s in self.shards:
            s.close()


def _main(argv=None) -> int:
    """`python -m paper_1305_0036_b200.sharded --N 28 --world 4 [--peer-memory]`: time the sharded path with all shards on ONE
    GPU (LocalCluster) next to the single-context path -- what the sharding costs in local work, exchange included as
    device copies; it says nothing about NVLink."""
    import argparse
    import json
    import time
    import torch
    from . import workloads as W
    ap = argparse.ArgumentParser(description=_main.__doc__)
    ap.add_argument("--N", type=int, default=28)
    ap.add_argument("--world", type=int, default=4)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--peer-memory", action="store_true")
    a = ap.parse_args(argv)
    w = W.grid_like(a.N, seed=8, tau=0.01, n_steps=1, state_seed=9, cols=6 if a.N >= 24 else None)
    ts = B.TrotterSuzuki(a.N, w.h, w.J)
    ts.set_random_phase_state(0, seed=9)
    ts.evolve(w.tau, 1, 4)
    torch.cuda.synchronize()
    t = time.perf_counter()
    ts.evolve(w.tau, a.steps, 4)
    torch.cuda.synchronize()
    one = (time.perf_counter() - t) / a.steps
    ts.close()
    del ts
    torch.cuda.empty_cache()
    cl = LocalCluster(a.N, w.h, w.J, a.world, peer_memory=a.peer_memory)
    for s in cl.shards:
        s.buf[0].fill_(2.0 ** (-a.N / 2.0))
    cl.evolve(w.tau, 1, 4)
    t = time.perf_counter()
    cl.evolve(w.tau, a.steps, 4)
    sh = (time.perf_counter() - t) / a.steps
    print(json.dumps({"N": a.N, "shards_on_one_gpu": a.world, "peer_memory": a.peer_memory, "single_context_ms_per_step": one * 1e3,
                      "sharded_ms_per_step": sh * 1e3, "ratio": sh / one, "norm2_after": cl.norm2()}))
    cl.close()
    return 0


if __name__ == "__main__":
    raise SystemExit(_main())
