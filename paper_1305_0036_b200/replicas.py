"""Host-side logic of the multi-GPU arm (replicas only).

The Trotter-Suzuki step on ONE state vector has an exchange step per sweep when sharded (SURVEY 8 e), which is not
built; what the paper itself runs in parallel is an ENSEMBLE of independent evolutions ("physical parallelization",
P:241): N ranks evolve N different random initial states under the same Hamiltonian, with no data-path collective.
This module holds only the rank bookkeeping around that (no arithmetic of the method): the per-rank state seed, the
max-over-ranks timing and the whole-job throughput.  It works with any torch.distributed backend (nccl on the GPU
box, gloo in the CPU tests).
"""
from __future__ import annotations

from typing import List, Optional


def replica_state_seed(base_seed: Optional[int], rank: int) -> int:
    """Seed of the initial state of ensemble member `rank` (rank 0 keeps the workload's own seed)."""
    return int(base_seed or 0) + 1000 * int(rank)


def max_over_ranks(value: float, device=None) -> float:
    """MAX all-reduce of a host scalar (timings are taken on each device; the job takes as long as its slowest rank)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def gather_scalars(value: float, device=None) -> List[float]:
    """All ranks' values of a host scalar, in rank order (used to report per-replica observables)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return [float(value)]
    t = torch.tensor([float(value)], dtype=torch.float64, device=device if device is not None else "cpu")
    out = [torch.zeros_like(t) for _ in range(dist.get_world_size())]
    dist.all_gather(out, t)
    return [float(x.item()) for x in out]


def whole_job_steps_per_s(steps_per_rank: int, world: int, ms_max: float) -> float:
    """Aggregate throughput of `world` replicas that each did `steps_per_rank` steps in at most ms_max milliseconds."""
    return world * steps_per_rank / (ms_max * 1e-3)
