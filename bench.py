#!/usr/bin/env python
"""bench.py -- Trotter-Suzuki steps/s at N = 30 on B200 (BASELINE.json metric), with roofline and CPU baseline.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--N 30] [--no-e2e] [--no-cpu]

A "step" is one 4th-order Trotter-Suzuki step U_4(tau) (20 global rotations + 20 merged diagonals) of
the whole 2^N complex128 state of the metric workload (workloads.config("M"): 5x6 open XYZ lattice, N = 30, 16 GiB).
Prints ONE JSON line (rank 0).  Multi-GPU (torchrun): the path does not shard without an exchange step (DESIGN.md
"Multi-GPU"), so N ranks run N independent replicas (ensemble members) -- "scaling": "weak", no collective on
the data path; value = total steps/s over all ranks, time = max over ranks.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_1305_0036_b200 import replicas as R  # noqa: E402
from paper_1305_0036_b200 import workloads as W  # noqa: E402

METRIC = "trotter_steps_per_sec"
UNIT = "steps/s"
N_SWEEPS_PER_STEP = 20


def workload_for(N: int, kind: str = "grid") -> W.Workload:
    if kind == "chain":          # Heisenberg chain, random z fields (config-1 recipe at size N)
        return W.chain_like(N, seed=8, tau=0.01, n_steps=5)
    if kind == "dipolar":        # all-to-all dipolar network, random product state (config-3 recipe at size N)
        return W.dipolar_like(N, seed=8, tau=0.005, n_steps=5)
    if N == 30:
        return W.config("M")
    return W.grid_like(N, seed=8, tau=0.01, n_steps=5, state_seed=9, cols=6 if N >= 24 else None)


def measured_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md, MEASURED_PEAKS.json absent)"


# ----------------------------------------------------------------------------------------------- clocks sampling
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.proc = None
        self.lines = []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append((time.time(), line.strip()))

    def stop(self, t0: float, t1: float) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        for ts, line in self.lines:
            if ts < t0 or ts > t1 + 0.2:
                continue
            f = [x.strip() for x in line.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples inside the timed region"]}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(mx)), "power_w_max": float(max(pw)),
                "samples": len(sm), "reasons": sorted(reasons)}


# ----------------------------------------------------------------------------------------------- CPU oracle legs
def oracle_sample(N_metric: int, w_metric: W.Workload):
    """One 4th-order step of the SAME lattice recipe at a size the oracle finishes in ~10-30 s, scaled to the metric
    size by the oracle's own cost model (work per step ~ N 2^N)."""
    from oracle import ts_oracle as O
    Ns = min(N_metric, 24)
    ws = w_metric if Ns == N_metric else W.grid_like(Ns, seed=8, tau=w_metric.tau, n_steps=1, state_seed=9, cols=6)
    psi = ws.state()
    O.evolve(psi, Ns, ws.h, ws.J, ws.tau, 0, 4, True)          # loads the library
    t = time.perf_counter()
    O.evolve(psi, Ns, ws.h, ws.J, ws.tau, 1, 4, True)
    dt = time.perf_counter() - t
    scale = (2.0 ** (Ns - N_metric)) * (Ns / N_metric)
    return {"steps_per_s_sample": 1.0 / dt, "value": scale / dt, "N_sample": Ns, "seconds": dt,
            "cores": O.num_threads(),
            "sample": f"1 U4 step of the same open-lattice XYZ recipe at N={Ns} (oracle as it stands, OpenMP), "
                      f"scaled by 2^({Ns}-{N_metric})*{Ns}/{N_metric} to N={N_metric}"}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    w = workload_for(args.N)
    times = []
    info = None
    for i in range(args.warmup + args.steps):
        info = oracle_sample(args.N, w)
        if i >= args.warmup:
            times.append(info["seconds"])
        if sum(times) > 150:           # keep the whole run within a few minutes
            break
    n_done = len(times)
    scale = (2.0 ** (info["N_sample"] - args.N)) * (info["N_sample"] / args.N)
    value = scale * n_done / sum(times)
    out = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
           "steps": n_done, "warmup": args.warmup, "ms_per_step": 1e3 / value, "higher_is_better": True,
           "scaling": "weak", "vs_baseline": None, "dtype": "f64 (complex128)", "data": "synthetic",
           "config": {"workload": w.name, "N": args.N, "order": 4, "tau": w.tau},
           "cpu_baseline": {"value": value, "unit": UNIT, "cores": info["cores"], "kind": "oracle",
                            "sample": info["sample"]},
           "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(out))


# ----------------------------------------------------------------------------------------------- our arm
def fill_pinned_state(w: W.Workload, host):
    """Write the workload's initial state (same numbers as Workload.state()) into a pinned complex128 tensor."""
    hv = host.numpy()
    for first, chunk in w.state_chunks(chunk_log2=22):
        hv[first:first + chunk.size] = chunk


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_1305_0036_b200 import binding as B

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    N = args.N
    w = workload_for(N, args.workload)
    if world > 1:                      # independent ensemble members: same Hamiltonian, different random state
        w.state_seed = R.replica_state_seed(w.state_seed, rank)
    dim = 1 << N
    ts = B.TrotterSuzuki(N, w.h, w.J, device=str(dev))
    if args.plan:
        ts.set_plan(*[int(x) for x in args.plan.split(",")])
    host = torch.empty(dim, dtype=torch.complex128, pin_memory=True)
    fill_pinned_state(w, host)
    ts.set_state(host)
    torch.cuda.synchronize()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident timing
    ts.set_profiling(os.environ.get('TS_BENCH_NOPROF', '0') != '1')
    for _ in range(max(args.warmup, 3)):
        ts.evolve(w.tau, 1, 4)
    barrier()
    ts.reset_profile()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
        time.sleep(0.3)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    t0 = time.time()
    e0.record()
    ts.evolve(w.tau, args.steps, 4)
    e1.record()
    barrier()
    t1 = time.time()
    ms = e0.elapsed_time(e1)
    prof = ts.get_profile()
    clocks = sampler.stop(t0, t1) if rank == 0 else None
    norm2 = ts.norm2()
    ms = R.max_over_ranks(ms, dev)
    steps_per_s = R.whole_job_steps_per_s(args.steps, world, ms)

    # ---- end to end through the C ABI with host buffers: H2D of the state + 1 step + D2H of <S^z_j>
    e2e = None
    if not args.no_e2e:
        ts.set_profiling(False)
        n_e2e = max(1, min(args.steps, 3))
        barrier()
        te = time.perf_counter()
        for _ in range(n_e2e):
            ts.set_state(host)                       # pinned host -> device, 16 * 2^N bytes
            ts.evolve(w.tau, 1, 4)
            sz = ts.expect_all(B.Z)                  # device -> host, N doubles (synchronises)
        barrier()
        te = time.perf_counter() - te
        te = R.max_over_ranks(te, dev)
        e2e = {"value": R.whole_job_steps_per_s(n_e2e, world, te * 1e3), "unit": UNIT, "h2d_bytes_per_step": 16 * dim,
               "d2h_bytes_per_step": 8 * N, "steps": n_e2e,
               "what": "ts_set_state(pinned host) + ts_evolve(1 step) + ts_expect_all(z) per step"}

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel (fused tile pass): algorithmic bytes = read + write of the state once
    peak, peak_src = measured_peak()
    # Algorithmic bytes: 32 B per amplitude per tile pass (read + write of the state once).  A
    # "tile_chunk3" launch does the work of THREE tile passes (high . fused low . high) and is credited with three
    # passes' bytes, SURVEY 8(d)'s per-pass figure; because it keeps each 32 MiB chunk in L2 between them it needs only
    # ONE HBM round trip ("hbm_round_trip_bytes_per_launch"): fewer bytes moved than credited is the point of it.
    pass_bytes = 32.0 * dim
    passes_per_launch = {"tile_fused": 1, "tile_single": 1, "tile_chunk3": 3, "naive_rot": 1, "naive_diag": 1}
    dom = max(passes_per_launch, key=lambda k: prof[k]["ms"])
    alg_bytes = pass_bytes * passes_per_launch[dom]
    dms = prof[dom]["ms"] / max(prof[dom]["launches"], 1)
    achieved = alg_bytes / (dms * 1e-3) / 1e9 if dms > 0 else 0.0
    kern_ms = {k: v for k, v in prof.items() if v["launches"]}
    launches = sum(v["launches"] for v in prof.values())
    round_trips = prof["tile_fused"]["launches"] + prof["tile_single"]["launches"] + prof["tile_chunk3"]["launches"]
    tile_passes = prof["tile_fused"]["launches"] + prof["tile_single"]["launches"] + 3 * prof["tile_chunk3"]["launches"]
    step_ms = ms / args.steps
    traffic = None                    # dram__bytes_read + write of the dominant kernel from the committed ncu capture (N = 30)
    try:                              # (values and the command that produced them: profiles/r01b_pipeline_and_l2_blocking.md)
        with open(os.path.join(ROOT, "profiles", "r01b_traffic.csv")) as f:
            for line in f.read().splitlines()[1:]:
                k, rd, wr = line.split(",")
                if N == 30 and k == dom:
                    traffic = float(rd) + float(wr)
    except Exception:
        traffic = None
    roofline = {"bound": "hbm", "kernel": dom, "achieved": achieved, "peak": peak, "unit": "GB/s",
                "frac": achieved / peak, "peak_source": peak_src, "traffic": traffic,
                "alg_bytes_per_launch": alg_bytes, "tile_passes_per_launch": passes_per_launch[dom],
                "hbm_round_trip_bytes_per_launch": pass_bytes, "avg_launch_ms": dms,
                "step_gbs_over_tile_passes": tile_passes * pass_bytes / (ms * 1e-3) / 1e9,
                "step_gbs_over_hbm_round_trips": round_trips * pass_bytes / (ms * 1e-3) / 1e9,
                "contract_model_frac_of_8TBs": (N_SWEEPS_PER_STEP * (1 + -(-(N - 13) // 10) if N > 13 else 1)
                                                * pass_bytes / 8e12) / (step_ms * 1e-3)}
    cpu = None
    if not args.no_cpu:
        s = oracle_sample(N, workload_for(N))      # (always the lattice recipe: the oracle's cost does not depend on it)
        cpu = {"value": s["value"], "unit": UNIT, "cores": s["cores"], "kind": "oracle", "sample": s["sample"],
               "sample_steps_per_s": s["steps_per_s_sample"]}

    out = {"metric": METRIC, "value": steps_per_s, "unit": UNIT, "n_gpus": world, "steps": args.steps,
           "warmup": max(args.warmup, 3), "ms_per_step": step_ms, "higher_is_better": True, "scaling": "weak",
           "vs_baseline": None, "dtype": "f64 (complex128)", "data": "synthetic",
           "config": {"workload": w.name, "N": N, "order": 4, "tau": w.tau, "state_bytes": 16 * dim,
                      "plan": ts.describe_plan(), "l2": "state (16*2^N B) is larger than L2; no flush needed",
                      "parallelism": f"replicas x{world}" if world > 1 else "1 GPU"},
           "spin_amplitude_updates_per_sec": steps_per_s * N_SWEEPS_PER_STEP * N * dim,
           "amplitude_steps_per_sec": steps_per_s * dim,
           "norm2_after": norm2,
           "gpu_launches": launches, "kernels": kern_ms, "clocks": clocks, "roofline": roofline,
           "cpu_baseline": cpu, "e2e": e2e}
    print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--N", type=int, default=30)
    ap.add_argument("--workload", default="grid", choices=["grid", "chain", "dipolar"],
                    help="Hamiltonian family (north_star: chains, lattices, all-to-all); the metric line is the default grid")
    ap.add_argument("--plan", default="", help="mode,run_bits,max_group_bits (ts_set_plan)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
