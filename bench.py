#!/usr/bin/env python
"""bench.py -- Trotter-Suzuki steps/s at N = 30 on B200 (BASELINE.json metric), with roofline and CPU baseline.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--N 30] [--config 1|2|3|4|5]
                    [--repeats 5] [--no-e2e] [--no-cpu] [--cpu-full]

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


def tiled_plan(ts) -> bool:
    return "tiled" in ts.describe_plan() and "kernels=v2" in ts.describe_plan()


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
def cpu_info():
    model = "unknown"
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.startswith("model name"):
                    model = line.split(":", 1)[1].strip()
                    break
    except Exception:
        pass
    return {"cpu_model": model, "nproc": os.cpu_count(), "OMP_NUM_THREADS": os.environ.get("OMP_NUM_THREADS", "unset")}


def oracle_steps_per_s(Ns: int, n_steps: int):
    """The oracle as it stands (plain C + OpenMP on all host cores) on the open-lattice XYZ recipe at size Ns:
    n_steps single 4th-order steps, each timed; returns (median steps/s, [seconds])."""
    from oracle import ts_oracle as O
    ws = W.grid_like(Ns, seed=8, tau=0.01, n_steps=1, state_seed=9, cols=6 if Ns >= 24 else None)
    psi = ws.state()
    O.evolve(psi, Ns, ws.h, ws.J, ws.tau, 0, 4, True)          # loads the library
    secs = []
    for _ in range(n_steps):
        t = time.perf_counter()
        O.evolve(psi, Ns, ws.h, ws.J, ws.tau, 1, 4, True)
        secs.append(time.perf_counter() - t)
    return 1.0 / float(np.median(secs)), secs


def oracle_baseline(N_metric: int, full: bool):
    """BASELINE.md's CPU-baseline plan: measured at N = 22 (3 steps, median) and N = 27 (1 step by default so that the
    run stays within minutes; 3 steps, median, with --cpu-full), and the metric size extrapolated from the largest
    measured size by the oracle's own cost model (work per step ~ N 2^N), labelled as such."""
    from oracle import ts_oracle as O
    sizes = [(min(22, N_metric), 3)]
    if N_metric > 22:
        sizes.append((min(27, N_metric), 3 if full else 1))
    measured = {}
    for Ns, k in sizes:
        v, secs = oracle_steps_per_s(Ns, k)
        measured[f"N={Ns}"] = {"steps_per_s": v, "seconds_per_step": [round(x, 3) for x in secs], "steps_timed": k}
    Nl = sizes[-1][0]
    scale = (2.0 ** (Nl - N_metric)) * (Nl / N_metric)
    value = measured[f"N={Nl}"]["steps_per_s"] * scale
    info = cpu_info()
    out = {"value": value, "unit": UNIT, "cores": O.num_threads(), "kind": "oracle", "measured": measured,
           "extrapolated": Nl != N_metric,
           "sample": (f"oracle as it stands (plain C, OpenMP, {O.num_threads()} threads) on the same open-lattice XYZ recipe: "
                      + ", ".join(f"{k}: {v['steps_timed']} step(s), median" for k, v in measured.items())
                      + (f"; N={N_metric} value EXTRAPOLATED from N={Nl} by 2^({Nl}-{N_metric})*{Nl}/{N_metric}"
                         if Nl != N_metric else "")),
           **info}
    return out


def run_reference(args):
    """The reference arm of this tier IS the oracle (there is no reference program): K timed single steps of the oracle, as
    it stands, on a bounded sample of the workload -- the same lattice recipe at N = 24, ~5 s per step on 16 cores, so
    that `--steps 20 --warmup 5` ends within a few minutes -- scaled to the metric size by its cost model (~ N 2^N)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import ts_oracle as O
    w = workload_for(args.N)
    Ns = min(24, args.N)
    ws = w if Ns == args.N else W.grid_like(Ns, seed=8, tau=w.tau, n_steps=1, state_seed=9, cols=6)
    psi = ws.state()
    O.evolve(psi, Ns, ws.h, ws.J, ws.tau, 0, 4, True)          # loads the library
    times = []
    for i in range(args.warmup + args.steps):
        t = time.perf_counter()
        O.evolve(psi, Ns, ws.h, ws.J, ws.tau, 1, 4, True)
        dt = time.perf_counter() - t
        if i >= args.warmup:
            times.append(dt)
        if sum(times) > 150:                   # keep the whole run within a few minutes
            break
    if not times:
        times = [dt]
    n_done = len(times)
    scale = (2.0 ** (Ns - args.N)) * (Ns / args.N)
    value = scale * n_done / sum(times)
    sample = (f"{n_done} timed oracle step(s) at N={Ns} (open-lattice XYZ recipe, plain C + OpenMP, {O.num_threads()} threads)"
              + (f", EXTRAPOLATED to N={args.N} by 2^({Ns}-{args.N})*{Ns}/{args.N}" if Ns != args.N else ""))
    out = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
           "steps": n_done, "warmup": args.warmup, "ms_per_step": 1e3 / value, "higher_is_better": True,
           "scaling": "weak", "vs_baseline": None, "dtype": "f64 (complex128)", "data": "synthetic",
           "config": {"workload": w.name, "N": args.N, "order": 4, "tau": w.tau},
           "cpu_baseline": {"value": value, "unit": UNIT, "cores": O.num_threads(), "kind": "oracle", "sample": sample,
                            "extrapolated": Ns != args.N, **cpu_info()},
           "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(out))


# ----------------------------------------------------------------------------------------------- our arm
def fill_pinned_state(w: W.Workload, host):
    """Write the workload's initial state (same numbers as Workload.state()) into a pinned complex128 tensor."""
    hv = host.numpy()
    for first, chunk in w.state_chunks(chunk_log2=22):
        hv[first:first + chunk.size] = chunk


def kernel_sources_hash() -> str:
    """SHA-256 over the device code of the tile kernels (ts_tile_v2.cuh, ts_tile_kernel.cuh and their instantiation units):
    an ncu capture under profiles/ is only quoted for the kernels it was taken from."""
    import hashlib
    d = os.path.join(ROOT, "paper_1305_0036_b200", "csrc")
    hsh = hashlib.sha256()
    for name in sorted(os.listdir(d)):
        if name in ("ts_tile_v2.cuh", "ts_tile_kernel.cuh", "ts_tile_cfgG.cu") or (name.startswith("ts_v2") and name.endswith(".cu")):
            with open(os.path.join(d, name), "rb") as f:
                hsh.update(name.encode() + b"\0" + f.read())
    return hsh.hexdigest()[:16]


def recorded_traffic(kernel_class: str, N: int):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of `kernel_class` from the newest committed ncu capture
    (profiles/r02_traffic.csv: columns class,N,dram_read_bytes,dram_write_bytes,sources_hash,commit), or None when that
    capture belongs to other kernel sources than the ones being timed."""
    try:
        with open(os.path.join(ROOT, "profiles", "r02_traffic.csv")) as f:
            rows = [ln.strip().split(",") for ln in f if ln.strip() and not ln.startswith("#")]
    except Exception:
        return None
    cur = kernel_sources_hash()
    for r in rows[1:]:
        if len(r) >= 6 and r[0] == kernel_class and int(r[1]) == N:
            if r[4] != cur:
                return None
            return {"bytes": float(r[2]) + float(r[3]), "read": float(r[2]), "write": float(r[3]), "commit": r[5],
                    "sources_hash": r[4]}
    return None


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

    if args.config:
        w = W.config(int(args.config))     # BASELINE configs 1-5 (parity-test cases; timed here on request only)
        N = w.N
    else:
        N = args.N
        w = workload_for(N, args.workload)
    if world > 1:                      # independent ensemble members: same Hamiltonian, different random state
        w.state_seed = R.replica_state_seed(w.state_seed, rank)
    dim = 1 << N
    ts = B.TrotterSuzuki(N, w.h, w.J, device=str(dev))
    if args.plan:
        ts.set_plan(*[int(x) for x in args.plan.split(",")])
    if args.groups:
        ts.set_plan_groups([int(x) for x in args.groups.split(",")])
    for kv in args.opt:
        k, v = kv.split("=")
        ts.set_option(getattr(B, "OPT_" + k.upper()), int(v))
    host = None
    if args.device_state:              # profiling / tuning runs: the eq. A.1 state generated on the device (timing does
        ts.set_random_phase_state(0, seed=9)   # not depend on the values); no host buffer, hence no e2e leg
        args.no_e2e = True
    else:
        host = torch.empty(dim, dtype=torch.complex128, pin_memory=True)
        fill_pinned_state(w, host)
        ts.set_state(host)
    torch.cuda.synchronize()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident timing: `repeats` regions of exactly K steps each, every region bracketed by a barrier and a
    # device synchronisation on both sides and timed with CUDA events on the stream the kernels run on; the value is
    # taken from the MEDIAN region (max over ranks of each region).  The state (16 * 2^N bytes) is larger than L2 for
    # N >= 24; for smaller N the L2 is flushed before every region.
    # The timed regions run WITHOUT the library's per-launch events (two event records per launch cost ~35 % at N = 16,
    # where a launch lasts a few microseconds); the per-kernel-class breakdown comes from one extra, profiled region of
    # the same K steps right after them.
    ts.set_profiling(False)
    for _ in range(max(args.warmup, 3)):
        ts.evolve(w.tau, 1, 4)
    barrier()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev) if 16 * dim < (256 << 20) else None
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
        time.sleep(0.3)
    region_ms, prof = [], None
    t0 = time.time()
    for rep in range(max(args.repeats, 1)):
        if flush is not None:
            flush.fill_(rep)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        e0.record()
        ts.evolve(w.tau, args.steps, 4)
        e1.record()
        barrier()
        region_ms.append(R.max_over_ranks(e0.elapsed_time(e1), dev))
    t1 = time.time()
    clocks = sampler.stop(t0, t1) if rank == 0 else None
    ts.set_profiling(True)
    ts.reset_profile()
    barrier()
    ts.evolve(w.tau, args.steps, 4)        # profiled region: per-kernel-class CUDA-event times and launch counts
    barrier()
    prof = ts.get_profile()
    ts.set_profiling(False)
    eff_khz = ts.get_option(B.OPT_LAST_LAUNCH_KHZ) if tiled_plan(ts) else None     # the last launch of the profiled region
    norm2 = ts.norm2()
    ms = float(np.median(region_ms))
    steps_per_s = R.whole_job_steps_per_s(args.steps, world, ms)

    # ---- transport ceiling, measured in the same run: the same launches with TS_OPT_PROBE = 1 (every tile travels through
    # the kernels' pipeline -- TMA in, TMA out, ticket scheduling, chunk dependencies -- but the arithmetic is skipped, so
    # the state is left as it is).  What the step would cost if the SM-side work were free.
    ceiling = None
    if tiled_plan(ts) and not args.no_ceiling:
        ts.set_option(B.OPT_PROBE, 1)
        ts.set_profiling(True)
        ts.evolve(w.tau, 1, 4)
        ts.reset_profile()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        e0.record()
        ts.evolve(w.tau, args.steps, 4)
        e1.record()
        barrier()
        cms = R.max_over_ranks(e0.elapsed_time(e1), dev) / args.steps
        cprof = ts.get_profile()
        ceil_khz = ts.get_option(B.OPT_LAST_LAUNCH_KHZ)
        ts.set_option(B.OPT_PROBE, 0)
        ts.set_profiling(False)
        ceiling = {"what": "same launches, copy only (TS_OPT_PROBE=1): tile transport without the arithmetic",
                   "ms_per_step": cms, "effective_sm_mhz_last_launch": ceil_khz / 1e3,
                   "kernel_avg_ms": {k: v["ms"] / v["launches"] for k, v in cprof.items() if v["launches"] and k.startswith("tile")}}
        ts.reset_profile()

    # ---- observable reductions, timed one by one with CUDA events: read-only passes over the state
    observables = None
    if args.observables:
        ts.set_profiling(False)
        observables = {}

        def timed(name, fn, passes):
            fn()                                     # warm-up (allocates scratch)
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize()
            a.record()
            fn()
            b.record()
            torch.cuda.synchronize()
            t = a.elapsed_time(b)
            observables[name] = {"ms": t, "state_reads": passes, "gbs": passes * 16.0 * dim / (t * 1e-3) / 1e9}
        ngroups = ts.describe_plan().count("H[") + 1 if "tiled" in ts.describe_plan() else N
        timed("norm2", ts.norm2, 1)
        timed("expect_all_z", lambda: ts.expect_all(B.Z), 1)
        timed("expect_all_x", lambda: ts.expect_all(B.X), ngroups)
        timed("expect_x_site0", lambda: ts.expect(B.X, 0), 1)
        timed("correlate_zz", lambda: ts.correlate(B.Z, 0, N - 1), 1)
        timed("correlate_xx", lambda: ts.correlate(B.X, 0, N - 1), 1)
        timed("total_sz", ts.total_sz, 1)

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

    # ---- roofline.  Unit = one amplitude; algorithmic bytes = 32 B per amplitude per HBM ROUND TRIP of
    # the state (16 B read + 16 B written), and every tile launch -- a fused pass, a single pass, or an L2-blocked triple
    # launch, which performs three tile passes on L2-resident chunks -- makes exactly one round trip of all 2^N
    # amplitudes.  So achieved = 32 * 2^N / launch time is what the HBM had to deliver, NOT a credit for passes: the
    # three passes' worth (SURVEY 8 d's contract figure) is reported separately as `credited_*`.
    peak, peak_src = measured_peak()
    rt_bytes = 32.0 * dim
    tile_classes = ("tile_fused", "tile_single", "tile_chunk3")
    timed = {k: prof[k] for k in tile_classes + ("naive_rot", "naive_diag", "small") if prof[k]["launches"]}
    dom = max(timed, key=lambda k: timed[k]["ms"]) if timed else "tile_fused"
    dms = prof[dom]["ms"] / max(prof[dom]["launches"], 1)
    achieved = rt_bytes / (dms * 1e-3) / 1e9 if dms > 0 else 0.0
    kern = {}
    for k, v in prof.items():
        if not v["launches"]:
            continue
        kern[k] = dict(v)
        if k in tile_classes and v["ms"] > 0:
            kern[k]["avg_ms"] = v["ms"] / v["launches"]
            kern[k]["hbm_gbs"] = v["launches"] * rt_bytes / (v["ms"] * 1e-3) / 1e9
            kern[k]["credited_gbs"] = v["state_passes"] * rt_bytes / (v["ms"] * 1e-3) / 1e9
    launches = sum(v["launches"] for v in prof.values())
    step_ms = ms / args.steps
    round_trips = sum(prof[k]["launches"] for k in tile_classes) / args.steps
    tile_passes = sum(prof[k]["state_passes"] for k in tile_classes) / args.steps
    tr = recorded_traffic(dom, N)
    hbm_resident = 16 * dim > (126 << 20)
    roofline = {"bound": "hbm", "kernel": dom, "achieved": achieved, "peak": peak, "unit": "GB/s",
                "frac": achieved / peak, "peak_source": peak_src,
                "traffic": tr["bytes"] if tr else None, "traffic_capture": tr,
                "frac_dram_actual": (tr["bytes"] / (dms * 1e-3) / 1e9 / peak) if (tr and dms > 0) else None,
                "alg_bytes_per_launch": rt_bytes, "avg_launch_ms": dms,
                "credited_tile_passes_per_launch": prof[dom]["state_passes"] / max(prof[dom]["launches"], 1),
                "credited_gbs": kern.get(dom, {}).get("credited_gbs"),
                "step": {"hbm_round_trips": round_trips, "tile_passes": tile_passes,
                         "bytes_moved": round_trips * rt_bytes, "gbs": round_trips * rt_bytes / (step_ms * 1e-3) / 1e9,
                         "frac_of_peak": round_trips * rt_bytes / (step_ms * 1e-3) / 1e9 / peak,
                         "floor_round_trips": N_SWEEPS_PER_STEP,
                         "contract_model_frac_of_8TBs": (N_SWEEPS_PER_STEP * (1 + -(-(N - 13) // 10) if N > 13 else 1)
                                                         * rt_bytes / 8e12) / (step_ms * 1e-3)},
                "transport_ceiling": ceiling,
                "frac_of_transport_ceiling": (ceiling["ms_per_step"] / step_ms) if ceiling else None,
                "note": ("frac = HBM bytes of the dominant launch / its time / peak.  The L2-blocked launch makes three tile "
                         "passes per HBM round trip and L2-resident passes move at most ~7.7 TB/s on this part, so its HBM "
                         "fraction cannot reach 1; transport_ceiling is the measured bound of the same launches without "
                         "arithmetic; clocks.reasons says whether the run hit the power cap") if hbm_resident
                        else "state fits in L2: absolute steps/s is the figure, not an HBM fraction"}
    cpu = None
    if not args.no_cpu:
        cpu = oracle_baseline(N, args.cpu_full)     # (the lattice recipe: the oracle's cost does not depend on the Hamiltonian)

    out = {"metric": METRIC, "value": steps_per_s, "unit": UNIT, "n_gpus": world, "steps": args.steps,
           "warmup": max(args.warmup, 3), "ms_per_step": step_ms, "higher_is_better": True, "scaling": "weak",
           "vs_baseline": None, "dtype": "f64 (complex128)", "data": "synthetic",
           "config": {"workload": w.name + ("+device_state" if args.device_state else ""), "N": N, "order": 4, "tau": w.tau,
                      "state_bytes": 16 * dim,
                      "plan": ts.describe_plan(),
                      "l2": ("state (16*2^N B) is larger than L2; no flush needed" if flush is None
                             else "L2 flushed (256 MiB write) before every timed region"),
                      "parallelism": f"replicas x{world}" if world > 1 else "1 GPU"},
           "timing": {"regions": len(region_ms), "region_ms": [round(x, 3) for x in region_ms], "value_from": "median region",
                      "steps_per_region": args.steps},
           "spin_amplitude_updates_per_sec": steps_per_s * N_SWEEPS_PER_STEP * N * dim,
           "amplitude_steps_per_sec": steps_per_s * dim,
           "norm2_after": norm2, "library": B.version(), "kernel_sources_hash": kernel_sources_hash(),
           "gpu_launches": launches, "kernels": kern, "clocks": clocks,
           "effective_sm_mhz_last_launch": (eff_khz / 1e3) if eff_khz else None, "roofline": roofline,
           "cpu_baseline": cpu, "e2e": e2e}
    if observables is not None:
        out["observables"] = observables
    print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


def run_sharded(args):
    """One state vector of N + log2(world) spins sharded over the ranks: per-GPU memory fixed at 2^N
    amplitudes ("weak" in memory; the work per step grows with the system).  Launch under torchrun; one rank degenerates to
    the unfused single-GPU sequence.  No >1-GPU box was available to this build: unmeasured beyond world = 1."""
    import torch
    import torch.distributed as dist
    from paper_1305_0036_b200 import sharded as S
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    g = S.log2_exact(world)
    Nt = args.N + g
    w = W.grid_like(Nt, seed=8, tau=0.01, n_steps=1, state_seed=9, cols=6 if Nt >= 24 else None)
    sh = S.ShardedTrotterSuzuki(Nt, w.h, w.J, rank, world, device=str(dev))
    sh.buf[0].fill_(2.0 ** (-Nt / 2.0))              # uniform superposition: timing does not depend on the values
    for _ in range(max(args.warmup, 1)):
        sh.evolve(w.tau, 1, 4)
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    sh.evolve(w.tau, args.steps, 4)
    e1.record()
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    ms = R.max_over_ranks(e0.elapsed_time(e1), dev) / args.steps
    nrm = sh.local_norm2()
    if world > 1:
        t = torch.tensor([nrm], device=dev, dtype=torch.float64)
        dist.all_reduce(t)
        nrm = float(t.item())
    if rank == 0:
        print(json.dumps({"metric": METRIC, "mode": "sharded", "value": 1e3 / ms, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                          "warmup": max(args.warmup, 1), "ms_per_step": ms, "higher_is_better": True, "scaling": "weak",
                          "dtype": "f64 (complex128)", "data": "synthetic", "norm2_after": nrm,
                          "config": {"workload": w.name, "N": Nt, "local_spins": args.N, "order": 4, "tau": w.tau,
                                     "parallelism": f"state sharded x{world}: all-to-all index-bit swap per sweep (NCCL)"}}))
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
    ap.add_argument("--groups", default="", help="bits of the high groups, bottom to top (ts_set_plan_groups), e.g. 9,9")
    ap.add_argument("--opt", action="append", default=[], help="KEY=VALUE for ts_set_option, e.g. kernel=0, chunk=0")
    ap.add_argument("--config", default="", help="time BASELINE config 1..5 instead of the metric workload")
    ap.add_argument("--repeats", type=int, default=5, help="timed regions of K steps each; the value is their median")
    ap.add_argument("--cpu-full", action="store_true", help="oracle: 3 steps (median) at N = 27 instead of 1")
    ap.add_argument("--observables", action="store_true", help="also time the observable reductions (row a6)")
    ap.add_argument("--device-state", action="store_true",
                    help="initial state generated on the device (eq. A.1) instead of the seeded host state: for ncu / tuning runs")
    ap.add_argument("--sharded", action="store_true",
                    help="one state vector of N + log2(world) spins sharded over the ranks instead of independent replicas")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-ceiling", action="store_true", help="skip the copy-only (transport ceiling) measurement")
    ap.add_argument("--no-cpu", action="store_true")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    elif args.sharded:
        run_sharded(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
