"""Brute-force plan tuner (SURVEY 8 f NEXT-4).

The paper: "we developed a small tool that does a brute force search for the fastest series of rotations [...] The best
configuration for each number of spins is stored in a file and read at the start of the simulation".  Here the
search space is what the C ABI exposes: the split of the N - 12 high index bits into groups (`ts_set_plan_groups`: how
many bits each tile pass butterflies, hence run lengths and passes per sweep), whether the group above A is run as an
L2-blocked triple launch (`TS_OPT_CHUNK`), and the kernel family (`TS_OPT_KERNEL`).  Every candidate is
timed on the device with CUDA events (median of `repeats` runs of `steps` 4th-order steps on a random state; throughput
does not depend on the values), and the winner per N is written as one line of a plan file that `ts_load_plan_file` /
the `TS_PLAN_FILE` environment variable read back.

    python -m paper_1305_0036_b200.tuner --N 24 27 30 --out plans/b200.plan [--steps 2] [--repeats 3] [--max-groups 4]

Argument marshalling and timing only: every candidate runs the library's own kernels.
"""
from __future__ import annotations

import argparse
import json
import sys
from typing import Iterable, List, Sequence, Tuple

import numpy as np

MAX_GROUP_BITS = 10         # runs of >= 64 bytes: 9 bits = 128-byte runs, 10 bits = 64-byte runs (ts_v2_H10.cu)


def compositions(total: int, max_part: int = MAX_GROUP_BITS, max_parts: int = 4) -> Iterable[Tuple[int, ...]]:
    """All ordered splits of `total` high bits into 1..max_parts groups of 1..max_part bits (bottom to top)."""
    if total == 0:
        yield ()
        return

    def rec(left: int, parts: Tuple[int, ...]):
        if left == 0:
            yield parts
            return
        if len(parts) == max_parts:
            return
        for p in range(min(max_part, left), 0, -1):
            yield from rec(left - p, parts + (p,))
    yield from rec(total, ())


def candidates(N: int, max_groups: int = 4, max_splits: int = 12) -> List[dict]:
    """Candidate plans for N >= 13: every split of the high bits with the fewest or fewest + 1 groups (each extra group is
    an extra HBM round trip per sweep), most promising first -- fewer groups, a larger group above A (bigger L2 chunk),
    longer shortest runs -- cut at `max_splits` splits so that the search stays within minutes at N = 30."""
    rem = N - 12
    comps = list(compositions(rem, MAX_GROUP_BITS, max_groups))
    if comps:
        gmin = min(len(c) for c in comps)
        comps = [c for c in comps if len(c) <= gmin + 1]
        # most promising first: fewest groups, a full 9-bit group above A (the 32-MiB chunk of the L2-blocked launch), then
        # the largest first group, then the longest shortest run
        comps.sort(key=lambda c: (len(c), 0 if (c and c[0] == 9) else 1, -c[0] if c else 0, max(c) if c else 0))
        comps = comps[:max_splits]
    out = []
    for groups in comps:
        chunk_possible = len(groups) >= 2 and groups[0] <= 9 and 12 + groups[0] <= 21
        for chunk in ((1, 0) if chunk_possible else (0,)):
            for kernel in (1,):          # the warp-specialised TMA kernels (ts_tile_v2.cuh)
                out.append({"groups": list(groups), "chunk": chunk, "l2_promotion": 0, "kernel": kernel})
    return out


def plan_line(N: int, plan: dict) -> str:
    cmin = 12 + plan["groups"][0] if (plan["chunk"] and plan["groups"]) else 21      # the chunk this plan was timed with
    return (f"N={N} groups={','.join(str(b) for b in plan['groups'])} kernel={plan['kernel']} chunk={plan['chunk']} "
            f"chunk_max_log2=21 chunk_min_log2={min(cmin, 21)} l2_promotion={plan['l2_promotion']}")


def time_plan(ts, B, plan: dict, tau: float, steps: int, repeats: int) -> float:
    """Median milliseconds per 4th-order step of `plan` on the state currently held by `ts`."""
    import torch
    ts.set_option(B.OPT_KERNEL, plan["kernel"])
    ts.set_option(B.OPT_CHUNK, plan["chunk"])
    ts.set_option(B.OPT_CHUNK_MIN_LOG2, 13)       # a candidate with chunk = 1 is timed WITH the triple launch, whatever its chunk size
    ts.set_option(B.OPT_L2_PROMOTION, plan["l2_promotion"])
    ts.set_plan_groups(plan["groups"])
    ts.evolve(tau, 1, 4)                      # builds the phase tables, warms up
    torch.cuda.synchronize()
    ms = []
    for _ in range(repeats):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        ts.evolve(tau, steps, 4)
        e1.record()
        torch.cuda.synchronize()
        ms.append(e0.elapsed_time(e1) / steps)
    return float(np.median(ms))


def tune(N: int, steps: int = 2, repeats: int = 3, max_groups: int = 4, max_splits: int = 12,
         verbose: bool = True) -> Tuple[dict, List[dict]]:
    import torch
    from . import binding as B
    rng = np.random.Generator(np.random.PCG64(N))      # every h and J entry non-zero; values only fill tables
    h = rng.normal(0.0, 0.5, (3, N))
    J = np.zeros((3, N, N))
    for a in range(3):
        J[a][np.triu_indices(N, 1)] = rng.normal(0.0, 1.0 / np.sqrt(N), N * (N - 1) // 2)
    ts = B.TrotterSuzuki(N, h, J)
    ts.set_random_phase_state(0, seed=N)       # any normalised state: timing is data-independent
    results = []
    for plan in candidates(N, max_groups, max_splits):
        try:
            ms = time_plan(ts, B, plan, 0.01, steps, repeats)
        except B.TSError as e:                 # a split this build cannot run
            if verbose:
                print(f"  N={N} {plan}: skipped ({e})", file=sys.stderr)
            continue
        results.append(dict(plan, ms_per_step=ms))
        if verbose:
            print(f"  N={N} groups={plan['groups']} chunk={plan['chunk']} kernel={plan['kernel']}: "
                  f"{ms:.3f} ms/step", file=sys.stderr)
    ts.close()
    del ts
    torch.cuda.empty_cache()
    best = min(results, key=lambda r: r["ms_per_step"])
    return best, results


def main(argv: Sequence[str] = None) -> int:
    ap = argparse.ArgumentParser(description=__doc__, formatter_class=argparse.RawDescriptionHelpFormatter)
    ap.add_argument("--N", type=int, nargs="+", required=True)
    ap.add_argument("--out", required=True, help="plan file to write (one line per N)")
    ap.add_argument("--steps", type=int, default=2)
    ap.add_argument("--repeats", type=int, default=3)
    ap.add_argument("--max-groups", type=int, default=4)
    ap.add_argument("--max-splits", type=int, default=12, help="splits of the high bits tried per N")
    ap.add_argument("--json", default="", help="also write every timing to this JSON file")
    args = ap.parse_args(argv)
    lines = ["# ts_b200 plan file: written by paper_1305_0036_b200.tuner (brute-force search, P:171)"]
    everything = {}
    for N in args.N:
        if N < 13:
            continue
        best, results = tune(N, args.steps, args.repeats, args.max_groups, args.max_splits)
        everything[N] = results
        lines.append(f"# N={N}: best of {len(results)} candidates, {best['ms_per_step']:.3f} ms/step")
        lines.append(plan_line(N, best))
    with open(args.out, "w") as f:
        f.write("\n".join(lines) + "\n")
    if args.json:
        with open(args.json, "w") as f:
            json.dump(everything, f, indent=1)
    print("\n".join(lines))
    return 0


if __name__ == "__main__":
    raise SystemExit(main())
