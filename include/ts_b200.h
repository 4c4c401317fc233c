/*
 * ts_b200.h -- C ABI of libts_b200.so: the Trotter-Suzuki time step of arXiv:1305.0036 on one B200 (sm_100a).
 *
 * "P:<n>" = line n of the paper text; "A<n>" = a reading listed in DESIGN.md.
 *
 * What the library computes: for the spin-1/2 Hamiltonian of eq. 1
 *     H = sum_j sum_a h^a_j S^a_j + sum_{j != k} sum_a J^a_{jk} S^a_j S^a_k ,   a = x, y, z,  S = Pauli / 2,
 * the state |psi> = sum_k c_k |k> (eq. 2; 2^N complex doubles) is advanced by the 2nd- or 4th-order
 * Trotter-Suzuki product formulas of P:54-58 in the paper's XYZ decomposition (eq. 6-10): diagonal
 * phase sweeps exp(-i t E_a(k)) and per-spin pair rotations X, Y of eq. 5.
 *
 * Conventions (identical in the oracle):
 *   - spin j (0-based) <-> bit j of the amplitude index k; bit = 1 is "up" (S^z = +1/2), 0 is "down".
 *   - amplitudes are interleaved (re, im) IEEE doubles; amplitude k is at byte offset 16 k.
 *   - alpha: TS_X = 0, TS_Y = 1, TS_Z = 2.  h is [3][N] row-major, J is [3][N][N] row-major.
 *   - J need not be symmetric: the coupling of the unordered pair {j,k} is J[a][j][k] + J[a][k][j]; J[a][j][j] is
 *     ignored (A1).
 *   - U_1(t) = exp(-itH_x) exp(-itH_y) exp(-itH_z) (A6),  U_2(t) = U_1^dag(-t/2) U_1(t/2),
 *     U_4(t) = U_2(at) U_2(at) U_2((1-4a)t) U_2(at) U_2(at),  a = 1/(4 - 4^(1/3)).
 *   - no normalisation is ever applied; expectation values are <psi|S^a_j|psi>, not divided by <psi|psi>.
 *
 * Every call returns a status (TS_OK = 0 or a negative TS_ERR_*) and never throws or aborts.  Pointer arguments are
 * HOST pointers unless the comment says "device".  A context is not thread-safe: use one per host thread.
 * All work runs on the context's CUDA stream (default: the legacy default stream; see ts_set_stream).  Calls that
 * return scalars to the host synchronise that stream; ts_evolve and the state setters do not (except host copies).
 * There is no CPU fallback: every call that touches the state fails with TS_ERR_CUDA when no CUDA device is usable.
 */
#ifndef TS_B200_H
#define TS_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct ts_ctx ts_ctx; /* opaque; owns the device tables and (unless a buffer is bound) the state */

enum { TS_OK = 0, TS_ERR_ARG = -1, TS_ERR_NOMEM = -2, TS_ERR_CUDA = -3, TS_ERR_NOSTATE = -4 };
enum { TS_X = 0, TS_Y = 1, TS_Z = 2 };
enum { TS_HOST = 0, TS_DEVICE = 1 };
/* ts_set_plan modes */
enum { TS_PLAN_AUTO = 0, TS_PLAN_NAIVE = 1, TS_PLAN_TILED = 2 };
/* ts_get_profile kernel classes */
enum { TS_KC_TILE_FUSED = 0,   /* tile pass: sweep . diagonal . sweep in one HBM round trip  */
       TS_KC_TILE_SINGLE = 1,  /* tile pass: one sweep's butterflies on one bit group (+ optional diagonal) */
       TS_KC_NAIVE_ROT = 2,    /* one-bit pair rotation, one launch per spin (the paper's basic kernel) */
       TS_KC_NAIVE_DIAG = 3,   /* per-amplitude O(N^2) phase correction */
       TS_KC_REDUCE = 4,       /* observable / norm reductions */
       TS_KC_SETUP = 5,        /* phase-table construction, state initialisation */
       TS_KC_TILE_CHUNK = 6,   /* three tile passes (high . fused low . high) in one L2-blocked launch: 1 HBM round trip */
       TS_KC_SMALL = 7,        /* N <= 12: a whole ts_evolve call in one single-CTA launch */
       TS_KC_COUNT = 8 };

/* Problem statement (eq. 1).  N in [1, 33].  h: [3][N], J: [3][N][N]; both are COPIED.
 * Errors: TS_ERR_ARG (null pointer, N out of range, non-finite h or J), TS_ERR_CUDA (no device), TS_ERR_NOMEM. */
int ts_create(ts_ctx** out, int N, const double* h, const double* J);

/* Frees the tables and the state if the library owns it.  NULL is accepted. */
int ts_destroy(ts_ctx* ctx);

/* Use this CUDA stream (a cudaStream_t passed as void*; NULL = legacy default stream) for all later work. */
int ts_set_stream(ts_ctx* ctx, void* cuda_stream);

/* Bind a caller-owned DEVICE buffer of 2^N complex128 (16 * 2^N bytes, 16-byte aligned) as the state vector
 * (P:109).  The library evolves it IN PLACE and never frees it.  Any library-owned state is released. */
int ts_bind_state(ts_ctx* ctx, void* dev_amps);

/* Copy 2^N amplitudes into the state (eq. 2).  where = TS_HOST: amps is a host pointer (pinned or pageable;
 * synchronous for pageable memory); TS_DEVICE: a device pointer (device-to-device copy).  If no buffer is bound the
 * library allocates its own.  Errors: TS_ERR_ARG, TS_ERR_NOMEM. */
int ts_set_state(ts_ctx* ctx, const void* amps, int where);

/* Copy `count` amplitudes to positions first .. first+count-1 of the state (chunked upload: an N = 32 state is 64 GiB,
 * larger than most host buffers).  Allocates like ts_set_state; amplitudes outside the range are left as they are.
 * Errors: TS_ERR_ARG (range outside [0, 2^N)), TS_ERR_NOMEM. */
int ts_set_state_range(ts_ctx* ctx, const void* amps, uint64_t first, uint64_t count, int where);

/* State := basis state |k>  (c_k = 1, all others 0); allocates like ts_set_state.  k < 2^N. */
int ts_set_basis_state(ts_ctx* ctx, uint64_t k);

/* Copy amplitudes first .. first+count-1 to dst (host or device as `where`); synchronises for TS_HOST. */
int ts_get_state(ts_ctx* ctx, void* dst, uint64_t first, uint64_t count, int where);

/* psi <- [U_order(tau)]^n_steps psi  with order = 2 or 4; tau may be negative (echo, eq. 11);
 * n_steps = 0 is a no-op.  Asynchronous on the stream.  One 4th-order step is 20 global rotations ("sweeps") and
 * 20 merged diagonals; see DESIGN.md "Sequencer".  Errors: TS_ERR_ARG (order, n_steps < 0, non-finite tau),
 * TS_ERR_NOSTATE, TS_ERR_CUDA. */
int ts_evolve(ts_ctx* ctx, double tau, int64_t n_steps, int order);

/* n_steps single steps U_order(tau), recording an observable after EVERY step (magnitudes followed in time;
 * BASELINE config 2 records <S^z_1>(t)) without a host round trip per step: the reductions write rows of a device
 * trace, copied once at the end.  alpha = TS_Z, j = -1: out[n_steps][N] = <S^z_s> of all sites; alpha = TS_Z, j >= 0:
 * out[n_steps]; alpha = TS_X / TS_Y: one site j, out[n_steps].  Steps are applied one by one (the state after each
 * step is needed), so the diagonals at step boundaries are not merged: round-off differs from ts_evolve(tau, n_steps)
 * at the 1e-15 level.  Synchronises at the end.  Errors: as ts_evolve, TS_ERR_NOMEM. */
int ts_evolve_observe(ts_ctx* ctx, double tau, int64_t n_steps, int order, int alpha, int j, double* out);

/* out[0] = <psi|S^alpha_j|psi>, j 0-based (reading A15).  Synchronises. */
int ts_expect(ts_ctx* ctx, int alpha, int j, double* out);

/* out[j] = <psi|S^alpha_j|psi> for all j < N (host array of N doubles).  Synchronises. */
int ts_expect_all(ts_ctx* ctx, int alpha, double* out);

/* out[0] = <psi|psi>.  Synchronises. */
int ts_norm2(ts_ctx* ctx, double* out);

/* out[0], out[1] = Re, Im of <phi|psi> where phi is a DEVICE buffer of 2^N complex128 (eq. 11). */
int ts_overlap(ts_ctx* ctx, const void* dev_phi, double* out);

/* out[0] = <psi| S^alpha_j S^alpha_k |psi>, j != k (two-site correlator: the "non-local physical magnitudes" of P:203;
 * formulas in csrc/ts_reduce.cu, reading A15).  One read-only pass.  Synchronises.  Errors: TS_ERR_ARG (j = k, range). */
int ts_correlate(ts_ctx* ctx, int alpha, int j, int k, double* out);

/* out[0] = sum_j <psi|S^z_j|psi>, the total magnetisation (conserved by polarisation-conserving Hamiltonians;
 * its spurious drift is the paper's second accuracy test).  One pass.  Synchronises. */
int ts_total_sz(ts_ctx* ctx, double* out);

/* out[0] = <psi|H|psi> for the Hamiltonian of eq. 1.  <H_z> is a weighted sum of |c_k|^2; <H_x> and <H_y> are
 * the same sums in the frames rotated by Y^dag and X^dag (eq. 7, 10), so the call applies four global rotations to the
 * state and undoes them exactly up to round-off: the state returns changed by <= ~1e-15 relative.  The energies are
 * evaluated from the O(N^2) definition -- an observable, not part of the time step.  Synchronises. */
int ts_energy(ts_ctx* ctx, double* out);

/* State := the "one spin up, the rest at infinite temperature" pure state of eq. A.1:
 *   |up>_u (x) sum_j 2^{-(N-1)/2} exp(i phi_j) |beta_j>,  phi_j = 2 pi u_j,
 * u_j = (j+1)-th output of SplitMix64 seeded with `seed`, top 53 bits (a counter-based stream, so ensemble members
 * are reproducible from (seed) alone; the oracle restates the same generator).  Allocates like ts_set_state. */
int ts_set_random_phase_state(ts_ctx* ctx, int up_spin, uint64_t seed);

/* Loschmidt echo with Sigma = 0 (eq. 11): keeps a device copy psi_0 of the current state, applies
 * [U_order(tau)]^n then [U_order(-tau)]^n, and returns out[0] = M_LE = |<psi_0|psi>|^2, out[1], out[2] = Re, Im of the
 * overlap.  For a perfectly accurate computation M_LE = 1: the deviation measures floating-point round-off only
 * (P:215).  Needs 16 * 2^N bytes of scratch.  Synchronises.  Errors: as ts_evolve, TS_ERR_NOMEM. */
int ts_loschmidt_echo(ts_ctx* ctx, double tau, int64_t n_steps, int order, double* out /*[3]*/);

/* Execution plan.  mode: TS_PLAN_AUTO (N <= 12: one single-CTA launch per ts_evolve; N >= 13: tiled), TS_PLAN_NAIVE (one launch per spin rotation
 * and per diagonal: the paper's basic scheme, kept as bring-up path and A/B baseline), TS_PLAN_TILED.
 * run_bits: number s of lowest index bits kept inside every high-bit tile (runs of 2^s * 16 bytes),
 * 0 = default (3).  max_group_bits: upper bound on butterflied bits per high-bit pass, 0 = as many as fit
 * (12 - s); smaller values force more passes (used by tests to exercise multi-group plans at small N).
 * Errors: TS_ERR_ARG when the combination cannot be planned for this N. */
int ts_set_plan(ts_ctx* ctx, int mode, int run_bits, int max_group_bits);

/* Explicit plan: the number of index bits of every high group, bottom to top (group k butterflies the high_bits[k]
 * spins above group k-1; group A = spins 0..11 is implied).  sum(high_bits) must be N - 12, each entry in [1, 11];
 * entries <= 10 (runs of >= 64 bytes; 9 = the 128-byte runs of P:165-167) run on the pipelined TMA kernels.  This is what the tuner
 * (paper_1305_0036_b200/tuner.py; "a brute force search for the fastest series of rotations ... stored in a
 * file") searches over and what a stored plan file sets.  N >= 12 only.  Errors: TS_ERR_ARG. */
int ts_set_plan_groups(ts_ctx* ctx, int n_high, const int* high_bits);

/* Execution options (all have defaults; the tuner and the A/B benchmarks set them).
 *   TS_OPT_KERNEL          2 (default): automatic -- the warp-specialised persistent TMA kernels when every SM
 *                          walks more than two tiles (N >= 21 on a B200), else one CTA per tile with register loads (the
 *                          pipeline's set-up does not pay for one or two tiles); 1: TMA kernels always; 0: never
 *   TS_OPT_CHUNK           1 (default): [high . fused low . high] as one L2-blocked launch where the plan allows; 0: off
 *   TS_OPT_CHUNK_MAX_LOG2  largest chunk of the L2-blocked launch, log2 amplitudes (default 21 = 32 MiB), 13..26
 *   TS_OPT_CHUNK_MIN_LOG2  smallest chunk the L2-blocked launch is used for (default 21: only a full 9-bit group above A; with
 *                          smaller chunks the per-chunk hand-overs between CTAs cost more than the HBM round trips they
 *                          save, profiles/r02_tuner.md); the tests lower it to 13 to exercise those hand-overs
 *   TS_OPT_GRAPH           1 (default): for N <= TS_OPT_GRAPH_MAX_N (default 21: L2-resident, launch-bound states) a
 *                          ts_evolve call of >= 4 steps captures the launches of one step into a CUDA graph and replays it;
 *                          0: every launch goes to the stream one by one.  Off while profiling is on.
 *   TS_OPT_GRAPH_MAX_N     see above (12..33).   TS_OPT_GRAPH_REPLAYS (read-only): graph replays so far
 *   TS_OPT_LAST_LAUNCH_KHZ (read-only, synchronises): the SM clock the last persistent tile launch really ran at, in kHz: SM
 *                          cycles / wall nanoseconds between the start and the last ticket of CTA 0's loader
 *   TS_OPT_L2_PROMOTION    tensor-map L2 promotion of the high groups: 0 none (default), 1: 128 B, 2: 256 B
 *   TS_OPT_SMALL           1 (default): under TS_PLAN_AUTO, N <= 12 runs a whole ts_evolve call as one single-CTA launch
 *                          (state in shared memory; small systems are latency-bound); 0: tiled / naive plans
 *   TS_OPT_DIAG_SOURCE     TS_PLAN_NAIVE only: 0 (default) each diagonal evaluates the O(N^2) energy per amplitude;
 *                          1: the paper's pre-computed variant: three 2^N-element energy vectors (+24 bytes per
 *                          amplitude), built on first use -- the A/B experiment of DESIGN.md 7.5
 *   TS_OPT_MAX_CTAS        upper bound on the grid of the persistent tile kernels (0, default: one CTA per SM); small values
 *                          make every CTA walk many tiles -- used by the tests to exercise buffer reuse at small N
 *   TS_OPT_L2_HINTS        1 (default): the L2-blocked launch marks its TMA transfers with L2 eviction priorities (a chunk's
 *                          intermediate writes "evict last", its final writes and first reads "evict first"); 0: none
 *   TS_OPT_PAIR            1 (default): a scheduling ticket of a high-group pass is a pair of adjacent tiles (their 128-byte
 *                          rows are the halves of 256-byte segments: DRAM page locality); 0: single tiles
 *   TS_OPT_PROBE           0 (default); 1: MEASUREMENT ONLY -- the tile kernels move every tile through their pipeline (TMA
 *                          in, TMA out) but skip the arithmetic, so the state is left unchanged by ts_evolve: the copy
 *                          ceiling of each pass's access pattern (bench.py --opt probe=1); 2 / 3: the fused
 *                          passes and the (Y^dag, Y) triple launch of the N = 30 plan run with only their arithmetic / only
 *                          their shared-memory layout exchanges (wrong results by construction; time attribution only)
 * Errors: TS_ERR_ARG (unknown key, value out of range). */
enum { TS_OPT_KERNEL = 0, TS_OPT_CHUNK = 1, TS_OPT_CHUNK_MAX_LOG2 = 2, TS_OPT_L2_PROMOTION = 3, TS_OPT_SMALL = 4,
       TS_OPT_DIAG_SOURCE = 5, TS_OPT_MAX_CTAS = 6, TS_OPT_L2_HINTS = 7, TS_OPT_PAIR = 8, TS_OPT_PROBE = 9,
       TS_OPT_CHUNK_MIN_LOG2 = 10, TS_OPT_GRAPH = 11, TS_OPT_GRAPH_MAX_N = 12, TS_OPT_GRAPH_REPLAYS = 13,
       TS_OPT_LAST_LAUNCH_KHZ = 14 };
int ts_set_option(ts_ctx* ctx, int key, int value);
int ts_get_option(ts_ctx* ctx, int key, int* value);

/* Apply the line for this context's N of a plan file written by the tuner ("stored in a file"):
 *     N=30 groups=9,9 kernel=1 chunk=1 chunk_max_log2=21 chunk_min_log2=21 l2_promotion=0
 * (text; '#' starts a comment line; keys other than N may be omitted).  No line for this N: TS_OK, nothing changes.
 * ts_create applies the file named by the environment variable TS_PLAN_FILE, if set, the same way.
 * Errors: TS_ERR_ARG (file cannot be opened, or the line does not describe a valid plan for N). */
int ts_load_plan_file(ts_ctx* ctx, const char* path);

/* Human-readable description of the current plan (groups, passes per sweep) into buf (NUL-terminated). */
int ts_describe_plan(ts_ctx* ctx, char* buf, int buflen);

/* Per-kernel-class device timing.  enable != 0: every later launch is bracketed by CUDA events on the stream.
 * ts_get_profile synchronises, then writes, for class c in [0, TS_KC_COUNT): launches[c], ms[c] (sum of event
 * durations) since the last ts_reset_profile.  Launch counts are kept even when timing is disabled (ms = 0). */
int ts_set_profiling(ts_ctx* ctx, int enable);
int ts_get_profile(ts_ctx* ctx, int64_t* launches /*[TS_KC_COUNT]*/, double* ms /*[TS_KC_COUNT]*/);
int ts_reset_profile(ts_ctx* ctx);
/* state_passes[c]: tile passes over the WHOLE state performed by the launches of class c since the last reset (1 per tile
 * pass launch, 3 per L2-blocked triple launch, 0 for the other classes): what bench.py turns into bytes. */
int ts_get_profile_passes(ts_ctx* ctx, double* state_passes /*[TS_KC_COUNT]*/);

/* Static string for a status code. */
const char* ts_strerror(int status);

/* Library build info: "ts_b200 <version> sm_100a ..." */
const char* ts_version(void);

/* ---- one state vector sharded over 2^g GPUs (SURVEY 8 e, 8 f NEXT-5; beyond the paper, whose limit was device memory).
 * Rank `rank` holds the 2^(N-g) amplitudes whose top g index bits equal `rank`; once per sweep the ranks swap the g rank
 * bits with the top g local bits (an all-to-all; see csrc/ts_shard.cu for the two spin layouts and the effective local
 * Hamiltonian of a shard).  The shard object owns two ordinary contexts, one per spin layout.
 *   ts_shard_create   h [3][N], J [3][N][N] of the FULL system (copied); log2_ranks = g in 0..8, 2g <= N, N - g <= 33.
 *   ts_shard_bind     two DEVICE buffers of 2^(N-g) complex128 each (caller-owned): the shard's amplitudes are in buf0, in
 *                     layout 0 (local index = low N-g bits of the global index); buf1 is the exchange target.
 *   ts_shard_evolve   psi <- U_order(tau)^n psi, collectively: EVERY rank must make the same call.  `exchange(user, src,
 *                     dst)` must perform the index-bit swap of this rank's 2^(N-g) amplitudes from device buffer src to
 *                     device buffer dst (block rho' of src, 2^(N-2g) amplitudes, goes to rank rho'; block rho' of dst
 *                     receives from rank rho') on the shard's stream or ordered with it, and return 0; it is called 20
 *                     times per 4th-order step (4 per 2nd-order step), an even number, so after the call the amplitudes
 *                     are again in layout 0 and in the buffer they started in.  g = 0: exchange may be NULL.
 *   ts_shard_bind_peers  PEER-MEMORY MODE: bufs0[r], bufs1[r] = the two buffers of rank r (r < 2^g) as DEVICE pointers valid on
 *                     this rank's device (peer-mapped over NVLink: CUDA IPC handles, or plain pointers when the ranks share
 *                     a process or a device); entry [rank] must be this shard's own buffers.  The exchange and the pass over
 *                     the arriving spins then run as ONE kernel that gathers its tiles from the peers' shards, and
 *                     `exchange` is only called as a barrier, with src = dst = NULL: it must return once every rank's work
 *                     queued so far is ordered before what this rank queues next (e.g. a 1-element all-reduce on the
 *                     stream).  Needs shards of >= 13 spins whose top bit group has >= g bits, g <= 5.  NULL, NULL: back to
 *                     the exchange mode.
 *   ts_shard_info     local spin count, current layout (0 / 1) and current buffer (0 / 1).
 *   ts_shard_spin_map spin_of_bit[N]: the spin on each local bit (first N-g entries), then on each rank bit, in `config`.
 *   ts_shard_ctx      the context of a layout: for the read-only calls (ts_expect_all, ts_norm2, ts_get_state) on this
 *                     rank's amplitudes; sums over ranks are the caller's (an all-reduce).  Do not evolve it directly.
 * Errors: TS_ERR_ARG, TS_ERR_NOMEM, TS_ERR_CUDA (also when the callback fails), TS_ERR_NOSTATE (nothing bound). */
typedef struct ts_shard ts_shard;
typedef int (*ts_exchange_fn)(void* user, void* src_dev, void* dst_dev);
int ts_shard_create(ts_shard** out, int N, const double* h, const double* J, int log2_ranks, int rank);
int ts_shard_destroy(ts_shard* s);
int ts_shard_bind(ts_shard* s, void* buf0_dev, void* buf1_dev);
int ts_shard_bind_peers(ts_shard* s, const void* const* bufs0_dev, const void* const* bufs1_dev);
int ts_shard_set_stream(ts_shard* s, void* cuda_stream);
int ts_shard_evolve(ts_shard* s, double tau, int64_t n_steps, int order, ts_exchange_fn exchange, void* user);
int ts_shard_info(ts_shard* s, int* n_local, int* config, int* buffer);
int ts_shard_spin_map(ts_shard* s, int config, int* spin_of_bit /*[N]*/);
ts_ctx* ts_shard_ctx(ts_shard* s, int config);

#ifdef __cplusplus
}
#endif
#endif /* TS_B200_H */
