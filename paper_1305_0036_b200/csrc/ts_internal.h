// ts_internal.h -- shared declarations of the CUDA path (host side).  Not part of the public ABI.
//
// Layers: ts_api.cu (C ABI, context, sequencer, plan) -> launchers in ts_tile.cu (tile passes + phase
// tables), ts_naive.cu (one-bit rotations, brute-force diagonal, stored-phase diagonal), ts_small.cu (single-CTA
// path for N <= 12), ts_reduce.cu (observables).  Nothing here is shared with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <vector>

#include "../../include/ts_b200.h"

#define TS_MAX_N 33
#define TS_TILE_LOG2 12                 // amplitudes per tile = 4096 (64 KiB)
#define TS_TILE_THREADS 128             // 32 amplitudes per thread
#define TS_MAX_FIXED (TS_MAX_N - TS_TILE_LOG2)

// Sweep kinds: eq. 5 re-indexed to bit order (A7), unnormalised (A13).  c0: bit = 0, c1: bit = 1.
//   YDAG: (c0, c1) <- (c0 - c1, c0 + c1)        Y: (c0, c1) <- (c0 + c1, c1 - c0)
//   XDAG: (c0, c1) <- (c0 - i c1, c1 - i c0)    X: (c0, c1) <- (c0 + i c1, c1 + i c0)
enum { SW_YDAG = 0, SW_Y = 1, SW_XDAG = 2, SW_X = 3, SW_NONE = 4 };

// One merged diagonal D_alpha(t) with an exact power-of-two scale 2^scale_pow.
struct DiagOp {
    int present;     // 0: identity
    int alpha;       // TS_X / TS_Y / TS_Z
    double t;        // c_k <- c_k * 2^scale_pow * exp(-i t E_alpha(k))
    int scale_pow;   // 0 or -N
};

// One group of index bits handled by one tile pass.
// Tile = 2^12 amplitudes: in-tile bit f < s  <-> spin f ("run" bits), f >= s <-> spin g0 + (f - s).
// The low group A has s = 12, g0 = 12 (the tile is contiguous) and butterflies all 12 bits.
struct TileGroup {
    int s;        // run bits (A: 12)
    int g0;       // first spin of the group (A: 12, i.e. the tile is contiguous)
    int is_low;   // group A: butterflies all 12 tile bits; otherwise the 12 - s group bits
};

// Phase tables of one (diagonal kind, tile group, kernel family), see ts_tile_kernel.cuh.  Built on first use, cached
// in the context; handles stay valid until ts_tile_free_tables.
struct DiagTables {
    int alpha, scale_pow, group, layout;   // layout: 0 = k_tile_pass register layout, 1 = v2 (ts_tile_v2.cuh)
    double t;
    double2* d_thread;       // device: TT[128] followed by WT[5][128]
    double2* d_tile_phase;   // device: [ntiles][32]
    double2 RR[32];          // host (passed to the kernel in its parameters)
};

// Cached CUtensorMap (128 bytes, kept opaque here so that this header does not need <cuda.h>).
struct TensorMapSlot {
    int valid;
    alignas(64) unsigned char bytes[128];
    TensorMapSlot() : valid(0) {}
};

struct ProfileRec { int kc; cudaEvent_t e0, e1; };

struct ts_ctx {
    int N;
    int device;
    int num_sms;
    cudaStream_t stream;
    double h[3][TS_MAX_N];
    double Jeff[3][TS_MAX_N][TS_MAX_N];   // symmetric, zero diagonal: Jeff[j][k] = J[j][k] + J[k][j]  (A1)
    double e0[3];     // energy offset added to E_alpha(k) by every diagonal: 0 for ts_create; for a shard context
                      // (ts_shard_create) the fields and couplings of the spins that sit on the rank bits
    double* d_h;      // [3][TS_MAX_N]
    double* d_Jeff;   // [3][TS_MAX_N][TS_MAX_N]
    double2* psi;     // 2^N amplitudes (device)
    int owns_psi;
    // plan
    int plan_mode, run_bits, max_group_bits;
    std::vector<int> explicit_groups;    // ts_set_plan_groups: bits of each high group, bottom to top (empty: automatic)
    std::vector<TileGroup> groups;
    int use_small;                       // N <= 12 under TS_PLAN_AUTO: the single-CTA path (ts_small.cu)
    // execution options (ts_set_option)
    int opt_kernel;                      // 0: k_tile_pass only, 1: v2 pipelined kernels where the geometry allows, 2: v2 from three tiles per SM on
    int opt_chunk;                       // 1: L2-blocked triple launches
    int opt_chunk_max_log2;              // largest chunk (log2 amplitudes)
    int opt_chunk_min_log2;              // smallest chunk the triple launch is used for (profiles/r02_tuner.md)
    int opt_small;                       // 1: single-CTA path for N <= 12
    int opt_diag_source;                 // 0: factorised on-the-fly tables, 1: stored 2^N phase vectors, naive plan only
    int opt_l2_promotion;                // tensor-map L2 promotion of the high groups: 0 none, 1 128 B, 2 256 B
    int opt_max_ctas;                    // upper bound on the persistent kernels' grid (0: one CTA per SM)
    int opt_l2_hints;                    // L2 eviction priorities on the TMA transfers of the L2-blocked launch
    int opt_graph;                       // 1: small states replay one step's launches from a CUDA graph (ts_api.cu)
    int opt_graph_max_n;                 // largest N that does so
    int top_bits_only;                   // > 0 (transient, ts_shard.cu): a high-group pass's FIRST sweep butterflies only the group's top so-many bits
    int dry_run;                         // launchers build / look up their phase tables and return without launching
    cudaGraphExec_t g_exec;              // the graph of the last graph-mode ts_evolve call (released lazily, after g_done)
    cudaEvent_t g_done;
    cudaStream_t g_stream;               // capture-only stream
    unsigned int* d_row_ctr;             // next trace row (ts_evolve_observe replayed from a graph)
    int64_t graph_replays;               // graph launches so far (each = one 4th-order step's launches)
    int opt_pair;                        // tickets of a high group are pairs of adjacent tiles
    int opt_groups;                      // compute groups per CTA of the persistent kernels (2; 1 = experiment)
    int opt_probe;                       // copy-only tile passes (the compute groups skip the tile body): pipeline ceilings
    unsigned int* d_sched;               // [2] ticket counter + finished-CTA counter of the persistent kernels (zero between launches)
    unsigned int* d_chunk_ctr;           // done counters of the triple launch
    size_t chunk_ctr_cap;
    std::vector<TensorMapSlot> tmaps;    // per group, for the bound state pointer tmap_psi
    void* tmap_psi;
    // phase tables, built on demand and cached (invalidated when the plan changes)
    std::vector<DiagTables*> tabs;
    double* d_energy[3];                 // the stored energy vectors E_x, E_y, E_z of the table variant, built on demand
    // reduction scratch
    double* d_red;
    size_t red_cap;   // in doubles
    double* d_trace;  // ts_evolve_observe rows
    size_t trace_cap;
    // profiling
    int profiling;
    int64_t launches[TS_KC_COUNT];
    double ms_acc[TS_KC_COUNT];
    double tiles_acc[TS_KC_COUNT];       // tile passes x tiles performed per class, in units of whole-state passes
    std::vector<ProfileRec> recs;
    std::vector<cudaEvent_t> ev_pool;
};

// ---- profiling helpers (ts_api.cu).  `state_passes`: tile passes over the whole state this launch performs
// (1 for a tile pass, 3 for a triple launch, N-bit fractions for the rest are not counted: 0).
void ts_prof_begin(ts_ctx* c, int kc, double state_passes = 0.0);
void ts_prof_end(ts_ctx* c);

// One global rotation (sweep) of the whole local state, optionally followed by the exact scaling 2^scale_pow: every group
// of the plan once (tiled), or one launch per spin (ts_api.cu).
cudaError_t ts_apply_sweep_all(ts_ctx* c, int kind, int scale_pow, int skip_last_group = 0);

// ---- naive path (ts_naive.cu)
cudaError_t ts_naive_rotate(ts_ctx* c, int j, int kind);
cudaError_t ts_naive_diag(ts_ctx* c, const DiagOp& d);
void ts_naive_free_stored(ts_ctx* c);

// ---- single-CTA path for small N (ts_small.cu): the whole ts_evolve call in one launch
#define TS_SMALL_MAX_N 12
cudaError_t ts_small_evolve(ts_ctx* c, double tau, int64_t n_steps, int order);
cudaError_t ts_small_init(void);

// ---- tiled path (ts_tile.cu)
cudaError_t ts_tile_get_tables(ts_ctx* c, const DiagOp& d, int group, int layout, const DiagTables** out);
void ts_tile_free_tables(ts_ctx* c);
// which phase-table layout the pass (group, kind1, kind2) will use (0 / 1), i.e. which kernel family runs it
int ts_tile_layout_for(const ts_ctx* c, int group, int kind1, int kind2);
cudaError_t ts_tile_pass(ts_ctx* c, int group, int kind1, const DiagOp* d /*or NULL*/, int kind2);
cudaError_t ts_tile_pass_p2p(ts_ctx* c, int group, int kind, const DiagOp* d, int kind2, const double2* const* peers, int gbits,
                             int rank, double2* dst);
bool ts_tile_chunk_supported(const ts_ctx* c, int gh, int ka, int kb);
// [H(gh) single ka] [A fused ka . D . kb] [H(gh) single kb] in one L2-blocked launch
cudaError_t ts_tile_chunk_triple(ts_ctx* c, int gh, int ka, const DiagOp& d, int kb);
cudaError_t ts_tile_init(void);   // registers the kernels, sets max dynamic shared memory on all of them (once per process)

// ---- reductions (ts_reduce.cu)
cudaError_t ts_reduce_expect_z_all(ts_ctx* c, double* out_host /*[N]*/);
cudaError_t ts_reduce_expect_xy(ts_ctx* c, int alpha, int j, double* out_host);
cudaError_t ts_reduce_expect_xy_all(ts_ctx* c, double* out_x /*[N] or NULL*/, double* out_y /*[N] or NULL*/);   // tiled plans
cudaError_t ts_reduce_norm2(ts_ctx* c, double* out_host);
cudaError_t ts_reduce_overlap(ts_ctx* c, const double2* phi, double* out_host /*[2]*/);
cudaError_t ts_reduce_corr(ts_ctx* c, int alpha, int j, int k, double* out_host);   // <S^a_j S^a_k>
cudaError_t ts_reduce_energy_diag(ts_ctx* c, int alpha, double* out_host);   // sum_k E_alpha(k) |c_k|^2 of the state AS STORED
cudaError_t ts_fill_basis(ts_ctx* c, uint64_t k);
cudaError_t ts_fill_random_phase(ts_ctx* c, int up_spin, uint64_t seed);
#define TS_TRACE_STRIDE (TS_MAX_N + 1)
cudaError_t ts_reduce_trace_row(ts_ctx* c, int alpha, int j, double* dev_row /*[TS_TRACE_STRIDE]*/, unsigned int* row_ctr = nullptr);
cudaError_t ts_set_u32(ts_ctx* c, unsigned int* p, unsigned int v);
