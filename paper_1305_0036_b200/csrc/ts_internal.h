// ts_internal.h -- shared declarations of the CUDA path (host side).  Not part of the public ABI.
//
// Layers: ts_api.cu (C ABI, context, sequencer, plan) -> launchers in ts_tile.cu
// (tile passes + phase tables), ts_naive.cu (one-bit rotations, brute-force diagonal), ts_reduce.cu (observables).
// Nothing here is shared with oracle/.
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

// Phase tables of one (diagonal kind, tile group), see ts_tile_kernel.cuh.  Built on first use, cached in the context.
struct DiagTables {
    int alpha, scale_pow, group;
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
    cudaStream_t stream;
    double h[3][TS_MAX_N];
    double Jeff[3][TS_MAX_N][TS_MAX_N];   // symmetric, zero diagonal: Jeff[j][k] = J[j][k] + J[k][j]  (A1)
    double* d_h;      // [3][TS_MAX_N]
    double* d_Jeff;   // [3][TS_MAX_N][TS_MAX_N]
    double2* psi;     // 2^N amplitudes (device)
    int owns_psi;
    // plan
    int plan_mode, run_bits, max_group_bits;
    int chunk_log2, chunks_per_launch;   // L2 blocking (0 = off)
    int chunk_mode, chunk_max_log2;      // L2-blocked triple launches (ts_tile_chunk.cuh): on/off, largest chunk (log2 amplitudes)
    uint32_t* d_sched;                   // job-block order of the triple launch, for sched_nchunks chunks
    unsigned int* d_chunk_ctr;           // ticket + done counters
    uint32_t sched_nchunks;
    int pipe_mode;                       // 1: persistent TMA-pipelined tile kernels (ts_tile_pipe.cuh), 0: one CTA per tile
    std::vector<TensorMapSlot> tmaps;    // per group, for the bound state pointer tmap_psi
    void* tmap_psi;
    std::vector<TileGroup> groups;
    // phase tables, built on demand and cached (invalidated when the plan changes)
    std::vector<DiagTables> tabs;
    // reduction scratch
    double* d_red;
    size_t red_cap;   // in doubles
    // profiling
    int profiling;
    int64_t launches[TS_KC_COUNT];
    double ms_acc[TS_KC_COUNT];
    std::vector<ProfileRec> recs;
    std::vector<cudaEvent_t> ev_pool;
};

// ---- profiling helpers (ts_api.cu)
void ts_prof_begin(ts_ctx* c, int kc);
void ts_prof_end(ts_ctx* c);

// ---- naive path (ts_naive.cu)
cudaError_t ts_naive_rotate(ts_ctx* c, int j, int kind);
cudaError_t ts_naive_diag(ts_ctx* c, const DiagOp& d);

// ---- tiled path (ts_tile.cu)
cudaError_t ts_tile_get_tables(ts_ctx* c, const DiagOp& d, int group, const DiagTables** out);
void ts_tile_free_tables(ts_ctx* c);
// tile_count = 0: all tiles; otherwise the window [tile_base, tile_base + tile_count)
cudaError_t ts_tile_pass(ts_ctx* c, int group, int kind1, const DiagTables* tabs /*or NULL*/, int kind2,
                         uint64_t tile_base, uint64_t tile_count);
bool ts_tile_chunk_supported(const ts_ctx* c, int gh, int ka, int kb);
// [H(gh) single ka] [A fused ka . D(tabs) . kb] [H(gh) single kb] in one L2-blocked launch
cudaError_t ts_tile_chunk_triple(ts_ctx* c, int gh, int ka, const DiagTables* tabs, int kb);
cudaError_t ts_tile_init(void);   // registers the kernels, sets max dynamic shared memory on all of them

// ---- reductions (ts_reduce.cu)
cudaError_t ts_reduce_expect_z_all(ts_ctx* c, double* out_host /*[N]*/);
cudaError_t ts_reduce_expect_xy(ts_ctx* c, int alpha, int j, double* out_host);
cudaError_t ts_reduce_norm2(ts_ctx* c, double* out_host);
cudaError_t ts_reduce_overlap(ts_ctx* c, const double2* phi, double* out_host /*[2]*/);
cudaError_t ts_fill_basis(ts_ctx* c, uint64_t k);
#define TS_TRACE_STRIDE (TS_MAX_N + 1)
cudaError_t ts_reduce_trace_row(ts_ctx* c, int alpha, int j, double* dev_row /*[TS_TRACE_STRIDE]*/);
