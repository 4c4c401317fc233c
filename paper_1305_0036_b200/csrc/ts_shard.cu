// ts_shard.cu -- one state vector sharded over G = 2^g GPUs (SURVEY 8 e, 8 f NEXT-5): N = 33 .. 36 spins, beyond one B200.
//
// Rank rho holds the 2^n amplitudes (n = N - g) whose top g index bits equal rho.  Diagonals and butterflies on the n
// local bits are independent per shard; the butterflies on the g RANK bits pair amplitudes of different GPUs.  Once per
// sweep the ranks therefore swap the g rank bits with the top g local bits ("index-bit swap", an all-to-all in which
// rank rho sends the block with top local bits rho' to rank rho' and files what it receives from rho' under top local
// bits rho'), butterfly the g spins that have just become local, and do NOT swap back: which spin sits on which bit is
// tracked instead.  The swap is an involution, so there are exactly two spin layouts ("configurations"):
//     configuration 0:  local bit b <-> spin b (b < n);                     rank bit r <-> spin n + r
//     configuration 1:  local bit b <-> spin b (b < n - g), local bit n - g + r <-> spin n + r;  rank bit r <-> spin n - g + r
// For each configuration the shard owns an ordinary context (ts_create) over its n local spins whose Hamiltonian is the
// one its amplitudes see: fields shifted by the couplings to the spins frozen on the rank bits (sigma_r = bit_r(rho) - 1/2),
//     h'_b = h_{s(b)} + sum_r Jeff_{s(b) s(r)} sigma_r,      J'_{bb'} = J_{s(b) s(b')},
//     e0   = sum_r h_{s(r)} sigma_r + sum_{r<r'} Jeff_{s(r) s(r')} sigma_r sigma_r'      (a rank-dependent phase: it matters)
// with s(.) the configuration's bit -> spin map.  Every factor of the product formula (eq. 6-10) then acts on the
// shard exactly as it acts on the full vector.
//
// One sweep i of kind k_i, from configuration c:    [rotation k_i on all n local spins of c]  ->  exchange  ->
// [rotation k_i on the g top local spins of c^1]  ->  [diagonal D_i in c^1].  20 sweeps per 4th-order step: an even number
// of exchanges, so every whole step ends in configuration 0 and in the buffer it started from.
//
// The exchange itself is the caller's: a callback that moves 2^n amplitudes from `src` to `dst` (both device buffers on
// this rank) through whatever joins the ranks -- NCCL all-to-all over NVLink in paper_1305_0036_b200/sharded.py, plain
// copies between the shards of one GPU in the single-GPU test.  Everything else (sequence, rotations, diagonals) is this
// library's own kernels.  Per sweep a shard makes one tile pass per bit group: the top group's pass is the ARRIVAL pass,
// [sweep i on the g arrived spins] . D_i . [sweep i+1 on the whole top group] (its first sweep restricted to the group's top
// g bits), so sweep i+1's local passes start below it.
//
// PEER-MEMORY MODE (ts_shard_bind_peers; NVLink 5 / NVSwitch gives every GPU load/store access to every peer's HBM): the
// exchange and the pass over the arrivals are ONE kernel (k_tile_pass_p2p, ts_tile_kernel.cuh).  The arrival pass's tiles
// are gathered straight from the peers' shards -- the rows whose top g row bits equal rho' are loaded from rank rho' at
// the position that has this rank's number in those bits, which is exactly what the all-to-all would have delivered --
// rotated, multiplied by the diagonal and stored into this rank's other buffer.  No collective moves data; what is left of
// the callback is a barrier (src = dst = NULL): "every rank has finished its local sweep".  One barrier per sweep
// suffices: a rank overwrites the buffer its peers read from only in its NEXT arrival pass, i.e. after the next barrier.
#include <math.h>
#include <string.h>

#include <new>

#include "ts_internal.h"

struct ts_shard {
    int N, g, n, rank;
    ts_ctx* cfg[2];
    double2* buf[2];
    int cur_cfg, cur_buf;
    const double2* peer[2][256];     // peer-memory mode: buffer 0 / 1 of every rank as mapped into this device (else peer[0][0] = NULL)
};

namespace {

int spin_of_local(const ts_shard* s, int cfg, int b)
{
    if (cfg == 0 || b < s->n - s->g) return b;
    return s->n + (b - (s->n - s->g));
}
int spin_of_rankbit(const ts_shard* s, int cfg, int r) { return cfg == 0 ? s->n + r : s->n - s->g + r; }

int make_cfg(ts_shard* s, int cfg, const double* h, const double* J)
{
    const int N = s->N, n = s->n, g = s->g;
    double* hl = new (std::nothrow) double[3 * (size_t)n];
    double* Jl = new (std::nothrow) double[3 * (size_t)n * n];
    if (!hl || !Jl) { delete[] hl; delete[] Jl; return TS_ERR_NOMEM; }
    double e0[3];
    for (int a = 0; a < 3; ++a) {
        const double* ha = h + (size_t)a * N;
        const double* Ja = J + (size_t)a * N * N;
        auto jeff = [&](int p, int q) { return Ja[(size_t)p * N + q] + Ja[(size_t)q * N + p]; };
        for (int b = 0; b < n; ++b) {
            const int sb = spin_of_local(s, cfg, b);
            double f = ha[sb];
            for (int r = 0; r < g; ++r) f += jeff(sb, spin_of_rankbit(s, cfg, r)) * ((double)((s->rank >> r) & 1) - 0.5);
            hl[(size_t)a * n + b] = f;
            for (int b2 = 0; b2 < n; ++b2)
                Jl[((size_t)a * n + b) * n + b2] = (b == b2) ? 0.0 : Ja[(size_t)sb * N + spin_of_local(s, cfg, b2)];
        }
        double e = 0.0;
        for (int r = 0; r < g; ++r) {
            const int sr = spin_of_rankbit(s, cfg, r);
            const double sg = (double)((s->rank >> r) & 1) - 0.5;
            double f = ha[sr];
            for (int r2 = 0; r2 < r; ++r2) f += jeff(sr, spin_of_rankbit(s, cfg, r2)) * ((double)((s->rank >> r2) & 1) - 0.5);
            e += sg * f;
        }
        e0[a] = e;
    }
    int st = ts_create(&s->cfg[cfg], n, hl, Jl);
    delete[] hl; delete[] Jl;
    if (st != TS_OK) return st;
    for (int a = 0; a < 3; ++a) s->cfg[cfg]->e0[a] = e0[a];
    return TS_OK;
}

// The whole local sweep of a context: one tile pass per bit group (the top one left out when the previous arrival pass has
// done it already), or one launch per spin for shards below 12 spins.
cudaError_t local_sweep(ts_ctx* c, int kind, bool top_group_done)
{
    return ts_apply_sweep_all(c, kind, 0, top_group_done ? 1 : 0);
}

// Can the arrival pass be the top bit group's tile pass?  (A shard of >= 13 spins whose top group has at least g bits.)
bool arrival_is_a_tile_pass(const ts_ctx* c, int g)
{
    return c->groups.size() >= 2 && TS_TILE_LOG2 - c->groups.back().s >= g;
}

// The g spins that arrived with an exchange sit on the top g local bits, i.e. on the top bits of the plan's last bit
// group: their rotation (sweep `kind`), the diagonal that follows the sweep and the NEXT sweep's butterflies on the whole
// group (`kind2`, SW_NONE after the last sweep) are ONE tile pass of that group.  (Shards below 13 spins, or a top group
// with fewer than g bits: one launch per spin, then the diagonal; kind2 must be SW_NONE.)
cudaError_t rotate_arrivals_then_diagonal(ts_ctx* c, int kind, int g, const DiagOp& d, int kind2)
{
    if (arrival_is_a_tile_pass(c, g)) {
        c->top_bits_only = g;
        cudaError_t e = ts_tile_pass(c, (int)c->groups.size() - 1, kind, d.present ? &d : nullptr, kind2);
        c->top_bits_only = 0;
        return e;
    }
    cudaError_t e = cudaSuccess;
    for (int j = c->N - g; j < c->N && e == cudaSuccess; ++j) e = ts_naive_rotate(c, j, kind);
    if (e != cudaSuccess || !d.present) return e;
    if (!c->groups.empty()) return ts_tile_pass(c, 0, SW_NONE, &d, SW_NONE);
    return ts_naive_diag(c, d);
}

cudaError_t diagonal(ts_ctx* c, const DiagOp& d)
{
    if (!d.present) return cudaSuccess;
    if (!c->groups.empty()) return ts_tile_pass(c, 0, SW_NONE, &d, SW_NONE);
    return ts_naive_diag(c, d);
}

int cuda_status(cudaError_t e)
{
    if (e == cudaSuccess) return TS_OK;
    if (e == cudaErrorMemoryAllocation) return TS_ERR_NOMEM;
    return TS_ERR_CUDA;
}

} // namespace

extern "C" {

int ts_shard_create(ts_shard** out, int N, const double* h, const double* J, int log2_ranks, int rank)
{
    if (!out) return TS_ERR_ARG;
    *out = nullptr;
    const int g = log2_ranks;
    if (!h || !J || g < 0 || g > 8 || N - g < 1 || N - g > TS_MAX_N || 2 * g > N || rank < 0 || rank >= (1 << g)) return TS_ERR_ARG;
    for (int i = 0; i < 3 * N; ++i) if (!isfinite(h[i])) return TS_ERR_ARG;
    for (int64_t i = 0; i < (int64_t)3 * N * N; ++i) if (!isfinite(J[i])) return TS_ERR_ARG;
    ts_shard* s = new (std::nothrow) ts_shard();
    if (!s) return TS_ERR_NOMEM;
    s->N = N; s->g = g; s->n = N - g; s->rank = rank;
    s->cfg[0] = s->cfg[1] = nullptr; s->buf[0] = s->buf[1] = nullptr; s->cur_cfg = 0; s->cur_buf = 0;
    s->peer[0][0] = nullptr;
    int st = make_cfg(s, 0, h, J);
    if (st == TS_OK) st = make_cfg(s, 1, h, J);
    if (st != TS_OK) { ts_shard_destroy(s); return st; }
    // partial operations run unfused: the tiled plan for n >= 12 (tile passes per group), one launch per spin below
    for (int c = 0; c < 2 && st == TS_OK; ++c)
        st = ts_set_plan(s->cfg[c], s->n >= TS_TILE_LOG2 ? TS_PLAN_TILED : TS_PLAN_NAIVE, 0, 0);
    if (st != TS_OK) { ts_shard_destroy(s); return st; }
    *out = s;
    return TS_OK;
}

int ts_shard_destroy(ts_shard* s)
{
    if (!s) return TS_OK;
    if (s->cfg[0]) ts_destroy(s->cfg[0]);
    if (s->cfg[1]) ts_destroy(s->cfg[1]);
    delete s;
    return TS_OK;
}

int ts_shard_bind(ts_shard* s, void* buf0, void* buf1)
{
    if (!s || !buf0 || !buf1 || buf0 == buf1) return TS_ERR_ARG;
    s->buf[0] = (double2*)buf0; s->buf[1] = (double2*)buf1;
    s->cur_cfg = 0; s->cur_buf = 0;
    int st = ts_bind_state(s->cfg[0], buf0);
    if (st == TS_OK) st = ts_bind_state(s->cfg[1], buf0);
    return st;
}

int ts_shard_bind_peers(ts_shard* s, const void* const* bufs0, const void* const* bufs1)
{
    if (!s) return TS_ERR_ARG;
    if (!bufs0 || !bufs1) { s->peer[0][0] = nullptr; return TS_OK; }          // back to the exchange callback
    if (!s->buf[0] || s->g < 1 || s->g > 5) return TS_ERR_ARG;
    // the arrival pass is the top bit group's tile pass: the shard must have one, with at least g bits
    const ts_ctx* c = s->cfg[0];
    if (c->groups.size() < 2 || TS_TILE_LOG2 - c->groups.back().s < s->g) return TS_ERR_ARG;
    for (int r = 0; r < (1 << s->g); ++r) {
        if (!bufs0[r] || !bufs1[r]) return TS_ERR_ARG;
        s->peer[0][r] = (const double2*)bufs0[r];
        s->peer[1][r] = (const double2*)bufs1[r];
    }
    if (s->peer[0][s->rank] != s->buf[0] || s->peer[1][s->rank] != s->buf[1]) { s->peer[0][0] = nullptr; return TS_ERR_ARG; }
    return TS_OK;
}

int ts_shard_set_stream(ts_shard* s, void* stream)
{
    if (!s) return TS_ERR_ARG;
    int st = ts_set_stream(s->cfg[0], stream);
    if (st == TS_OK) st = ts_set_stream(s->cfg[1], stream);
    return st;
}

int ts_shard_info(ts_shard* s, int* n_local, int* config, int* buffer)
{
    if (!s) return TS_ERR_ARG;
    if (n_local) *n_local = s->n;
    if (config) *config = s->cur_cfg;
    if (buffer) *buffer = s->cur_buf;
    return TS_OK;
}

int ts_shard_spin_map(ts_shard* s, int config, int* spin_of_bit)
{
    if (!s || !spin_of_bit || config < 0 || config > 1) return TS_ERR_ARG;
    for (int b = 0; b < s->n; ++b) spin_of_bit[b] = spin_of_local(s, config, b);
    for (int r = 0; r < s->g; ++r) spin_of_bit[s->n + r] = spin_of_rankbit(s, config, r);
    return TS_OK;
}

ts_ctx* ts_shard_ctx(ts_shard* s, int config) { return (s && config >= 0 && config <= 1) ? s->cfg[config] : nullptr; }

int ts_shard_evolve(ts_shard* s, double tau, int64_t n_steps, int order, ts_exchange_fn exchange, void* user)
{
    if (!s || !isfinite(tau) || n_steps < 0 || (order != 2 && order != 4) || (s->g > 0 && !exchange)) return TS_ERR_ARG;
    if (!s->buf[0]) return TS_ERR_NOSTATE;
    if (n_steps == 0) return TS_OK;
    // the merged Suzuki sequence of ts_api.cu: D_z(s/2) . X^dag . D_y(s/2) . Y^dag . D_x(s) . Y . D_y(s/2) . X . D_z(s/2), the
    // trailing D_z merged with the next leading one, 2^-N (N of the FULL system: every sweep butterflies all N spins)
    // after each backward sweep
    const double a = 1.0 / (4.0 - cbrt(4.0));
    const int64_t n_sub = n_steps * (order == 4 ? 5 : 1), M = 4 * n_sub;
    auto sub = [&](int64_t u) -> double {
        if (u < 0 || u >= n_sub) return 0.0;
        if (order == 2) return tau;
        return ((u % 5) == 2) ? (1.0 - 4.0 * a) * tau : a * tau;
    };
    static const int kinds[4] = {SW_XDAG, SW_YDAG, SW_Y, SW_X};
    cudaError_t e = cudaSuccess;
    DiagOp d; d.present = 1; d.alpha = TS_Z; d.t = 0.5 * sub(0); d.scale_pow = 0;
    e = diagonal(s->cfg[s->cur_cfg], d);
    const bool fuse = s->g > 0 && arrival_is_a_tile_pass(s->cfg[0], s->g);
    bool top_done = false;               // the top group's butterflies of this sweep were done by the last arrival pass
    for (int64_t i = 1; i <= M && e == cudaSuccess; ++i) {
        const int kind = kinds[(i - 1) & 3];
        const int kind2 = (fuse && i < M) ? kinds[i & 3] : SW_NONE;
        e = local_sweep(s->cfg[s->cur_cfg], kind, top_done);
        if (e != cudaSuccess) break;
        const int64_t u = (i - 1) >> 2;
        const double su = sub(u);
        switch ((i - 1) & 3) {
        case 0: d.alpha = TS_Y; d.t = 0.5 * su; d.scale_pow = 0; break;
        case 1: d.alpha = TS_X; d.t = su; d.scale_pow = 0; break;
        case 2: d.alpha = TS_Y; d.t = 0.5 * su; d.scale_pow = -s->N; break;
        default: d.alpha = TS_Z; d.t = 0.5 * su + 0.5 * sub(u + 1); d.scale_pow = -s->N; break;
        }
        if (s->g > 0 && s->peer[0][0]) {
            // peer-memory mode: barrier, then the arrival pass gathers its tiles from the peers' current buffers
            if (exchange(user, nullptr, nullptr) != 0) return TS_ERR_CUDA;
            double2* dst = s->buf[s->cur_buf ^ 1];
            ts_ctx* cn = s->cfg[s->cur_cfg ^ 1];
            ts_bind_state(cn, (void*)dst);
            e = ts_tile_pass_p2p(cn, (int)cn->groups.size() - 1, kind, &d, kind2, s->peer[s->cur_buf], s->g, s->rank, dst);
            s->cur_buf ^= 1; s->cur_cfg ^= 1;
            ts_bind_state(s->cfg[0], (void*)dst);
            ts_bind_state(s->cfg[1], (void*)dst);
            top_done = (kind2 != SW_NONE);
        } else if (s->g > 0) {
            double2* src = s->buf[s->cur_buf];
            double2* dst = s->buf[s->cur_buf ^ 1];
            if (exchange(user, (void*)src, (void*)dst) != 0) return TS_ERR_CUDA;
            s->cur_buf ^= 1; s->cur_cfg ^= 1;
            ts_bind_state(s->cfg[0], (void*)dst);
            ts_bind_state(s->cfg[1], (void*)dst);
            e = rotate_arrivals_then_diagonal(s->cfg[s->cur_cfg], kind, s->g, d, kind2);
            top_done = (kind2 != SW_NONE);
        } else {
            e = diagonal(s->cfg[s->cur_cfg], d);
        }
    }
    return cuda_status(e);
}

} // extern "C"
