// ts_api.cu -- C ABI (include/ts_b200.h), context, plan and the Suzuki sequencer (SURVEY 8 a1, 8 b).
//
// Sequencer.  With U_1(t) = exp(-itH_x) exp(-itH_y) exp(-itH_z) (eq. 3/6/8; A6) and
// U_2(s) = U_1^dag(-s/2) U_1(s/2):
//     U_2(s) = e^{-i s/2 H_z} e^{-i s/2 H_y} e^{-i s H_x} e^{-i s/2 H_y} e^{-i s/2 H_z}.
// With e^{-itH_y} = X D_y(t) X^dag, e^{-itH_x} = Y D_x(t) Y^dag (eq. 7, 10) and because the
// global rotation X (a product of single-spin rotations about x) commutes with H_x, the apply order becomes
//     D_z(s/2) . X^dag . D_y(s/2) . Y^dag . D_x(s) . Y . D_y(s/2) . X . D_z(s/2)
// i.e. 4 sweeps and 5 diagonals per U_2; the trailing D_z merges with the next leading D_z.  Sweeps are unnormalised;
// the exact factor 2^-N rides on the diagonal that follows each "backward" sweep (Y and X), so the norm only sees
// random round-off (A13).  U_4 = five U_2 with s = (a, a, 1-4a, a, a) tau: 20 sweeps + 20 diagonals per
// step in steady state.
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <new>
#include <string>

#include "ts_internal.h"

namespace {

struct Seq {
    int order, N;
    int64_t n_sub, M;     // sub-steps (U_2 applications), sweeps
    double tau, a;
    Seq(int order_, int N_, double tau_, int64_t n_steps) : order(order_), N(N_), tau(tau_)
    {
        a = 1.0 / (4.0 - cbrt(4.0));
        n_sub = n_steps * (order == 4 ? 5 : 1);
        M = 4 * n_sub;
    }
    double sub(int64_t u) const
    {
        if (u < 0 || u >= n_sub) return 0.0;
        if (order == 2) return tau;
        return ((u % 5) == 2) ? (1.0 - 4.0 * a) * tau : a * tau;
    }
    int kind(int64_t i) const     // sweep i = 1 .. M
    {
        static const int k[4] = {SW_XDAG, SW_YDAG, SW_Y, SW_X};
        return k[(i - 1) & 3];
    }
    DiagOp diag(int64_t i) const  // diagonal after sweep i (i = 0: before the first sweep)
    {
        DiagOp d; d.present = 1;
        if (i == 0) { d.alpha = TS_Z; d.t = 0.5 * sub(0); d.scale_pow = 0; return d; }
        const int64_t u = (i - 1) >> 2;
        const double s = sub(u);
        switch ((i - 1) & 3) {
        case 0: d.alpha = TS_Y; d.t = 0.5 * s; d.scale_pow = 0; break;
        case 1: d.alpha = TS_X; d.t = s; d.scale_pow = 0; break;
        case 2: d.alpha = TS_Y; d.t = 0.5 * s; d.scale_pow = -N; break;
        default: d.alpha = TS_Z; d.t = 0.5 * s + 0.5 * sub(u + 1); d.scale_pow = -N; break;
        }
        return d;
    }
};

int build_plan(ts_ctx* c)
{
    c->groups.clear();
    const int N = c->N;
    int mode = c->plan_mode;
    if (mode == TS_PLAN_AUTO) mode = (N >= TS_TILE_LOG2) ? TS_PLAN_TILED : TS_PLAN_NAIVE;
    if (mode == TS_PLAN_NAIVE) return TS_OK;
    if (N < TS_TILE_LOG2) return TS_ERR_ARG;
    const int s_min = c->run_bits > 0 ? c->run_bits : 3;
    if (s_min < 1 || s_min > TS_TILE_LOG2 - 1) return TS_ERR_ARG;
    int mgmax = TS_TILE_LOG2 - s_min;
    if (c->max_group_bits > 0 && c->max_group_bits < mgmax) mgmax = c->max_group_bits;
    TileGroup A; A.s = TS_TILE_LOG2; A.g0 = TS_TILE_LOG2; A.is_low = 1;
    c->groups.push_back(A);
    const int rem = N - TS_TILE_LOG2;
    if (rem > 0) {
        const int ng = (rem + mgmax - 1) / mgmax;
        int g0 = TS_TILE_LOG2;
        for (int i = 0; i < ng; ++i) {
            const int mg = rem / ng + (i < rem % ng ? 1 : 0);    // balanced split: longer runs for everyone
            TileGroup g; g.s = TS_TILE_LOG2 - mg; g.g0 = g0; g.is_low = 0;
            c->groups.push_back(g);
            g0 += mg;
        }
    }
    return TS_OK;
}

bool tiled(const ts_ctx* c) { return !c->groups.empty(); }

int cuda_status(cudaError_t e)
{
    if (e == cudaSuccess) return TS_OK;
    if (e == cudaErrorMemoryAllocation) return TS_ERR_NOMEM;
    return TS_ERR_CUDA;
}

int ensure_state(ts_ctx* c)
{
    if (c->psi) return TS_OK;
    void* p = nullptr;
    cudaError_t e = cudaMalloc(&p, sizeof(double2) << c->N);
    if (e != cudaSuccess) { cudaGetLastError(); return TS_ERR_NOMEM; }
    c->psi = (double2*)p;
    c->owns_psi = 1;
    return TS_OK;
}

} // namespace

void ts_prof_begin(ts_ctx* c, int kc)
{
    c->launches[kc]++;
    if (!c->profiling) return;
    ProfileRec r; r.kc = kc;
    for (cudaEvent_t* e : {&r.e0, &r.e1}) {
        if (!c->ev_pool.empty()) { *e = c->ev_pool.back(); c->ev_pool.pop_back(); }
        else cudaEventCreate(e);
    }
    cudaEventRecord(r.e0, c->stream);
    c->recs.push_back(r);
}

void ts_prof_end(ts_ctx* c)
{
    if (!c->profiling || c->recs.empty()) return;
    cudaEventRecord(c->recs.back().e1, c->stream);
}

extern "C" {

const char* ts_strerror(int s)
{
    switch (s) {
    case TS_OK: return "ok";
    case TS_ERR_ARG: return "invalid argument";
    case TS_ERR_NOMEM: return "out of (device) memory";
    case TS_ERR_CUDA: return "CUDA error or no usable CUDA device";
    case TS_ERR_NOSTATE: return "no state vector set";
    default: return "unknown status";
    }
}

const char* ts_version(void) { return "ts_b200 0.1 sm_100a tile=2^12 regs=32amp/thread"; }

int ts_create(ts_ctx** out, int N, const double* h, const double* J)
{
    if (!out) return TS_ERR_ARG;
    *out = nullptr;
    if (!h || !J || N < 1 || N > TS_MAX_N) return TS_ERR_ARG;
    for (int i = 0; i < 3 * N; ++i) if (!isfinite(h[i])) return TS_ERR_ARG;
    for (int64_t i = 0; i < (int64_t)3 * N * N; ++i) if (!isfinite(J[i])) return TS_ERR_ARG;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) { cudaGetLastError(); return TS_ERR_CUDA; }
    ts_ctx* c = new (std::nothrow) ts_ctx();
    if (!c) return TS_ERR_NOMEM;
    c->N = N;
    cudaGetDevice(&c->device);
    c->stream = 0;
    memset(c->h, 0, sizeof(c->h));
    memset(c->Jeff, 0, sizeof(c->Jeff));
    for (int a = 0; a < 3; ++a) {
        for (int j = 0; j < N; ++j) c->h[a][j] = h[a * N + j];
        for (int j = 0; j < N; ++j)
            for (int k = 0; k < N; ++k)
                if (j != k) c->Jeff[a][j][k] = J[((size_t)a * N + j) * N + k] + J[((size_t)a * N + k) * N + j];
    }
    c->psi = nullptr; c->owns_psi = 0;
    c->plan_mode = TS_PLAN_AUTO; c->run_bits = 0; c->max_group_bits = 0;
    c->chunk_log2 = getenv("TS_CHUNK_LOG2") ? atoi(getenv("TS_CHUNK_LOG2")) : 0;
    c->chunks_per_launch = getenv("TS_CHUNKS_PER_LAUNCH") ? atoi(getenv("TS_CHUNKS_PER_LAUNCH")) : 1;
    c->pipe_mode = getenv("TS_PIPE") ? atoi(getenv("TS_PIPE")) : 1;
    c->chunk_mode = getenv("TS_CHUNK3") ? atoi(getenv("TS_CHUNK3")) : 2;
    c->chunk_max_log2 = getenv("TS_CHUNK3_MAX_LOG2") ? atoi(getenv("TS_CHUNK3_MAX_LOG2")) : 21;
    c->d_sched = nullptr; c->d_chunk_ctr = nullptr; c->sched_nchunks = 0;
    c->tmap_psi = nullptr;
    c->d_red = nullptr; c->red_cap = 0;
    c->profiling = 0;
    memset(c->launches, 0, sizeof(c->launches));
    memset(c->ms_acc, 0, sizeof(c->ms_acc));
    cudaError_t e = cudaMalloc(&c->d_h, sizeof(c->h));
    if (e == cudaSuccess) e = cudaMalloc(&c->d_Jeff, sizeof(c->Jeff));
    if (e == cudaSuccess) e = cudaMemcpy(c->d_h, c->h, sizeof(c->h), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(c->d_Jeff, c->Jeff, sizeof(c->Jeff), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = ts_tile_init();
    if (e != cudaSuccess) { cudaGetLastError(); ts_destroy(c); return cuda_status(e); }
    int st = build_plan(c);
    if (st != TS_OK) { ts_destroy(c); return st; }
    *out = c;
    return TS_OK;
}

int ts_destroy(ts_ctx* c)
{
    if (!c) return TS_OK;
    if (c->psi && c->owns_psi) cudaFree(c->psi);
    if (c->d_h) cudaFree(c->d_h);
    if (c->d_Jeff) cudaFree(c->d_Jeff);
    ts_tile_free_tables(c);
    if (c->d_red) cudaFree(c->d_red);
    if (c->d_sched) cudaFree(c->d_sched);
    if (c->d_chunk_ctr) cudaFree(c->d_chunk_ctr);
    for (auto& r : c->recs) { cudaEventDestroy(r.e0); cudaEventDestroy(r.e1); }
    for (auto& e : c->ev_pool) cudaEventDestroy(e);
    delete c;
    return TS_OK;
}

int ts_set_stream(ts_ctx* c, void* s)
{
    if (!c) return TS_ERR_ARG;
    c->stream = (cudaStream_t)s;
    return TS_OK;
}

int ts_bind_state(ts_ctx* c, void* dev)
{
    if (!c || !dev || ((uintptr_t)dev & 15)) return TS_ERR_ARG;
    if (c->psi && c->owns_psi) cudaFree(c->psi);
    c->psi = (double2*)dev;
    c->owns_psi = 0;
    return TS_OK;
}

int ts_set_state(ts_ctx* c, const void* amps, int where)
{
    if (!c || !amps || (where != TS_HOST && where != TS_DEVICE)) return TS_ERR_ARG;
    int st = ensure_state(c);
    if (st != TS_OK) return st;
    cudaError_t e = cudaMemcpyAsync(c->psi, amps, sizeof(double2) << c->N,
                                    where == TS_HOST ? cudaMemcpyHostToDevice : cudaMemcpyDeviceToDevice, c->stream);
    return cuda_status(e);
}

int ts_set_state_range(ts_ctx* c, const void* amps, uint64_t first, uint64_t count, int where)
{
    if (!c || !amps || (where != TS_HOST && where != TS_DEVICE)) return TS_ERR_ARG;
    const uint64_t dim = (uint64_t)1 << c->N;
    if (first > dim || count > dim - first) return TS_ERR_ARG;
    int st = ensure_state(c);
    if (st != TS_OK) return st;
    if (count == 0) return TS_OK;
    cudaError_t e = cudaMemcpyAsync(c->psi + first, amps, count * sizeof(double2),
                                    where == TS_HOST ? cudaMemcpyHostToDevice : cudaMemcpyDeviceToDevice, c->stream);
    return cuda_status(e);
}

int ts_set_basis_state(ts_ctx* c, uint64_t k)
{
    if (!c || k >= ((uint64_t)1 << c->N)) return TS_ERR_ARG;
    int st = ensure_state(c);
    if (st != TS_OK) return st;
    return cuda_status(ts_fill_basis(c, k));
}

int ts_get_state(ts_ctx* c, void* dst, uint64_t first, uint64_t count, int where)
{
    if (!c || !dst || (where != TS_HOST && where != TS_DEVICE)) return TS_ERR_ARG;
    if (!c->psi) return TS_ERR_NOSTATE;
    const uint64_t dim = (uint64_t)1 << c->N;
    if (first > dim || count > dim - first) return TS_ERR_ARG;
    if (count == 0) return TS_OK;
    cudaError_t e = cudaMemcpyAsync(dst, c->psi + first, count * sizeof(double2),
                                    where == TS_HOST ? cudaMemcpyDeviceToHost : cudaMemcpyDeviceToDevice, c->stream);
    if (e == cudaSuccess && where == TS_HOST) e = cudaStreamSynchronize(c->stream);
    return cuda_status(e);
}

int ts_set_plan(ts_ctx* c, int mode, int run_bits, int max_group_bits)
{
    if (!c || mode < TS_PLAN_AUTO || mode > TS_PLAN_TILED || run_bits < 0 || max_group_bits < 0) return TS_ERR_ARG;
    const int om = c->plan_mode, orb = c->run_bits, omg = c->max_group_bits;
    c->plan_mode = mode; c->run_bits = run_bits; c->max_group_bits = max_group_bits;
    cudaStreamSynchronize(c->stream);
    ts_tile_free_tables(c);          // tables depend on the group geometry
    c->tmaps.clear();
    int st = build_plan(c);
    if (st != TS_OK) { c->plan_mode = om; c->run_bits = orb; c->max_group_bits = omg; build_plan(c); }
    return st;
}

int ts_describe_plan(ts_ctx* c, char* buf, int buflen)
{
    if (!c || !buf || buflen < 1) return TS_ERR_ARG;
    std::string s;
    char tmp[128];
    if (!tiled(c)) {
        snprintf(tmp, sizeof tmp, "naive: N=%d, %d one-bit rotation launches + 1 diagonal launch per sweep", c->N, c->N);
        s = tmp;
    } else {
        const int g = (int)c->groups.size();
        snprintf(tmp, sizeof tmp, "tiled: N=%d, tile=2^%d, %d group(s), %d HBM round trip(s) per sweep:", c->N,
                 TS_TILE_LOG2, g, g > 1 ? g - 1 : 1);
        s = tmp;
        for (const TileGroup& t : c->groups) {
            if (t.is_low) snprintf(tmp, sizeof tmp, " A[spins 0..11]");
            else snprintf(tmp, sizeof tmp, " H[spins %d..%d, run 2^%d]", t.g0, t.g0 + TS_TILE_LOG2 - t.s - 1, t.s);
            s += tmp;
        }
    }
    snprintf(buf, buflen, "%s", s.c_str());
    return TS_OK;
}

int ts_evolve(ts_ctx* c, double tau, int64_t n_steps, int order)
{
    if (!c || !isfinite(tau) || n_steps < 0 || (order != 2 && order != 4)) return TS_ERR_ARG;
    if (!c->psi) return TS_ERR_NOSTATE;
    if (n_steps == 0) return TS_OK;
    const Seq q(order, c->N, tau, n_steps);
    cudaError_t e = cudaSuccess;

    if (!tiled(c)) {
        e = ts_naive_diag(c, q.diag(0));
        for (int64_t i = 1; i <= q.M && e == cudaSuccess; ++i) {
            for (int j = 0; j < c->N && e == cudaSuccess; ++j) e = ts_naive_rotate(c, j, q.kind(i));
            if (e == cudaSuccess) e = ts_naive_diag(c, q.diag(i));
        }
        return cuda_status(e);
    }

    // ---- pass list: one entry per HBM round trip (or per L2 round trip inside a blocked run)
    struct Pass { int gi, k1, k2; DiagOp d; };
    std::vector<Pass> passes;
    auto push = [&](int gi, int k1, const DiagOp* d, int k2) {
        Pass ps; ps.gi = gi; ps.k1 = k1; ps.k2 = k2;
        if (d) ps.d = *d; else ps.d.present = 0;
        passes.push_back(ps);
    };
    const int g = (int)c->groups.size();
    for (int64_t i = 1; i <= q.M; ++i) {
        const bool fwd = (i & 1);
        if (g == 1) {
            const DiagOp d0 = q.diag(i - 1);
            push(0, SW_NONE, &d0, q.kind(i));
            if (i == q.M) { const DiagOp dm = q.diag(q.M); push(0, SW_NONE, &dm, SW_NONE); }
            continue;
        }
        for (int pos = 0; pos < g; ++pos) {
            const int gi = fwd ? pos : g - 1 - pos;
            const bool first = (pos == 0), last = (pos == g - 1);
            if (first && i > 1) continue;                              // done by the previous fused pass
            if (last && i < q.M) {                                     // sweep i . D_i . sweep i+1 on the same group
                const DiagOp d = q.diag(i);
                push(gi, q.kind(i), &d, q.kind(i + 1));
            } else if (first && i == 1) {
                const DiagOp d = q.diag(0);
                push(gi, SW_NONE, &d, q.kind(1));
            } else if (last && i == q.M) {
                const DiagOp d = q.diag(q.M);
                push(gi, q.kind(i), &d, SW_NONE);
            } else {
                push(gi, q.kind(i), nullptr, SW_NONE);
            }
        }
    }

    auto launch = [&](const Pass& ps, uint64_t tile_base, uint64_t tile_count) -> cudaError_t {
        const DiagTables* tb = nullptr;
        if (ps.d.present) {
            cudaError_t ee = ts_tile_get_tables(c, ps.d, ps.gi, &tb);
            if (ee != cudaSuccess) return ee;
        }
        return ts_tile_pass(c, ps.gi, ps.k1, tb, ps.k2, tile_base, tile_count);
    };

    // ---- execution.  L2 blocking: consecutive passes whose groups all lie below spin
    // `chunk_log2` act inside aligned chunks of 2^chunk_log2 amplitudes (closed-set argument of P:141 applied to the
    // chunk), so such a run is executed chunk window by chunk window: the window is read from HBM by the first pass,
    // stays in the 126 MB L2 for the passes in between and is written back once.
    const int C = c->chunk_log2;
    const uint64_t ntiles = (uint64_t)1 << (c->N - TS_TILE_LOG2);
    auto top_spin = [&](int gi) { const TileGroup& t = c->groups[gi]; return t.is_low ? TS_TILE_LOG2 - 1 : t.g0 + TS_TILE_LOG2 - t.s - 1; };
    size_t ip = 0;
    while (ip < passes.size() && e == cudaSuccess) {
        // [H single ka] [A fused ka . D . kb] [H single kb]  ->  one L2-blocked launch (ts_tile_chunk.cuh)
        if (ip + 2 < passes.size()) {
            const Pass &p0 = passes[ip], &p1 = passes[ip + 1], &p2 = passes[ip + 2];
            if (p0.gi == p2.gi && p1.gi == 0 && p0.k2 == SW_NONE && !p0.d.present && p2.k2 == SW_NONE && !p2.d.present &&
                p1.d.present && p1.k1 == p0.k1 && p1.k2 == p2.k1 && ts_tile_chunk_supported(c, p0.gi, p1.k1, p1.k2)) {
                const DiagTables* tb = nullptr;
                e = ts_tile_get_tables(c, p1.d, 0, &tb);
                if (e == cudaSuccess) e = ts_tile_chunk_triple(c, p0.gi, p1.k1, tb, p1.k2);
                ip += 3;
                continue;
            }
        }
        size_t jp = ip;
        if (C > 0 && C < c->N)
            while (jp < passes.size() && top_spin(passes[jp].gi) < C) ++jp;
        if (jp - ip >= 2) {
            const uint64_t win = ((uint64_t)1 << (C - TS_TILE_LOG2)) * (uint64_t)(c->chunks_per_launch > 0 ? c->chunks_per_launch : 1);
            for (uint64_t tb0 = 0; tb0 < ntiles && e == cudaSuccess; tb0 += win) {
                const uint64_t cnt = (ntiles - tb0 < win) ? ntiles - tb0 : win;
                for (size_t k = ip; k < jp && e == cudaSuccess; ++k) e = launch(passes[k], tb0, cnt);
            }
            ip = jp;
        } else {
            e = launch(passes[ip], 0, 0);
            ++ip;
        }
    }
    return cuda_status(e);
}

int ts_evolve_observe(ts_ctx* c, double tau, int64_t n_steps, int order, int alpha, int j, double* out)
{
    if (!c || !out || !isfinite(tau) || n_steps < 0 || (order != 2 && order != 4) || alpha < TS_X || alpha > TS_Z) return TS_ERR_ARG;
    if (alpha == TS_Z ? (j < -1 || j >= c->N) : (j < 0 || j >= c->N)) return TS_ERR_ARG;
    if (!c->psi) return TS_ERR_NOSTATE;
    if (n_steps == 0) return TS_OK;
    double* d_trace = nullptr;
    cudaError_t e = cudaMalloc(&d_trace, sizeof(double) * TS_TRACE_STRIDE * (size_t)n_steps);
    if (e != cudaSuccess) { cudaGetLastError(); return TS_ERR_NOMEM; }
    int st = TS_OK;
    for (int64_t k = 0; k < n_steps && st == TS_OK; ++k) {
        st = ts_evolve(c, tau, 1, order);
        if (st == TS_OK) st = cuda_status(ts_reduce_trace_row(c, alpha, j < 0 ? 0 : j, d_trace + (size_t)k * TS_TRACE_STRIDE));
    }
    std::vector<double> host;
    if (st == TS_OK) {
        host.resize((size_t)TS_TRACE_STRIDE * n_steps);
        e = cudaMemcpyAsync(host.data(), d_trace, sizeof(double) * host.size(), cudaMemcpyDeviceToHost, c->stream);
        if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
        st = cuda_status(e);
    } else {
        cudaStreamSynchronize(c->stream);
    }
    cudaFree(d_trace);
    if (st != TS_OK) return st;
    for (int64_t k = 0; k < n_steps; ++k) {
        const double* row = host.data() + (size_t)k * TS_TRACE_STRIDE;
        if (alpha == TS_Z) {
            if (j < 0) for (int s = 0; s < c->N; ++s) out[(size_t)k * c->N + s] = row[1 + s] - 0.5 * row[0];
            else out[k] = row[1 + j] - 0.5 * row[0];
        } else {
            out[k] = (alpha == TS_X) ? row[0] : row[1];
        }
    }
    return TS_OK;
}

int ts_expect(ts_ctx* c, int alpha, int j, double* out)
{
    if (!c || !out || alpha < TS_X || alpha > TS_Z || j < 0 || j >= c->N) return TS_ERR_ARG;
    if (!c->psi) return TS_ERR_NOSTATE;
    if (alpha == TS_Z) {
        double v[TS_MAX_N];
        cudaError_t e = ts_reduce_expect_z_all(c, v);
        if (e != cudaSuccess) return cuda_status(e);
        *out = v[j];
        return TS_OK;
    }
    return cuda_status(ts_reduce_expect_xy(c, alpha, j, out));
}

int ts_expect_all(ts_ctx* c, int alpha, double* out)
{
    if (!c || !out || alpha < TS_X || alpha > TS_Z) return TS_ERR_ARG;
    if (!c->psi) return TS_ERR_NOSTATE;
    if (alpha == TS_Z) return cuda_status(ts_reduce_expect_z_all(c, out));
    for (int j = 0; j < c->N; ++j) {
        cudaError_t e = ts_reduce_expect_xy(c, alpha, j, out + j);
        if (e != cudaSuccess) return cuda_status(e);
    }
    return TS_OK;
}

int ts_norm2(ts_ctx* c, double* out)
{
    if (!c || !out) return TS_ERR_ARG;
    if (!c->psi) return TS_ERR_NOSTATE;
    return cuda_status(ts_reduce_norm2(c, out));
}

int ts_overlap(ts_ctx* c, const void* dev_phi, double* out)
{
    if (!c || !out || !dev_phi) return TS_ERR_ARG;
    if (!c->psi) return TS_ERR_NOSTATE;
    return cuda_status(ts_reduce_overlap(c, (const double2*)dev_phi, out));
}

int ts_set_profiling(ts_ctx* c, int enable)
{
    if (!c) return TS_ERR_ARG;
    c->profiling = enable ? 1 : 0;
    return TS_OK;
}

int ts_get_profile(ts_ctx* c, int64_t* launches, double* ms)
{
    if (!c || !launches || !ms) return TS_ERR_ARG;
    cudaError_t e = cudaStreamSynchronize(c->stream);
    if (e != cudaSuccess) return cuda_status(e);
    for (auto& r : c->recs) {
        float f = 0.f;
        if (cudaEventElapsedTime(&f, r.e0, r.e1) == cudaSuccess) c->ms_acc[r.kc] += f;
        else cudaGetLastError();
        c->ev_pool.push_back(r.e0);
        c->ev_pool.push_back(r.e1);
    }
    c->recs.clear();
    for (int k = 0; k < TS_KC_COUNT; ++k) { launches[k] = c->launches[k]; ms[k] = c->ms_acc[k]; }
    return TS_OK;
}

int ts_reset_profile(ts_ctx* c)
{
    if (!c) return TS_ERR_ARG;
    int64_t l[TS_KC_COUNT]; double m[TS_KC_COUNT];
    int st = ts_get_profile(c, l, m);      // drains pending records
    memset(c->launches, 0, sizeof(c->launches));
    memset(c->ms_acc, 0, sizeof(c->ms_acc));
    return st;
}

} // extern "C"
