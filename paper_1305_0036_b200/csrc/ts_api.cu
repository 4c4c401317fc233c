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
    c->use_small = 0;
    const int N = c->N;
    int mode = c->plan_mode;
    if (mode == TS_PLAN_AUTO) {
        if (N <= TS_SMALL_MAX_N && c->opt_small) { c->use_small = 1; return TS_OK; }
        mode = (N >= TS_TILE_LOG2) ? TS_PLAN_TILED : TS_PLAN_NAIVE;
    }
    if (mode == TS_PLAN_NAIVE) return TS_OK;
    if (N < TS_TILE_LOG2) return TS_ERR_ARG;
    TileGroup A; A.s = TS_TILE_LOG2; A.g0 = TS_TILE_LOG2; A.is_low = 1;
    c->groups.push_back(A);
    const int rem = N - TS_TILE_LOG2;
    std::vector<int> bits;
    if (!c->explicit_groups.empty()) {
        // ts_set_plan_groups: the caller (tests, the tuner, a plan file) names the bits of every high group
        int sum = 0;
        for (int mg : c->explicit_groups) {
            if (mg < 1 || mg > TS_TILE_LOG2 - 1) return TS_ERR_ARG;
            sum += mg;
        }
        if (sum != rem) return TS_ERR_ARG;
        bits = c->explicit_groups;
    } else if (rem > 0) {
        const int s_min = c->run_bits > 0 ? c->run_bits : 3;
        if (s_min < 1 || s_min > TS_TILE_LOG2 - 1) return TS_ERR_ARG;
        int mgmax = TS_TILE_LOG2 - s_min;
        if (c->max_group_bits > 0 && c->max_group_bits < mgmax) mgmax = c->max_group_bits;
        int left = rem;
        if (c->run_bits == 0 && c->max_group_bits == 0 && rem == 2 * (mgmax + 1)) {
            // N = 32: two groups of TEN bits (64-byte runs, no L2-blocked launch: the chunk would be 64 MiB) beat 9 + 6 + 5
            // with its extra tile pass per sweep: 1 272 vs 1 392 ms per step (profiles/r02_ab_and_sizes.md)
            bits.push_back(mgmax + 1);
            bits.push_back(mgmax + 1);
            left = 0;
        } else if (c->run_bits == 0 && c->max_group_bits == 0 && rem > mgmax) {
            // default plan: the group right above A takes as many bits as a pass can (9), so that A + that group is a
            // 32-MiB chunk the L2-blocked triple launch keeps on chip (ts_tile_v2.cuh) at every N >= 22 ...
            bits.push_back(mgmax);
            left -= mgmax;
        }
        // ... and the bits above are split evenly: the longest runs for every remaining pass.  One bit too
        // many for a single group (N = 31) is still ONE group, with 64-byte runs: measured 597 vs 673 ms per step against
        // two groups of five (profiles/r02_ab_and_sizes.md) -- a tile pass more per sweep costs more than short runs do.
        const bool ten = (c->run_bits == 0 && c->max_group_bits == 0 && left == mgmax + 1);
        const int ng = left == 0 ? 0 : ten ? 1 : (left + mgmax - 1) / mgmax;
        for (int i = 0; i < ng; ++i) bits.push_back(left / ng + (i < left % ng ? 1 : 0));
    }
    int g0 = TS_TILE_LOG2;
    for (int mg : bits) {
        TileGroup g; g.s = TS_TILE_LOG2 - mg; g.g0 = g0; g.is_low = 0;
        c->groups.push_back(g);
        g0 += mg;
    }
    return TS_OK;
}

bool tiled(const ts_ctx* c) { return !c->groups.empty(); }

int env_int(const char* name, int dflt)
{
    const char* v = getenv(name);
    return v ? atoi(v) : dflt;
}

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

// The executable graph of the last graph-mode call is destroyed once its replays have completed.
void graph_release(ts_ctx* c)
{
    if (!c->g_exec) return;
    if (c->g_done) cudaEventSynchronize(c->g_done);
    cudaGraphExecDestroy(c->g_exec);
    c->g_exec = nullptr;
}

// ---- the tiled path's launch stream -------------------------------------------------------------------------------
// Passes are generated sweep by sweep (the paper's runs are 5e5 .. 5e6 steps: no list of them is ever
// materialised for a long run) and emitted through a three-entry window in which the pattern
//     [H1 single ka] [A fused ka . D . kb] [H1 single kb]   ->   one L2-blocked launch (ts_tile_v2.cuh)
// is recognised.  A command is one launch: a tile pass or a triple launch.
struct Cmd {
    int triple;        // 1: ts_tile_chunk_triple(gi, k1, d, k2), 0: ts_tile_pass(gi, k1, d or none, k2)
    int gi, k1, k2;
    DiagOp d;
    bool operator==(const Cmd& o) const
    {
        return triple == o.triple && gi == o.gi && k1 == o.k1 && k2 == o.k2 && d.present == o.d.present &&
               (!d.present || (d.alpha == o.d.alpha && d.t == o.d.t && d.scale_pow == o.d.scale_pow));
    }
};

template <class Emit>
cudaError_t generate(ts_ctx* c, const Seq& q, Emit&& emit)
{
    struct Pass { int gi, k1, k2; DiagOp d; };
    const int g = (int)c->groups.size();
    int64_t sweep = 1;                 // next sweep to expand
    int pos = 0;                       // next position within it
    Pass win[4];
    int nwin = 0;
    cudaError_t e = cudaSuccess;
    auto refill = [&]() {
        while (nwin < 3 && sweep <= q.M) {
            const int64_t i = sweep;
            Pass ps; ps.d.present = 0; ps.gi = 0; ps.k1 = SW_NONE; ps.k2 = SW_NONE;
            bool out = true;
            if (g == 1) {
                if (pos == 0) { ps.d = q.diag(i - 1); ps.k2 = q.kind(i); }
                else { ps.d = q.diag(q.M); }                                // trailing diagonal after the last sweep
                ++pos;
                if (pos > (i == q.M ? 1 : 0)) { ++sweep; pos = 0; }
            } else {
                const bool fwd = (i & 1);
                const bool first = (pos == 0), last = (pos == g - 1);
                ps.gi = fwd ? pos : g - 1 - pos;
                if (first && i > 1) out = false;                               // done by the previous fused pass
                else if (last && i < q.M) { ps.k1 = q.kind(i); ps.d = q.diag(i); ps.k2 = q.kind(i + 1); }
                else if (first && i == 1) { ps.d = q.diag(0); ps.k2 = q.kind(1); }
                else if (last && i == q.M) { ps.k1 = q.kind(i); ps.d = q.diag(q.M); }
                else ps.k1 = q.kind(i);
                if (++pos == g) { ++sweep; pos = 0; }
            }
            if (out) win[nwin++] = ps;
        }
    };
    for (;;) {
        refill();
        if (nwin == 0 || e != cudaSuccess) break;
        int used = 1;
        Cmd cmd;
        if (nwin >= 3) {
            const Pass &p0 = win[0], &p1 = win[1], &p2 = win[2];
            if (p0.gi == p2.gi && p1.gi == 0 && p0.k2 == SW_NONE && !p0.d.present && p2.k2 == SW_NONE && !p2.d.present &&
                p1.d.present && p1.k1 == p0.k1 && p1.k2 == p2.k1 && ts_tile_chunk_supported(c, p0.gi, p1.k1, p1.k2)) {
                cmd.triple = 1; cmd.gi = p0.gi; cmd.k1 = p1.k1; cmd.k2 = p1.k2; cmd.d = p1.d;
                used = 3;
            }
        }
        if (used == 1) { cmd.triple = 0; cmd.gi = win[0].gi; cmd.k1 = win[0].k1; cmd.k2 = win[0].k2; cmd.d = win[0].d; }
        e = emit(cmd);
        for (int k = used; k < nwin; ++k) win[k - used] = win[k];
        nwin -= used;
    }
    return e;
}

cudaError_t execute(ts_ctx* c, const Cmd& cmd)
{
    if (cmd.triple) return ts_tile_chunk_triple(c, cmd.gi, cmd.k1, cmd.d, cmd.k2);
    return ts_tile_pass(c, cmd.gi, cmd.k1, cmd.d.present ? &cmd.d : nullptr, cmd.k2);
}

bool coop_refused(cudaError_t e)
{
    return e == cudaErrorCooperativeLaunchTooLarge || e == cudaErrorLaunchOutOfResources || e == cudaErrorNotSupported;
}

// Small, L2-resident states are launch-bound (a tile pass at N = 16 lasts ~5 us, the gap between two
// dependent launches about as long).  The launch stream of a run is periodic, head + unit x (n - 2) + tail with `unit` =
// one 4th-order step, so the unit is captured ONCE into a CUDA graph and replayed.  The decomposition is found by
// generating the streams of 2, 3 and 4 steps on the host and is checked on the 4-step stream before it is trusted.
bool split_periodic(ts_ctx* c, const Seq& q, std::vector<Cmd>& head, std::vector<Cmd>& unit, std::vector<Cmd>& tail)
{
    std::vector<Cmd> L[3];
    for (int k = 0; k < 3; ++k) {
        const Seq qk(q.order, q.N, q.tau, 2 + k);
        if (generate(c, qk, [&](const Cmd& cmd) { L[k].push_back(cmd); return cudaSuccess; }) != cudaSuccess) return false;
    }
    if (L[1].size() <= L[0].size() || L[2].size() - L[1].size() != L[1].size() - L[0].size()) return false;
    const size_t P = L[1].size() - L[0].size();
    size_t S = 0;                                       // common suffix of the 2- and 3-step streams
    while (S < L[0].size() && L[0][L[0].size() - 1 - S] == L[1][L[1].size() - 1 - S]) ++S;
    if (S == 0 || S >= L[0].size()) return false;
    const size_t H = L[0].size() - S;
    head.assign(L[0].begin(), L[0].begin() + H);
    tail.assign(L[0].begin() + H, L[0].end());
    unit.assign(L[1].begin() + H, L[1].begin() + H + P);
    std::vector<Cmd> check(head);                       // head + unit + unit + tail must be the 4-step stream
    check.insert(check.end(), unit.begin(), unit.end());
    check.insert(check.end(), unit.begin(), unit.end());
    check.insert(check.end(), tail.begin(), tail.end());
    if (check.size() != L[2].size()) return false;
    for (size_t k = 0; k < check.size(); ++k) if (!(check[k] == L[2][k])) return false;
    return true;
}

int evolve_tiled(ts_ctx* c, const Seq& q)
{
    cudaError_t e = cudaSuccess;
    auto run = [&](const Cmd& cmd) -> cudaError_t {
        cudaError_t r = execute(c, cmd);
        if (cmd.triple && coop_refused(r)) {
            // not all CTAs can be co-resident here (MPS, a shared GPU): run the three passes one by one from now on
            cudaGetLastError();
            c->opt_chunk = 0;
            r = ts_tile_pass(c, cmd.gi, cmd.k1, nullptr, SW_NONE);
            if (r == cudaSuccess) r = ts_tile_pass(c, 0, cmd.k1, &cmd.d, cmd.k2);
            if (r == cudaSuccess) r = ts_tile_pass(c, cmd.gi, cmd.k2, nullptr, SW_NONE);
        }
        return r;
    };
    const int64_t n_steps = q.n_sub / (q.order == 4 ? 5 : 1);
    const bool graph_ok = c->opt_graph && !c->profiling && c->N <= c->opt_graph_max_n && n_steps >= 4;
    std::vector<Cmd> head, unit, tail;
    if (graph_ok && split_periodic(c, q, head, unit, tail)) {
        for (const Cmd& cmd : head) { e = run(cmd); if (e != cudaSuccess) return cuda_status(e); }
        // every phase table of the unit exists before the capture starts (building one allocates and launches)
        c->dry_run = 1;
        for (const Cmd& cmd : unit) { e = execute(c, cmd); if (e != cudaSuccess) break; }
        c->dry_run = 0;
    c->top_bits_only = 0;
        if (e != cudaSuccess) return cuda_status(e);
        graph_release(c);
        int64_t l0[TS_KC_COUNT]; double t0[TS_KC_COUNT];
        memcpy(l0, c->launches, sizeof(l0)); memcpy(t0, c->tiles_acc, sizeof(t0));
        cudaGraph_t graph = nullptr;
        cudaGraphExec_t gexec = nullptr;
        bool captured = false;
        // capture on a stream of our own (the caller's may be the legacy default stream, which cannot be captured); nothing
        // runs there: the graph is launched into the caller's stream
        cudaStream_t user = c->stream;
        if (!c->g_stream && cudaStreamCreateWithFlags(&c->g_stream, cudaStreamNonBlocking) != cudaSuccess) c->g_stream = nullptr;
        if (c->g_stream && cudaStreamBeginCapture(c->g_stream, cudaStreamCaptureModeThreadLocal) == cudaSuccess) {
            c->stream = c->g_stream;
            cudaError_t ce = cudaSuccess;
            for (const Cmd& cmd : unit) { ce = execute(c, cmd); if (ce != cudaSuccess) break; }
            cudaError_t ee = cudaStreamEndCapture(c->g_stream, &graph);
            c->stream = user;
            if (ce == cudaSuccess && ee == cudaSuccess && graph && cudaGraphInstantiate(&gexec, graph, 0) == cudaSuccess)
                captured = true;
        }
        cudaGetLastError();
        if (graph) cudaGraphDestroy(graph);
        int64_t left = n_steps - 2;
        if (captured) {
            // the capture went through the launchers once: count its launches once per replay
            for (int k = 0; k < TS_KC_COUNT; ++k) {
                c->launches[k] = l0[k] + (c->launches[k] - l0[k]) * left;
                c->tiles_acc[k] = t0[k] + (c->tiles_acc[k] - t0[k]) * (double)left;
            }
            c->graph_replays += left;
            for (; left > 0 && e == cudaSuccess; --left) e = cudaGraphLaunch(gexec, c->stream);
            c->g_exec = gexec;
            if (!c->g_done) cudaEventCreateWithFlags(&c->g_done, cudaEventDisableTiming);
            if (c->g_done) cudaEventRecord(c->g_done, c->stream);
        } else {
            memcpy(c->launches, l0, sizeof(l0)); memcpy(c->tiles_acc, t0, sizeof(t0));
            if (gexec) cudaGraphExecDestroy(gexec);
        }
        for (; left > 0 && e == cudaSuccess; --left)  // capture refused: the same launches, one by one
            for (const Cmd& cmd : unit) { e = run(cmd); if (e != cudaSuccess) break; }
        for (const Cmd& cmd : tail) { if (e != cudaSuccess) break; e = run(cmd); }
        return cuda_status(e);
    }
    e = generate(c, q, run);
    return cuda_status(e);
}

} // namespace

void ts_prof_begin(ts_ctx* c, int kc, double state_passes)
{
    c->launches[kc]++;
    c->tiles_acc[kc] += state_passes;
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

const char* ts_version(void) { return "ts_b200 0.3 sm_100a tile=2^12 regs=32amp/thread kernels=v2(tma-in/out,warp-specialised,ticket-scheduled)+v1"; }

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
    c->e0[0] = c->e0[1] = c->e0[2] = 0.0;
    for (int a = 0; a < 3; ++a) {
        for (int j = 0; j < N; ++j) c->h[a][j] = h[a * N + j];
        for (int j = 0; j < N; ++j)
            for (int k = 0; k < N; ++k)
                if (j != k) c->Jeff[a][j][k] = J[((size_t)a * N + j) * N + k] + J[((size_t)a * N + k) * N + j];
    }
    c->psi = nullptr; c->owns_psi = 0;
    c->plan_mode = TS_PLAN_AUTO; c->run_bits = 0; c->max_group_bits = 0;
    // execution options: defaults, overridable once per context from the environment (A/B runs of bench.py) and at
    // any time through ts_set_option
    c->opt_kernel = env_int("TS_KERNEL", 2);
    c->opt_chunk = env_int("TS_CHUNK3", 1);
    c->opt_chunk_max_log2 = env_int("TS_CHUNK3_MAX_LOG2", 21);
    c->opt_chunk_min_log2 = env_int("TS_CHUNK3_MIN_LOG2", 21);
    c->opt_small = env_int("TS_SMALL", 1);
    c->opt_diag_source = 0;
    c->opt_l2_promotion = env_int("TS_L2_PROMOTION", 0);
    c->opt_max_ctas = 0;
    c->opt_l2_hints = env_int("TS_L2_HINTS", 1);
    c->opt_pair = env_int("TS_PAIR", 1);
    c->opt_graph = env_int("TS_GRAPH", 1);
    c->opt_graph_max_n = 21;
    c->dry_run = 0;
    c->top_bits_only = 0;
    c->g_exec = nullptr; c->g_done = nullptr; c->g_stream = nullptr; c->d_row_ctr = nullptr;
    c->graph_replays = 0;
    c->opt_probe = 0;
    c->opt_groups = env_int("TS_GROUPS", 2);
    if (c->opt_groups < 1 || c->opt_groups > 2) c->opt_groups = 2;
    c->d_chunk_ctr = nullptr; c->chunk_ctr_cap = 0;
    c->d_sched = nullptr;
    c->d_energy[0] = c->d_energy[1] = c->d_energy[2] = nullptr;
    c->tmap_psi = nullptr;
    c->d_red = nullptr; c->red_cap = 0;
    c->d_trace = nullptr; c->trace_cap = 0;
    c->profiling = 0;
    memset(c->launches, 0, sizeof(c->launches));
    memset(c->ms_acc, 0, sizeof(c->ms_acc));
    memset(c->tiles_acc, 0, sizeof(c->tiles_acc));
    if (cudaDeviceGetAttribute(&c->num_sms, cudaDevAttrMultiProcessorCount, c->device) != cudaSuccess || c->num_sms < 1) {
        cudaGetLastError(); delete c; return TS_ERR_CUDA;
    }
    cudaError_t e = cudaMalloc(&c->d_h, sizeof(c->h));
    if (e == cudaSuccess) e = cudaMalloc(&c->d_Jeff, sizeof(c->Jeff));
    if (e == cudaSuccess) e = cudaMemcpy(c->d_h, c->h, sizeof(c->h), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(c->d_Jeff, c->Jeff, sizeof(c->Jeff), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMalloc(&c->d_sched, 8 * sizeof(unsigned int));     // [0..1] tickets, [2..5] clock probe
    if (e == cudaSuccess) e = cudaMemset(c->d_sched, 0, 8 * sizeof(unsigned int));   // kernels leave the tickets at zero
    if (e == cudaSuccess) e = ts_tile_init();
    if (e == cudaSuccess) e = ts_small_init();
    if (e != cudaSuccess) { cudaGetLastError(); ts_destroy(c); return cuda_status(e); }
    int st = build_plan(c);
    if (st != TS_OK) { ts_destroy(c); return st; }
    const char* pf = getenv("TS_PLAN_FILE");       // a tuned plan (paper_1305_0036_b200/tuner.py) for this size, if any
    if (pf && *pf) {
        st = ts_load_plan_file(c, pf);
        if (st != TS_OK) { ts_destroy(c); return st; }
    }
    *out = c;
    return TS_OK;
}

int ts_destroy(ts_ctx* c)
{
    if (!c) return TS_OK;
    graph_release(c);
    if (c->g_done) cudaEventDestroy(c->g_done);
    if (c->g_stream) cudaStreamDestroy(c->g_stream);
    if (c->d_row_ctr) cudaFree(c->d_row_ctr);
    if (c->psi && c->owns_psi) cudaFree(c->psi);
    if (c->d_h) cudaFree(c->d_h);
    if (c->d_Jeff) cudaFree(c->d_Jeff);
    ts_tile_free_tables(c);
    ts_naive_free_stored(c);
    if (c->d_red) cudaFree(c->d_red);
    if (c->d_chunk_ctr) cudaFree(c->d_chunk_ctr);
    if (c->d_sched) cudaFree(c->d_sched);
    if (c->d_trace) cudaFree(c->d_trace);
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
    const std::vector<int> oeg = c->explicit_groups;
    c->plan_mode = mode; c->run_bits = run_bits; c->max_group_bits = max_group_bits;
    c->explicit_groups.clear();
    cudaStreamSynchronize(c->stream);
    ts_tile_free_tables(c);          // tables depend on the group geometry
    c->tmaps.clear();
    int st = build_plan(c);
    if (st != TS_OK) { c->plan_mode = om; c->run_bits = orb; c->max_group_bits = omg; c->explicit_groups = oeg; build_plan(c); }
    return st;
}

int ts_set_plan_groups(ts_ctx* c, int n_high, const int* high_bits)
{
    if (!c || n_high < 0 || (n_high > 0 && !high_bits) || c->N < TS_TILE_LOG2) return TS_ERR_ARG;
    if ((n_high == 0) != (c->N == TS_TILE_LOG2)) return TS_ERR_ARG;
    const int om = c->plan_mode;
    const std::vector<int> oeg = c->explicit_groups;
    c->plan_mode = TS_PLAN_TILED;
    c->explicit_groups.assign(high_bits, high_bits + n_high);
    cudaStreamSynchronize(c->stream);
    ts_tile_free_tables(c);
    c->tmaps.clear();
    int st = build_plan(c);
    if (st != TS_OK) { c->plan_mode = om; c->explicit_groups = oeg; build_plan(c); }
    return st;
}

int ts_set_option(ts_ctx* c, int key, int value)
{
    if (!c) return TS_ERR_ARG;
    switch (key) {
    case TS_OPT_KERNEL: if (value < 0 || value > 2) return TS_ERR_ARG; c->opt_kernel = value; break;
    case TS_OPT_CHUNK: if (value < 0 || value > 1) return TS_ERR_ARG; c->opt_chunk = value; break;
    case TS_OPT_CHUNK_MAX_LOG2: if (value < TS_TILE_LOG2 + 1 || value > 26) return TS_ERR_ARG; c->opt_chunk_max_log2 = value; break;
    case TS_OPT_L2_PROMOTION: if (value < 0 || value > 2) return TS_ERR_ARG; c->opt_l2_promotion = value; c->tmaps.clear(); break;
    case TS_OPT_MAX_CTAS: if (value < 0) return TS_ERR_ARG; c->opt_max_ctas = value; break;
    case TS_OPT_L2_HINTS: if (value < 0 || value > 1) return TS_ERR_ARG; c->opt_l2_hints = value; break;
    case TS_OPT_PAIR: if (value < 0 || value > 1) return TS_ERR_ARG; c->opt_pair = value; break;
    case TS_OPT_GRAPH: if (value < 0 || value > 1) return TS_ERR_ARG; c->opt_graph = value; break;
    case TS_OPT_GRAPH_MAX_N: if (value < TS_TILE_LOG2 || value > TS_MAX_N) return TS_ERR_ARG; c->opt_graph_max_n = value; break;
    case TS_OPT_CHUNK_MIN_LOG2: if (value < TS_TILE_LOG2 + 1 || value > 26) return TS_ERR_ARG; c->opt_chunk_min_log2 = value; break;
    case TS_OPT_PROBE: if (value < 0 || value > 3) return TS_ERR_ARG; c->opt_probe = value; break;
    case TS_OPT_DIAG_SOURCE:
        if (value < 0 || value > 1) return TS_ERR_ARG;
        c->opt_diag_source = value;
        if (!value) { cudaStreamSynchronize(c->stream); ts_naive_free_stored(c); }
        break;
    case TS_OPT_SMALL:
        if (value < 0 || value > 1) return TS_ERR_ARG;
        c->opt_small = value;
        cudaStreamSynchronize(c->stream);
        ts_tile_free_tables(c);
        c->tmaps.clear();
        return build_plan(c);
    default: return TS_ERR_ARG;
    }
    // phase tables are keyed by the kernel family that reads them, so nothing cached goes stale
    return TS_OK;
}

int ts_get_option(ts_ctx* c, int key, int* value)
{
    if (!c || !value) return TS_ERR_ARG;
    switch (key) {
    case TS_OPT_KERNEL: *value = c->opt_kernel; break;
    case TS_OPT_CHUNK: *value = c->opt_chunk; break;
    case TS_OPT_CHUNK_MAX_LOG2: *value = c->opt_chunk_max_log2; break;
    case TS_OPT_L2_PROMOTION: *value = c->opt_l2_promotion; break;
    case TS_OPT_SMALL: *value = c->opt_small; break;
    case TS_OPT_DIAG_SOURCE: *value = c->opt_diag_source; break;
    case TS_OPT_MAX_CTAS: *value = c->opt_max_ctas; break;
    case TS_OPT_L2_HINTS: *value = c->opt_l2_hints; break;
    case TS_OPT_PAIR: *value = c->opt_pair; break;
    case TS_OPT_GRAPH: *value = c->opt_graph; break;
    case TS_OPT_GRAPH_MAX_N: *value = c->opt_graph_max_n; break;
    case TS_OPT_LAST_LAUNCH_KHZ: {
        // effective SM clock of the last persistent tile launch: cycles / nanoseconds seen by CTA 0's loader (synchronises)
        unsigned long long v[2] = {0, 0};
        if (cudaStreamSynchronize(c->stream) != cudaSuccess ||
            cudaMemcpy(v, c->d_sched + 2, sizeof(v), cudaMemcpyDeviceToHost) != cudaSuccess) { cudaGetLastError(); return TS_ERR_CUDA; }
        *value = v[1] ? (int)((double)v[0] / (double)v[1] * 1e6) : 0;
        break;
    }
    case TS_OPT_GRAPH_REPLAYS: *value = (int)(c->graph_replays > 0x7fffffff ? 0x7fffffff : c->graph_replays); break;
    case TS_OPT_CHUNK_MIN_LOG2: *value = c->opt_chunk_min_log2; break;
    case TS_OPT_PROBE: *value = c->opt_probe; break;
    default: return TS_ERR_ARG;
    }
    return TS_OK;
}

// Plan file (the tuned sequence of rotations per N "stored in a file"): text, one line per system size,
//     N=30 groups=9,9 kernel=1 chunk=1 chunk_max_log2=21 chunk_min_log2=21 l2_promotion=0
// `groups` = bits of every high group, bottom to top (ts_set_plan_groups); the other keys are ts_set_option values and
// may be omitted.  Lines starting with '#' are comments.  Returns TS_OK and leaves the context untouched when the file
// has no line for this N.
int ts_load_plan_file(ts_ctx* c, const char* path)
{
    if (!c || !path) return TS_ERR_ARG;
    FILE* f = fopen(path, "r");
    if (!f) return TS_ERR_ARG;
    char line[512];
    int st = TS_OK;
    while (fgets(line, sizeof line, f)) {
        if (line[0] == '#') continue;
        int n = -1;
        std::vector<int> groups;
        int kernel = -1, chunk = -1, cmax = -1, cmin = -1, prom = -1;
        bool have_groups = false;
        for (char* tok = strtok(line, " \t\r\n"); tok; tok = strtok(nullptr, " \t\r\n")) {
            if (!strncmp(tok, "N=", 2)) n = atoi(tok + 2);
            else if (!strncmp(tok, "groups=", 7)) {
                have_groups = true;
                for (const char* p = tok + 7; *p;) {
                    groups.push_back(atoi(p));
                    while (*p && *p != ',') ++p;
                    if (*p == ',') ++p;
                }
            }
            else if (!strncmp(tok, "kernel=", 7)) kernel = atoi(tok + 7);
            else if (!strncmp(tok, "chunk=", 6)) chunk = atoi(tok + 6);
            else if (!strncmp(tok, "chunk_max_log2=", 15)) cmax = atoi(tok + 15);
            else if (!strncmp(tok, "chunk_min_log2=", 15)) cmin = atoi(tok + 15);
            else if (!strncmp(tok, "l2_promotion=", 13)) prom = atoi(tok + 13);
        }
        if (n != c->N) continue;
        if (kernel >= 0 && st == TS_OK) st = ts_set_option(c, TS_OPT_KERNEL, kernel);
        if (chunk >= 0 && st == TS_OK) st = ts_set_option(c, TS_OPT_CHUNK, chunk);
        if (cmax >= 0 && st == TS_OK) st = ts_set_option(c, TS_OPT_CHUNK_MAX_LOG2, cmax);
        if (cmin >= 0 && st == TS_OK) st = ts_set_option(c, TS_OPT_CHUNK_MIN_LOG2, cmin);
        if (prom >= 0 && st == TS_OK) st = ts_set_option(c, TS_OPT_L2_PROMOTION, prom);
        if (have_groups && st == TS_OK && c->N >= TS_TILE_LOG2 + 1) st = ts_set_plan_groups(c, (int)groups.size(), groups.data());
        break;
    }
    fclose(f);
    return st;
}

int ts_describe_plan(ts_ctx* c, char* buf, int buflen)
{
    if (!c || !buf || buflen < 1) return TS_ERR_ARG;
    std::string s;
    char tmp[128];
    if (c->use_small) {
        snprintf(tmp, sizeof tmp, "small: N=%d, one CTA, state and energy tables in shared memory, one launch per ts_evolve", c->N);
        s = tmp;
    } else if (!tiled(c)) {
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
        snprintf(tmp, sizeof tmp, "; kernels=%s", ts_tile_layout_for(c, 0, SW_YDAG, SW_Y) ? "v2" : "v1");
        s += tmp;
        if (ts_tile_chunk_supported(c, 1, SW_YDAG, SW_Y)) {
            const TileGroup& t = c->groups[1];
            snprintf(tmp, sizeof tmp, "; L2-blocked triple launch on chunks of 2^%d", t.g0 + TS_TILE_LOG2 - t.s);
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

    if (c->use_small) return cuda_status(ts_small_evolve(c, tau, n_steps, order));
    if (!tiled(c)) {
        e = ts_naive_diag(c, q.diag(0));
        for (int64_t i = 1; i <= q.M && e == cudaSuccess; ++i) {
            for (int j = 0; j < c->N && e == cudaSuccess; ++j) e = ts_naive_rotate(c, j, q.kind(i));
            if (e == cudaSuccess) e = ts_naive_diag(c, q.diag(i));
        }
        return cuda_status(e);
    }

    return evolve_tiled(c, q);
}

int ts_evolve_observe(ts_ctx* c, double tau, int64_t n_steps, int order, int alpha, int j, double* out)
{
    if (!c || !out || !isfinite(tau) || n_steps < 0 || (order != 2 && order != 4) || alpha < TS_X || alpha > TS_Z) return TS_ERR_ARG;
    if (alpha == TS_Z ? (j < -1 || j >= c->N) : (j < 0 || j >= c->N)) return TS_ERR_ARG;
    if (!c->psi) return TS_ERR_NOSTATE;
    if (n_steps == 0) return TS_OK;
    cudaError_t e = cudaSuccess;
    const size_t need = (size_t)TS_TRACE_STRIDE * (size_t)n_steps;
    if (c->trace_cap < need) {
        if (c->d_trace) { cudaStreamSynchronize(c->stream); cudaFree(c->d_trace); }
        c->d_trace = nullptr; c->trace_cap = 0;
        e = cudaMalloc(&c->d_trace, sizeof(double) * need);
        if (e != cudaSuccess) { cudaGetLastError(); return TS_ERR_NOMEM; }
        c->trace_cap = need;
    }
    double* d_trace = c->d_trace;
    int st = TS_OK;
    int64_t k = 0;
    // Small states (launch-bound): the first step runs launch by launch (it builds every phase table and the
    // reduction scratch), then [one step + the row's reduction] is captured once and replayed; the row index lives on
    // the device and advances with every replay.
    if (c->opt_graph && !c->profiling && c->N <= c->opt_graph_max_n && n_steps >= 4) {
        st = ts_evolve(c, tau, 1, order);
        if (st == TS_OK) st = cuda_status(ts_reduce_trace_row(c, alpha, j < 0 ? 0 : j, d_trace));
        k = 1;
        if (st == TS_OK && !c->d_row_ctr && cudaMalloc(&c->d_row_ctr, sizeof(unsigned int)) != cudaSuccess) { cudaGetLastError(); c->d_row_ctr = nullptr; }
        if (st == TS_OK && c->d_row_ctr) {
            graph_release(c);
            cudaStream_t user = c->stream;
            cudaGraph_t graph = nullptr;
            cudaGraphExec_t gexec = nullptr;
            int64_t l0[TS_KC_COUNT]; double t0[TS_KC_COUNT];
            memcpy(l0, c->launches, sizeof(l0)); memcpy(t0, c->tiles_acc, sizeof(t0));
            bool captured = false;
            if (!c->g_stream && cudaStreamCreateWithFlags(&c->g_stream, cudaStreamNonBlocking) != cudaSuccess) c->g_stream = nullptr;
            if (c->g_stream && cudaStreamBeginCapture(c->g_stream, cudaStreamCaptureModeThreadLocal) == cudaSuccess) {
                c->stream = c->g_stream;
                int cs = ts_evolve(c, tau, 1, order);
                if (cs == TS_OK) cs = cuda_status(ts_reduce_trace_row(c, alpha, j < 0 ? 0 : j, d_trace, c->d_row_ctr));
                cudaError_t ee = cudaStreamEndCapture(c->g_stream, &graph);
                c->stream = user;
                if (cs == TS_OK && ee == cudaSuccess && graph && cudaGraphInstantiate(&gexec, graph, 0) == cudaSuccess) captured = true;
            }
            cudaGetLastError();
            if (graph) cudaGraphDestroy(graph);
            if (captured) {
                const int64_t left = n_steps - 1;
                for (int q = 0; q < TS_KC_COUNT; ++q) {
                    c->launches[q] = l0[q] + (c->launches[q] - l0[q]) * left;
                    c->tiles_acc[q] = t0[q] + (c->tiles_acc[q] - t0[q]) * (double)left;
                }
                cudaError_t e2 = ts_set_u32(c, c->d_row_ctr, 1u);
                for (; k < n_steps && e2 == cudaSuccess; ++k) e2 = cudaGraphLaunch(gexec, c->stream);
                c->graph_replays += left;
                c->g_exec = gexec;
                if (!c->g_done) cudaEventCreateWithFlags(&c->g_done, cudaEventDisableTiming);
                if (c->g_done) cudaEventRecord(c->g_done, c->stream);
                st = cuda_status(e2);
            } else {
                memcpy(c->launches, l0, sizeof(l0)); memcpy(c->tiles_acc, t0, sizeof(t0));
                if (gexec) cudaGraphExecDestroy(gexec);
            }
        }
    }
    for (; k < n_steps && st == TS_OK; ++k) {
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
    if (tiled(c))       // one pass per bit group of the plan (every tile holds both members of the group's pairs)
        return cuda_status(ts_reduce_expect_xy_all(c, alpha == TS_X ? out : nullptr, alpha == TS_Y ? out : nullptr));
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

int ts_correlate(ts_ctx* c, int alpha, int j, int k, double* out)
{
    if (!c || !out || alpha < TS_X || alpha > TS_Z || j < 0 || j >= c->N || k < 0 || k >= c->N || j == k) return TS_ERR_ARG;
    if (!c->psi) return TS_ERR_NOSTATE;
    return cuda_status(ts_reduce_corr(c, alpha, j, k, out));
}

int ts_total_sz(ts_ctx* c, double* out)
{
    if (!c || !out) return TS_ERR_ARG;
    if (!c->psi) return TS_ERR_NOSTATE;
    double v[TS_MAX_N];
    cudaError_t e = ts_reduce_expect_z_all(c, v);
    if (e != cudaSuccess) return cuda_status(e);
    double s = 0.0;
    for (int j = 0; j < c->N; ++j) s += v[j];
    *out = s;
    return TS_OK;
}

} // extern "C"

// One global rotation (sweep) of the state, optionally followed by the exact scaling 2^scale_pow: every group of the
// plan once (tiled), or one launch per spin (naive / small-N contexts).
cudaError_t ts_apply_sweep_all(ts_ctx* c, int kind, int scale_pow, int skip_last_group)
{
    cudaError_t e = cudaSuccess;
    DiagOp d; d.present = (scale_pow != 0); d.alpha = TS_Z; d.t = 0.0; d.scale_pow = scale_pow;
    if (!tiled(c)) {
        for (int j = 0; j < c->N && e == cudaSuccess; ++j) e = ts_naive_rotate(c, j, kind);
        if (e == cudaSuccess && d.present) e = ts_naive_diag(c, d);
        return e;
    }
    const int g = (int)c->groups.size() - (skip_last_group ? 1 : 0);      // (skipped: done by a fused pass before)
    for (int gi = 0; gi < g && e == cudaSuccess; ++gi)
        e = ts_tile_pass(c, gi, kind, (gi == g - 1 && d.present) ? &d : nullptr, SW_NONE);
    return e;
}

extern "C" {

int ts_energy(ts_ctx* c, double* out)
{
    if (!c || !out) return TS_ERR_ARG;
    if (!c->psi) return TS_ERR_NOSTATE;
    // <H> = <H_z> + <H_x> + <H_y>;  <psi|H_x|psi> = sum_k E_x(k) |(Y^dag psi)_k|^2 and <psi|H_y|psi> = sum_k E_y(k)
    // |(X^dag psi)_k|^2 (eq. 7, 10: P:81-84), the unnormalised sweeps carrying a factor 2^N in |.|^2.
    double ez = 0.0, ex = 0.0, ey = 0.0;
    cudaError_t e = ts_reduce_energy_diag(c, TS_Z, &ez);
    if (e == cudaSuccess) e = ts_apply_sweep_all(c, SW_YDAG, 0);
    if (e == cudaSuccess) e = ts_reduce_energy_diag(c, TS_X, &ex);
    if (e == cudaSuccess) e = ts_apply_sweep_all(c, SW_Y, -c->N);           // back: Y Y^dag = 2^N, removed exactly
    if (e == cudaSuccess) e = ts_apply_sweep_all(c, SW_XDAG, 0);
    if (e == cudaSuccess) e = ts_reduce_energy_diag(c, TS_Y, &ey);
    if (e == cudaSuccess) e = ts_apply_sweep_all(c, SW_X, -c->N);
    if (e != cudaSuccess) return cuda_status(e);
    const double sc = ldexp(1.0, -c->N);
    *out = ez + sc * (ex + ey);
    return TS_OK;
}

int ts_set_random_phase_state(ts_ctx* c, int up_spin, uint64_t seed)
{
    if (!c || up_spin < 0 || up_spin >= c->N) return TS_ERR_ARG;
    int st = ensure_state(c);
    if (st != TS_OK) return st;
    return cuda_status(ts_fill_random_phase(c, up_spin, seed));
}

int ts_loschmidt_echo(ts_ctx* c, double tau, int64_t n_steps, int order, double* out)
{
    if (!c || !out || !isfinite(tau) || n_steps < 0 || (order != 2 && order != 4)) return TS_ERR_ARG;
    if (!c->psi) return TS_ERR_NOSTATE;
    double2* psi0 = nullptr;
    const size_t bytes = sizeof(double2) << c->N;
    if (cudaMalloc(&psi0, bytes) != cudaSuccess) { cudaGetLastError(); return TS_ERR_NOMEM; }
    cudaError_t e = cudaMemcpyAsync(psi0, c->psi, bytes, cudaMemcpyDeviceToDevice, c->stream);
    int st = cuda_status(e);
    if (st == TS_OK) st = ts_evolve(c, tau, n_steps, order);
    if (st == TS_OK) st = ts_evolve(c, -tau, n_steps, order);
    double ov[2] = {0.0, 0.0};
    if (st == TS_OK) st = cuda_status(ts_reduce_overlap(c, psi0, ov));
    else cudaStreamSynchronize(c->stream);
    cudaFree(psi0);
    if (st != TS_OK) return st;
    out[0] = ov[0] * ov[0] + ov[1] * ov[1];
    out[1] = ov[0];
    out[2] = ov[1];
    return TS_OK;
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

int ts_get_profile_passes(ts_ctx* c, double* state_passes)
{
    if (!c || !state_passes) return TS_ERR_ARG;
    for (int k = 0; k < TS_KC_COUNT; ++k) state_passes[k] = c->tiles_acc[k];
    return TS_OK;
}

int ts_reset_profile(ts_ctx* c)
{
    if (!c) return TS_ERR_ARG;
    int64_t l[TS_KC_COUNT]; double m[TS_KC_COUNT];
    int st = ts_get_profile(c, l, m);      // drains pending records
    memset(c->launches, 0, sizeof(c->launches));
    memset(c->ms_acc, 0, sizeof(c->ms_acc));
    memset(c->tiles_acc, 0, sizeof(c->tiles_acc));
    return st;
}

} // extern "C"
