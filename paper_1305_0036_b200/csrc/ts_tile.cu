// ts_tile.cu -- launcher of the tile passes and construction of their phase tables.
// The kernel itself is in ts_tile_kernel.cuh; its instantiations are in ts_tile_cfg*.cu.
#include <math.h>
#include <string.h>

#include <cudaTypedefs.h>
#include <stdio.h>
#include <stdlib.h>

#include "ts_tile_chunk.cuh"
#include "ts_tile_pipe.cuh"

namespace {

tile_kernel_t g_tab[TS_CFG_COUNT][5][5];
pipe_kernel_t g_pipe[TS_CFG_COUNT][5][5];
chunk_kernel_t g_chunk[TS_CFG_COUNT][2];
chunk_pipe_kernel_t g_chunk_pipe[TS_CFG_COUNT][2];
bool g_registered = false;
int g_num_sms = 0;
PFN_cuTensorMapEncodeTiled_v12000 g_encode = nullptr;

// Geometry of the diagonal-time layout of one group: which spins sit on register bits (R), thread bits (T) and
// outside the tile (X).
struct PhaseGeom {
    double t;
    int N, nfixed;
    int rspin[5], tspin[7], xspin[TS_MAX_FIXED];
};

inline int spin_of_fbit(const TileGroup& g, int f) { return f < g.s ? f : g.g0 + (f - g.s); }
inline int n_bfly(const TileGroup& g) { return g.is_low ? TS_TILE_LOG2 : TS_TILE_LOG2 - g.s; }
inline bool two_stage(const TileGroup& g) { return n_bfly(g) > 5; }

int cfg_of(const TileGroup& g)
{
    if (g.is_low) return TS_CFG_A;
    switch (n_bfly(g)) {
    case 7: return TS_CFG_H7;
    case 8: return TS_CFG_H8;
    case 9: return TS_CFG_H9;
    case 10: return TS_CFG_H10;
    default: return TS_CFG_GENERIC;
    }
}

PhaseGeom make_geom(const ts_ctx* c, const TileGroup& g, double t)
{
    PhaseGeom q;
    q.t = t; q.N = c->N; q.nfixed = c->N - TS_TILE_LOG2;
    const bool two = two_stage(g);
    for (int b = 0; b < 5; ++b) q.rspin[b] = spin_of_fbit(g, two ? 2 + b : 7 + b);
    for (int b = 0; b < 7; ++b) {
        const int f = two ? (b < 2 ? b : 5 + b) : b;     // layout 2: thread bits 0,1 -> f 0,1; 2..6 -> f 7..11
        q.tspin[b] = spin_of_fbit(g, f);
    }
    bool in_tile[TS_MAX_N] = {false};
    for (int f = 0; f < TS_TILE_LOG2; ++f) in_tile[spin_of_fbit(g, f)] = true;
    int nx = 0;
    for (int i = 0; i < TS_MAX_FIXED; ++i) q.xspin[i] = 0;
    for (int j = 0; j < c->N; ++j) if (!in_tile[j]) q.xspin[nx++] = j;    // ascending = tile-index bit order
    return q;
}

// TT[v], WT[0..4][v] for thread index v (one block of 128 threads).
__global__ void __launch_bounds__(128) k_build_thread_tables(double2* __restrict__ out, const PhaseGeom q,
                                                             const double* __restrict__ h,
                                                             const double* __restrict__ Jeff)
{
    const int v = threadIdx.x;
    double sg[7];
    for (int b = 0; b < 7; ++b) sg[b] = (double)((v >> b) & 1) - 0.5;
    double ET = 0.0;                              // fields and couplings among the thread spins
    for (int b = 0; b < 7; ++b) {
        double f = h[q.tspin[b]];
        for (int c = 0; c < b; ++c) f += Jeff[q.tspin[b] * TS_MAX_N + q.tspin[c]] * sg[c];
        ET += sg[b] * f;
    }
    double bsum = 0.0;
    for (int i = 0; i < 5; ++i) {
        double bi = 0.0;
        for (int b = 0; b < 7; ++b) bi += Jeff[q.rspin[i] * TS_MAX_N + q.tspin[b]] * sg[b];
        bsum += bi;
        double sn, cs;
        sincos(-q.t * bi, &sn, &cs);
        out[128 + i * 128 + v] = make_double2(cs, sn);
    }
    double sn, cs;
    sincos(-q.t * (ET - 0.5 * bsum), &sn, &cs);
    out[v] = make_double2(cs, sn);
}

// Tile-phase table: 32 entries per tile (layout in ts_tile_kernel.cuh); one thread per entry.
__global__ void __launch_bounds__(256) k_build_tile_phase(double2* __restrict__ out, uint64_t ntiles,
                                                          const PhaseGeom q, const double* __restrict__ h,
                                                          const double* __restrict__ Jeff)
{
    __shared__ double sJ[TS_MAX_N * TS_MAX_N];
    __shared__ double sh[TS_MAX_N];
    for (int i = threadIdx.x; i < TS_MAX_N * TS_MAX_N; i += blockDim.x) sJ[i] = Jeff[i];
    for (int i = threadIdx.x; i < TS_MAX_N; i += blockDim.x) sh[i] = h[i];
    __syncthreads();
    const uint64_t gid = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const uint64_t tau = gid >> 5;
    const int e = (int)(gid & 31);
    if (tau >= ntiles) return;
    const int nf = q.nfixed;
    auto a_of = [&](int j) {                      // a_j(tau) = sum_x Jeff_jx sigma_x(tau)
        double a = 0.0;
        for (int x = 0; x < nf; ++x) a = fma(sJ[j * TS_MAX_N + q.xspin[x]], (double)((tau >> x) & 1) - 0.5, a);
        return a;
    };
    double E = 0.0;
    if (e == 0) {
        for (int x = 0; x < nf; ++x) {
            const int sp = q.xspin[x];
            E = fma((double)((tau >> x) & 1) - 0.5, sh[sp] + 0.5 * a_of(sp), E);
        }
        double ar = 0.0;
        for (int i = 0; i < 5; ++i) ar += a_of(q.rspin[i]);
        E -= 0.5 * ar;
    } else if (e < 17) {
        const int v = e - 1;
        for (int b = 0; b < 4; ++b) E = fma((double)((v >> b) & 1) - 0.5, a_of(q.tspin[b]), E);
    } else if (e < 25) {
        const int v = e - 17;
        for (int b = 0; b < 3; ++b) E = fma((double)((v >> b) & 1) - 0.5, a_of(q.tspin[4 + b]), E);
    } else if (e < 30) {
        E = a_of(q.rspin[e - 25]);
    }
    double sn, cs;
    sincos(-q.t * E, &sn, &cs);
    out[gid] = make_double2(cs, sn);
}

// RR[r] = exp(-it E_R(r)) on the host, then dithered by one ulp so that the running sum of |z|^2 - 1 over the table
// stays within one ulp (error diffusion): RR is the one factor every amplitude of every tile multiplies by without a
// later re-normalisation, so a common modulus bias of ~1e-17 would add up linearly in the norm.
void build_RR(const ts_ctx* c, const PhaseGeom& q, int alpha, double2* RR)
{
    for (int r = 0; r < 32; ++r) {
        double ER = 0.0;
        for (int i = 0; i < 5; ++i) {
            const double si = (double)((r >> i) & 1) - 0.5;
            double f = c->h[alpha][q.rspin[i]];
            for (int k = 0; k < i; ++k) f += c->Jeff[alpha][q.rspin[i]][q.rspin[k]] * ((double)((r >> k) & 1) - 0.5);
            ER += si * f;
        }
        RR[r] = make_double2(cos(-q.t * ER), sin(-q.t * ER));
    }
    double S = 0.0;
    for (int r = 0; r < 32; ++r) {
        const double2 z = RR[r];
        double best = 0.0; double2 zb = z; bool have = false;
        for (int cand = 0; cand < 3; ++cand) {
            double2 zc = z;
            if (cand) {
                double& comp = (fabs(z.x) >= fabs(z.y)) ? zc.x : zc.y;
                comp = nextafter(comp, cand == 1 ? 2.0 : -2.0);
            }
            const double pp = zc.x * zc.x, ep = fma(zc.x, zc.x, -pp);
            const double qq = zc.y * zc.y, eq = fma(zc.y, zc.y, -qq);
            const double hi = pp >= qq ? pp : qq, lo = pp >= qq ? qq : pp;
            const double dl = ((hi - 1.0) + lo) + (ep + eq);            // |zc|^2 - 1, accurate
            if (!have || fabs(S + dl) < fabs(S + best)) { best = dl; zb = zc; have = true; }
        }
        S += best;
        RR[r] = zb;
    }
}

} // namespace

cudaError_t ts_tile_init(void)
{
    if (!g_registered) {
        memset(g_tab, 0, sizeof(g_tab));
        ts_tile_register_generic(&g_tab[TS_CFG_GENERIC]);
        ts_tile_register_A(&g_tab[TS_CFG_A]);
        ts_tile_register_H7(&g_tab[TS_CFG_H7]);
        ts_tile_register_H8(&g_tab[TS_CFG_H8]);
        ts_tile_register_H9(&g_tab[TS_CFG_H9]);
        ts_tile_register_H10(&g_tab[TS_CFG_H10]);
        memset(g_pipe, 0, sizeof(g_pipe));
        ts_pipe_register_generic(&g_pipe[TS_CFG_GENERIC]);
        ts_pipe_register_A(&g_pipe[TS_CFG_A]);
        ts_pipe_register_H7(&g_pipe[TS_CFG_H7]);
        ts_pipe_register_H8(&g_pipe[TS_CFG_H8]);
        ts_pipe_register_H9(&g_pipe[TS_CFG_H9]);
        ts_pipe_register_H10(&g_pipe[TS_CFG_H10]);
        memset(g_chunk, 0, sizeof(g_chunk));
        ts_chunk_register_H7(&g_chunk[TS_CFG_H7]);
        ts_chunk_register_H8(&g_chunk[TS_CFG_H8]);
        ts_chunk_register_H9(&g_chunk[TS_CFG_H9]);
        ts_chunk_register_H10(&g_chunk[TS_CFG_H10]);
        memset(g_chunk_pipe, 0, sizeof(g_chunk_pipe));
        ts_chunk_pipe_register_H7(&g_chunk_pipe[TS_CFG_H7]);
        ts_chunk_pipe_register_H8(&g_chunk_pipe[TS_CFG_H8]);
        ts_chunk_pipe_register_H9(&g_chunk_pipe[TS_CFG_H9]);
        ts_chunk_pipe_register_H10(&g_chunk_pipe[TS_CFG_H10]);
        g_registered = true;
    }
    if (!g_num_sms) {
        int dev = 0;
        cudaError_t e = cudaGetDevice(&dev);
        if (e == cudaSuccess) e = cudaDeviceGetAttribute(&g_num_sms, cudaDevAttrMultiProcessorCount, dev);
        if (e != cudaSuccess) return e;
    }
    if (!g_encode) {
        void* fn = nullptr;
        cudaDriverEntryPointQueryResult qr;
        cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qr);
        if (e != cudaSuccess) return e;
        if (qr != cudaDriverEntryPointSuccess || !fn) return cudaErrorNotSupported;
        g_encode = (PFN_cuTensorMapEncodeTiled_v12000)fn;
    }
    for (int cf = 0; cf < TS_CFG_COUNT; ++cf)
        for (int v = 0; v < 2; ++v)
            if (g_chunk[cf][v]) {
                cudaError_t e = cudaFuncSetAttribute((const void*)g_chunk[cf][v], cudaFuncAttributeMaxDynamicSharedMemorySize,
                                                     (int)(sizeof(double2) << TS_TILE_LOG2));
                if (e == cudaSuccess)
                    e = cudaFuncSetAttribute((const void*)g_chunk_pipe[cf][v], cudaFuncAttributeMaxDynamicSharedMemorySize, TS_PIPE_SMEM);
                if (e != cudaSuccess) return e;
            }
    for (int cf = 0; cf < TS_CFG_COUNT; ++cf)
        for (int k1 = 0; k1 < 5; ++k1)
            for (int k2 = 0; k2 < 5; ++k2)
                if (g_pipe[cf][k1][k2]) {
                    cudaError_t e = cudaFuncSetAttribute((const void*)g_pipe[cf][k1][k2],
                                                         cudaFuncAttributeMaxDynamicSharedMemorySize, TS_PIPE_SMEM);
                    if (e != cudaSuccess) return e;
                }
    for (int cf = 0; cf < TS_CFG_COUNT; ++cf)
        for (int k1 = 0; k1 < 5; ++k1)
            for (int k2 = 0; k2 < 5; ++k2)
                if (g_tab[cf][k1][k2]) {
                    cudaError_t e = cudaFuncSetAttribute((const void*)g_tab[cf][k1][k2],
                                                         cudaFuncAttributeMaxDynamicSharedMemorySize,
                                                         (int)(sizeof(double2) << TS_TILE_LOG2));
                    if (e != cudaSuccess) return e;
                }
    return cudaSuccess;
}

void ts_tile_free_tables(ts_ctx* c)
{
    for (auto& tb : c->tabs) {
        if (tb.d_thread) cudaFree(tb.d_thread);
        if (tb.d_tile_phase) cudaFree(tb.d_tile_phase);
    }
    c->tabs.clear();
}

cudaError_t ts_tile_get_tables(ts_ctx* c, const DiagOp& d, int group, const DiagTables** out)
{
    for (const auto& tb : c->tabs)
        if (tb.alpha == d.alpha && tb.scale_pow == d.scale_pow && tb.group == group && tb.t == d.t) {
            *out = &tb;
            return cudaSuccess;
        }
    if (c->tabs.size() >= 48) {                 // cap the cache: queued launches may still read the old tables
        cudaError_t e = cudaStreamSynchronize(c->stream);
        if (e != cudaSuccess) return e;
        ts_tile_free_tables(c);
    }
    const TileGroup& g = c->groups[group];
    const PhaseGeom q = make_geom(c, g, d.t);
    const uint64_t ntiles = (uint64_t)1 << (c->N - TS_TILE_LOG2);
    DiagTables tb;
    tb.alpha = d.alpha; tb.scale_pow = d.scale_pow; tb.group = group; tb.t = d.t;
    tb.d_thread = nullptr; tb.d_tile_phase = nullptr;
    cudaError_t e = cudaMalloc(&tb.d_thread, sizeof(double2) * 6 * 128);
    if (e == cudaSuccess) e = cudaMalloc(&tb.d_tile_phase, sizeof(double2) * 32 * ntiles);
    if (e != cudaSuccess) {
        if (tb.d_thread) cudaFree(tb.d_thread);
        return e;
    }
    build_RR(c, q, d.alpha, tb.RR);
    const double* dh = c->d_h + d.alpha * TS_MAX_N;
    const double* dJ = c->d_Jeff + (size_t)d.alpha * TS_MAX_N * TS_MAX_N;
    ts_prof_begin(c, TS_KC_SETUP);
    k_build_thread_tables<<<1, 128, 0, c->stream>>>(tb.d_thread, q, dh, dJ);
    const uint64_t nthreads = ntiles * 32;
    k_build_tile_phase<<<(unsigned)((nthreads + 255) / 256), 256, 0, c->stream>>>(tb.d_tile_phase, ntiles, q, dh, dJ);
    ts_prof_end(c);
    c->launches[TS_KC_SETUP]++;
    e = cudaGetLastError();
    c->tabs.push_back(tb);
    *out = &c->tabs.back();
    return e;
}

static void fill_pipe_geom(const TileGroup& g, uint64_t ntiles, PipeGeom* pg)
{
    pg->ntiles = ntiles;
    pg->is_low = g.is_low;
    const int m = TS_TILE_LOG2 - g.s;                  // rows per tile = 2^m (A: one row)
    pg->row_bytes = g.is_low ? TS_PIPE_HALF_BYTES : (16 << g.s);
    pg->rows_half = g.is_low ? 1 : (1 << (m - 1));
    pg->tensor = (!g.is_low && g.s <= 7) ? 1 : 0;      // box inner dimension <= 256 doubles
    pg->box_rows = pg->rows_half < 256 ? pg->rows_half : 256;
    pg->nbox = pg->rows_half / pg->box_rows;
    pg->dbg = nullptr;
    pg->pf = getenv("TS_PF") ? atoi(getenv("TS_PF")) : 0;    // measured: L2 prefetches cost TMA issue time, slower at any distance
}

// Tensor map of a high group with short runs: the state seen as [hi][2^m rows][2^g0 amplitudes = 2^(g0+1) doubles];
// one box = {2^s amplitudes, <= 256 rows, 1} (runs of 2^s consecutive elements, strided rows).
cudaError_t ts_tile_tensor_map(ts_ctx* c, int group, CUtensorMap* out)
{
    if (c->tmap_psi != (void*)c->psi || c->tmaps.size() != c->groups.size()) {
        c->tmaps.assign(c->groups.size(), TensorMapSlot());
        c->tmap_psi = (void*)c->psi;
    }
    TensorMapSlot& sl = c->tmaps[group];
    if (!sl.valid) {
        const TileGroup& g = c->groups[group];
        const int m = TS_TILE_LOG2 - g.s;
        const int rows_half = 1 << (m - 1);
        const int top = c->N - g.g0 - m;                     // index bits above the group
        cuuint64_t dims[3] = {(cuuint64_t)2 << g.g0, (cuuint64_t)1 << m, (cuuint64_t)1 << top};
        cuuint64_t strides[2] = {(cuuint64_t)16 << g.g0, (cuuint64_t)16 << (g.g0 + m)};
        cuuint32_t box[3] = {(cuuint32_t)2 << g.s, (cuuint32_t)(rows_half < 256 ? rows_half : 256), 1};
        cuuint32_t estr[3] = {1, 1, 1};
        CUtensorMap tm;
        CUresult r = g_encode(&tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, (void*)c->psi, dims, strides, box, estr,
                              CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                              CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r != CUDA_SUCCESS) return cudaErrorInvalidValue;
        memcpy(sl.bytes, &tm, sizeof(tm));
        sl.valid = 1;
    }
    memcpy(out, sl.bytes, sizeof(CUtensorMap));
    return cudaSuccess;
}

cudaError_t ts_tile_pass(ts_ctx* c, int group, int kind1, const DiagTables* tb, int kind2, uint64_t tile_base,
                         uint64_t tile_count)
{
    const TileGroup& g = c->groups[group];
    TilePassParams p;
    p.psi = c->psi;
    p.tile_base = tile_base;
    p.tile_phase = nullptr; p.TT = nullptr; p.WT = nullptr; p.scale = 1.0;
    if (tb) {
        p.tile_phase = tb->d_tile_phase;
        p.TT = tb->d_thread;
        p.WT = tb->d_thread + 128;
        p.scale = ldexp(1.0, tb->scale_pow);
        memcpy(p.RR, tb->RR, sizeof(p.RR));
    } else {
        for (int r = 0; r < 32; ++r) p.RR[r] = make_double2(1.0, 0.0);
    }
    p.s = g.s; p.g0 = g.g0;
    const int nb = n_bfly(g);
    p.two_stage = two_stage(g) ? 1 : 0;
    p.nshfl = g.is_low ? 2 : 0;
    if (g.is_low) { p.bf1 = 31u; p.bf2 = 31u; }
    else if (nb <= 5) { p.bf1 = (31u << (5 - nb)) & 31u; p.bf2 = 0u; }          // top nb bits of f 7..11
    else { p.bf1 = 31u; p.bf2 = (31u << (10 - nb)) & 31u; }                       // top nb-5 bits of f 2..6
    const uint64_t ntiles = tile_count ? tile_count : (uint64_t)1 << (c->N - TS_TILE_LOG2);
    const size_t smem = p.two_stage ? (sizeof(double2) << TS_TILE_LOG2) : 0;
    tile_kernel_t k = g_tab[cfg_of(g)][kind1][kind2];
    if (!k) k = g_tab[TS_CFG_GENERIC][kind1][kind2];
    if (!k) return cudaErrorInvalidValue;
    const bool fused = (kind1 != SW_NONE && kind2 != SW_NONE);
    if (c->pipe_mode == 2 || (c->pipe_mode == 1 && fused)) {
        pipe_kernel_t pk = g_pipe[cfg_of(g)][kind1][kind2];
        if (!pk) pk = g_pipe[TS_CFG_GENERIC][kind1][kind2];
        if (!pk) return cudaErrorInvalidValue;
        PipeGeom pg;
        fill_pipe_geom(g, ntiles, &pg);
        CUtensorMap tm;
        memset(&tm, 0, sizeof(tm));
        if (pg.tensor) {
            cudaError_t e = ts_tile_tensor_map(c, group, &tm);
            if (e != cudaSuccess) return e;
        }
        if (getenv("TS_DEBUG")) { cudaMalloc(&pg.dbg, 64); cudaMemset(pg.dbg, 0, 64); }
        const uint64_t grid = ntiles < (uint64_t)g_num_sms ? ntiles : (uint64_t)g_num_sms;
        ts_prof_begin(c, fused ? TS_KC_TILE_FUSED : TS_KC_TILE_SINGLE);
        pk<<<(unsigned)grid, TS_PIPE_THREADS, TS_PIPE_SMEM, c->stream>>>(p, tm, pg);
        ts_prof_end(c);
        if (getenv("TS_DEBUG")) {
            cudaError_t e = cudaStreamSynchronize(c->stream);
            fprintf(stderr, "pipe pass: group %d (s=%d g0=%d low=%d) k1=%d k2=%d diag=%d tensor=%d rows_half=%d row_bytes=%d "
                    "box_rows=%d nbox=%d grid=%llu ntiles=%llu -> %s\n", group, g.s, g.g0, g.is_low, kind1, kind2, tb != nullptr,
                    pg.tensor, pg.rows_half, pg.row_bytes, pg.box_rows, pg.nbox, (unsigned long long)grid,
                    (unsigned long long)ntiles, cudaGetErrorString(e));
            unsigned long long hd[5] = {0, 0, 0, 0, 0};
            if (e == cudaSuccess) cudaMemcpy(hd, pg.dbg, sizeof(hd), cudaMemcpyDeviceToHost);
            fprintf(stderr, "    landed-vs-global mismatches %llu (first: tile %llu reg %llu thread %llu slot %llu)\n", hd[0], hd[1],
                    hd[2], hd[3], hd[4]);
            cudaFree(pg.dbg);
            if (e != cudaSuccess) return e;
        }
        return cudaGetLastError();
    }
    ts_prof_begin(c, fused ? TS_KC_TILE_FUSED : TS_KC_TILE_SINGLE);
    k<<<(unsigned)ntiles, TS_TILE_THREADS, smem, c->stream>>>(p);
    ts_prof_end(c);
    return cudaGetLastError();
}

namespace {

void fill_params(const ts_ctx* c, const TileGroup& g, const DiagTables* tb, TilePassParams* p)
{
    p->psi = c->psi;
    p->tile_base = 0;
    p->tile_phase = nullptr; p->TT = nullptr; p->WT = nullptr; p->scale = 1.0;
    if (tb) {
        p->tile_phase = tb->d_tile_phase;
        p->TT = tb->d_thread;
        p->WT = tb->d_thread + 128;
        p->scale = ldexp(1.0, tb->scale_pow);
        memcpy(p->RR, tb->RR, sizeof(p->RR));
    } else {
        for (int r = 0; r < 32; ++r) p->RR[r] = make_double2(1.0, 0.0);
    }
    p->s = g.s; p->g0 = g.g0;
    const int nb = n_bfly(g);
    p->two_stage = two_stage(g) ? 1 : 0;
    p->nshfl = g.is_low ? 2 : 0;
    if (g.is_low) { p->bf1 = 31u; p->bf2 = 31u; }
    else if (nb <= 5) { p->bf1 = (31u << (5 - nb)) & 31u; p->bf2 = 0u; }
    else { p->bf1 = 31u; p->bf2 = (31u << (10 - nb)) & 31u; }
}

} // namespace

// Can [H(gh) single ka] [A fused ka . D . kb] [H(gh) single kb] run as one L2-blocked launch?
bool ts_tile_chunk_supported(const ts_ctx* c, int gh, int ka, int kb)
{
    if (c->chunk_mode == 0 || gh < 1 || gh >= (int)c->groups.size() || !c->groups[0].is_low) return false;
    const TileGroup& g = c->groups[gh];
    if (g.g0 != TS_TILE_LOG2) return false;                            // the group right above A
    const int C = g.g0 + (TS_TILE_LOG2 - g.s);                         // chunk = spins 0 .. C-1
    if (C >= c->N || C > c->chunk_max_log2) return false;
    // mode 2 (default): only the pipelined kernel, which needs >= 512 tiles per chunk and >= 2 chunks; mode 1: ticket kernel
    if (c->chunk_mode == 2 && (C - TS_TILE_LOG2 < 9 || c->N - C < 1)) return false;
    const int v = (ka == SW_YDAG && kb == SW_Y) ? 0 : (ka == SW_X && kb == SW_XDAG) ? 1 : -1;
    return v >= 0 && g_chunk[cfg_of(g)][v] != nullptr;
}

cudaError_t ts_tile_chunk_triple(ts_ctx* c, int gh, int ka, const DiagTables* tb, int kb)
{
    const TileGroup& g = c->groups[gh];
    const int C = g.g0 + (TS_TILE_LOG2 - g.s);
    const uint32_t nchunks = 1u << (c->N - C);
    const bool piped = (c->chunk_mode == 2 && C - TS_TILE_LOG2 >= 9 && nchunks >= 2);
    // The pipelined kernel issues the loads of a job ~1.5 tiles ahead, from a thread that still has earlier jobs to run:
    // a dependency must lie at least one block (> 3 grid widths of jobs) back or it would wait for itself.  So its order
    // is  P1(0) P1(1) P2(0) P2(1) P3(0) | P1(c) P3(c-1) P2(c) ...  and the last P3 runs as an ordinary pass afterwards.
    const uint32_t nblocks = piped ? 3 * nchunks - 1 : 3 * nchunks;
    const uint32_t key = nchunks * 2 + (piped ? 1 : 0);
    if (c->sched_nchunks != key) {
        if (c->d_sched) cudaFree(c->d_sched);
        if (c->d_chunk_ctr) cudaFree(c->d_chunk_ctr);
        c->d_sched = nullptr; c->d_chunk_ctr = nullptr; c->sched_nchunks = 0;
        std::vector<uint32_t> sched;
        auto P = [](uint32_t phase, uint32_t chunk) { return phase | (chunk << 2); };
        if (piped) {
            sched.push_back(P(0, 0)); sched.push_back(P(0, 1)); sched.push_back(P(1, 0)); sched.push_back(P(1, 1));
            sched.push_back(P(2, 0));
            for (uint32_t k = 2; k < nchunks; ++k) { sched.push_back(P(0, k)); sched.push_back(P(2, k - 1)); sched.push_back(P(1, k)); }
        } else {
            // P1(0) P2(0) | P1(k) P3(k-1) P2(k) ... | P3(last)
            sched.push_back(P(0, 0)); sched.push_back(P(1, 0));
            for (uint32_t k = 1; k < nchunks; ++k) { sched.push_back(P(0, k)); sched.push_back(P(2, k - 1)); sched.push_back(P(1, k)); }
            sched.push_back(P(2, nchunks - 1));
        }
        if (sched.size() != nblocks) return cudaErrorInvalidValue;
        cudaError_t e = cudaMalloc(&c->d_sched, sizeof(uint32_t) * nblocks);
        if (e == cudaSuccess) e = cudaMalloc(&c->d_chunk_ctr, sizeof(unsigned int) * (64 + 2 * (size_t)nchunks));
        if (e == cudaSuccess) e = cudaMemcpyAsync(c->d_sched, sched.data(), sizeof(uint32_t) * nblocks, cudaMemcpyHostToDevice, c->stream);
        if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);    // `sched` is a temporary
        if (e != cudaSuccess) return e;
        c->sched_nchunks = key;
    }
    ChunkParams q;
    fill_params(c, g, nullptr, &q.h);
    fill_params(c, c->groups[0], tb, &q.a);
    q.sched = c->d_sched;
    q.ticket = c->d_chunk_ctr;
    q.done = c->d_chunk_ctr + 64;
    q.nblocks = nblocks; q.nchunks = nchunks; q.tiles_log2 = (uint32_t)(C - TS_TILE_LOG2);
    cudaError_t e = cudaMemsetAsync(c->d_chunk_ctr, 0, sizeof(unsigned int) * (64 + 2 * (size_t)nchunks), c->stream);
    if (e != cudaSuccess) return e;
    const int v = (ka == SW_YDAG) ? 0 : 1;
    const uint64_t jobs = (uint64_t)nblocks << q.tiles_log2;
    if (piped) {
        PipeGeom pg;
        fill_pipe_geom(g, jobs, &pg);
        CUtensorMap tm;
        memset(&tm, 0, sizeof(tm));
        if (pg.tensor) {
            e = ts_tile_tensor_map(c, gh, &tm);
            if (e != cudaSuccess) return e;
        }
        const uint64_t grid1 = jobs < (uint64_t)g_num_sms ? jobs : (uint64_t)g_num_sms;
        ts_prof_begin(c, TS_KC_TILE_CHUNK);
        // cooperative launch: the CTAs wait on one another's progress, so they must all be resident (else: error, not a hang)
        void* args[3] = {(void*)&q, (void*)&tm, (void*)&pg};
        e = cudaLaunchCooperativeKernel((const void*)g_chunk_pipe[cfg_of(g)][v], dim3((unsigned)grid1), dim3(TS_PIPE_THREADS), args,
                                        TS_PIPE_SMEM, c->stream);
        ts_prof_end(c);
        if (e != cudaSuccess) return e;
        // the last chunk's third phase
        return ts_tile_pass(c, gh, kb, nullptr, SW_NONE, (uint64_t)(nchunks - 1) << q.tiles_log2, (uint64_t)1 << q.tiles_log2);
    }
    chunk_kernel_t k = g_chunk[cfg_of(g)][v];
    uint64_t grid = 2 * (uint64_t)g_num_sms;
    if (grid > jobs) grid = jobs;
    ts_prof_begin(c, TS_KC_TILE_CHUNK);
    k<<<(unsigned)grid, TS_TILE_THREADS, sizeof(double2) << TS_TILE_LOG2, c->stream>>>(q);
    ts_prof_end(c);
    return cudaGetLastError();
}
