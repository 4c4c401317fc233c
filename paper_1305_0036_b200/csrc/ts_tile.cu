// ts_tile.cu -- launchers of the tile passes and construction of their phase tables.
// Kernels: ts_tile_v2.cuh (warp-specialised TMA pipeline, the production path; instantiated in ts_v2_*.cu) and
// ts_tile_kernel.cuh (one CTA per tile, register loads: fallback for geometries v2 does not take, and A/B baseline).
#include <math.h>
#include <string.h>

#include <cudaTypedefs.h>

#include <mutex>

#include "ts_tile_v2.cuh"

namespace {

tile_kernel_t g_tab[5][5];                 // k_tile_pass, run-time butterfly masks
tile_kernel_t g_p2p[5][5];                 // k_tile_pass_p2p (sharded state vector: tiles gathered from peer memory)
v2_kernel_t g_v2[4][5][5];                 // [type][k1][k2]: group A, high group (run-time masks), high group of 9 bits, of 10 bits
v2_chunk_kernel_t g_v2_chunk[2][2];        // [9-bit high group][(Y^dag, Y), (X, X^dag)]
v2_chunk_kernel_t g_probe_chunk[2];        // measurement builds (ts_v2_probe.cu): [arithmetic only, exchanges only]
v2_kernel_t g_probe_H[2], g_probe_A[2];
PFN_cuTensorMapEncodeTiled_v12000 g_encode = nullptr;
std::once_flag g_once;
cudaError_t g_init_status = cudaSuccess;

// Geometry of the diagonal-time layout of one group: which spins sit on register bits (R), thread bits (T) and
// outside the tile (X).
struct PhaseGeom {
    double t, e0;        // time of the diagonal; energy offset of the context (shards: the spins on the rank bits)
    int N, nfixed;
    int nr, nt;          // register bits / thread bits at diagonal time (5 + 7)
    int rec;             // entries of a tile-phase record (32)
    int rspin[5], tspin[8], xspin[TS_MAX_FIXED];
};

inline int spin_of_fbit(const TileGroup& g, int f) { return f < g.s ? f : g.g0 + (f - g.s); }
inline int n_bfly(const TileGroup& g) { return g.is_low ? TS_TILE_LOG2 : TS_TILE_LOG2 - g.s; }
inline bool two_stage(const TileGroup& g) { return n_bfly(g) > 5; }
inline bool v2_geometry_ok(const TileGroup& g) { return g.is_low || (g.s >= 2 && g.s <= 11); }   // s = 2: the ten-bit kernels
inline int nib(uint32_t pack, int i) { return (int)((pack >> (4 * i)) & 15u); }
inline int v2_type(const TileGroup& g) { return g.is_low ? 0 : (g.s == 3 ? 2 : (g.s == 2 ? 3 : 1)); }     // kernel table index

// layout 0: k_tile_pass.  layout 1: v2 (ts_tile_v2.cuh: the diagonal is applied in A2', H2 or H1).
PhaseGeom make_geom(const ts_ctx* c, const TileGroup& g, double t, int layout)
{
    PhaseGeom q;
    q.t = t; q.e0 = 0.0; q.N = c->N; q.nfixed = c->N - TS_TILE_LOG2;
    q.nr = 5; q.nt = TS_TILE_LOG2 - q.nr; q.rec = 32;
    for (int b = 0; b < 5; ++b) q.rspin[b] = 0;
    for (int b = 0; b < 8; ++b) q.tspin[b] = 0;
    const bool two = two_stage(g);
    if (layout == 0) {
        for (int b = 0; b < 5; ++b) q.rspin[b] = spin_of_fbit(g, two ? 2 + b : 7 + b);
        for (int b = 0; b < 7; ++b) {
            const int f = two ? (b < 2 ? b : 5 + b) : b;     // layout 2: thread bits 0,1 -> f 0,1; 2..6 -> f 7..11
            q.tspin[b] = spin_of_fbit(g, f);
        }
    } else {
        const bool ten = (!g.is_low && g.s == 2);
        const uint32_t RP = g.is_low ? TS_V2_A2S_R : ten ? TS_V2_H2X_R : (two ? TS_V2_H2_R : TS_V2_H1_R);
        const uint32_t TP = g.is_low ? TS_V2_A2S_T : ten ? TS_V2_H2X_T : (two ? TS_V2_H2_T : TS_V2_H1_T);
        for (int b = 0; b < 5; ++b) q.rspin[b] = spin_of_fbit(g, nib(RP, b));
        for (int b = 0; b < 7; ++b) q.tspin[b] = spin_of_fbit(g, nib(TP, b));
    }
    bool in_tile[TS_MAX_N] = {false};
    for (int f = 0; f < TS_TILE_LOG2; ++f) in_tile[spin_of_fbit(g, f)] = true;
    int nx = 0;
    for (int i = 0; i < TS_MAX_FIXED; ++i) q.xspin[i] = 0;
    for (int j = 0; j < c->N; ++j) if (!in_tile[j]) q.xspin[nx++] = j;    // ascending = tile-index bit order
    return q;
}

// TT[v], WT[0..nr-1][v] for thread index v (one block of 2^nt threads); out = TT[2^nt] followed by WT[nr][2^nt].
__global__ void __launch_bounds__(256) k_build_thread_tables(double2* __restrict__ out, const PhaseGeom q,
                                                             const double* __restrict__ h,
                                                             const double* __restrict__ Jeff)
{
    const int v = threadIdx.x;
    const int GT = 1 << q.nt;
    double sg[8];
    for (int b = 0; b < q.nt; ++b) sg[b] = (double)((v >> b) & 1) - 0.5;
    double ET = 0.0;                              // fields and couplings among the thread spins
    for (int b = 0; b < q.nt; ++b) {
        double f = h[q.tspin[b]];
        for (int c = 0; c < b; ++c) f += Jeff[q.tspin[b] * TS_MAX_N + q.tspin[c]] * sg[c];
        ET += sg[b] * f;
    }
    double bsum = 0.0;
    for (int i = 0; i < q.nr; ++i) {
        double bi = 0.0;
        for (int b = 0; b < q.nt; ++b) bi += Jeff[q.rspin[i] * TS_MAX_N + q.tspin[b]] * sg[b];
        bsum += bi;
        double sn, cs;
        sincos(-q.t * bi, &sn, &cs);
        out[GT + i * GT + v] = make_double2(cs, sn);
    }
    double sn, cs;
    sincos(-q.t * (ET - 0.5 * bsum), &sn, &cs);
    out[v] = make_double2(cs, sn);
}

// Tile-phase table: q.rec entries per tile, one thread per entry:
//   [0] tp0;  [1..16] the four low thread bits;  [17 .. 16 + 2^(nt-4)] the remaining thread bits;  then nr entries tpW;
//   the rest is padding (1).  (Layout and meaning in ts_tile_kernel.cuh.)
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
    const uint64_t tau = gid / (uint64_t)q.rec;
    const int e = (int)(gid % (uint64_t)q.rec);
    if (tau >= ntiles) return;
    const int nf = q.nfixed;
    const int nhi = q.nt - 4, wofs = 17 + (1 << nhi);
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
        for (int i = 0; i < q.nr; ++i) ar += a_of(q.rspin[i]);
        E -= 0.5 * ar;
        E += q.e0;
    } else if (e < 17) {
        const int v = e - 1;
        for (int b = 0; b < 4; ++b) E = fma((double)((v >> b) & 1) - 0.5, a_of(q.tspin[b]), E);
    } else if (e < wofs) {
        const int v = e - 17;
        for (int b = 0; b < nhi; ++b) E = fma((double)((v >> b) & 1) - 0.5, a_of(q.tspin[4 + b]), E);
    } else if (e < wofs + q.nr) {
        E = a_of(q.rspin[e - wofs]);
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
    const int nrr = 1 << q.nr;
    for (int r = nrr; r < 32; ++r) RR[r] = make_double2(1.0, 0.0);
    for (int r = 0; r < nrr; ++r) {
        double ER = 0.0;
        for (int i = 0; i < q.nr; ++i) {
            const double si = (double)((r >> i) & 1) - 0.5;
            double f = c->h[alpha][q.rspin[i]];
            for (int k = 0; k < i; ++k) f += c->Jeff[alpha][q.rspin[i]][q.rspin[k]] * ((double)((r >> k) & 1) - 0.5);
            ER += si * f;
        }
        RR[r] = make_double2(cos(-q.t * ER), sin(-q.t * ER));
    }
    double S = 0.0;
    for (int r = 0; r < nrr; ++r) {
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

void init_once()
{
    memset(g_tab, 0, sizeof(g_tab));
    ts_tile_register_generic(&g_tab);
    memset(g_p2p, 0, sizeof(g_p2p));
    ts_tile_register_p2p(&g_p2p);
    memset(g_v2, 0, sizeof(g_v2));
    ts_v2_register_A(&g_v2[0]);
    ts_v2_register_Hf(&g_v2[1]);
    ts_v2_register_Hs(&g_v2[1]);
    ts_v2_register_H9f(&g_v2[2]);
    ts_v2_register_H9s(&g_v2[2]);
    ts_v2_register_H10(&g_v2[3]);
    memset(g_v2_chunk, 0, sizeof(g_v2_chunk));
    ts_v2_register_chunk0(g_v2_chunk);
    ts_v2_register_chunk1(g_v2_chunk);
    ts_v2_register_chunk0_h9(g_v2_chunk);
    ts_v2_register_chunk1_h9(g_v2_chunk);
    ts_v2_register_probe(g_probe_chunk, g_probe_H, g_probe_A);
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult qr;
    cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qr);
    if (e == cudaSuccess && (qr != cudaDriverEntryPointSuccess || !fn)) e = cudaErrorNotSupported;
    if (e != cudaSuccess) { g_init_status = e; return; }
    g_encode = (PFN_cuTensorMapEncodeTiled_v12000)fn;
    for (int ty = 0; ty < 4 && e == cudaSuccess; ++ty)
        for (int k1 = 0; k1 < 5 && e == cudaSuccess; ++k1)
            for (int k2 = 0; k2 < 5 && e == cudaSuccess; ++k2)
                if (g_v2[ty][k1][k2])
                    e = cudaFuncSetAttribute((const void*)g_v2[ty][k1][k2], cudaFuncAttributeMaxDynamicSharedMemorySize, TS_V2_SMEM);
    for (int hm = 0; hm < 2 && e == cudaSuccess; ++hm)
        for (int v = 0; v < 2 && e == cudaSuccess; ++v)
            if (g_v2_chunk[hm][v])
                e = cudaFuncSetAttribute((const void*)g_v2_chunk[hm][v], cudaFuncAttributeMaxDynamicSharedMemorySize, TS_V2_SMEM);
    for (int m = 0; m < 2 && e == cudaSuccess; ++m) {
        e = cudaFuncSetAttribute((const void*)g_probe_chunk[m], cudaFuncAttributeMaxDynamicSharedMemorySize, TS_V2_SMEM);
        if (e == cudaSuccess) e = cudaFuncSetAttribute((const void*)g_probe_H[m], cudaFuncAttributeMaxDynamicSharedMemorySize, TS_V2_SMEM);
        if (e == cudaSuccess) e = cudaFuncSetAttribute((const void*)g_probe_A[m], cudaFuncAttributeMaxDynamicSharedMemorySize, TS_V2_SMEM);
    }
    for (int k1 = 0; k1 < 5 && e == cudaSuccess; ++k1)
        for (int k2 = 0; k2 < 5 && e == cudaSuccess; ++k2)
            if (g_tab[k1][k2])
                e = cudaFuncSetAttribute((const void*)g_tab[k1][k2], cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)(sizeof(double2) << TS_TILE_LOG2));
    for (int k1 = 0; k1 < 5 && e == cudaSuccess; ++k1)
        for (int k2 = 0; k2 < 5 && e == cudaSuccess; ++k2)
            if (g_p2p[k1][k2])
                e = cudaFuncSetAttribute((const void*)g_p2p[k1][k2], cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)(sizeof(double2) << TS_TILE_LOG2));
    g_init_status = e;
}

void fill_v1_params(const ts_ctx* c, const TileGroup& g, const DiagTables* tb, TilePassParams* p)
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
    for (int k = 0; k < 8; ++k) p->peers[k] = nullptr;
    p->dst = nullptr; p->p2p_gbits = 0; p->p2p_rank = 0;
    p->s = g.s; p->g0 = g.g0;
    // butterflied bits: all of the group's, or (c->top_bits_only > 0) only its top `top_bits_only` ones; the layouts the
    // tile moves through -- and with them the diagonal's tables -- are those of the whole group either way
    const int nb = (c->top_bits_only > 0 && !g.is_low) ? c->top_bits_only : n_bfly(g);
    p->two_stage = two_stage(g) ? 1 : 0;
    p->nshfl = g.is_low ? 2 : 0;
    auto masks = [&](int bits, unsigned& m1, unsigned& m2) {
        if (g.is_low) { m1 = 31u; m2 = 31u; }
        else if (bits <= 5) { m1 = (31u << (5 - bits)) & 31u; m2 = 0u; }          // top `bits` bits of f 7..11 (layout 1)
        else { m1 = 31u; m2 = (31u << (10 - bits)) & 31u; }                        // + top bits-5 bits of f 2..6
    };
    masks(nb, p->bf1, p->bf2);
    masks(n_bfly(g), p->bf1b, p->bf2b);       // a second sweep in the same pass always takes all of the group's bits
}

void fill_v2_geom(const TileGroup& g, V2Geom* q, int top_bits_only = 0)
{
    q->type = g.is_low ? 0 : 1;
    q->s = g.s; q->g0 = g.g0;
    q->m = g.is_low ? 0 : TS_TILE_LOG2 - g.s;
    q->nmid = g.g0 - g.s;
    q->unit_log2 = g.s < 3 ? g.s : 3;
    q->box_rows_log2 = (q->m - 1 < 8) ? q->m - 1 : 8;
    q->two_stage = (!g.is_low && q->m > 5) ? 1 : 0;
    q->mask1 = 0u; q->mask2 = 0u;
    if (!g.is_low) {
        const int mb = top_bits_only > 0 ? top_bits_only : q->m;          // f bits 12 - mb .. 11 are butterflied
        q->mask1 = tsk::v2_h_mask1(mb);
        q->mask2 = tsk::v2_h_mask2(mb);     // (H2 register bit 4 = f 7 is a filler)
    }
}

void fill_v2_diag(const DiagTables* tb, V2Diag* d)
{
    d->tile_phase = nullptr; d->tables = nullptr; d->scale = 1.0;
    if (tb) {
        d->tile_phase = tb->d_tile_phase;
        d->tables = tb->d_thread;            // TT[128], WT[5][128], RR[32]
        d->scale = ldexp(1.0, tb->scale_pow);
    }
}

// Tensor map of one group for the v2 kernels (SWIZZLE_128B, rows of 16 doubles = 8 amplitudes = 128 B):
//   group A:    the state as [2^(N-3) rows][16 doubles], box {16, 256}  (half a contiguous tile);
//   high group: the state as [2^top][2^m rows][2^(g0-3) units][16 doubles], box {16, 2^(s-3), 2^(m-1), 1}: half a tile
//               = 2^(m-1) strided rows of 2^s consecutive amplitudes.
cudaError_t v2_tensor_map(ts_ctx* c, int group, CUtensorMap* out)
{
    if (c->tmap_psi != (void*)c->psi || c->tmaps.size() != c->groups.size()) {
        c->tmaps.assign(c->groups.size(), TensorMapSlot());
        c->tmap_psi = (void*)c->psi;
    }
    TensorMapSlot& sl = c->tmaps[group];
    if (!sl.valid) {
        const TileGroup& g = c->groups[group];
        CUtensorMap tm;
        CUresult r;
        cuuint32_t estr[4] = {1, 1, 1, 1};
        if (g.is_low) {
            cuuint64_t dims[2] = {16, (cuuint64_t)1 << (c->N - 3)};
            cuuint64_t strides[1] = {128};
            cuuint32_t box[2] = {16, 256};
            r = g_encode(&tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, (void*)c->psi, dims, strides, box, estr,
                         CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_NONE,
                         CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        } else {
            const int m = TS_TILE_LOG2 - g.s;
            const int top = c->N - g.g0 - m;                     // index bits above the group
            const int u = g.s < 3 ? g.s : 3;                     // unit = 2^u amplitudes (128 bytes; 64 for runs of 4)
            const int rows_log2 = (m - 1 < 8) ? m - 1 : 8;       // a box dimension cannot exceed 256
            cuuint64_t dims[4] = {(cuuint64_t)2 << u, (cuuint64_t)1 << (g.g0 - u), (cuuint64_t)1 << m, (cuuint64_t)1 << top};
            cuuint64_t strides[3] = {(cuuint64_t)16 << u, (cuuint64_t)16 << g.g0, (cuuint64_t)16 << (g.g0 + m)};
            cuuint32_t box[4] = {(cuuint32_t)2 << u, (cuuint32_t)1 << (g.s - u), (cuuint32_t)1 << rows_log2, 1};
            const CUtensorMapL2promotion prom = c->opt_l2_promotion == 2 ? CU_TENSOR_MAP_L2_PROMOTION_L2_256B
                                              : c->opt_l2_promotion == 1 ? CU_TENSOR_MAP_L2_PROMOTION_L2_128B
                                                                         : CU_TENSOR_MAP_L2_PROMOTION_NONE;
            r = g_encode(&tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, (void*)c->psi, dims, strides, box, estr,
                         CU_TENSOR_MAP_INTERLEAVE_NONE, g.s < 3 ? CU_TENSOR_MAP_SWIZZLE_64B : CU_TENSOR_MAP_SWIZZLE_128B, prom,
                         CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        }
        if (r != CUDA_SUCCESS) return cudaErrorInvalidValue;
        memcpy(sl.bytes, &tm, sizeof(tm));
        sl.valid = 1;
    }
    memcpy(out, sl.bytes, sizeof(CUtensorMap));
    return cudaSuccess;
}

} // namespace

cudaError_t ts_tile_init(void)
{
    std::call_once(g_once, init_once);
    return g_init_status;
}

void ts_tile_free_tables(ts_ctx* c)
{
    for (DiagTables* tb : c->tabs) {
        if (tb->d_thread) cudaFree(tb->d_thread);
        if (tb->d_tile_phase) cudaFree(tb->d_tile_phase);
        delete tb;
    }
    c->tabs.clear();
}

cudaError_t ts_tile_get_tables(ts_ctx* c, const DiagOp& d, int group, int layout, const DiagTables** out)
{
    for (const DiagTables* tb : c->tabs)
        if (tb->alpha == d.alpha && tb->scale_pow == d.scale_pow && tb->group == group && tb->layout == layout && tb->t == d.t) {
            *out = tb;
            return cudaSuccess;
        }
    if (c->tabs.size() >= 48) {                 // cap the cache: queued launches may still read the old tables
        cudaError_t e = cudaStreamSynchronize(c->stream);
        if (e != cudaSuccess) return e;
        ts_tile_free_tables(c);
    }
    const TileGroup& g = c->groups[group];
    PhaseGeom q = make_geom(c, g, d.t, layout);
    q.e0 = c->e0[d.alpha];
    const uint64_t ntiles = (uint64_t)1 << (c->N - TS_TILE_LOG2);
    const int GT = 1 << q.nt, nrr = 1 << q.nr;
    const size_t n_thread_tab = (size_t)(1 + q.nr) * GT;          // TT, WT[nr]; RR[2^nr] follows
    DiagTables* tb = new DiagTables();
    tb->alpha = d.alpha; tb->scale_pow = d.scale_pow; tb->group = group; tb->layout = layout; tb->t = d.t;
    tb->d_thread = nullptr; tb->d_tile_phase = nullptr;
    cudaError_t e = cudaMalloc(&tb->d_thread, sizeof(double2) * (n_thread_tab + nrr));
    if (e == cudaSuccess) e = cudaMalloc(&tb->d_tile_phase, sizeof(double2) * (size_t)q.rec * ntiles);
    if (e != cudaSuccess) {
        if (tb->d_thread) cudaFree(tb->d_thread);
        delete tb;
        return e;
    }
    build_RR(c, q, d.alpha, tb->RR);
    e = cudaMemcpyAsync(tb->d_thread + n_thread_tab, tb->RR, sizeof(double2) * nrr, cudaMemcpyHostToDevice, c->stream);   // (tb is heap-allocated and lives as long as the cache entry)
    if (e != cudaSuccess) { cudaFree(tb->d_thread); cudaFree(tb->d_tile_phase); delete tb; return e; }
    const double* dh = c->d_h + d.alpha * TS_MAX_N;
    const double* dJ = c->d_Jeff + (size_t)d.alpha * TS_MAX_N * TS_MAX_N;
    ts_prof_begin(c, TS_KC_SETUP);
    k_build_thread_tables<<<1, GT, 0, c->stream>>>(tb->d_thread, q, dh, dJ);
    const uint64_t nthreads = ntiles * (uint64_t)q.rec;
    k_build_tile_phase<<<(unsigned)((nthreads + 255) / 256), 256, 0, c->stream>>>(tb->d_tile_phase, ntiles, q, dh, dJ);
    ts_prof_end(c);
    c->launches[TS_KC_SETUP]++;
    e = cudaGetLastError();
    c->tabs.push_back(tb);
    *out = tb;
    return e;
}

int ts_tile_layout_for(const ts_ctx* c, int group, int kind1, int kind2)
{
    const TileGroup& g = c->groups[group];
    if (c->opt_kernel == 0 || !v2_geometry_ok(g)) return 0;
    // automatic choice: the persistent pipeline pays once every SM walks several tiles; with at most two tiles per SM
    // (N <= 20 on 148 SMs) the one-CTA-per-tile kernel is faster (no pipeline set-up: 283 vs 361 us per step at N = 20)
    if (c->opt_kernel == 2 && (((uint64_t)1 << (c->N - TS_TILE_LOG2)) <= 2ull * (uint64_t)c->num_sms)) return 0;
    if (c->top_bits_only > 0 && !g.is_low && (kind2 != SW_NONE || g.s < 3)) return 0;   // separate masks per sweep: k_tile_pass only
    return g_v2[(c->top_bits_only > 0 && !g.is_low) ? 1 : v2_type(g)][kind1][kind2] ? 1 : 0;
}

cudaError_t ts_tile_pass(ts_ctx* c, int group, int kind1, const DiagOp* d, int kind2)
{
    const TileGroup& g = c->groups[group];
    const int layout = ts_tile_layout_for(c, group, kind1, kind2);
    const DiagTables* tb = nullptr;
    if (d && d->present) {
        cudaError_t e = ts_tile_get_tables(c, *d, group, layout, &tb);
        if (e != cudaSuccess) return e;
    }
    const uint64_t ntiles = (uint64_t)1 << (c->N - TS_TILE_LOG2);
    const bool fused = (kind1 != SW_NONE && kind2 != SW_NONE);
    if (layout >= 1) {
        V2Pass p;
        const int tbo = g.is_low ? 0 : c->top_bits_only;
        fill_v2_geom(g, &p.g, tbo);
        fill_v2_diag(tb, &p.d);
        p.ntiles = ntiles;
        p.sched = c->d_sched;
        p.pair_log2 = (c->opt_pair && !g.is_low && g.g0 > g.s && ntiles >= 2) ? 1u : 0u;   // adjacent tiles exist (nmid >= 1)
        p.probe = (c->opt_probe == 1);
        p.ngroups = c->opt_groups;
        v2_kernel_t kern = g_v2[tbo > 0 ? 1 : v2_type(g)][kind1][kind2];   // (a bit subset needs the run-time-mask kernels)
        if (c->opt_probe >= 2) {                       // measurement builds exist for the fused passes of the N = 30 plan
            if (v2_type(g) == 2 && fused) kern = g_probe_H[c->opt_probe - 2];     // (the kinds do not change the cost)
            if (v2_type(g) == 0 && fused) kern = g_probe_A[c->opt_probe - 2];
        }
        CUtensorMap tm;
        cudaError_t e = v2_tensor_map(c, group, &tm);
        if (e != cudaSuccess) return e;
        const uint64_t cap = (c->opt_max_ctas > 0 && c->opt_max_ctas < c->num_sms) ? (uint64_t)c->opt_max_ctas : (uint64_t)c->num_sms;
        const uint64_t grid = ntiles < cap ? ntiles : cap;
        if (c->dry_run) return cudaSuccess;
        ts_prof_begin(c, fused ? TS_KC_TILE_FUSED : TS_KC_TILE_SINGLE, 1.0);
        kern<<<(unsigned)grid, TS_V2_THREADS, TS_V2_SMEM, c->stream>>>(p, tm);
        ts_prof_end(c);
        return cudaGetLastError();
    }
    TilePassParams p;
    fill_v1_params(c, g, tb, &p);
    tile_kernel_t k = g_tab[kind1][kind2];
    if (!k) return cudaErrorInvalidValue;
    const size_t smem = p.two_stage ? (sizeof(double2) << TS_TILE_LOG2) : 0;
    if (c->dry_run) return cudaSuccess;
    ts_prof_begin(c, fused ? TS_KC_TILE_FUSED : TS_KC_TILE_SINGLE, 1.0);
    k<<<(unsigned)ntiles, TS_TILE_THREADS, smem, c->stream>>>(p);
    ts_prof_end(c);
    return cudaGetLastError();
}

// Sharded state vector (ts_shard.cu): sweep `kind`'s butterflies on the top `gbits` bits of `group` (the spins that would
// have arrived with the all-to-all), the diagonal, and sweep `kind2`'s butterflies on all of the group's bits (SW_NONE: none),
// the tiles gathered straight from the peers' shards.
cudaError_t ts_tile_pass_p2p(ts_ctx* c, int group, int kind, const DiagOp* d, int kind2, const double2* const* peers, int gbits,
                             int rank, double2* dst)
{
    const TileGroup& g = c->groups[group];
    if (g.is_low || gbits < 1 || gbits > 5 || TS_TILE_LOG2 - g.s < gbits || !g_p2p[kind][kind2]) return cudaErrorInvalidValue;
    const DiagTables* tb = nullptr;
    if (d && d->present) {
        cudaError_t e = ts_tile_get_tables(c, *d, group, 0, &tb);
        if (e != cudaSuccess) return e;
    }
    TilePassParams p;
    c->top_bits_only = gbits;
    fill_v1_params(c, g, tb, &p);
    c->top_bits_only = 0;
    for (int k = 0; k < (1 << gbits); ++k) p.peers[k] = peers[k];
    p.dst = dst; p.p2p_gbits = gbits; p.p2p_rank = rank;
    const uint64_t ntiles = (uint64_t)1 << (c->N - TS_TILE_LOG2);
    const size_t smem = p.two_stage ? (sizeof(double2) << TS_TILE_LOG2) : 0;
    ts_prof_begin(c, kind2 != SW_NONE ? TS_KC_TILE_FUSED : TS_KC_TILE_SINGLE, 1.0);
    g_p2p[kind][kind2]<<<(unsigned)ntiles, TS_TILE_THREADS, smem, c->stream>>>(p);
    ts_prof_end(c);
    return cudaGetLastError();
}

// Can [H(gh) single ka] [A fused ka . D . kb] [H(gh) single kb] run as one L2-blocked launch?
bool ts_tile_chunk_supported(const ts_ctx* c, int gh, int ka, int kb)
{
    if (c->opt_chunk == 0 || c->opt_kernel == 0 || gh != 1 || (int)c->groups.size() < 3 || !c->groups[0].is_low) return false;
    if (ts_tile_layout_for(c, 0, ka, kb) == 0) return false;           // the TMA kernels are not in use at this size
    const TileGroup& g = c->groups[gh];
    if (g.g0 != TS_TILE_LOG2 || !v2_geometry_ok(g) || g.s < 3) return false;     // the group right above A, 128-byte runs
    const int C = g.g0 + (TS_TILE_LOG2 - g.s);                         // chunk = spins 0 .. C-1
    if (C >= c->N || C > c->opt_chunk_max_log2) return false;          // at least two chunks, each small enough for L2
    if (C < c->opt_chunk_min_log2) return false;                       // small chunks: the hand-overs cost more than the round trips
    const int v = (ka == SW_YDAG && kb == SW_Y) ? 0 : (ka == SW_X && kb == SW_XDAG) ? 1 : -1;
    return v >= 0 && g_v2_chunk[g.s == 3 ? 1 : 0][v] != nullptr;
}

cudaError_t ts_tile_chunk_triple(ts_ctx* c, int gh, int ka, const DiagOp& d, int kb)
{
    const TileGroup& g = c->groups[gh];
    const int C = g.g0 + (TS_TILE_LOG2 - g.s);
    const uint32_t nchunks = 1u << (c->N - C);
    const DiagTables* tb = nullptr;
    cudaError_t e = cudaSuccess;
    if (d.present) {
        e = ts_tile_get_tables(c, d, 0, 1, &tb);
        if (e != cudaSuccess) return e;
    }
    if (c->dry_run) return cudaSuccess;
    const size_t nctr = 2 * (size_t)nchunks;
    if (c->chunk_ctr_cap < nctr) {
        e = cudaStreamSynchronize(c->stream);                          // queued launches may still use the old counters
        if (e != cudaSuccess) return e;
        if (c->d_chunk_ctr) cudaFree(c->d_chunk_ctr);
        c->d_chunk_ctr = nullptr; c->chunk_ctr_cap = 0;
        e = cudaMalloc(&c->d_chunk_ctr, sizeof(unsigned int) * nctr);
        if (e != cudaSuccess) return e;
        c->chunk_ctr_cap = nctr;
    }
    V2Chunk q;
    fill_v2_geom(g, &q.gh);
    fill_v2_geom(c->groups[0], &q.ga);
    fill_v2_diag(tb, &q.d);
    q.done = c->d_chunk_ctr;
    q.sched = c->d_sched;
    q.probe = (c->opt_probe == 1);
    q.ngroups = c->opt_groups;
    q.nchunks = nchunks; q.tiles_log2 = (uint32_t)(C - TS_TILE_LOG2);
    q.l2_hints = c->opt_l2_hints;
    e = cudaMemsetAsync(c->d_chunk_ctr, 0, sizeof(unsigned int) * nctr, c->stream);
    if (e != cudaSuccess) return e;
    CUtensorMap tmA, tmH;
    e = v2_tensor_map(c, 0, &tmA);
    if (e == cudaSuccess) e = v2_tensor_map(c, gh, &tmH);
    if (e != cudaSuccess) return e;
    const int v = (ka == SW_YDAG) ? 0 : 1;
    const uint64_t jobs = (uint64_t)(3u * nchunks) << q.tiles_log2;
    const uint64_t cap = (c->opt_max_ctas > 0 && c->opt_max_ctas < c->num_sms) ? (uint64_t)c->opt_max_ctas : (uint64_t)c->num_sms;
    const uint64_t grid = jobs < cap ? jobs : cap;
    ts_prof_begin(c, TS_KC_TILE_CHUNK, 3.0);
    // cooperative launch: the loaders wait on other CTAs' progress, so all CTAs must be resident (else: error, not a hang)
    void* args[3] = {(void*)&q, (void*)&tmA, (void*)&tmH};
    const void* kern = (const void*)g_v2_chunk[g.s == 3 ? 1 : 0][v];
    if (c->opt_probe >= 2 && g.s == 3) kern = (const void*)g_probe_chunk[c->opt_probe - 2];
    e = cudaLaunchCooperativeKernel(kern, dim3((unsigned)grid), dim3(TS_V2_THREADS), args, TS_V2_SMEM, c->stream);
    ts_prof_end(c);
    return e;
}
