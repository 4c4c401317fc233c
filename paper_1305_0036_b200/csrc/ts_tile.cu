// ts_tile.cu -- the production hot path: tile passes.
//
// One launch = one HBM round trip of the whole state.  Each CTA (128 threads) owns one closed tile of 2^12
// amplitudes (the set of states with the spins outside the tile fixed "is closed under the pairing operation
// that flips any spin which is not in F"), holds it in REGISTERS (32 amplitudes per thread) and applies
//
//      [butterflies of sweep K1 on the tile's group bits] . [diagonal D] . [butterflies of sweep K2 on the same bits]
//
// before storing it back in place.  Fusing the last bit group of one global rotation with the first bit group of the
// next (butterflies on different bits commute, so a sweep may visit its groups in any order) removes one round trip
// per sweep; the diagonal in between is applied on the fly ("the phase correction is performed when the
// rotation kernel reads elements from memory") from factorised phase tables instead of the paper's three 2^N
// vectors.
//
// Tile geometry (TileGroup): in-tile bit f < s <-> spin f (runs of 2^s consecutive amplitudes);
// f >= s <-> spin g0 + f - s.  Register/thread layouts, with t = threadIdx.x (7 bits) and r = register index (5 bits):
//   layout 1 (global load/store, coalesced):  f = t | r << 7                      registers hold f bits 7..11
//   layout 2 (after one shared-memory exchange): f = (t & 3) | r << 2 | (t >> 2) << 7   registers hold f bits 2..6
// Group A (f = spins 0..11) additionally butterflies f bits 0,1 (lane bits 0,1 in layout 2) by warp shuffles.
// Shared-memory slot of f is f ^ ((f >> 5) & 7): conflict-free 128-bit accesses in both layouts.
#include "ts_internal.h"

namespace {

struct TilePassParams {
    double2* psi;
    const DiagDesc* desc;   // NULL: no diagonal in this pass
    const double* h;        // [TS_MAX_N]            of desc's alpha
    const double* Jeff;     // [TS_MAX_N][TS_MAX_N]  of desc's alpha
    int N, s, g0;
    int two_stage;          // layout 2 is used (more than 5 butterflied bits)
    int nshfl;              // 2 for group A, else 0
    unsigned bf1, bf2;      // which register bits are butterflied in layout 1 / layout 2
};

__device__ __forceinline__ double2 cmul(double2 a, double2 b)
{
    return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}

template <int KIND>
__device__ __forceinline__ void pair_update(double& r0, double& i0, double& r1, double& i1)
{
    const double a = r0, b = i0, c = r1, d = i1;
    if (KIND == SW_YDAG)      { r0 = a - c; i0 = b - d; r1 = a + c; i1 = b + d; }
    else if (KIND == SW_Y)    { r0 = a + c; i0 = b + d; r1 = c - a; i1 = d - b; }
    else if (KIND == SW_XDAG) { r0 = a + d; i0 = b - c; r1 = c + b; i1 = d - a; }
    else if (KIND == SW_X)    { r0 = a - d; i0 = b + c; r1 = c - b; i1 = d + a; }
}

// Butterflies on the register bits selected by `mask` (uniform across the grid).
template <int KIND>
__device__ __forceinline__ void bfly_regs(double (&re)[32], double (&im)[32], unsigned mask)
{
    if (KIND == SW_NONE) return;
#pragma unroll
    for (int b = 0; b < 5; ++b) {
        if (mask & (1u << b)) {
#pragma unroll
            for (int r = 0; r < 32; ++r)
                if (!(r & (1 << b))) pair_update<KIND>(re[r], im[r], re[r | (1 << b)], im[r | (1 << b)]);
        }
    }
}

// Butterfly on lane bit lb: each lane holds one member of the pair and fetches the other by shuffle.
template <int KIND>
__device__ __forceinline__ void bfly_lane(double (&re)[32], double (&im)[32], int lb, int lane)
{
    if (KIND == SW_NONE) return;
    const int up = (lane >> lb) & 1;      // this lane holds c1
    // YDAG: c0' = c0 - c1, c1' = c0 + c1 -> mine + sg * partner with sg = up ? +1 : -1;  Y: sg = up ? -1 : +1
    const double sg = (KIND == SW_YDAG) ? (up ? 1.0 : -1.0) : (up ? -1.0 : 1.0);
#pragma unroll
    for (int r = 0; r < 32; ++r) {
        const double pr = __shfl_xor_sync(0xffffffffu, re[r], 1 << lb);
        const double pi = __shfl_xor_sync(0xffffffffu, im[r], 1 << lb);
        if (KIND == SW_YDAG || KIND == SW_Y) { re[r] = fma(sg, pr, re[r]); im[r] = fma(sg, pi, im[r]); }
        else if (KIND == SW_XDAG)            { re[r] = re[r] + pi; im[r] = im[r] - pr; }   // mine - i partner
        else                                 { re[r] = re[r] - pi; im[r] = im[r] + pr; }   // mine + i partner
    }
}

__device__ __forceinline__ int slot_of(int f) { return f ^ ((f >> 5) & 7); }
__device__ __forceinline__ int f_layout1(int t, int r) { return t | (r << 7); }
__device__ __forceinline__ int f_layout2(int t, int r) { return (t & 3) | (r << 2) | ((t >> 2) << 7); }

template <bool FROM1>
__device__ __forceinline__ void exchange(double2* sm, double (&re)[32], double (&im)[32], int t)
{
    // registers (layout FROM1 ? 1 : 2) -> shared -> registers (the other layout)
    __syncthreads();     // earlier readers of the buffer are done
#pragma unroll
    for (int r = 0; r < 32; ++r) {
        const int f = FROM1 ? f_layout1(t, r) : f_layout2(t, r);
        sm[slot_of(f)] = make_double2(re[r], im[r]);
    }
    __syncthreads();
#pragma unroll
    for (int r = 0; r < 32; ++r) {
        const int f = FROM1 ? f_layout2(t, r) : f_layout1(t, r);
        const double2 v = sm[slot_of(f)];
        re[r] = v.x; im[r] = v.y;
    }
}

// Per-tile phase preparation.  With X = spins outside the tile (fixed by the tile index tau),
// T = spins on thread bits, R = spins on register bits at diagonal time:
//   a_j   = sum_{x in X} Jeff_jx sigma_x(tau)                                          (effective field from X)
//   sph[0]      = exp(-it [E_X(tau) - 1/2 sum_{i in R} a_i])
//   sph[1+v]    = exp(-it sum_{b<4} sigma_b(v) a_{T_b}),  v < 16      (thread bits 0..3)
//   sph[17+v]   = exp(-it sum_{b<3} sigma_b(v) a_{T_{4+b}}),  v < 8   (thread bits 4..6)
//   sph[25+i]   = exp(-it a_{R_i}),  i < 5
__device__ __forceinline__ void tile_phase_prep(const TilePassParams& p, uint64_t tau, int t, double* s_a,
                                                double2* s_ph)
{
    const DiagDesc* __restrict__ d = p.desc;
    const int nfixed = d->nfixed;
    if (t < p.N) {
        double a = 0.0;
        const double* __restrict__ row = p.Jeff + (size_t)t * TS_MAX_N;
        for (int x = 0; x < nfixed; ++x) {
            const double sg = (double)((tau >> x) & 1) - 0.5;
            a = fma(row[d->xspin[x]], sg, a);
        }
        s_a[t] = a;
    }
    __syncthreads();
    if (t < 30) {
        double E = 0.0;
        if (t == 0) {
            for (int x = 0; x < nfixed; ++x) {
                const int sp = d->xspin[x];
                const double sg = (double)((tau >> x) & 1) - 0.5;
                E = fma(sg, p.h[sp] + 0.5 * s_a[sp], E);
            }
            double ar = 0.0;
            for (int i = 0; i < 5; ++i) ar += s_a[d->rspin[i]];
            E -= 0.5 * ar;
        } else if (t < 17) {
            const int v = t - 1;
            for (int b = 0; b < 4; ++b) E = fma((double)((v >> b) & 1) - 0.5, s_a[d->tspin[b]], E);
        } else if (t < 25) {
            const int v = t - 17;
            for (int b = 0; b < 3; ++b) E = fma((double)((v >> b) & 1) - 0.5, s_a[d->tspin[4 + b]], E);
        } else {
            E = s_a[d->rspin[t - 25]];
        }
        double sn, cs;
        sincos(-d->t * E, &sn, &cs);
        s_ph[t] = make_double2(cs, sn);
    }
}

// z / |z| to first order (|z|^2 = 1 + O(1e-15)): removes the modulus bias that table entries shared by many
// amplitudes would otherwise add to the norm at every diagonal.
__device__ __forceinline__ double2 cunit(double2 z)
{
    const double f = fma(-0.5, fma(z.x, z.x, z.y * z.y), 1.5);
    return make_double2(z.x * f, z.y * f);
}

// c_r <- c_r * P[r],  P[r] = scale * base * RR[r] * prod_i w_i^{r_i}   (depth-first product tree: 31 + 32 + 32 cmul)
__device__ __forceinline__ void apply_diag(const TilePassParams& p, int t, const double2* s_ph,
                                           double (&re)[32], double (&im)[32])
{
    const DiagDesc* __restrict__ d = p.desc;
    double2 base = cmul(s_ph[0], d->TT[t]);
    base = cmul(base, s_ph[1 + (t & 15)]);
    base = cunit(cmul(base, s_ph[17 + (t >> 4)]));
    const double scale = d->scale;          // exact power of two
    base.x *= scale; base.y *= scale;
    double2 w[5];
#pragma unroll
    for (int i = 0; i < 5; ++i) w[i] = cunit(cmul(s_ph[25 + i], d->WT[i][t]));
#pragma unroll
    for (int b4 = 0; b4 < 2; ++b4) {
        const double2 q4 = b4 ? cmul(base, w[4]) : base;
#pragma unroll
        for (int b3 = 0; b3 < 2; ++b3) {
            const double2 q3 = b3 ? cmul(q4, w[3]) : q4;
#pragma unroll
            for (int b2 = 0; b2 < 2; ++b2) {
                const double2 q2 = b2 ? cmul(q3, w[2]) : q3;
#pragma unroll
                for (int b1 = 0; b1 < 2; ++b1) {
                    const double2 q1 = b1 ? cmul(q2, w[1]) : q2;
#pragma unroll
                    for (int b0 = 0; b0 < 2; ++b0) {
                        const double2 q0 = b0 ? cmul(q1, w[0]) : q1;
                        const int r = b0 | (b1 << 1) | (b2 << 2) | (b3 << 3) | (b4 << 4);
                        const double2 ph = cmul(q0, d->RR[r]);
                        const double2 c = cmul(make_double2(re[r], im[r]), ph);
                        re[r] = c.x; im[r] = c.y;
                    }
                }
            }
        }
    }
}

template <int K1, int K2>
__global__ void __launch_bounds__(TS_TILE_THREADS, 2) k_tile_pass(const TilePassParams p)
{
    extern __shared__ double2 sm[];          // 4096 slots when p.two_stage
    __shared__ double s_a[TS_MAX_N];
    __shared__ double2 s_ph[32];

    const int t = threadIdx.x;
    const int lane = t & 31;
    const uint64_t tau = blockIdx.x;
    const int s = p.s, g0 = p.g0;
    const int nmid = g0 - s;
    const uint64_t base = ((tau & (((uint64_t)1 << nmid) - 1)) << s) | ((tau >> nmid) << (g0 + TS_TILE_LOG2 - s));
    const uint64_t runmask = ((uint64_t)1 << s) - 1;

    // global element offset of in-tile index f: run bits stay, group bits move up to g0
    uint64_t offb[5];
#pragma unroll
    for (int b = 0; b < 5; ++b) {
        const uint64_t f = (uint64_t)1 << (7 + b);
        offb[b] = (f & runmask) | ((f >> s) << g0);
    }
    const uint64_t offt = ((uint64_t)t & runmask) | (((uint64_t)t >> s) << g0);
    double2* __restrict__ gp = p.psi + base + offt;

    double re[32], im[32];
#pragma unroll
    for (int r = 0; r < 32; ++r) {
        uint64_t o = 0;
#pragma unroll
        for (int b = 0; b < 5; ++b) if (r & (1 << b)) o |= offb[b];
        const double2 v = __ldcs(gp + o);
        re[r] = v.x; im[r] = v.y;
    }

    if (p.desc) tile_phase_prep(p, tau, t, s_a, s_ph);   // overlaps the loads in flight

    // ---- sweep K1
    bfly_regs<K1>(re, im, p.bf1);
    if (p.two_stage) {
        exchange<true>(sm, re, im, t);
        bfly_regs<K1>(re, im, p.bf2);
        if (p.nshfl) { bfly_lane<K1>(re, im, 0, lane); bfly_lane<K1>(re, im, 1, lane); }
    }
    // ---- diagonal
    if (p.desc) {
        __syncthreads();                     // s_ph complete
        apply_diag(p, t, s_ph, re, im);
    }
    // ---- sweep K2 (mirror order)
    if (p.two_stage) {
        if (p.nshfl) { bfly_lane<K2>(re, im, 1, lane); bfly_lane<K2>(re, im, 0, lane); }
        bfly_regs<K2>(re, im, p.bf2);
        exchange<false>(sm, re, im, t);
    }
    bfly_regs<K2>(re, im, p.bf1);

#pragma unroll
    for (int r = 0; r < 32; ++r) {
        uint64_t o = 0;
#pragma unroll
        for (int b = 0; b < 5; ++b) if (r & (1 << b)) o |= offb[b];
        __stcs(gp + o, make_double2(re[r], im[r]));
    }
}

// ------------------------------------------------------------------------------------------------ phase tables
struct DescHeader {
    double t, scale;
    int alpha, N, nfixed;
    int rspin[5], tspin[7], xspin[TS_MAX_FIXED];
};

// One block of 128 threads: thread v fills TT[v], WT[0..4][v] and (v < 32) RR[v]; thread 0 writes the header.
__global__ void __launch_bounds__(128) k_build_desc(DiagDesc* __restrict__ out, const DescHeader hd,
                                                    const double* __restrict__ h, const double* __restrict__ Jeff)
{
    const int v = threadIdx.x;
    if (v == 0) {
        out->t = hd.t; out->scale = hd.scale; out->alpha = hd.alpha; out->N = hd.N; out->nfixed = hd.nfixed;
        for (int i = 0; i < 5; ++i) out->rspin[i] = hd.rspin[i];
        for (int i = 0; i < 7; ++i) out->tspin[i] = hd.tspin[i];
        for (int i = 0; i < TS_MAX_FIXED; ++i) out->xspin[i] = hd.xspin[i];
    }
    double sg[7];
    for (int b = 0; b < 7; ++b) sg[b] = (double)((v >> b) & 1) - 0.5;
    // E_T(v): fields and pair couplings among the thread spins
    double ET = 0.0;
    for (int b = 0; b < 7; ++b) {
        double f = h[hd.tspin[b]];
        for (int c = 0; c < b; ++c) f += Jeff[hd.tspin[b] * TS_MAX_N + hd.tspin[c]] * sg[c];
        ET += sg[b] * f;
    }
    double bsum = 0.0;
    for (int i = 0; i < 5; ++i) {
        double bi = 0.0;
        for (int b = 0; b < 7; ++b) bi += Jeff[hd.rspin[i] * TS_MAX_N + hd.tspin[b]] * sg[b];
        bsum += bi;
        double sn, cs;
        sincos(-hd.t * bi, &sn, &cs);
        out->WT[i][v] = make_double2(cs, sn);
    }
    {
        double sn, cs;
        sincos(-hd.t * (ET - 0.5 * bsum), &sn, &cs);
        out->TT[v] = make_double2(cs, sn);
    }
    if (v < 32) {
        double ER = 0.0;
        for (int i = 0; i < 5; ++i) {
            const double si = (double)((v >> i) & 1) - 0.5;
            double f = h[hd.rspin[i]];
            for (int c = 0; c < i; ++c) f += Jeff[hd.rspin[i] * TS_MAX_N + hd.rspin[c]] * ((double)((v >> c) & 1) - 0.5);
            ER += si * f;
        }
        double sn, cs;
        sincos(-hd.t * ER, &sn, &cs);
        out->RR[v] = make_double2(cs, sn);
    }
    // RR is the one table every amplitude of every tile multiplies by un-normalised: dither its entries by one ulp so
    // that the running sum of |z|^2 - 1 over the table stays within one ulp (error diffusion), i.e. its mean modulus
    // bias is ~1e-18 instead of ~1e-17.  The angle changes by <= 1 ulp.
    __syncthreads();
    if (v == 0) {
        double S = 0.0;
        for (int r = 0; r < 32; ++r) {
            double2 z = out->RR[r];
            double best = 0.0; double2 zb = z; bool have = false;
            for (int cand = 0; cand < 3; ++cand) {
                double2 zc = z;
                if (cand) {
                    const bool bigx = fabs(z.x) >= fabs(z.y);
                    double& comp = bigx ? zc.x : zc.y;
                    comp = (cand == 1) ? nextafter(comp, 2.0) : nextafter(comp, -2.0);
                }
                const double pp = zc.x * zc.x, ep = fma(zc.x, zc.x, -pp);
                const double qq = zc.y * zc.y, eq = fma(zc.y, zc.y, -qq);
                const double hi = pp >= qq ? pp : qq, lo = pp >= qq ? qq : pp;
                const double dl = ((hi - 1.0) + lo) + (ep + eq);        // |zc|^2 - 1, accurate
                if (!have || fabs(S + dl) < fabs(S + best)) { best = dl; zb = zc; have = true; }
            }
            S += best;
            out->RR[r] = zb;
        }
    }
}

inline int spin_of_fbit(const TileGroup& g, int f) { return f < g.s ? f : g.g0 + (f - g.s); }
inline int n_bfly(const TileGroup& g) { return g.is_low ? TS_TILE_LOG2 : TS_TILE_LOG2 - g.s; }
inline bool two_stage(const TileGroup& g) { return n_bfly(g) > 5; }

typedef void (*tile_kernel_t)(const TilePassParams);

template <int K1, int K2> tile_kernel_t kptr() { return k_tile_pass<K1, K2>; }

tile_kernel_t pick_kernel(int k1, int k2)
{
#define ROW(K1)                                                                                                   \
    switch (k2) {                                                                                                 \
    case SW_YDAG: return kptr<K1, SW_YDAG>();                                                                     \
    case SW_Y:    return kptr<K1, SW_Y>();                                                                        \
    case SW_XDAG: return kptr<K1, SW_XDAG>();                                                                     \
    case SW_X:    return kptr<K1, SW_X>();                                                                        \
    default:      return kptr<K1, SW_NONE>();                                                                     \
    }
    switch (k1) {
    case SW_YDAG: ROW(SW_YDAG)
    case SW_Y:    ROW(SW_Y)
    case SW_XDAG: ROW(SW_XDAG)
    case SW_X:    ROW(SW_X)
    default:      ROW(SW_NONE)
    }
#undef ROW
    return nullptr;
}

} // namespace

cudaError_t ts_tile_init(void)
{
    for (int k1 = 0; k1 <= SW_NONE; ++k1)
        for (int k2 = 0; k2 <= SW_NONE; ++k2) {
            cudaError_t e = cudaFuncSetAttribute((const void*)pick_kernel(k1, k2),
                                                 cudaFuncAttributeMaxDynamicSharedMemorySize,
                                                 (int)(sizeof(double2) << TS_TILE_LOG2));
            if (e != cudaSuccess) return e;
        }
    return cudaSuccess;
}

cudaError_t ts_tile_build_desc(ts_ctx* c, DiagDesc* d_dst, const DiagOp& d, const TileGroup& g)
{
    DescHeader hd;
    hd.t = d.t;
    hd.scale = ldexp(1.0, d.scale_pow);
    hd.alpha = d.alpha;
    hd.N = c->N;
    hd.nfixed = c->N - TS_TILE_LOG2;
    const bool two = two_stage(g);
    for (int b = 0; b < 5; ++b) hd.rspin[b] = spin_of_fbit(g, two ? 2 + b : 7 + b);
    for (int b = 0; b < 7; ++b) {
        const int f = two ? (b < 2 ? b : 5 + b) : b;     // layout 2: thread bits 0,1 -> f 0,1; 2..6 -> f 7..11
        hd.tspin[b] = spin_of_fbit(g, f);
    }
    bool in_tile[TS_MAX_N] = {false};
    for (int f = 0; f < TS_TILE_LOG2; ++f) in_tile[spin_of_fbit(g, f)] = true;
    int nx = 0;
    for (int i = 0; i < TS_MAX_FIXED; ++i) hd.xspin[i] = 0;
    for (int j = 0; j < c->N; ++j) if (!in_tile[j]) hd.xspin[nx++] = j;    // ascending = tile-index bit order
    ts_prof_begin(c, TS_KC_SETUP);
    k_build_desc<<<1, 128, 0, c->stream>>>(d_dst, hd, c->d_h + d.alpha * TS_MAX_N,
                                           c->d_Jeff + (size_t)d.alpha * TS_MAX_N * TS_MAX_N);
    ts_prof_end(c);
    return cudaGetLastError();
}

cudaError_t ts_tile_pass(ts_ctx* c, const TileGroup& g, int kind1, const DiagDesc* d_desc, int kind2, int alpha)
{
    TilePassParams p;
    p.psi = c->psi;
    p.desc = d_desc;
    p.h = c->d_h + alpha * TS_MAX_N;
    p.Jeff = c->d_Jeff + (size_t)alpha * TS_MAX_N * TS_MAX_N;
    p.N = c->N; p.s = g.s; p.g0 = g.g0;
    const int nb = n_bfly(g);
    p.two_stage = two_stage(g) ? 1 : 0;
    p.nshfl = g.is_low ? 2 : 0;
    if (g.is_low) { p.bf1 = 31u; p.bf2 = 31u; }
    else if (nb <= 5) { p.bf1 = (31u << (5 - nb)) & 31u; p.bf2 = 0u; }          // top nb bits of f 7..11
    else { p.bf1 = 31u; p.bf2 = (31u << (10 - nb)) & 31u; }                       // top nb-5 bits of f 2..6
    const uint64_t ntiles = (uint64_t)1 << (c->N - TS_TILE_LOG2);
    const size_t smem = p.two_stage ? (sizeof(double2) << TS_TILE_LOG2) : 0;
    tile_kernel_t k = pick_kernel(kind1, kind2);
    const bool fused = (kind1 != SW_NONE && kind2 != SW_NONE);
    ts_prof_begin(c, fused ? TS_KC_TILE_FUSED : TS_KC_TILE_SINGLE);
    k<<<(unsigned)ntiles, TS_TILE_THREADS, smem, c->stream>>>(p);
    ts_prof_end(c);
    return cudaGetLastError();
}
