// ts_tile_kernel.cuh -- the tile-pass arithmetic and its first kernel, k_tile_pass: one CTA per tile,
// loads and stores straight from registers.  The production kernels (ts_tile_v2.cuh) reuse the butterfly and
// phase-table code below and differ in how tiles travel; k_tile_pass stays as the fallback for geometries they do not
// take and as the A/B baseline.  Included by ts_tile_cfgG.cu, ts_tile_v2.cuh and ts_tile.cu.
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
//
// Diagonal.  With X = spins outside the tile (fixed by the tile index tau), T = the 7 spins on thread
// bits and R = the 5 spins on register bits at diagonal time, sigma = bit - 1/2, and
//   a_j(tau) = sum_{x in X} Jeff_jx sigma_x(tau),   b_i(t) = sum_{j in T} Jeff_ij sigma_j(t)
// the phase of amplitude (tau, t, r) is
//   P = scale * [tp0 * tpLN0[t & 15] * tpLN1[t >> 4] * TT[t]] * RR[r] * prod_{i<5} (tpW_i * WT_i[t])^{r_i}
//   tp0      = exp(-i t [E_X(tau) - 1/2 sum_{i in R} a_i])            per tile     (tile-phase table, 32 entries/tile)
//   tpLN0[v] = exp(-i t sum_{b<4} sigma_b(v) a_{T_b}),  tpLN1[v] = same for thread bits 4..6      per tile
//   tpW_i    = exp(-i t a_{R_i})                                       per tile
//   TT[t]    = exp(-i t [E_T(t) - 1/2 sum_i b_i(t)]),  WT_i[t] = exp(-i t b_i(t))                  per (kind, group)
//   RR[r]    = exp(-i t E_R(r))                                        per (kind, group), passed in the parameters
// All table entries are built once per (diagonal kind, group) with full-accuracy sincos; the hot kernel only does
// complex multiplications: 8 per thread + (31 + 32 + 32)/32 per amplitude.
#pragma once
#include "ts_internal.h"

struct TilePassParams {
    double2* psi;
    uint64_t tile_base;          // first tile of this launch (L2-blocked runs launch a window of tiles)
    const double2* tile_phase;   // [ntiles][32]   (NULL: no diagonal in this pass)
    const double2* TT;           // [128]
    const double2* WT;           // [5][128]
    double scale;                // exact power of two
    int s, g0;
    int two_stage;               // layout 2 is used (more than 5 butterflied bits)     (generic kernel only)
    int nshfl;                   // 2 for group A, else 0                                  (generic kernel only)
    unsigned bf1, bf2;           // butterflied register bits in layout 1 / layout 2, sweep K1   (generic kernel only)
    unsigned bf1b, bf2b;         // the same for sweep K2 (equal to bf1, bf2 except in a sharded sweep's arrival pass)
    double2 RR[32];              // read straight from the constant bank
    // ---- peer-memory pass of a sharded state vector (k_tile_pass_p2p, ts_shard.cu): the tile's rows whose top `p2p_gbits`
    // row bits equal rho are LOADED from peers[rho] -- rank rho's shard as mapped into this device, read over NVLink --
    // at the position that has this rank's number in those bits (the all-to-all index-bit swap folded into the load), and
    // the finished tile is stored to `dst` (this rank's other buffer).  Unused (gbits = 0) by the in-place passes.
    const double2* peers[8];
    double2* dst;
    int p2p_gbits, p2p_rank;
};

typedef void (*tile_kernel_t)(const TilePassParams);

// registry filled by ts_tile_cfgG.cu
void ts_tile_register_generic(tile_kernel_t (*tab)[5][5]);
void ts_tile_register_p2p(tile_kernel_t (*tab)[5][5]);   // [k1][k2]: k_tile_pass_p2p

#ifdef __CUDACC__
namespace tsk {

__device__ __forceinline__ double2 cmul(double2 a, double2 b)
{
    return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}

// z / |z| to first order (|z|^2 = 1 + O(1e-15)): removes the modulus bias that table entries shared by many
// amplitudes would otherwise add to the norm at every diagonal.
__device__ __forceinline__ double2 cunit(double2 z)
{
    const double f = fma(-0.5, fma(z.x, z.x, z.y * z.y), 1.5);
    return make_double2(z.x * f, z.y * f);
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

// Butterflies on the register bits selected by MASK (compile time) or `mask` (MASK < 0, uniform across the grid).
template <int KIND, int MASK>
__device__ __forceinline__ void bfly_regs(double (&re)[32], double (&im)[32], unsigned mask)
{
    if (KIND == SW_NONE) return;
#pragma unroll
    for (int b = 0; b < 5; ++b) {
        if (MASK >= 0 ? ((MASK >> b) & 1) != 0 : (mask & (1u << b)) != 0) {
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
    if (!FROM1) __syncthreads();     // readers of the first exchange are done
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

// c_r <- c_r * P[r]   (depth-first product tree: 31 + 32 + 32 complex multiplications per thread)
__device__ __forceinline__ void apply_diag(const TilePassParams& p, double2 base, const double2 (&w)[5],
                                           double (&re)[32], double (&im)[32])
{
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
                        const double2 ph = cmul(q0, p.RR[r]);
                        const double2 c = cmul(make_double2(re[r], im[r]), ph);
                        re[r] = c.x; im[r] = c.y;
                    }
                }
            }
        }
    }
}

// One tile: load (layout 1), sweep K1, diagonal, sweep K2, store in place.  CG bit 0: bypass L1 on the loads
// (ld.global.cg); bit 1: keep the stores in L2 (st.global.cg) instead of streaming them out (st.global.cs).
template <int K1, int K2, int BF1, int BF2, int NSHFL, int CG, bool P2P = false>
__device__ __forceinline__ void tile_body(const TilePassParams& p, const uint64_t tau, double2* sm)
{
    constexpr bool GENERIC = (BF1 < 0);
    const bool two_stage = GENERIC ? (p.two_stage != 0) : (BF2 != 0);
    const int nshfl = GENERIC ? p.nshfl : NSHFL;

    const int t = threadIdx.x;
    const int lane = t & 31;
    const int s = p.s, g0 = p.g0;
    const int nmid = g0 - s;
    const uint64_t base_idx =
        ((tau & (((uint64_t)1 << nmid) - 1)) << s) | ((tau >> nmid) << (g0 + TS_TILE_LOG2 - s));
    const uint64_t runmask = ((uint64_t)1 << s) - 1;

    // global element offset of in-tile index f: run bits stay, group bits move up to g0
    uint64_t offb[5];
#pragma unroll
    for (int b = 0; b < 5; ++b) {
        const uint64_t f = (uint64_t)1 << (7 + b);
        offb[b] = (f & runmask) | ((f >> s) << g0);
    }
    const uint64_t offt = ((uint64_t)t & runmask) | (((uint64_t)t >> s) << g0);
    double2* __restrict__ gp = p.psi + base_idx + offt;

    double re[32], im[32];
    if (P2P) {
        // register bits 5 - gbits .. 4 are the tile's top row bits: they name the peer the row comes from; in the peer's
        // shard the row sits where those bits spell THIS rank
        const int lowb = 5 - p.p2p_gbits;
        uint64_t rank_off = 0;
#pragma unroll
        for (int b = 0; b < 5; ++b) if (b >= lowb && ((p.p2p_rank >> (b - lowb)) & 1)) rank_off |= offb[b];
        const uint64_t toff = base_idx + offt + rank_off;
#pragma unroll
        for (int r = 0; r < 32; ++r) {
            uint64_t o = 0;
#pragma unroll
            for (int b = 0; b < 5; ++b) if ((r & (1 << b)) && b < lowb) o |= offb[b];
            const double2 v = __ldcs(p.peers[r >> lowb] + toff + o);
            re[r] = v.x; im[r] = v.y;
        }
    } else {
#pragma unroll
        for (int r = 0; r < 32; ++r) {
            uint64_t o = 0;
#pragma unroll
            for (int b = 0; b < 5; ++b) if (r & (1 << b)) o |= offb[b];
            const double2 v = (CG & 1) ? __ldcg(gp + o) : __ldcs(gp + o);
            re[r] = v.x; im[r] = v.y;
        }
    }

    // phase factors of this thread (loads overlap the data loads in flight)
    double2 base = make_double2(1.0, 0.0), w[5];
    const bool has_diag = (p.tile_phase != nullptr);
    if (has_diag) {
        const double2* __restrict__ tp = p.tile_phase + (tau << 5);
        base = cmul(__ldg(tp), __ldg(p.TT + t));
        base = cmul(base, __ldg(tp + 1 + (t & 15)));
        base = cunit(cmul(base, __ldg(tp + 17 + (t >> 4))));
        base.x *= p.scale; base.y *= p.scale;
#pragma unroll
        for (int i = 0; i < 5; ++i) w[i] = cunit(cmul(__ldg(tp + 25 + i), __ldg(p.WT + i * 128 + t)));
    }

    // ---- sweep K1
    bfly_regs<K1, BF1>(re, im, p.bf1);
    if (two_stage) {
        exchange<true>(sm, re, im, t);
        bfly_regs<K1, BF2>(re, im, p.bf2);
        if (nshfl) { bfly_lane<K1>(re, im, 0, lane); bfly_lane<K1>(re, im, 1, lane); }
    }
    // ---- diagonal
    if (has_diag) apply_diag(p, base, w, re, im);
    // ---- sweep K2 (mirror order)
    if (two_stage) {
        if (nshfl) { bfly_lane<K2>(re, im, 1, lane); bfly_lane<K2>(re, im, 0, lane); }
        bfly_regs<K2, BF2>(re, im, p.bf2b);
        exchange<false>(sm, re, im, t);
    }
    bfly_regs<K2, BF1>(re, im, p.bf1b);

    double2* __restrict__ sp = P2P ? (p.dst + base_idx + offt) : gp;
#pragma unroll
    for (int r = 0; r < 32; ++r) {
        uint64_t o = 0;
#pragma unroll
        for (int b = 0; b < 5; ++b) if (r & (1 << b)) o |= offb[b];
        if (CG & 2) __stcg(sp + o, make_double2(re[r], im[r]));
        else __stcs(sp + o, make_double2(re[r], im[r]));
    }
}

template <int K1, int K2, int BF1, int BF2, int NSHFL, int MINB>
__global__ void __launch_bounds__(TS_TILE_THREADS, MINB) k_tile_pass(const __grid_constant__ TilePassParams p)
{
    extern __shared__ double2 sm[];          // 4096 slots when layout 2 is used
    tile_body<K1, K2, BF1, BF2, NSHFL, 0>(p, p.tile_base + blockIdx.x, sm);
}

// Sweep K1's butterflies on the top p2p_gbits bits of the group, the diagonal, then sweep K2's butterflies on ALL of the
// group's bits (the next sweep starts with this group); tiles gathered from peer memory.
template <int K1, int K2>
__global__ void __launch_bounds__(TS_TILE_THREADS, 2) k_tile_pass_p2p(const __grid_constant__ TilePassParams p)
{
    extern __shared__ double2 sm[];
    tile_body<K1, K2, -1, -1, 0, 0, true>(p, p.tile_base + blockIdx.x, sm);
}

} // namespace tsk
#endif
