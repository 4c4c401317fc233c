// ts_tile_v3.cuh -- the v2 tile pipeline (ts_tile_v2.cuh: loader warp, storer warp, three in-place 64-KiB tile buffers, TMA
// in and out with the 128-byte swizzle) with SIXTEEN amplitudes per thread instead of 32.
//
// Why: ncu on the 32-amplitude kernels shows nothing saturated -- FP64 pipe ~30 %, issue slots 30-38 %, shared-memory
// pipe < 50 % -- with only two compute warps per scheduler (232 registers per thread): each warp's instruction stream
// (LDS burst -> 320 dependent-by-level DADDs -> STS burst -> barrier ...) leaves its scheduler idle most of the time.
// With 16 amplitudes per thread a tile is worked on by 256 threads (8 warps) at ~112 registers, so an SM holds 16 compute
// warps = four per scheduler, the same two tiles in flight.  Twelve tile bits = three layouts of four register bits, so
// group A needs no warp shuffles at all: K1 in A1, A2, A3; diagonal in A3; K2 in A3, A2, A1 (four in-place exchanges, the
// same shared-memory traffic as two exchanges plus four shuffle rounds).
//
// Register layouts (f bit of each of the 4 register bits / 8 thread bits; every layout keeps one of {f0|f3}, {f1|f4},
// {f2|f5} on each of the three low lane bits = conflict-free 128-bit accesses under slot(f) = f ^ ((f >> 3) & 7)):
//   A1: regs {3,4,5,11}   threads {0,1,2,6,7,8,9,10}      A2: regs {0,1,2,10}  threads {3,4,5,6,7,8,9,11}
//   A3: regs {6,7,8,9}    threads {0,1,2,3,4,5,10,11}
//   H1: regs {8,9,10,11}  threads {0,...,7}                H2: regs {4,5,6,7}   threads {0,1,2,3,8,9,10,11}
// A high group with m group bits butterflies f >= s = 12 - m: f8..11 in H1, f_max(s,4)..7 in H2 (m > 4), and for m = 9 the
// one remaining bit f3 = lane bit 3 of H2 by a warp shuffle.  The diagonal is applied in A3 / H2 (m > 4) / H1.
//
// Phase tables (ts_tile.cu builds them for this geometry): per tile a record of 40 entries -- [0] tp0, [1..16] the four
// low thread bits, [17..32] the four high thread bits, [33..36] the register bits -- and per launch TT[256], WT[4][256],
// RR[16] (1296 entries) in shared memory.
#pragma once
#include "ts_tile_v2.cuh"

#define TS_V3_GROUP_THREADS 256
#define TS_V3_THREADS 640                 // 16 compute warps (two tile groups) + one producer warpgroup
#define TS_V3_REGS_COMPUTE 112            // setmaxnreg: 512 x 112 + 128 x 24 = 60 416 <= 640 x 96 allocated at launch
#define TS_V3_REGS_PRODUCER 24
#define TS_V3_REC 40                      // entries of a tile-phase record (640 bytes)
#define TS_V3_TAB_ENTRIES (5 * 256 + 16)
#define TS_V3_OFF_TP (TS_V2_NBUF * TS_V2_TILE_BYTES)
#define TS_V3_OFF_BAR (TS_V3_OFF_TP + TS_V2_NBUF * TS_V3_REC * 16)
#define TS_V3_OFF_TAB (TS_V3_OFF_BAR + 128)
#define TS_V3_TAB_BYTES (TS_V3_TAB_ENTRIES * 16)
#define TS_V3_SMEM (TS_V3_OFF_TAB + TS_V3_TAB_BYTES)

#define TS_V3_A1_R 0xB543u
#define TS_V3_A1_T 0xA9876210u
#define TS_V3_A2_R 0xA210u
#define TS_V3_A2_T 0xB9876543u
#define TS_V3_A3_R 0x9876u
#define TS_V3_A3_T 0xBA543210u
#define TS_V3_H1_R 0xBA98u
#define TS_V3_H1_T 0x76543210u
#define TS_V3_H2_R 0x7654u
#define TS_V3_H2_T 0xBA983210u

// tab[type][k1][k2]; type 0: group A, 1: high group (run-time masks), 2: high group with 9 group bits
void ts_v3_register_A(v2_kernel_t (*tab)[5][5]);
void ts_v3_register_Hf(v2_kernel_t (*tab)[5][5]);
void ts_v3_register_Hs(v2_kernel_t (*tab)[5][5]);
void ts_v3_register_H9(v2_kernel_t (*tab)[5][5]);
void ts_v3_register_chunk0(v2_chunk_kernel_t (*tab)[2]);
void ts_v3_register_chunk1(v2_chunk_kernel_t (*tab)[2]);
void ts_v3_register_chunk0_h9(v2_chunk_kernel_t (*tab)[2]);
void ts_v3_register_chunk1_h9(v2_chunk_kernel_t (*tab)[2]);

// Butterflied register bits of a high group with m group bits in H1 (bit i <-> f 8 + i) and H2 (bit i <-> f 4 + i).
__host__ __device__ constexpr unsigned v3_h_mask1(int m) { unsigned k = 0; for (int i = 0; i < 4; ++i) if (8 + i >= 12 - m) k |= 1u << i; return k; }
__host__ __device__ constexpr unsigned v3_h_mask2(int m) { unsigned k = 0; for (int i = 0; i < 4; ++i) if (4 + i >= 12 - m) k |= 1u << i; return k; }

#ifdef __CUDACC__
namespace tsk {

template <uint32_t RP, uint32_t TP>
struct V3Layout {
    static __device__ __forceinline__ uint32_t thread_off(int t)
    {
        uint32_t f = 0;
#pragma unroll
        for (int i = 0; i < 8; ++i) f |= (uint32_t)((t >> i) & 1) << ((TP >> (4 * i)) & 15u);
        return (f ^ ((f >> 3) & 7u)) << 4;
    }
    static __host__ __device__ constexpr uint32_t reg_slot(int r)
    {
        uint32_t f = 0;
        for (int i = 0; i < 4; ++i) f |= (uint32_t)((r >> i) & 1) << ((RP >> (4 * i)) & 15u);
        return f ^ ((f >> 3) & 7u);
    }
    static __device__ __forceinline__ double2* ptr(unsigned char* buf, uint32_t toff, int r)
    {
        const uint32_t c = reg_slot(r);
        return reinterpret_cast<double2*>(buf + ((toff ^ ((c & 7u) << 4)) + ((c & ~7u) << 4)));
    }
    static __device__ __forceinline__ void load(unsigned char* buf, uint32_t toff, double (&re)[16], double (&im)[16])
    {
#pragma unroll
        for (int r = 0; r < 16; ++r) {
            const double2 v = *ptr(buf, toff, r);
            re[r] = v.x; im[r] = v.y;
        }
    }
    static __device__ __forceinline__ void store(unsigned char* buf, uint32_t toff, const double (&re)[16], const double (&im)[16])
    {
#pragma unroll
        for (int r = 0; r < 16; ++r) *ptr(buf, toff, r) = make_double2(re[r], im[r]);
    }
};

template <int KIND, int MASK>
__device__ __forceinline__ void v3_bfly_regs(double (&re)[16], double (&im)[16], unsigned mask)
{
    if (KIND == SW_NONE) return;
#pragma unroll
    for (int b = 0; b < 4; ++b) {
        if (MASK >= 0 ? ((MASK >> b) & 1) != 0 : (mask & (1u << b)) != 0) {
#pragma unroll
            for (int r = 0; r < 16; ++r)
                if (!(r & (1 << b))) pair_update<KIND>(re[r], im[r], re[r | (1 << b)], im[r | (1 << b)]);
        }
    }
}

// Butterfly on lane bit lb: each lane holds one member of the pair and fetches the other by shuffle.
template <int KIND>
__device__ __forceinline__ void v3_bfly_lane(double (&re)[16], double (&im)[16], int lb, int lane)
{
    if (KIND == SW_NONE) return;
    const int up = (lane >> lb) & 1;
    const double sg = (KIND == SW_YDAG) ? (up ? 1.0 : -1.0) : (up ? -1.0 : 1.0);
#pragma unroll
    for (int r = 0; r < 16; ++r) {
        const double pr = __shfl_xor_sync(0xffffffffu, re[r], 1 << lb);
        const double pi = __shfl_xor_sync(0xffffffffu, im[r], 1 << lb);
        if (KIND == SW_YDAG || KIND == SW_Y) { re[r] = fma(sg, pr, re[r]); im[r] = fma(sg, pi, im[r]); }
        else if (KIND == SW_XDAG)            { re[r] = re[r] + pi; im[r] = im[r] - pr; }
        else                                 { re[r] = re[r] - pi; im[r] = im[r] + pr; }
    }
}

__device__ __forceinline__ void v3_group_sync(int grp)
{
    asm volatile("bar.sync %0, %1;" ::"r"(grp + 1), "r"(TS_V3_GROUP_THREADS) : "memory");
}

// c_r <- c_r * [scale tp0 TT[t] LN0 LN1] * RR[r] * prod_i (tpW_i WT_i[t])^{r_i}
__device__ __forceinline__ void v3_diag(const double scale, const double2* tp, const double2* tab, const int t, double (&re)[16],
                                        double (&im)[16])
{
    double2 base = cmul(tp[0], tab[t]);
    base = cmul(base, tp[1 + (t & 15)]);
    base = cunit(cmul(base, tp[17 + (t >> 4)]));
    base.x *= scale; base.y *= scale;
    double2 w[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) w[k] = cunit(cmul(tp[33 + k], tab[256 + k * 256 + t]));
    const double2* RR = tab + 1280;
#pragma unroll
    for (int b3 = 0; b3 < 2; ++b3) {
        const double2 q3 = b3 ? cmul(base, w[3]) : base;
#pragma unroll
        for (int b2 = 0; b2 < 2; ++b2) {
            const double2 q2 = b2 ? cmul(q3, w[2]) : q3;
#pragma unroll
            for (int b1 = 0; b1 < 2; ++b1) {
                const double2 q1 = b1 ? cmul(q2, w[1]) : q2;
#pragma unroll
                for (int b0 = 0; b0 < 2; ++b0) {
                    const double2 q0 = b0 ? cmul(q1, w[0]) : q1;
                    const int r = b0 | (b1 << 1) | (b2 << 2) | (b3 << 3);
                    const double2 ph = cmul(q0, RR[r]);
                    const double2 c = cmul(make_double2(re[r], im[r]), ph);
                    re[r] = c.x; im[r] = c.y;
                }
            }
        }
    }
}

// ------------------------------------------------------------------------------------------------ tile bodies
template <int K1, int K2>
__device__ __forceinline__ void v3_body_A(unsigned char* buf, const bool diag, const double scale, const double2* tp,
                                          const double2* tab, const int t, const int grp)
{
    using L1 = V3Layout<TS_V3_A1_R, TS_V3_A1_T>;
    using L2 = V3Layout<TS_V3_A2_R, TS_V3_A2_T>;
    using L3 = V3Layout<TS_V3_A3_R, TS_V3_A3_T>;
    const uint32_t o1 = L1::thread_off(t), o2 = L2::thread_off(t), o3 = L3::thread_off(t);
    double re[16], im[16];
    if (K1 != SW_NONE) {
        L1::load(buf, o1, re, im);
        v3_bfly_regs<K1, 15>(re, im, 0u);              // f 3,4,5,11
        L1::store(buf, o1, re, im);
        v3_group_sync(grp);
        L2::load(buf, o2, re, im);
        v3_bfly_regs<K1, 15>(re, im, 0u);              // f 0,1,2,10
        L2::store(buf, o2, re, im);
        v3_group_sync(grp);
    }
    L3::load(buf, o3, re, im);
    v3_bfly_regs<K1, 15>(re, im, 0u);                  // f 6,7,8,9
    if (diag) v3_diag(scale, tp, tab, t, re, im);
    v3_bfly_regs<K2, 15>(re, im, 0u);
    L3::store(buf, o3, re, im);
    if (K2 != SW_NONE) {
        v3_group_sync(grp);
        L2::load(buf, o2, re, im);
        v3_bfly_regs<K2, 15>(re, im, 0u);
        L2::store(buf, o2, re, im);
        v3_group_sync(grp);
        L1::load(buf, o1, re, im);
        v3_bfly_regs<K2, 15>(re, im, 0u);
        L1::store(buf, o1, re, im);
    }
}

// M > 0: number of group bits known at compile time; M = -1: from g (g.mask1 / g.mask2 / g.two_stage / g.s).
template <int K1, int K2, int M>
__device__ __forceinline__ void v3_body_H(unsigned char* buf, const V2Geom& g, const bool diag, const double scale, const double2* tp,
                                          const double2* tab, const int t, const int grp)
{
    using L1 = V3Layout<TS_V3_H1_R, TS_V3_H1_T>;
    using L2 = V3Layout<TS_V3_H2_R, TS_V3_H2_T>;
    constexpr bool CT = (M > 0);
    constexpr int MK1 = CT ? (int)v3_h_mask1(M > 0 ? M : 1) : -1;
    constexpr int MK2 = CT ? (int)v3_h_mask2(M > 0 ? M : 1) : -1;
    const uint32_t o1 = L1::thread_off(t), o2 = L2::thread_off(t);
    const bool two = CT ? (M > 4) : (g.two_stage != 0);
    const bool shf = CT ? (M == 9) : (g.s == 3);       // f3 = lane bit 3 of H2
    const int lane = t & 31;
    double re[16], im[16];
    L1::load(buf, o1, re, im);
    v3_bfly_regs<K1, MK1>(re, im, g.mask1);
    if (two) {
        L1::store(buf, o1, re, im);
        v3_group_sync(grp);
        L2::load(buf, o2, re, im);
        v3_bfly_regs<K1, MK2>(re, im, g.mask2);
        if (shf) v3_bfly_lane<K1>(re, im, 3, lane);
    }
    if (diag) v3_diag(scale, tp, tab, t, re, im);
    if (K2 != SW_NONE) {
        if (two) {
            if (shf) v3_bfly_lane<K2>(re, im, 3, lane);
            v3_bfly_regs<K2, MK2>(re, im, g.mask2);
            L2::store(buf, o2, re, im);
            v3_group_sync(grp);
            L1::load(buf, o1, re, im);
        }
        v3_bfly_regs<K2, MK1>(re, im, g.mask1);
        L1::store(buf, o1, re, im);
    } else {
        if (two) L2::store(buf, o2, re, im);
        else L1::store(buf, o1, re, im);
    }
}

__device__ __forceinline__ void v3_init_barriers(const uint32_t sBar)
{
    for (int k = 0; k < TS_V2_NBUF; ++k) {
        v2_mbar_init(sBar + 8 * k, 1);                                    // full
        v2_mbar_init(sBar + 8 * (TS_V2_NBUF + k), TS_V3_GROUP_THREADS);   // done
        v2_mbar_init(sBar + 8 * (2 * TS_V2_NBUF + k), 1);                 // free
    }
    v2_mbar_init(sBar + 8 * 3 * TS_V2_NBUF, 1);                           // tab
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    v2_fence_async_smem();
}

// ------------------------------------------------------------------------------------------------ one tile pass
// Same protocol as k_tile_v2 (see ts_tile_v2.cuh); warps 0..15 compute (group = warp / 8), warp 16 loads, warp 17 stores.
template <int TYPE, int K1, int K2>
__global__ void __launch_bounds__(TS_V3_THREADS, 1)
k_tile_v3(const __grid_constant__ V2Pass p, const __grid_constant__ CUtensorMap tmap)
{
    extern __shared__ __align__(1024) unsigned char smraw[];
    const uint32_t sBase = v2_smem_u32(smraw);
    const uint32_t sBar = sBase + TS_V3_OFF_BAR;
    const int warp = threadIdx.x >> 5;
    const uint64_t G = gridDim.x;
    const uint64_t n_cta = (p.ntiles > blockIdx.x) ? (p.ntiles - blockIdx.x + G - 1) / G : 0;
    const bool has_diag = (p.d.tile_phase != nullptr);

    if (threadIdx.x == 0) {
        if (sBase & 1023u) __trap();
        v3_init_barriers(sBar);
    }
    __syncthreads();

    if (warp >= 16) {                                  // ---- producer warpgroup
        v2_regs_dec<TS_V3_REGS_PRODUCER>();
        if (warp == 16 && (threadIdx.x & 31) == 0) {   // ---- loader
            if (has_diag) {
                v2_mbar_expect_tx(sBar + 8 * 3 * TS_V2_NBUF, TS_V3_TAB_BYTES);
                v2_bulk_load(sBase + TS_V3_OFF_TAB, p.d.tables, TS_V3_TAB_BYTES, sBar + 8 * 3 * TS_V2_NBUF);
            }
            for (uint64_t j = 0; j < n_cta; ++j) {
                const uint32_t b = (uint32_t)(j % TS_V2_NBUF), use = (uint32_t)(j / TS_V2_NBUF);
                if (use > 0) v2_mbar_wait(sBar + 8 * (2 * TS_V2_NBUF + b), (use - 1) & 1u);
                const uint64_t tile = blockIdx.x + j * G;
                const uint32_t bar = sBar + 8 * b;
                v2_mbar_expect_tx(bar, TS_V2_TILE_BYTES + (has_diag ? TS_V3_REC * 16u : 0u));
                if (has_diag)
                    v2_bulk_load(sBase + TS_V3_OFF_TP + b * (TS_V3_REC * 16u), p.d.tile_phase + tile * TS_V3_REC, TS_V3_REC * 16u, bar);
                v2_issue_load(p.g, &tmap, tile, sBase + b * TS_V2_TILE_BYTES, bar);
            }
        } else if (warp == 17 && (threadIdx.x & 31) == 0) {   // ---- storer
            for (uint64_t j = 0; j < n_cta; ++j) {
                const uint32_t b = (uint32_t)(j % TS_V2_NBUF), use = (uint32_t)(j / TS_V2_NBUF);
                v2_mbar_wait(sBar + 8 * (TS_V2_NBUF + b), use & 1u);
                v2_issue_store(p.g, &tmap, blockIdx.x + j * G, sBase + b * TS_V2_TILE_BYTES);
                v2_store_commit();
                v2_store_wait_read();
                v2_mbar_arrive(sBar + 8 * (2 * TS_V2_NBUF + b));
            }
            v2_store_wait_all();
        }
    } else {                                           // ---- compute warpgroups
        v2_regs_inc<TS_V3_REGS_COMPUTE>();
        const int grp = warp >> 3;
        const int t = threadIdx.x & (TS_V3_GROUP_THREADS - 1);
        const double2* tab = reinterpret_cast<const double2*>(smraw + TS_V3_OFF_TAB);
        const double scale = p.d.scale;
        if (has_diag) v2_mbar_wait(sBar + 8 * 3 * TS_V2_NBUF, 0u);
        for (uint64_t j = grp; j < n_cta; j += 2) {
            const uint32_t b = (uint32_t)(j % TS_V2_NBUF), use = (uint32_t)(j / TS_V2_NBUF);
            v2_wait_full(sBar + 8 * b, sBar + 8 * (TS_V2_NBUF + b), use);
            unsigned char* buf = smraw + b * TS_V2_TILE_BYTES;
            const double2* tp = reinterpret_cast<const double2*>(smraw + TS_V3_OFF_TP + b * (TS_V3_REC * 16u));
            if constexpr (TYPE == 0) v3_body_A<K1, K2>(buf, has_diag, scale, tp, tab, t, grp);
            else if constexpr (TYPE == 2) v3_body_H<K1, K2, 9>(buf, p.g, has_diag, scale, tp, tab, t, grp);
            else v3_body_H<K1, K2, -1>(buf, p.g, has_diag, scale, tp, tab, t, grp);
            v2_fence_async_smem();
            v2_mbar_arrive(sBar + 8 * (TS_V2_NBUF + b));
        }
    }
}

// ------------------------------------------------------------------------------------------------ L2-blocked triple
// Same job order, dependency protocol and L2 priorities as k_chunk_v2 (ts_tile_v2.cuh).
template <int KA, int KB, int HM>
__global__ void __launch_bounds__(TS_V3_THREADS, 1)
k_chunk_v3(const __grid_constant__ V2Chunk q, const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmH)
{
    extern __shared__ __align__(1024) unsigned char smraw[];
    const uint32_t sBase = v2_smem_u32(smraw);
    const uint32_t sBar = sBase + TS_V3_OFF_BAR;
    const int warp = threadIdx.x >> 5;
    const uint32_t tl = q.tiles_log2, T = 1u << tl;
    const uint32_t nblocks = 3u * q.nchunks;
    const uint64_t total = (uint64_t)nblocks << tl;
    const uint64_t G = gridDim.x;
    const uint64_t n_cta = (total > blockIdx.x) ? (total - blockIdx.x + G - 1) / G : 0;
    const bool has_diag = (q.d.tile_phase != nullptr);

    auto job_of = [&](const uint64_t j, uint32_t& phase, uint32_t& c, uint64_t& tile) {
        const uint64_t n = blockIdx.x + j * G;
        const uint32_t B = (uint32_t)(n >> tl);
        if (B == nblocks - 1) { phase = 2; c = q.nchunks - 1; }
        else if (B < 5) { phase = (B < 2) ? 0u : (B < 4 ? 1u : 2u); c = (B == 1 || B == 3) ? 1u : 0u; }
        else {
            const uint32_t k = B - 5, r = k % 3;
            c = 2 + k / 3;
            if (r == 0) phase = 0; else if (r == 1) { phase = 2; c -= 1; } else phase = 1;
        }
        tile = ((uint64_t)c << tl) | (n & (T - 1));
    };

    if (threadIdx.x == 0) {
        if (sBase & 1023u) __trap();
        v3_init_barriers(sBar);
    }
    __syncthreads();

    if (warp >= 16) {                                  // ---- producer warpgroup
        v2_regs_dec<TS_V3_REGS_PRODUCER>();
        if (warp == 16 && (threadIdx.x & 31) == 0) {   // ---- loader
            if (has_diag) {
                v2_mbar_expect_tx(sBar + 8 * 3 * TS_V2_NBUF, TS_V3_TAB_BYTES);
                v2_bulk_load(sBase + TS_V3_OFF_TAB, q.d.tables, TS_V3_TAB_BYTES, sBar + 8 * 3 * TS_V2_NBUF);
            }
            const uint64_t pol_ld[3] = {v2_policy(q.l2_hints ? 1 : 0), v2_policy(q.l2_hints ? 2 : 0), v2_policy(q.l2_hints ? 1 : 0)};
            uint32_t ok_key = 0xffffffffu;
            for (uint64_t j = 0; j < n_cta; ++j) {
                const uint32_t b = (uint32_t)(j % TS_V2_NBUF), use = (uint32_t)(j / TS_V2_NBUF);
                uint32_t phase, c; uint64_t tile;
                job_of(j, phase, c, tile);
                if (phase != 0) {
                    const uint32_t key = (phase << 28) | c;
                    if (key != ok_key) {
                        const unsigned int* dp = q.done + (size_t)(phase - 1) * q.nchunks + c;
                        while (v2_ld_acquire(dp) < T) __nanosleep(64);
                        ok_key = key;
                    }
                    v2_fence_async_all();
                }
                if (use > 0) v2_mbar_wait(sBar + 8 * (2 * TS_V2_NBUF + b), (use - 1) & 1u);
                const uint32_t bar = sBar + 8 * b;
                const bool tpl = has_diag && phase == 1;
                v2_mbar_expect_tx(bar, TS_V2_TILE_BYTES + (tpl ? TS_V3_REC * 16u : 0u));
                if (tpl)
                    v2_bulk_load(sBase + TS_V3_OFF_TP + b * (TS_V3_REC * 16u), q.d.tile_phase + tile * TS_V3_REC, TS_V3_REC * 16u, bar);
                if (phase == 1) v2_issue_load_h(q.ga, &tmA, tile, sBase + b * TS_V2_TILE_BYTES, bar, pol_ld[1]);
                else v2_issue_load_h(q.gh, &tmH, tile, sBase + b * TS_V2_TILE_BYTES, bar, pol_ld[phase]);
            }
        } else if (warp == 17 && (threadIdx.x & 31) == 0) {   // ---- storer
            const uint64_t pol_st[3] = {v2_policy(q.l2_hints ? 2 : 0), v2_policy(q.l2_hints ? 2 : 0), v2_policy(q.l2_hints ? 1 : 0)};
            for (uint64_t j = 0; j < n_cta; ++j) {
                const uint32_t b = (uint32_t)(j % TS_V2_NBUF), use = (uint32_t)(j / TS_V2_NBUF);
                uint32_t phase, c; uint64_t tile;
                job_of(j, phase, c, tile);
                v2_mbar_wait(sBar + 8 * (TS_V2_NBUF + b), use & 1u);
                if (phase == 1) v2_issue_store_h(q.ga, &tmA, tile, sBase + b * TS_V2_TILE_BYTES, pol_st[1]);
                else v2_issue_store_h(q.gh, &tmH, tile, sBase + b * TS_V2_TILE_BYTES, pol_st[phase]);
                v2_store_commit();
                v2_store_wait_read();
                v2_mbar_arrive(sBar + 8 * (2 * TS_V2_NBUF + b));
                if (phase != 2) {
                    v2_store_wait_all();
                    v2_fence_async_all();
                    __threadfence();
                    atomicAdd(q.done + (size_t)phase * q.nchunks + c, 1u);
                }
            }
            v2_store_wait_all();
        }
    } else {                                           // ---- compute warpgroups
        v2_regs_inc<TS_V3_REGS_COMPUTE>();
        const int grp = warp >> 3;
        const int t = threadIdx.x & (TS_V3_GROUP_THREADS - 1);
        const double2* tab = reinterpret_cast<const double2*>(smraw + TS_V3_OFF_TAB);
        const double scale = q.d.scale;
        if (has_diag) v2_mbar_wait(sBar + 8 * 3 * TS_V2_NBUF, 0u);
        for (uint64_t j = grp; j < n_cta; j += 2) {
            const uint32_t b = (uint32_t)(j % TS_V2_NBUF), use = (uint32_t)(j / TS_V2_NBUF);
            uint32_t phase, c; uint64_t tile;
            job_of(j, phase, c, tile);
            v2_wait_full(sBar + 8 * b, sBar + 8 * (TS_V2_NBUF + b), use);
            unsigned char* buf = smraw + b * TS_V2_TILE_BYTES;
            const double2* tp = reinterpret_cast<const double2*>(smraw + TS_V3_OFF_TP + b * (TS_V3_REC * 16u));
            if (phase == 0) v3_body_H<KA, SW_NONE, HM>(buf, q.gh, false, 1.0, tp, tab, t, grp);
            else if (phase == 1) v3_body_A<KA, KB>(buf, has_diag, scale, tp, tab, t, grp);
            else v3_body_H<KB, SW_NONE, HM>(buf, q.gh, false, 1.0, tp, tab, t, grp);
            v2_fence_async_smem();
            v2_mbar_arrive(sBar + 8 * (TS_V2_NBUF + b));
        }
    }
}

} // namespace tsk
#endif
