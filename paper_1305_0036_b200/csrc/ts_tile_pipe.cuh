// ts_tile_pipe.cuh -- the tile pass as a persistent, TMA-fed pipeline (DESIGN.md 7.1 "pipelined").
//
// Same mathematics, tile geometry, register layouts and phase tables as k_tile_pass (ts_tile_kernel.cuh); what
// changes is how tiles travel.  One CTA per SM walks over tiles b, b + G, b + 2G, ...; its 256 threads form two
// compute groups of 128 that take alternate tiles, so one group's shared-memory/shuffle phases overlap the other's
// FP64 phases.  Loads are asynchronous bulk copies (TMA) into a ring of three half-tile slots (32 KiB each):
//   * contiguous tiles (group A) and high groups with rows >= 4 KiB: 1-D cp.async.bulk per row;
//   * high groups with short runs (128-B runs at N = 30): one 3-D tensor-map box {run, rows, 1} per half tile,
// each completing on the slot's mbarrier; the 512-B tile-phase record rides on the first half's barrier.  A group
// reads a landed half into registers (layout 1 is linear in the slot, so the read is bank-conflict-free), and the
// same group then refills the slot with the half three positions ahead: HBM reads for the next tiles are always in
// flight while a tile is being computed -- the old kernel's load -> compute -> store phases did not overlap (9.2 ms
// per fused group-A pass against a 4.9 ms copy).  Stores go straight from registers (coalesced st.global.cs).
//
// Shared memory: 3 x 32 KiB ring + 2 x 64 KiB exchange buffers (one per group) + 3 x 512 B phase records + barriers.
#pragma once
#include <cuda.h>

#include "ts_tile_kernel.cuh"

#define TS_PIPE_THREADS 256
#define TS_PIPE_SLOTS 3
#define TS_PIPE_HALF_BYTES 32768
#define TS_PIPE_OFF_E (TS_PIPE_SLOTS * TS_PIPE_HALF_BYTES)
#define TS_PIPE_OFF_TP (TS_PIPE_OFF_E + 2 * 65536)
#define TS_PIPE_OFF_BAR (TS_PIPE_OFF_TP + TS_PIPE_SLOTS * 512)
#define TS_PIPE_SMEM (TS_PIPE_OFF_BAR + 128)

struct PipeGeom {
    uint64_t ntiles;      // tiles of this launch
    int is_low;           // contiguous tile: one 32 KiB bulk copy per half
    int tensor;           // 1: tensor-map boxes, 0: 1-D bulk copies per row
    int rows_half;        // rows per half tile
    int row_bytes;        // 16 << s
    int box_rows, nbox;   // tensor mode: boxes per half tile
    int pf;               // L2 prefetch distance in half tiles (0 = off): TMA prefetches into L2 cost no shared memory
    unsigned long long* dbg;   // TS_DEBUG: [0] mismatches between landed halves and direct global reads, [1..4] first one
};

typedef void (*pipe_kernel_t)(const TilePassParams, const CUtensorMap, const PipeGeom);

void ts_pipe_register_generic(pipe_kernel_t (*tab)[5][5]);
void ts_pipe_register_A(pipe_kernel_t (*tab)[5][5]);
void ts_pipe_register_H7(pipe_kernel_t (*tab)[5][5]);
void ts_pipe_register_H8(pipe_kernel_t (*tab)[5][5]);
void ts_pipe_register_H9(pipe_kernel_t (*tab)[5][5]);
void ts_pipe_register_H10(pipe_kernel_t (*tab)[5][5]);

#ifdef __CUDACC__
namespace tsk {

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity)
{
    uint32_t ok;
    do {
        asm volatile(
            "{\n\t.reg .pred p;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t}"
            : "=r"(ok)
            : "r"(bar), "r"(parity)
            : "memory");
    } while (!ok);
}
__device__ __forceinline__ void bulk_load(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
                 "l"(src), "r"(bytes), "r"(bar)
                 : "memory");
}
__device__ __forceinline__ void tensor_load_3d(uint32_t dst, const CUtensorMap* tm, uint32_t bar, int c0, int c1, int c2)
{
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];" ::"r"(dst),
        "l"(tm), "r"(bar), "r"(c0), "r"(c1), "r"(c2)
        : "memory");
}
__device__ __forceinline__ void bulk_prefetch_l2(const void* src, uint32_t bytes)
{
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(src), "r"(bytes) : "memory");
}
__device__ __forceinline__ void tensor_prefetch_l2_3d(const CUtensorMap* tm, int c0, int c1, int c2)
{
    asm volatile("cp.async.bulk.prefetch.tensor.3d.L2.global.tile [%0, {%1, %2, %3}];" ::"l"(tm), "r"(c0), "r"(c1), "r"(c2)
                 : "memory");
}
__device__ __forceinline__ void group_sync(int grp)
{
    asm volatile("bar.sync %0, %1;" ::"r"(grp + 1), "r"(TS_TILE_THREADS) : "memory");
}

template <bool FROM1>
__device__ __forceinline__ void exchange_g(double2* sm, double (&re)[32], double (&im)[32], int t, int grp)
{
    if (!FROM1) group_sync(grp);     // readers of the first exchange are done
#pragma unroll
    for (int r = 0; r < 32; ++r) {
        const int f = FROM1 ? f_layout1(t, r) : f_layout2(t, r);
        sm[slot_of(f)] = make_double2(re[r], im[r]);
    }
    group_sync(grp);
#pragma unroll
    for (int r = 0; r < 32; ++r) {
        const int f = FROM1 ? f_layout2(t, r) : f_layout1(t, r);
        const double2 v = sm[slot_of(f)];
        re[r] = v.x; im[r] = v.y;
    }
}

// Sweeps, diagonal and in-place store of one tile held in registers in layout 1 (used by k_tile_pipe and k_chunk_pipe).
// STCG: keep the stored lines in L2 (st.global.cg) instead of streaming them out (st.global.cs).
template <int K1, int K2, int BF1, int BF2, int NSHFL, bool STCG>
__device__ __forceinline__ void pipe_compute_store(const TilePassParams& p, const uint64_t tau, double (&re)[32], double (&im)[32],
                                                   const double2 base, const double2 (&w)[5], double2* E, const int t, const int grp)
{
    constexpr bool GENERIC = (BF1 < 0);
    const bool two_stage = GENERIC ? (p.two_stage != 0) : (BF2 != 0);
    const int nshfl = GENERIC ? p.nshfl : NSHFL;
    const int lane = t & 31;
    const bool has_diag = (p.tile_phase != nullptr);
    const int s = p.s, g0 = p.g0, nmid = g0 - s;
    const uint64_t runmask = ((uint64_t)1 << s) - 1;
    const uint64_t base_idx = ((tau & (((uint64_t)1 << nmid) - 1)) << s) | ((tau >> nmid) << (g0 + TS_TILE_LOG2 - s));

    // Single sweep of a high group with runs of >= 8 amplitudes and no diagonal: ONE exchange.  Layout 2H keeps the run
    // bits f0..2 on the lanes (f = (t & 7) | r << 3 | (t >> 3) << 8; registers hold f3..7), so the tile can be stored
    // straight from it in full 128-byte runs, exactly as coalesced as from layout 1.
    if (K2 == SW_NONE && NSHFL == 0 && !GENERIC && BF2 != 0 && (BF2 & 1) == 0 && !has_diag) {
        bfly_regs<K1, BF1>(re, im, p.bf1);
#pragma unroll
        for (int r = 0; r < 32; ++r) E[slot_of(f_layout1(t, r))] = make_double2(re[r], im[r]);
        group_sync(grp);
#pragma unroll
        for (int r = 0; r < 32; ++r) {
            const double2 v = E[slot_of((t & 7) | (r << 3) | ((t >> 3) << 8))];
            re[r] = v.x; im[r] = v.y;
        }
        bfly_regs<K1, ((BF2 >= 0 ? BF2 : 0) >> 1)>(re, im, 0u);          // f3..6 sit on register bits 0..3 here
        uint64_t ob[5];
#pragma unroll
        for (int b = 0; b < 5; ++b) {
            const uint64_t f = (uint64_t)1 << (3 + b);
            ob[b] = (f & runmask) | ((f >> s) << g0);
        }
        const uint64_t ft = (uint64_t)((t & 7) | ((t >> 3) << 8));
        double2* __restrict__ gq = p.psi + base_idx + ((ft & runmask) | ((ft >> s) << g0));
#pragma unroll
        for (int r = 0; r < 32; ++r) {
            uint64_t o = 0;
#pragma unroll
            for (int b = 0; b < 5; ++b) if (r & (1 << b)) o |= ob[b];
            if (STCG) __stcg(gq + o, make_double2(re[r], im[r]));
            else __stcs(gq + o, make_double2(re[r], im[r]));
        }
        return;      // (the two barriers of the next tile's landing reads separate these reads of E from its next writes)
    }

    // ---- sweep K1
    bfly_regs<K1, BF1>(re, im, p.bf1);
    if (two_stage) {
        exchange_g<true>(E, re, im, t, grp);
        bfly_regs<K1, BF2>(re, im, p.bf2);
        if (nshfl) { bfly_lane<K1>(re, im, 0, lane); bfly_lane<K1>(re, im, 1, lane); }
    }
    // ---- diagonal
    if (has_diag) apply_diag(p, base, w, re, im);
    // ---- sweep K2 (mirror order)
    if (two_stage) {
        if (nshfl) { bfly_lane<K2>(re, im, 1, lane); bfly_lane<K2>(re, im, 0, lane); }
        bfly_regs<K2, BF2>(re, im, p.bf2);
        exchange_g<false>(E, re, im, t, grp);
    }
    bfly_regs<K2, BF1>(re, im, p.bf1);

    // global element offset of in-tile index f: run bits stay, group bits move up to g0
    uint64_t offb[5];
#pragma unroll
    for (int b = 0; b < 5; ++b) {
        const uint64_t f = (uint64_t)1 << (7 + b);
        offb[b] = (f & runmask) | ((f >> s) << g0);
    }
    const uint64_t offt = ((uint64_t)t & runmask) | (((uint64_t)t >> s) << g0);
    double2* __restrict__ gp = p.psi + base_idx + offt;
#pragma unroll
    for (int r = 0; r < 32; ++r) {
        uint64_t o = 0;
#pragma unroll
        for (int b = 0; b < 5; ++b) if (r & (1 << b)) o |= offb[b];
        if (STCG) __stcg(gp + o, make_double2(re[r], im[r]));
        else __stcs(gp + o, make_double2(re[r], im[r]));
    }
}

// Per-thread phase factors from the tile-phase record `tp` (32 entries, in shared memory) and the thread tables.
__device__ __forceinline__ void pipe_thread_phase(const TilePassParams& p, const double2* tp, const int t, double2& base, double2 (&w)[5])
{
    base = cmul(tp[0], __ldg(p.TT + t));
    base = cmul(base, tp[1 + (t & 15)]);
    base = cunit(cmul(base, tp[17 + (t >> 4)]));
    base.x *= p.scale; base.y *= p.scale;
#pragma unroll
    for (int k = 0; k < 5; ++k) w[k] = cunit(cmul(tp[25 + k], __ldg(p.WT + k * 128 + t)));
}

template <int K1, int K2, int BF1, int BF2, int NSHFL>
__global__ void __launch_bounds__(TS_PIPE_THREADS, 1)
k_tile_pipe(const __grid_constant__ TilePassParams p, const __grid_constant__ CUtensorMap tmap, const PipeGeom g)
{
    extern __shared__ __align__(1024) unsigned char smraw[];
    constexpr bool GENERIC = (BF1 < 0);
    const bool two_stage = GENERIC ? (p.two_stage != 0) : (BF2 != 0);
    const int nshfl = GENERIC ? p.nshfl : NSHFL;

    const int grp = threadIdx.x >> 7;
    const int t = threadIdx.x & (TS_TILE_THREADS - 1);
    const int lane = t & 31;
    const uint32_t sL = smem_u32(smraw);
    const uint32_t sTP = smem_u32(smraw + TS_PIPE_OFF_TP);
    const uint32_t sBar = smem_u32(smraw + TS_PIPE_OFF_BAR);
    double2* E = reinterpret_cast<double2*>(smraw + TS_PIPE_OFF_E) + ((size_t)grp << TS_TILE_LOG2);
    const double2* TPs = reinterpret_cast<const double2*>(smraw + TS_PIPE_OFF_TP);
    // cons[x] = 1 + index (in this CTA's tile sequence) of the last tile whose first half group x has consumed
    volatile uint32_t* cons = reinterpret_cast<volatile uint32_t*>(smraw + TS_PIPE_OFF_BAR + 32);

    const int s = p.s, g0 = p.g0;
    const int nmid = g0 - s;
    const uint64_t midmask = ((uint64_t)1 << nmid) - 1;
    const bool has_diag = (p.tile_phase != nullptr);

    // tiles of this CTA: b, b + G, ...;  halves q = 2 i + h in ring order
    const uint64_t G = gridDim.x;
    const uint64_t n_cta = (g.ntiles > blockIdx.x) ? (g.ntiles - blockIdx.x + G - 1) / G : 0;
    const uint64_t n_half = 2 * n_cta;

    // half q of this CTA into L2 only (the ring holds 1.5 tiles, not enough bytes in flight to cover HBM latency)
    auto prefetch_half = [&](uint64_t q) {
        const uint64_t tau = p.tile_base + blockIdx.x + (q >> 1) * G;
        const int h = (int)(q & 1);
        const uint64_t mid = tau & midmask, hi = tau >> nmid;
        if (g.tensor) {
            for (int b = 0; b < g.nbox; ++b)
                tensor_prefetch_l2_3d(&tmap, (int)(mid << (s + 1)), h * g.rows_half + b * g.box_rows, (int)hi);
        } else {
            const uint64_t base_idx = (mid << s) | (hi << (g0 + TS_TILE_LOG2 - s));
            if (g.is_low) {
                bulk_prefetch_l2(p.psi + base_idx + (uint64_t)h * (TS_PIPE_HALF_BYTES / 16), TS_PIPE_HALF_BYTES);
            } else {
                for (int r = 0; r < g.rows_half; ++r)
                    bulk_prefetch_l2(p.psi + base_idx + ((uint64_t)(h * g.rows_half + r) << g0), g.row_bytes);
            }
        }
    };
    auto issue_load = [&](uint64_t q, int slot) {
        if (g.pf > 0 && q + g.pf < n_half) prefetch_half(q + g.pf);
        const uint64_t i = q >> 1;
        const int h = (int)(q & 1);
        const uint64_t tau = p.tile_base + blockIdx.x + i * G;
        const uint32_t bar = sBar + 8 * slot;
        const uint32_t dst = sL + slot * TS_PIPE_HALF_BYTES;
        const bool tp = has_diag && h == 0;
        mbar_expect_tx(bar, TS_PIPE_HALF_BYTES + (tp ? 512u : 0u));
        if (tp) bulk_load(sTP + slot * 512, p.tile_phase + (tau << 5), 512, bar);
        const uint64_t mid = tau & midmask, hi = tau >> nmid;
        if (g.tensor) {
            for (int b = 0; b < g.nbox; ++b)
                tensor_load_3d(dst + b * g.box_rows * g.row_bytes, &tmap, bar, (int)(mid << (s + 1)),
                               h * g.rows_half + b * g.box_rows, (int)hi);
        } else {
            const uint64_t base_idx = (mid << s) | (hi << (g0 + TS_TILE_LOG2 - s));
            if (g.is_low) {
                bulk_load(dst, p.psi + base_idx + (uint64_t)h * (TS_PIPE_HALF_BYTES / 16), TS_PIPE_HALF_BYTES, bar);
            } else {
                for (int r = 0; r < g.rows_half; ++r)
                    bulk_load(dst + r * g.row_bytes, p.psi + base_idx + ((uint64_t)(h * g.rows_half + r) << g0),
                              g.row_bytes, bar);
            }
        }
    };

    if (threadIdx.x == 0) {
        for (int k = 0; k < TS_PIPE_SLOTS; ++k) mbar_init(sBar + 8 * k, 1);
        cons[0] = 0; cons[1] = 0;
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        for (uint64_t q = TS_PIPE_SLOTS; q < (uint64_t)(TS_PIPE_SLOTS + g.pf) && q < n_half; ++q) prefetch_half(q);
        for (uint64_t q = 0; q < TS_PIPE_SLOTS && q < n_half; ++q) issue_load(q, (int)q);
    }
    __syncthreads();

    // global element offset of in-tile index f (stores): run bits stay, group bits move up to g0
    const uint64_t runmask = ((uint64_t)1 << s) - 1;
    uint64_t offb[5];
#pragma unroll
    for (int b = 0; b < 5; ++b) {
        const uint64_t f = (uint64_t)1 << (7 + b);
        offb[b] = (f & runmask) | ((f >> s) << g0);
    }
    const uint64_t offt = ((uint64_t)t & runmask) | (((uint64_t)t >> s) << g0);

    // ring position of this group's first half: q = 2 grp; slot = q % 3, use = q / 3
    uint32_t slot = (2 * grp) % TS_PIPE_SLOTS, use = (2 * grp) / TS_PIPE_SLOTS;

    for (uint64_t i = grp; i < n_cta; i += 2) {
        const uint64_t tau = p.tile_base + blockIdx.x + i * G;
        double re[32], im[32];
        double2 base = make_double2(1.0, 0.0), w[5];

#pragma unroll
        for (int h = 0; h < 2; ++h) {
            // A parity wait is only sound once the slot's PREVIOUS use has completed.  For h = 0 that use (half 1 of
            // tile i - 2) was consumed by this group; for h = 1 it is half 0 of tile i - 1, which belongs to the other
            // group and may still be in flight: wait until that group has consumed it.
            if (h == 1 && i > 0) while (cons[grp ^ 1] < (uint32_t)i) { }
            mbar_wait(sBar + 8 * slot, use & 1);
            const double2* Ls = reinterpret_cast<const double2*>(smraw + slot * TS_PIPE_HALF_BYTES);
#pragma unroll
            for (int r = 0; r < 16; ++r) {
                const double2 v = Ls[t | (r << 7)];
                re[16 * h + r] = v.x; im[16 * h + r] = v.y;
            }
            if (g.dbg) {                       // debug: landed data must equal what a direct global read returns
                const uint64_t bi = ((tau & midmask) << s) | ((tau >> nmid) << (g0 + TS_TILE_LOG2 - s));
                for (int r = 0; r < 16; ++r) {
                    uint64_t o = 0;
                    for (int b = 0; b < 5; ++b) if ((16 * h + r) & (1 << b)) o |= offb[b];
                    const double2 v = p.psi[bi + offt + o];
                    if (v.x != re[16 * h + r] || v.y != im[16 * h + r]) {
                        if (atomicAdd(g.dbg, 1ULL) == 0) { g.dbg[1] = tau; g.dbg[2] = 16 * h + r; g.dbg[3] = t; g.dbg[4] = slot; }
                    }
                }
            }
            if (h == 0 && has_diag) {
                pipe_thread_phase(p, TPs + slot * 32, t, base, w);
            }
            group_sync(grp);
            if (t == (h ? 32 : 0)) {     // the two halves are served by different warps: neither is late twice
                const uint64_t qn = 2 * i + h + TS_PIPE_SLOTS;
                if (qn < n_half) issue_load(qn, (int)slot);
                if (h == 0) cons[grp] = (uint32_t)i + 1;
            }
            // next half of this group: q + 1 (within the tile) or q + 3 (skipping the other group's tile)
            slot += 1; if (slot >= TS_PIPE_SLOTS) { slot -= TS_PIPE_SLOTS; use += 1; }
        }
        // skip the other group's two halves
        slot += 2; if (slot >= TS_PIPE_SLOTS) { slot -= TS_PIPE_SLOTS; use += 1; }

        pipe_compute_store<K1, K2, BF1, BF2, NSHFL, false>(p, tau, re, im, base, w, E, t, grp);
    }
}

#define TS_PIPE_REGISTER_CFG(NAME, BF1, BF2, NSHFL)                                                               \
    void ts_pipe_register_##NAME(pipe_kernel_t (*tab)[5][5])                                                      \
    {                                                                                                             \
        (*tab)[SW_XDAG][SW_YDAG] = tsk::k_tile_pipe<SW_XDAG, SW_YDAG, BF1, BF2, NSHFL>;                           \
        (*tab)[SW_YDAG][SW_Y]    = tsk::k_tile_pipe<SW_YDAG, SW_Y, BF1, BF2, NSHFL>;                              \
        (*tab)[SW_Y][SW_X]       = tsk::k_tile_pipe<SW_Y, SW_X, BF1, BF2, NSHFL>;                                 \
        (*tab)[SW_X][SW_XDAG]    = tsk::k_tile_pipe<SW_X, SW_XDAG, BF1, BF2, NSHFL>;                              \
        (*tab)[SW_YDAG][SW_NONE] = tsk::k_tile_pipe<SW_YDAG, SW_NONE, BF1, BF2, NSHFL>;                           \
        (*tab)[SW_Y][SW_NONE]    = tsk::k_tile_pipe<SW_Y, SW_NONE, BF1, BF2, NSHFL>;                              \
        (*tab)[SW_XDAG][SW_NONE] = tsk::k_tile_pipe<SW_XDAG, SW_NONE, BF1, BF2, NSHFL>;                           \
        (*tab)[SW_X][SW_NONE]    = tsk::k_tile_pipe<SW_X, SW_NONE, BF1, BF2, NSHFL>;                              \
        (*tab)[SW_NONE][SW_XDAG] = tsk::k_tile_pipe<SW_NONE, SW_XDAG, BF1, BF2, NSHFL>;                           \
    }

} // namespace tsk
#endif
