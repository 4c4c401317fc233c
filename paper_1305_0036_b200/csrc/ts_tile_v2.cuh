// ts_tile_v2.cuh -- the tile pass as a warp-specialised, TMA-in / TMA-out persistent kernel (
// DESIGN.md 7.2).  Same mathematics as k_tile_pass (ts_tile_kernel.cuh): a closed tile of 2^12 amplitudes is
// held in registers, 32 amplitudes per thread, and gets  [butterflies of sweep K1] . [diagonal D] . [butterflies of
// sweep K2]  on the bits of its group before it is written back in place.  What differs is how the tile travels:
//
//   * one CTA per SM, 10 warps: 8 compute warps = two groups of 128 threads that take alternate tiles, one LOADER warp
//     and one STORER warp (one elected lane each).  No compute thread ever forms a global address.
//   * three 64-KiB tile buffers in shared memory.  The loader fills a buffer with two TMA tensor boxes of 32 KiB
//     (cp.async.bulk.tensor, 128-byte swizzle, completion on the buffer's `full` mbarrier); a compute group works on it
//     IN PLACE -- the register<->register layout exchanges of the butterfly network go through the tile's own buffer,
//     every thread overwriting exactly the slots it read, so an exchange costs ONE group barrier -- and leaves the
//     finished tile in the buffer; the storer writes it back with two TMA tensor stores and hands the buffer back to
//     the loader when the store has read it.  Loads, stores and arithmetic of different tiles overlap without any
//     thread waiting on a memory instruction of its own.
//   * shared-memory slot of in-tile index f:  slot(f) = f ^ ((f >> 3) & 7)  -- exactly what TMA's SWIZZLE_128B writes
//     for rows of 8 amplitudes (128 B).  All register layouts below keep one of {f0|f3}, {f1|f4}, {f2|f5} on each of
//     the three low lane bits, which makes every 128-bit shared-memory access conflict-free under that swizzle.
//
//   * tiles are handed out DYNAMICALLY: the loader draws tickets from a global counter (one atomicAdd per ticket, fetched
//     one ticket ahead) and passes the tile index to the compute groups and the storer through a shared-memory slot per
//     buffer.  SMs do not run at the same speed (ncu, static assignment: fastest SM done after 5.6 ms, slowest after
//     7.9 ms of a 7.9 ms top-group pass, profiles/r02a_baseline.md), so a static split leaves a fifth of the chip idle at
//     the end of every pass.  A ticket of a high group is a PAIR of adjacent tiles (2p, 2p + 1): their 128-byte rows are
//     the two halves of 256-byte segments.
//
// In-tile index f (12 bits): group A (spins 0..11): f = spin.  High group (s run bits, m = 12 - s group bits):
// f < s <-> spin f, f >= s <-> spin g0 + f - s; the tile is 2^m rows of 2^s amplitudes at a stride of 2^g0.
//
// Register layouts (r = register index, 5 bits; t = thread index in the group, 7 bits; lists give the f bit of each
// register / thread bit):
//   A1: regs {3,4,5,10,11}  threads {0,1,2,8,9,6,7}        A2: regs {0,1,2,8,9}  threads {3,4,5,6,7,10,11}
//   H1: regs {7,8,9,10,11}  threads {0,1,2,3,4,5,6}        H2: regs {3,4,5,6,7}  threads {0,1,2,8,9,10,11}
//   H1x: regs {5,8,9,10,11} threads {0,1,2,3,4,6,7}        H2x: regs {2,3,4,6,7} threads {0,1,5,8,9,10,11}   (ten-bit group)
// Group A butterflies all 12 bits without warp shuffles: K1 on 5 bits in A1, 5 in A2, then A2 -> A2' (regs {0,1,2,6,7}:
// lane bits 3, 4 swapped with register bits 3, 4 -- an exchange INSIDE each warp's quarter of the buffer, __syncwarp only)
// and f6, f7 there; the diagonal in A2'; K2 on all five register bits of A2', the five of A1, and f8, f9 in A1'.  A high group butterflies f >= s: f7..11 in H1 and f_s..6 in H2 (m > 5 only; diagonal in H2, else H1).
#pragma once
#include <cuda.h>

#include "ts_tile_kernel.cuh"

#define TS_V2_THREADS 384                 // two compute warpgroups (8 warps) + one producer warpgroup (loader warp, storer warp, 2 idle)
#define TS_V2_REGS_COMPUTE 232            // setmaxnreg: 256 x 232 + 128 x 40 = 64 512 <= 65 536 registers
#define TS_V2_REGS_PRODUCER 40
#ifndef TS_V2_NBUF
#define TS_V2_NBUF 3
#endif
#define TS_V2_TILE_BYTES 65536
#define TS_V2_OFF_TP (TS_V2_NBUF * TS_V2_TILE_BYTES)         // 3 x 512 B tile-phase records
#define TS_V2_OFF_BAR (TS_V2_OFF_TP + TS_V2_NBUF * 512)      // full[3], done[3], free[3], tab mbarriers (80 B), then tile[3] (u32)
#define TS_V2_OFF_TILE (TS_V2_OFF_BAR + 112)                 // tile index of the job in each buffer (written by the loader)
// mbarriers (8 bytes each): full[3], done[3], free[3][half 0], free[3][half 1], tab
#define TS_V2_BAR_FULL(b) (8u * (b))
#define TS_V2_BAR_DONE(b) (8u * (TS_V2_NBUF + (b)))
#define TS_V2_BAR_FREE(b, h) (8u * ((2 + (h)) * TS_V2_NBUF + (b)))
#define TS_V2_BAR_TABLE (8u * 4 * TS_V2_NBUF)
#define TS_V2_END 0xffffffffu                                // "no more tiles" marker in a tile slot
#define TS_V2_OFF_TAB (TS_V2_OFF_BAR + 128)                  // per-launch phase tables: TT[128], WT[5][128], RR[32]
#define TS_V2_TAB_BYTES (800 * 16)
#define TS_V2_SMEM (TS_V2_OFF_TAB + TS_V2_TAB_BYTES)

#define TS_V2_A1_R 0xBA543u
#define TS_V2_A1_T 0x7698210u
#define TS_V2_A2_R 0x98210u
#define TS_V2_A2_T 0xBA76543u
// A2' / A1': A2 / A1 with lane bits 3, 4 and register bits 3, 4 swapped (an intra-warp exchange through the warp's own
// quarter of the tile buffer: no block barrier).  They put f6, f7 (resp. f8, f9) on register bits.
#define TS_V2_A2S_R 0x76210u
#define TS_V2_A2S_T 0xBA98543u
#define TS_V2_A1S_R 0x98543u
#define TS_V2_A1S_T 0x76BA210u
#define TS_V2_H1_R 0xBA987u
#define TS_V2_H1_T 0x6543210u
#define TS_V2_H2_R 0x76543u
#define TS_V2_H2_T 0xBA98210u
// a high group of TEN bits (runs of 4 amplitudes = 64 bytes, TMA's 64-byte swizzle): two full five-bit stages, f2 .. f11.
// (H1x is conflict-free under that swizzle; H2x, with f2 on a register bit, has two-way bank conflicts -- the LSU has the room)
#define TS_V2_H1X_R 0xBA985u
#define TS_V2_H1X_T 0x7643210u
#define TS_V2_H2X_R 0x76432u
#define TS_V2_H2X_T 0xBA98510u

// One tile group as the kernel sees it.
struct V2Geom {
    int type;               // 0: group A (contiguous tile), 1: high group
    int s, g0, m;           // high group: run bits, first spin, group bits (A: 12, 12, 0)
    int nmid;               // g0 - s: tile-index bits below the group
    int unit_log2;          // amplitudes per tensor-map unit (inner box dimension): min(3, s), i.e. 128 or 64 bytes
    int box_rows_log2;      // rows per TMA box: min(8, m - 1); a tile is 2^(m - box_rows_log2) boxes
    int two_stage;          // high group with m > 5: layouts H1 and H2
    unsigned mask1, mask2;  // butterflied register bits in H1 / H2
};

// Phase tables of the diagonal applied by a pass (see ts_tile_kernel.cuh for their meaning); tile_phase = NULL: none.
struct V2Diag {
    const double2* tile_phase;   // [ntiles][32]: one 512-byte record per tile, loaded with the tile
    const double2* tables;       // TT[128], WT[5][128], RR[32] (800 entries): copied to shared memory once per launch
    double scale;                // exact power of two
};

struct V2Pass {
    V2Geom g;
    V2Diag d;
    uint64_t ntiles;
    unsigned int* sched;         // [2]: next ticket, CTAs finished (both zero between launches: the last CTA resets them)
    uint32_t pair_log2;          // tiles per ticket = 2^pair_log2 (1: adjacent tile pairs of a high group)
    int probe;                   // 1: copy only -- the compute groups skip the tile body (TS_OPT_PROBE: pipeline ceilings)
    int ngroups;                 // compute groups in use: 2, or 1 (TS_OPT_GROUPS: one tile at a time in arithmetic, two buffers in transport)
};

// L2-blocked triple launch: [high group, sweep KA] [group A: KA . D . KB] [high group, sweep KB] chunk by chunk.
struct V2Chunk {
    V2Geom gh, ga;
    V2Diag d;
    unsigned int* done;          // [2][nchunks] tiles finished (and globally visible) of phase 1 / phase 2 of a chunk
    unsigned int* sched;         // [2]: next ticket, CTAs finished
    uint32_t nchunks, tiles_log2;
    int probe;
    int ngroups;
    int l2_hints;                // 1: eviction priorities on the TMA transfers (keep a chunk in L2 until its third phase wrote it)
};

typedef void (*v2_kernel_t)(const V2Pass, const CUtensorMap);
typedef void (*v2_chunk_kernel_t)(const V2Chunk, const CUtensorMap, const CUtensorMap);

// tab[type][k1][k2]; type 0: group A, 1: high group (run-time masks), 2: high group with 9 group bits, 3: with 10
void ts_v2_register_A(v2_kernel_t (*tab)[5][5]);
void ts_v2_register_Hf(v2_kernel_t (*tab)[5][5]);
void ts_v2_register_Hs(v2_kernel_t (*tab)[5][5]);
void ts_v2_register_H9f(v2_kernel_t (*tab)[5][5]);
void ts_v2_register_H9s(v2_kernel_t (*tab)[5][5]);
void ts_v2_register_H10(v2_kernel_t (*tab)[5][5]);
// tab[hm][v]: hm = 0: any high group, 1: 9 group bits;  v = 0: (Y^dag, Y), v = 1: (X, X^dag) -- the two kind pairs that
// meet at group A in the sweep order
void ts_v2_register_chunk0(v2_chunk_kernel_t (*tab)[2]);
void ts_v2_register_chunk1(v2_chunk_kernel_t (*tab)[2]);
void ts_v2_register_chunk0_h9(v2_chunk_kernel_t (*tab)[2]);
void ts_v2_register_chunk1_h9(v2_chunk_kernel_t (*tab)[2]);
// measurement builds of the N = 30 kernels (ts_v2_probe.cu): mode 1 = arithmetic only (no layout exchanges), 2 = exchanges
// only (no arithmetic); index [mode - 1].  chunk: (Y^dag, Y) with a 9-bit high group; fusedH: top group (X^dag, Y^dag);
// fusedA: group A (Y^dag, Y)
void ts_v2_register_probe(v2_chunk_kernel_t* chunk, v2_kernel_t* fusedH, v2_kernel_t* fusedA);

#ifdef __CUDACC__
namespace tsk {

// ------------------------------------------------------------------------------------------------ PTX wrappers
__device__ __forceinline__ uint32_t v2_smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void v2_mbar_init(uint32_t bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void v2_mbar_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void v2_mbar_arrive(uint32_t bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void v2_mbar_wait(uint32_t bar, uint32_t parity)
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
__device__ __forceinline__ void v2_bulk_load(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
                 "l"(src), "r"(bytes), "r"(bar)
                 : "memory");
}
__device__ __forceinline__ void v2_tma_load_2d(uint32_t dst, const CUtensorMap* tm, uint32_t bar, int c0, int c1)
{
    asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];" ::"r"(dst),
                 "l"(tm), "r"(bar), "r"(c0), "r"(c1)
                 : "memory");
}
__device__ __forceinline__ void v2_tma_load_4d(uint32_t dst, const CUtensorMap* tm, uint32_t bar, int c0, int c1, int c2, int c3)
{
    asm volatile(
        "cp.async.bulk.tensor.4d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6}], [%2];" ::"r"(dst),
        "l"(tm), "r"(bar), "r"(c0), "r"(c1), "r"(c2), "r"(c3)
        : "memory");
}
__device__ __forceinline__ void v2_tma_store_2d(const CUtensorMap* tm, uint32_t src, int c0, int c1)
{
    asm volatile("cp.async.bulk.tensor.2d.global.shared::cta.tile.bulk_group [%0, {%2, %3}], [%1];" ::"l"(tm), "r"(src), "r"(c0),
                 "r"(c1)
                 : "memory");
}
__device__ __forceinline__ void v2_tma_store_4d(const CUtensorMap* tm, uint32_t src, int c0, int c1, int c2, int c3)
{
    asm volatile("cp.async.bulk.tensor.4d.global.shared::cta.tile.bulk_group [%0, {%2, %3, %4, %5}], [%1];" ::"l"(tm), "r"(src),
                 "r"(c0), "r"(c1), "r"(c2), "r"(c3)
                 : "memory");
}
// L2 eviction-priority policies for the L2-blocked launch (createpolicy; 0: evict_normal, 1: evict_first, 2: evict_last)
__device__ __forceinline__ uint64_t v2_policy(int kind)
{
    uint64_t pol;
    if (kind == 1) asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    else if (kind == 2) asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol));
    else asm volatile("createpolicy.fractional.L2::evict_normal.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
__device__ __forceinline__ void v2_tma_load_2d_h(uint32_t dst, const CUtensorMap* tm, uint32_t bar, int c0, int c1, uint64_t pol)
{
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1, {%3, %4}], [%2], %5;" ::"r"(dst),
        "l"(tm), "r"(bar), "r"(c0), "r"(c1), "l"(pol)
        : "memory");
}
__device__ __forceinline__ void v2_tma_load_4d_h(uint32_t dst, const CUtensorMap* tm, uint32_t bar, int c0, int c1, int c2, int c3,
                                                 uint64_t pol)
{
    asm volatile(
        "cp.async.bulk.tensor.4d.shared::cluster.global.tile.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1, {%3, %4, %5, %6}], [%2], %7;" ::"r"(dst),
        "l"(tm), "r"(bar), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "l"(pol)
        : "memory");
}
__device__ __forceinline__ void v2_tma_store_2d_h(const CUtensorMap* tm, uint32_t src, int c0, int c1, uint64_t pol)
{
    asm volatile("cp.async.bulk.tensor.2d.global.shared::cta.tile.bulk_group.L2::cache_hint [%0, {%2, %3}], [%1], %4;" ::"l"(tm),
                 "r"(src), "r"(c0), "r"(c1), "l"(pol)
                 : "memory");
}
__device__ __forceinline__ void v2_tma_store_4d_h(const CUtensorMap* tm, uint32_t src, int c0, int c1, int c2, int c3, uint64_t pol)
{
    asm volatile("cp.async.bulk.tensor.4d.global.shared::cta.tile.bulk_group.L2::cache_hint [%0, {%2, %3, %4, %5}], [%1], %6;" ::"l"(tm),
                 "r"(src), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "l"(pol)
                 : "memory");
}
__device__ __forceinline__ void v2_store_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void v2_store_wait_read() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
__device__ __forceinline__ void v2_store_wait_read_but_one() { asm volatile("cp.async.bulk.wait_group.read 1;" ::: "memory"); }
__device__ __forceinline__ void v2_store_wait_all() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }
__device__ __forceinline__ void v2_fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void v2_fence_async_all() { asm volatile("fence.proxy.async;" ::: "memory"); }
__device__ __forceinline__ void v2_group_sync(int grp)
{
    asm volatile("bar.sync %0, %1;" ::"r"(grp + 1), "r"(TS_TILE_THREADS) : "memory");
}
template <int R> __device__ __forceinline__ void v2_regs_inc() { asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(R)); }
template <int R> __device__ __forceinline__ void v2_regs_dec() { asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(R)); }
__device__ __forceinline__ unsigned int v2_ld_acquire(const unsigned int* p)
{
    unsigned int v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}

// ------------------------------------------------------------------------------------------------ register layouts
// RP / TP: the f bit of register bit i / thread bit i, one nibble each.
// SWZ: 7 = TMA's 128-byte swizzle (slot = f ^ (f >> 3 & 7), rows of 128 bytes), 3 = its 64-byte swizzle (rows of 64 bytes)
template <uint32_t RP, uint32_t TP, uint32_t SWZ = 7u>
struct V2Layout {
    // byte offset (within a tile buffer) of the slot of the thread part of f
    static __device__ __forceinline__ uint32_t thread_off(int t)
    {
        uint32_t f = 0;
#pragma unroll
        for (int i = 0; i < 7; ++i) f |= (uint32_t)((t >> i) & 1) << ((TP >> (4 * i)) & 15u);
        return (f ^ ((f >> 3) & SWZ)) << 4;
    }
    static __host__ __device__ constexpr uint32_t reg_slot(int r)
    {
        uint32_t f = 0;
        for (int i = 0; i < 5; ++i) f |= (uint32_t)((r >> i) & 1) << ((RP >> (4 * i)) & 15u);
        return f ^ ((f >> 3) & SWZ);
    }
    // slot(f_t | f_r) = slot(f_t) ^ slot(f_r) (the swizzle is linear over bits); only the three low slot bits mix
    static __device__ __forceinline__ double2* ptr(unsigned char* buf, uint32_t toff, int r)
    {
        const uint32_t c = reg_slot(r);
        return reinterpret_cast<double2*>(buf + ((toff ^ ((c & 7u) << 4)) + ((c & ~7u) << 4)));
    }
    static __device__ __forceinline__ void load(unsigned char* buf, uint32_t toff, double (&re)[32], double (&im)[32])
    {
#pragma unroll
        for (int r = 0; r < 32; ++r) {
            const double2 v = *ptr(buf, toff, r);
            re[r] = v.x; im[r] = v.y;
        }
    }
    static __device__ __forceinline__ void store(unsigned char* buf, uint32_t toff, const double (&re)[32], const double (&im)[32])
    {
#pragma unroll
        for (int r = 0; r < 32; ++r) *ptr(buf, toff, r) = make_double2(re[r], im[r]);
    }
};

// Per-thread phase factors from the tile-phase record `tp` (32 entries) and the thread tables `tab` (TT, WT), both in
// shared memory.
__device__ __forceinline__ void v2_thread_phase(const double scale, const double2* tp, const double2* tab, const int t, double2& base,
                                                double2 (&w)[5])
{
    base = cmul(tp[0], tab[t]);
    base = cmul(base, tp[1 + (t & 15)]);
    base = cunit(cmul(base, tp[17 + (t >> 4)]));
    base.x *= scale; base.y *= scale;
#pragma unroll
    for (int k = 0; k < 5; ++k) w[k] = cunit(cmul(tp[25 + k], tab[128 + k * 128 + t]));
}

// c_r <- c_r * base * RR[r] * prod_i w_i^{r_i}   (depth-first product tree; RR = tab + 768, broadcast reads)
__device__ __forceinline__ void v2_apply_diag(const double2* RR, const double2 base, const double2 (&w)[5], double (&re)[32],
                                              double (&im)[32])
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
                        const double2 ph = cmul(q0, RR[r]);
                        const double2 c = cmul(make_double2(re[r], im[r]), ph);
                        re[r] = c.x; im[r] = c.y;
                    }
                }
            }
        }
    }
}

// Measurement builds without arithmetic: swap neighbouring registers after every shared-memory load, so that what is stored
// differs from what was loaded and the compiler cannot drop the exchange as a load followed by a store of the same value
// (it did: an earlier "exchanges only" build ran with 1 % shared-memory traffic).
template <bool ON>
__device__ __forceinline__ void v2_probe_touch(double (&re)[32], double (&im)[32])
{
    if (!ON) return;
#pragma unroll
    for (int r = 0; r < 32; r += 2) {
        const double a = re[r], b = im[r];
        re[r] = re[r + 1]; im[r] = im[r + 1];
        re[r + 1] = a; im[r + 1] = b;
    }
}

// ------------------------------------------------------------------------------------------------ tile bodies
// The tile is in `buf` (landed by TMA); on return the finished tile is in `buf` again, in the same slots.
// diag: apply the diagonal; tp: this tile's phase record; tab: the launch's thread tables (both in shared memory).
// MODE (measurement builds, ts_v2_probe.cu): bit 0 = do the arithmetic, bit 1 = do the layout exchanges; 3 = the product.
template <int K1, int K2, int MODE = 3>
__device__ __forceinline__ void v2_body_A(unsigned char* buf, const bool diag, const double scale, const double2* tp,
                                          const double2* tab, const int t, const int grp)
{
    constexpr bool AR = (MODE & 1) != 0, EX = (MODE & 2) != 0;
    using L1 = V2Layout<TS_V2_A1_R, TS_V2_A1_T>;
    using L2 = V2Layout<TS_V2_A2_R, TS_V2_A2_T>;
    using L1S = V2Layout<TS_V2_A1S_R, TS_V2_A1S_T>;
    using L2S = V2Layout<TS_V2_A2S_R, TS_V2_A2S_T>;
    const uint32_t o1 = L1::thread_off(t), o2 = L2::thread_off(t), o1s = L1S::thread_off(t), o2s = L2S::thread_off(t);
    double re[32], im[32];
    if (K1 != SW_NONE) {
        L1::load(buf, o1, re, im);
        v2_probe_touch<!AR>(re, im);
        if (AR) bfly_regs<K1, 31>(re, im, 0u);         // f 3,4,5,10,11
        if (EX) {
            L1::store(buf, o1, re, im);
            v2_group_sync(grp);
            L2::load(buf, o2, re, im);
            v2_probe_touch<!AR>(re, im);
        }
        if (AR) bfly_regs<K1, 31>(re, im, 0u);         // f 0,1,2,8,9
        if (EX) {
            L2::store(buf, o2, re, im);                // A2 -> A2': lanes <-> registers inside the warp's own quarter
            __syncwarp();
        }
    }
    if (EX || K1 == SW_NONE) L2S::load(buf, o2s, re, im);
    v2_probe_touch<!AR>(re, im);
    if (AR) bfly_regs<K1, 24>(re, im, 0u);             // f 6,7
    if (diag && AR) {
        double2 base, w[5];
        v2_thread_phase(scale, tp, tab, t, base, w);
        v2_apply_diag(tab + 768, base, w, re, im);
    }
    if (K2 != SW_NONE) {
        if (AR) bfly_regs<K2, 31>(re, im, 0u);         // f 0,1,2,6,7
        if (EX) {
            L2S::store(buf, o2s, re, im);
            v2_group_sync(grp);
            L1::load(buf, o1, re, im);
            v2_probe_touch<!AR>(re, im);
        }
        if (AR) bfly_regs<K2, 31>(re, im, 0u);         // f 3,4,5,10,11
        if (EX) {
            L1::store(buf, o1, re, im);                // A1 -> A1'
            __syncwarp();
            L1S::load(buf, o1s, re, im);
            v2_probe_touch<!AR>(re, im);
        }
        if (AR) bfly_regs<K2, 24>(re, im, 0u);         // f 8,9
        if (EX) L1S::store(buf, o1s, re, im);
        else if (K1 != SW_NONE) L1::store(buf, o1, re, im);
        else L2S::store(buf, o2s, re, im);
    } else {
        if (EX) L2S::store(buf, o2s, re, im);
        else L1::store(buf, o1, re, im);
    }
}

// Butterflied register bits of a high group with m group bits (s = 12 - m run bits): H1 register bit i <-> f 7 + i,
// H2 register bit i <-> f 3 + i for i < 4 (bit 4 = f 7 is a filler, done in H1).
__host__ __device__ constexpr unsigned v2_h_mask1(int m) { unsigned k = 0; for (int i = 0; i < 5; ++i) if (7 + i >= 12 - m) k |= 1u << i; return k; }
__host__ __device__ constexpr unsigned v2_h_mask2(int m) { unsigned k = 0; for (int i = 0; i < 4; ++i) if (3 + i >= 12 - m) k |= 1u << i; return k; }

// M > 0: the number of group bits is a compile-time constant (masks folded: no run-time branches around the butterfly
// levels); M = -1: taken from g at run time.
template <int K1, int K2, int M, int MODE = 3>
__device__ __forceinline__ void v2_body_H(unsigned char* buf, const V2Geom& g, const bool diag, const double scale, const double2* tp,
                                          const double2* tab, const int t, const int grp)
{
    constexpr bool AR = (MODE & 1) != 0, EX = (MODE & 2) != 0;
    constexpr bool TEN = (M == 10);                    // ten group bits: layouts H1x / H2x, all five register bits in both
    using L1 = V2Layout<TEN ? TS_V2_H1X_R : TS_V2_H1_R, TEN ? TS_V2_H1X_T : TS_V2_H1_T, TEN ? 3u : 7u>;
    using L2 = V2Layout<TEN ? TS_V2_H2X_R : TS_V2_H2_R, TEN ? TS_V2_H2X_T : TS_V2_H2_T, TEN ? 3u : 7u>;
    constexpr bool CT = (M > 0);
    constexpr int MK1 = TEN ? 31 : (CT ? (int)v2_h_mask1(M > 0 ? M : 1) : -1);
    constexpr int MK2 = TEN ? 31 : (CT ? (int)v2_h_mask2(M > 0 ? M : 1) : -1);
    const uint32_t o1 = L1::thread_off(t), o2 = L2::thread_off(t);
    const bool two = EX && (CT ? (M > 5) : (g.two_stage != 0));
    double re[32], im[32];
    L1::load(buf, o1, re, im);
    v2_probe_touch<!AR>(re, im);
    if (AR) bfly_regs<K1, MK1>(re, im, g.mask1);
    if (two) {
        L1::store(buf, o1, re, im);
        v2_group_sync(grp);
        L2::load(buf, o2, re, im);
        v2_probe_touch<!AR>(re, im);
    }
    if (AR && (two || !EX)) bfly_regs<K1, MK2>(re, im, g.mask2);
    if (diag && AR) {
        double2 base, w[5];
        v2_thread_phase(scale, tp, tab, t, base, w);
        v2_apply_diag(tab + 768, base, w, re, im);
    }
    if (K2 != SW_NONE) {
        if (AR && (two || !EX)) bfly_regs<K2, MK2>(re, im, g.mask2);
        if (two) {
            L2::store(buf, o2, re, im);
            v2_group_sync(grp);
            L1::load(buf, o1, re, im);
            v2_probe_touch<!AR>(re, im);
        }
        if (AR) bfly_regs<K2, MK1>(re, im, g.mask1);
        L1::store(buf, o1, re, im);
    } else {
        if (two) L2::store(buf, o2, re, im);
        else L1::store(buf, o1, re, im);
    }
}

// ------------------------------------------------------------------------------------------------ TMA issue
// Tensor maps (ts_tile.cu): group A: the state as [2^(N-3)] rows of 16 doubles, box {16, 256}; high group: the state as
// [top][2^m rows][2^(g0-u) units][2^(u+1) doubles] with u = unit_log2, box {2^(u+1), 2^(s-u), 2^box_rows_log2, 1}: a tile
// is 2 (m <= 9) or 4 (m = 10) boxes of consecutive rows, landing one after the other.
struct V2Boxes { int c1, c3, nbox, rows, bytes; };
__device__ __forceinline__ V2Boxes v2_tile_boxes(const V2Geom& g, const uint64_t tile)
{
    V2Boxes b;
    if (g.type == 0) { b.c1 = (int)(tile << 9); b.c3 = 0; b.nbox = 2; b.rows = 256; b.bytes = 32768; }
    else {
        const uint64_t mid = tile & (((uint64_t)1 << g.nmid) - 1);
        b.c1 = (int)(mid << (g.s - g.unit_log2));
        b.c3 = (int)(tile >> g.nmid);
        b.rows = 1 << g.box_rows_log2;
        b.nbox = 1 << (g.m - g.box_rows_log2);
        b.bytes = TS_V2_TILE_BYTES >> (g.m - g.box_rows_log2);
    }
    return b;
}
// `half` 0 / 1: the boxes of the first / second half of the tile (a buffer is refilled half by half, see the loader)
__device__ __forceinline__ void v2_issue_load(const V2Geom& g, const CUtensorMap* tm, const uint64_t tile, const uint32_t dst,
                                              const uint32_t bar, const int half)
{
    const V2Boxes b = v2_tile_boxes(g, tile);
    for (int q = half * (b.nbox >> 1); q < (half + 1) * (b.nbox >> 1); ++q) {
        if (g.type == 0) v2_tma_load_2d(dst + q * b.bytes, tm, bar, 0, b.c1 + q * b.rows);
        else v2_tma_load_4d(dst + q * b.bytes, tm, bar, 0, b.c1, q * b.rows, b.c3);
    }
}
__device__ __forceinline__ void v2_issue_load_h(const V2Geom& g, const CUtensorMap* tm, const uint64_t tile, const uint32_t dst,
                                                const uint32_t bar, const uint64_t pol, const int half)
{
    const V2Boxes b = v2_tile_boxes(g, tile);
    for (int q = half * (b.nbox >> 1); q < (half + 1) * (b.nbox >> 1); ++q) {
        if (g.type == 0) v2_tma_load_2d_h(dst + q * b.bytes, tm, bar, 0, b.c1 + q * b.rows, pol);
        else v2_tma_load_4d_h(dst + q * b.bytes, tm, bar, 0, b.c1, q * b.rows, b.c3, pol);
    }
}
__device__ __forceinline__ void v2_issue_store_h(const V2Geom& g, const CUtensorMap* tm, const uint64_t tile, const uint32_t src,
                                                 const uint64_t pol, const int half)
{
    const V2Boxes b = v2_tile_boxes(g, tile);
    for (int q = half * (b.nbox >> 1); q < (half + 1) * (b.nbox >> 1); ++q) {
        if (g.type == 0) v2_tma_store_2d_h(tm, src + q * b.bytes, 0, b.c1 + q * b.rows, pol);
        else v2_tma_store_4d_h(tm, src + q * b.bytes, 0, b.c1, q * b.rows, b.c3, pol);
    }
}
__device__ __forceinline__ void v2_issue_store(const V2Geom& g, const CUtensorMap* tm, const uint64_t tile, const uint32_t src,
                                               const int half)
{
    const V2Boxes b = v2_tile_boxes(g, tile);
    for (int q = half * (b.nbox >> 1); q < (half + 1) * (b.nbox >> 1); ++q) {
        if (g.type == 0) v2_tma_store_2d(tm, src + q * b.bytes, 0, b.c1 + q * b.rows);
        else v2_tma_store_4d(tm, src + q * b.bytes, 0, b.c1, q * b.rows, b.c3);
    }
}

// Compute threads wait for job j's tile: buffer b = j % 3, use u = j / 3.  A parity wait only tells "the barrier's current
// phase has parity p" (block) from "it has the other parity" (pass), so it is sound only while the barrier is known to be
// in phase u or u + 1.  `full[b]` could still be in phase u - 1 if the other group's job j - 3 had not even landed; so
// first wait until that job has been CONSUMED (done[b], phase u - 1: it cannot run ahead of phase u before this very
// job arrives on it, and this group saw phase u - 2 complete when it finished job j - 6), which implies that full[b]
// completed phase u - 1.  Then full[b] is in phase u or u + 1 and the wait below is exact.
__device__ __forceinline__ void v2_wait_full(const uint32_t bar_full, const uint32_t bar_done, const uint32_t use)
{
    if (use > 0) v2_mbar_wait(bar_done, (use - 1) & 1u);
    v2_mbar_wait(bar_full, use & 1u);
}

__device__ __forceinline__ void v2_init_barriers(const uint32_t sBar)
{
    for (int k = 0; k < TS_V2_NBUF; ++k) {
        v2_mbar_init(sBar + TS_V2_BAR_FULL(k), 2);                    // full: the loader's two expect_tx arrives (one per half)
        v2_mbar_init(sBar + TS_V2_BAR_DONE(k), TS_TILE_THREADS);      // done: every thread of the compute group
        v2_mbar_init(sBar + TS_V2_BAR_FREE(k, 0), 1);                 // free: the storer, once per half
        v2_mbar_init(sBar + TS_V2_BAR_FREE(k, 1), 1);
    }
    v2_mbar_init(sBar + TS_V2_BAR_TABLE, 1);                          // tab: the launch's thread tables have landed
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    v2_fence_async_smem();
}

// ------------------------------------------------------------------------------------------------ scheduling
// Tickets.  sched[0] is the next ticket; the loader (one lane) draws them with atomicAdd, always one ahead of the ticket
// it is loading so that the atomic's round trip to L2 is never on its critical path.  sched[1] counts CTAs whose loader is
// done; the last one sets both words back to zero, so every launch starts from 0 without a memset in between.
__device__ __forceinline__ uint32_t v2_ticket_next(unsigned int* sched) { return atomicAdd(sched, 1u); }
__device__ __forceinline__ void v2_ticket_finish(unsigned int* sched)
{
    __threadfence();
    if (atomicAdd(sched + 1, 1u) == gridDim.x - 1) {      // every other CTA has drawn its last ticket already
        sched[0] = 0u;
        sched[1] = 0u;
        __threadfence();
    }
}
// Effective SM clock of a launch: CTA 0's loader reads the SM cycle counter and the global nanosecond timer when it starts
// and when it has drawn its last ticket, and leaves both differences in sched[2..5].  Under a power cap the clock a
// sampling tool reports and the cycles the SMs really get can differ; this is the latter (TS_OPT_LAST_LAUNCH_KHZ).
__device__ __forceinline__ void v2_clock_read(unsigned long long& cyc, unsigned long long& ns)
{
    asm volatile("mov.u64 %0, %%clock64;" : "=l"(cyc));
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(ns));
}
__device__ __forceinline__ void v2_clock_leave(unsigned int* sched, const unsigned long long c0, const unsigned long long t0)
{
    unsigned long long c1, t1;
    v2_clock_read(c1, t1);
    unsigned long long* out = reinterpret_cast<unsigned long long*>(sched + 2);
    out[0] = c1 - c0;
    out[1] = t1 - t0;
}
__device__ __forceinline__ uint32_t v2_ld_tile(const unsigned char* smraw, uint32_t b)
{
    return *reinterpret_cast<const volatile uint32_t*>(smraw + TS_V2_OFF_TILE + 4u * b);
}
__device__ __forceinline__ void v2_st_tile(unsigned char* smraw, uint32_t b, uint32_t v)
{
    *reinterpret_cast<volatile uint32_t*>(smraw + TS_V2_OFF_TILE + 4u * b) = v;
}
// The loader's epilogue: two END markers, one for each compute group (local jobs j and j + 1 belong to different groups;
// the storer leaves at the first).  A marker completes the buffer's `full` phase with a plain arrive (no bytes expected).
__device__ __forceinline__ void v2_push_end(unsigned char* smraw, const uint32_t sBar, uint64_t j)
{
    for (int k = 0; k < 2; ++k, ++j) {
        const uint32_t b = (uint32_t)(j % TS_V2_NBUF), use = (uint32_t)(j / TS_V2_NBUF);
        if (use > 0) {
            v2_mbar_wait(sBar + TS_V2_BAR_FREE(b, 0), (use - 1) & 1u);
            v2_mbar_wait(sBar + TS_V2_BAR_FREE(b, 1), (use - 1) & 1u);
        }
        v2_st_tile(smraw, b, TS_V2_END);
        v2_mbar_arrive(sBar + TS_V2_BAR_FULL(b));
        v2_mbar_arrive(sBar + TS_V2_BAR_FULL(b));
    }
}

// ------------------------------------------------------------------------------------------------ one tile pass
// TYPE 0: group A, 1: high group (any m <= 9), 2: high group with m = 9 (masks folded), 3: high group with m = 10 (64-byte
// runs, layouts H1x / H2x).  MODE: see v2_body_A.
template <int TYPE, int K1, int K2, int MODE = 3>
__global__ void __launch_bounds__(TS_V2_THREADS, 1)
k_tile_v2(const __grid_constant__ V2Pass p, const __grid_constant__ CUtensorMap tmap)
{
    extern __shared__ __align__(1024) unsigned char smraw[];
    const uint32_t sBase = v2_smem_u32(smraw);
    const uint32_t sBar = sBase + TS_V2_OFF_BAR;
    const int warp = threadIdx.x >> 5;
    const bool has_diag = (p.d.tile_phase != nullptr);

    if (threadIdx.x == 0) {
        if (sBase & 1023u) __trap();                   // the 128-byte swizzle is a function of the shared address
        v2_init_barriers(sBar);
    }
    __syncthreads();

    if (warp >= 8) {                                   // ---- producer warpgroup: hands its registers to the compute warpgroups
        v2_regs_dec<TS_V2_REGS_PRODUCER>();
        if (warp == 8 && (threadIdx.x & 31) == 0) {    // ---- loader
            if (has_diag) {
                v2_mbar_expect_tx(sBar + TS_V2_BAR_TABLE, TS_V2_TAB_BYTES);
                v2_bulk_load(sBase + TS_V2_OFF_TAB, p.d.tables, TS_V2_TAB_BYTES, sBar + TS_V2_BAR_TABLE);
            }
            const uint32_t per = 1u << p.pair_log2;
            const uint64_t ntick = p.ntiles >> p.pair_log2;
            uint64_t j = 0;
            unsigned long long clk0 = 0, ns0 = 0;
            if (blockIdx.x == 0) v2_clock_read(clk0, ns0);
            uint32_t tk = v2_ticket_next(p.sched);
            while (tk < ntick) {
                const uint32_t nxt = v2_ticket_next(p.sched);
                for (uint32_t u = 0; u < per; ++u, ++j) {
                    // A buffer comes back half by half: the first half of the next tile is on its way while the store of
                    // the previous tile is still reading the second half (one buffer is all the transport has while both
                    // compute groups hold theirs, so its turn-around time is the pipeline's period).
                    const uint32_t b = (uint32_t)(j % TS_V2_NBUF), use = (uint32_t)(j / TS_V2_NBUF);
                    const uint64_t tile = ((uint64_t)tk << p.pair_log2) + u;
                    const uint32_t bar = sBar + TS_V2_BAR_FULL(b);
                    if (use > 0) v2_mbar_wait(sBar + TS_V2_BAR_FREE(b, 0), (use - 1) & 1u);
                    v2_st_tile(smraw, b, (uint32_t)tile);
                    v2_mbar_expect_tx(bar, TS_V2_TILE_BYTES / 2 + (has_diag ? 512u : 0u));
                    if (has_diag) v2_bulk_load(sBase + TS_V2_OFF_TP + b * 512u, p.d.tile_phase + (tile << 5), 512u, bar);
                    v2_issue_load(p.g, &tmap, tile, sBase + b * TS_V2_TILE_BYTES, bar, 0);
                    if (use > 0) v2_mbar_wait(sBar + TS_V2_BAR_FREE(b, 1), (use - 1) & 1u);
                    v2_mbar_expect_tx(bar, TS_V2_TILE_BYTES / 2);
                    v2_issue_load(p.g, &tmap, tile, sBase + b * TS_V2_TILE_BYTES, bar, 1);
                }
                tk = nxt;
            }
            v2_push_end(smraw, sBar, j);
            if (blockIdx.x == 0) v2_clock_leave(p.sched, clk0, ns0);
            v2_ticket_finish(p.sched);
        } else if (warp == 9 && (threadIdx.x & 31) == 0) {   // ---- storer
            for (uint64_t j = 0;; ++j) {
                const uint32_t b = (uint32_t)(j % TS_V2_NBUF), use = (uint32_t)(j / TS_V2_NBUF);
                v2_mbar_wait(sBar + TS_V2_BAR_DONE(b), use & 1u);
                const uint32_t tile = v2_ld_tile(smraw, b);
                if (tile == TS_V2_END) break;
                v2_issue_store(p.g, &tmap, tile, sBase + b * TS_V2_TILE_BYTES, 0);
                v2_store_commit();
                v2_issue_store(p.g, &tmap, tile, sBase + b * TS_V2_TILE_BYTES, 1);
                v2_store_commit();
                v2_store_wait_read_but_one();          // the first half has been read: it can be refilled
                v2_mbar_arrive(sBar + TS_V2_BAR_FREE(b, 0));
                v2_store_wait_read();
                v2_mbar_arrive(sBar + TS_V2_BAR_FREE(b, 1));
            }
            v2_store_wait_all();
        }
    } else {                                           // ---- compute warpgroups
        v2_regs_inc<TS_V2_REGS_COMPUTE>();
        const int grp = warp >> 2;
        const int t = threadIdx.x & (TS_TILE_THREADS - 1);
        const double2* tab = reinterpret_cast<const double2*>(smraw + TS_V2_OFF_TAB);
        const double scale = p.d.scale;
        if (has_diag) v2_mbar_wait(sBar + TS_V2_BAR_TABLE, 0u);
        if (grp >= p.ngroups) return;
        for (uint64_t j = grp;; j += p.ngroups) {
            const uint32_t b = (uint32_t)(j % TS_V2_NBUF), use = (uint32_t)(j / TS_V2_NBUF);
            v2_wait_full(sBar + TS_V2_BAR_FULL(b), sBar + TS_V2_BAR_DONE(b), use);
            const bool end = (v2_ld_tile(smraw, b) == TS_V2_END);
            if (!end && !p.probe) {
                unsigned char* buf = smraw + b * TS_V2_TILE_BYTES;
                const double2* tp = reinterpret_cast<const double2*>(smraw + TS_V2_OFF_TP + b * 512u);
                if constexpr (TYPE == 0) v2_body_A<K1, K2, MODE>(buf, has_diag, scale, tp, tab, t, grp);
                else if constexpr (TYPE == 2) v2_body_H<K1, K2, 9, MODE>(buf, p.g, has_diag, scale, tp, tab, t, grp);
                else if constexpr (TYPE == 3) v2_body_H<K1, K2, 10, MODE>(buf, p.g, has_diag, scale, tp, tab, t, grp);
                else v2_body_H<K1, K2, -1, MODE>(buf, p.g, has_diag, scale, tp, tab, t, grp);
                v2_fence_async_smem();                 // my shared-memory writes -> visible to the TMA store
            }
            v2_mbar_arrive(sBar + TS_V2_BAR_DONE(b));
            if (end) break;
        }
    }
}

// ------------------------------------------------------------------------------------------------ L2-blocked triple
// Jobs n = 0 .. 3 * nchunks * T - 1 (T = tiles per chunk) in blocks of one (phase, chunk):
//     P1(0) P1(1) P2(0) P2(1) P3(0) | P1(c) P3(c-1) P2(c), c = 2 .. nchunks-1 | P3(nchunks-1)
// P1 = high group, sweep KA (from HBM);  P2 = group A, KA . D . KB (from L2);  P3 = high group, sweep KB (from L2, then
// out to HBM).  A chunk is closed under all three (closed-set argument of P:141 applied to spins 0 .. C-1), so two
// chunks (64 MiB) live in the 126 MB L2 at any time and the state makes ONE HBM round trip for three tile passes.
// Job n is ticket n: tickets are drawn in increasing order and every CTA loads its tickets in the order it drew them.  A
// job of phase 2 / 3 may be LOADED once all T tiles of the previous phase of its chunk are stored and visible: the loader
// polls done[phase - 1][chunk] (acquire) before it issues the TMA load, the storer publishes a tile (release) once its TMA
// store has completed.  Only the loader ever waits on other CTAs; the compute groups and the storer keep draining the
// jobs already loaded.  The smallest unfinished ticket depends only on smaller tickets, all finished, and it is the
// oldest job of the CTA that drew it: the launch cannot deadlock as long as all CTAs are resident (cooperative launch).
template <int KA, int KB, int HM, int MODE = 3>
__global__ void __launch_bounds__(TS_V2_THREADS, 1)
k_chunk_v2(const __grid_constant__ V2Chunk q, const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmH)
{
    extern __shared__ __align__(1024) unsigned char smraw[];
    const uint32_t sBase = v2_smem_u32(smraw);
    const uint32_t sBar = sBase + TS_V2_OFF_BAR;
    const int warp = threadIdx.x >> 5;
    const uint32_t tl = q.tiles_log2, T = 1u << tl;
    const uint32_t nblocks = 3u * q.nchunks;
    const uint32_t total = nblocks << tl;
    const bool has_diag = (q.d.tile_phase != nullptr);

    auto job_of = [&](const uint32_t n, uint32_t& phase, uint32_t& c, uint64_t& tile) {
        const uint32_t B = n >> tl;
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
        v2_init_barriers(sBar);
    }
    __syncthreads();

    if (warp >= 8) {                                   // ---- producer warpgroup
        v2_regs_dec<TS_V2_REGS_PRODUCER>();
        if (warp == 8 && (threadIdx.x & 31) == 0) {    // ---- loader
            if (has_diag) {
                v2_mbar_expect_tx(sBar + TS_V2_BAR_TABLE, TS_V2_TAB_BYTES);
                v2_bulk_load(sBase + TS_V2_OFF_TAB, q.d.tables, TS_V2_TAB_BYTES, sBar + TS_V2_BAR_TABLE);
            }
            // L2 priorities: what phase 1 reads from HBM is about to be overwritten (evict first); what phases 1 and 2
            // write is read again from L2 (evict last); the third phase's reads are the last use of a line.
            const uint64_t pol_ld[3] = {v2_policy(q.l2_hints ? 1 : 0), v2_policy(q.l2_hints ? 2 : 0), v2_policy(q.l2_hints ? 1 : 0)};
            uint32_t ok_key = 0xffffffffu;             // (phase, chunk) whose dependency was last seen satisfied
            uint64_t j = 0;
            unsigned long long clk0 = 0, ns0 = 0;
            if (blockIdx.x == 0) v2_clock_read(clk0, ns0);
            uint32_t n = v2_ticket_next(q.sched);
            while (n < total) {
                const uint32_t nxt = v2_ticket_next(q.sched);
                const uint32_t b = (uint32_t)(j % TS_V2_NBUF), use = (uint32_t)(j / TS_V2_NBUF);
                uint32_t phase, c; uint64_t tile;
                job_of(n, phase, c, tile);
                if (phase != 0) {
                    const uint32_t key = (phase << 28) | c;
                    if (key != ok_key) {
                        const unsigned int* dp = q.done + (size_t)(phase - 1) * q.nchunks + c;
                        while (v2_ld_acquire(dp) < T) __nanosleep(64);
                        ok_key = key;
                    }
                    v2_fence_async_all();              // the TMA engine reads what other SMs' TMA stores wrote
                }
                const uint32_t bar = sBar + TS_V2_BAR_FULL(b);
                const bool tpl = has_diag && phase == 1;
                const V2Geom& gj = (phase == 1) ? q.ga : q.gh;
                const CUtensorMap* tmj = (phase == 1) ? &tmA : &tmH;
                if (use > 0) v2_mbar_wait(sBar + TS_V2_BAR_FREE(b, 0), (use - 1) & 1u);
                v2_st_tile(smraw, b, n);
                v2_mbar_expect_tx(bar, TS_V2_TILE_BYTES / 2 + (tpl ? 512u : 0u));
                if (tpl) v2_bulk_load(sBase + TS_V2_OFF_TP + b * 512u, q.d.tile_phase + (tile << 5), 512u, bar);
                v2_issue_load_h(gj, tmj, tile, sBase + b * TS_V2_TILE_BYTES, bar, pol_ld[phase], 0);
                if (use > 0) v2_mbar_wait(sBar + TS_V2_BAR_FREE(b, 1), (use - 1) & 1u);
                v2_mbar_expect_tx(bar, TS_V2_TILE_BYTES / 2);
                v2_issue_load_h(gj, tmj, tile, sBase + b * TS_V2_TILE_BYTES, bar, pol_ld[phase], 1);
                ++j;
                n = nxt;
            }
            v2_push_end(smraw, sBar, j);
            if (blockIdx.x == 0) v2_clock_leave(q.sched, clk0, ns0);
            v2_ticket_finish(q.sched);
        } else if (warp == 9 && (threadIdx.x & 31) == 0) {   // ---- storer
            const uint64_t pol_st[3] = {v2_policy(q.l2_hints ? 2 : 0), v2_policy(q.l2_hints ? 2 : 0), v2_policy(q.l2_hints ? 1 : 0)};
            for (uint64_t j = 0;; ++j) {
                const uint32_t b = (uint32_t)(j % TS_V2_NBUF), use = (uint32_t)(j / TS_V2_NBUF);
                v2_mbar_wait(sBar + TS_V2_BAR_DONE(b), use & 1u);
                const uint32_t n = v2_ld_tile(smraw, b);
                if (n == TS_V2_END) break;
                uint32_t phase, c; uint64_t tile;
                job_of(n, phase, c, tile);
                const V2Geom& gj = (phase == 1) ? q.ga : q.gh;
                const CUtensorMap* tmj = (phase == 1) ? &tmA : &tmH;
                v2_issue_store_h(gj, tmj, tile, sBase + b * TS_V2_TILE_BYTES, pol_st[phase], 0);
                v2_store_commit();
                v2_issue_store_h(gj, tmj, tile, sBase + b * TS_V2_TILE_BYTES, pol_st[phase], 1);
                v2_store_commit();
                v2_store_wait_read_but_one();          // a half can be refilled as soon as the store has read it
                v2_mbar_arrive(sBar + TS_V2_BAR_FREE(b, 0));
                v2_store_wait_read();
                v2_mbar_arrive(sBar + TS_V2_BAR_FREE(b, 1));
                if (phase != 2) {
                    // Publish only once the tile IS in global memory (L2).  (Not deferred to the next job: a publish
                    // that waited for this CTA's next job could wait for a job that depends on it.)
                    v2_store_wait_all();
                    v2_fence_async_all();
                    __threadfence();
                    atomicAdd(q.done + (size_t)phase * q.nchunks + c, 1u);
                }
            }
            v2_store_wait_all();
        }
    } else {                                           // ---- compute warpgroups
        v2_regs_inc<TS_V2_REGS_COMPUTE>();
        const int grp = warp >> 2;
        const int t = threadIdx.x & (TS_TILE_THREADS - 1);
        const double2* tab = reinterpret_cast<const double2*>(smraw + TS_V2_OFF_TAB);
        const double scale = q.d.scale;
        if (has_diag) v2_mbar_wait(sBar + TS_V2_BAR_TABLE, 0u);
        if (grp >= q.ngroups) return;
        for (uint64_t j = grp;; j += q.ngroups) {
            const uint32_t b = (uint32_t)(j % TS_V2_NBUF), use = (uint32_t)(j / TS_V2_NBUF);
            v2_wait_full(sBar + TS_V2_BAR_FULL(b), sBar + TS_V2_BAR_DONE(b), use);
            const uint32_t n = v2_ld_tile(smraw, b);
            const bool end = (n == TS_V2_END);
            if (!end && !q.probe) {
                const uint32_t B = n >> tl;
                // phase of block B (see job_of): 0 / 2 = high group, 1 = group A
                uint32_t phase;
                if (B == nblocks - 1) phase = 2;
                else if (B < 5) phase = (B < 2) ? 0u : (B < 4 ? 1u : 2u);
                else { const uint32_t r = (B - 5) % 3; phase = (r == 0) ? 0u : (r == 1 ? 2u : 1u); }
                unsigned char* buf = smraw + b * TS_V2_TILE_BYTES;
                const double2* tp = reinterpret_cast<const double2*>(smraw + TS_V2_OFF_TP + b * 512u);
                if (phase == 0) v2_body_H<KA, SW_NONE, HM, MODE>(buf, q.gh, false, 1.0, tp, tab, t, grp);
                else if (phase == 1) v2_body_A<KA, KB, MODE>(buf, has_diag, scale, tp, tab, t, grp);
                else v2_body_H<KB, SW_NONE, HM, MODE>(buf, q.gh, false, 1.0, tp, tab, t, grp);
                v2_fence_async_smem();
            }
            v2_mbar_arrive(sBar + TS_V2_BAR_DONE(b));
            if (end) break;
        }
    }
}

} // namespace tsk
#endif
