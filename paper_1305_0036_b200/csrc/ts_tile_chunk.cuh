// ts_tile_chunk.cuh -- L2-blocked execution of three consecutive tile passes in ONE launch.
//
// At N = 30 the passes of a step repeat the pattern  H1(sweep i) , A(sweep i . D_i . sweep i+1) , H1(sweep i+1) , H2(...)
// where A = spins 0..11 and H1 = spins 12..20.  The first three act inside aligned chunks of 2^21 amplitudes (32 MiB:
// the closed-set argument of P:141 applied to the chunk), so a chunk can be read from HBM once, stay in the 126 MB L2
// for the two passes in between, and be written back once: one HBM round trip instead of three.
//
// One persistent launch (2 CTAs per SM) executes all 3 x nchunks x 2^(C-12) tile jobs.  Jobs are handed out in a fixed
// order by a global ticket counter:  P1(0) P2(0) | P1(c) P3(c-1) P2(c) | ... | P3(last), in blocks of one (phase,
// chunk) = 512 tiles.  A phase of a chunk may start when all tiles of the previous phase of that chunk are done
// (done[phase][chunk] == tiles per chunk, published with __threadfence + atomicAdd); every dependency lies at least
// one block (512 jobs, ~1.7 waves of CTAs) back in the ticket order, so CTAs practically never wait, and since
// tickets are claimed in order a waiting CTA only ever waits for jobs already claimed by running CTAs (no deadlock,
// co-residency not required).  Two chunks (64 MiB) are live at any time.  Loads bypass L1 (another SM wrote the data
// in this launch); stores of phases 1 and 2 stay in L2 (st.global.cg), phase 3 streams out (st.global.cs).
#pragma once
#include "ts_tile_pipe.cuh"

struct ChunkParams {
    TilePassParams h;          // geometry of the high group (phases 1 and 3; no diagonal)
    TilePassParams a;          // group A with the diagonal's tables (phase 2)
    const uint32_t* sched;     // [nblocks]: phase | chunk << 2
    unsigned int* ticket;      // job counter (zeroed before the launch)
    unsigned int* done;        // [2][nchunks] (zeroed before the launch)
    uint32_t nblocks, nchunks, tiles_log2;
};

typedef void (*chunk_kernel_t)(const ChunkParams);
// pipelined variant (k_chunk_pipe): same job order, static round-robin over persistent CTAs, TMA-fed
typedef void (*chunk_pipe_kernel_t)(const ChunkParams, const CUtensorMap, const PipeGeom);
void ts_chunk_pipe_register_H7(chunk_pipe_kernel_t (*tab)[2]);
void ts_chunk_pipe_register_H8(chunk_pipe_kernel_t (*tab)[2]);
void ts_chunk_pipe_register_H9(chunk_pipe_kernel_t (*tab)[2]);
void ts_chunk_pipe_register_H10(chunk_pipe_kernel_t (*tab)[2]);
// tab[cfg][v]: v = 0: (Y^dag, Y), v = 1: (X, X^dag) -- the two kind pairs that meet at group A in the sweep order
void ts_chunk_register_H7(chunk_kernel_t (*tab)[2]);
void ts_chunk_register_H8(chunk_kernel_t (*tab)[2]);
void ts_chunk_register_H9(chunk_kernel_t (*tab)[2]);
void ts_chunk_register_H10(chunk_kernel_t (*tab)[2]);

#ifdef __CUDACC__
namespace tsk {

template <int KA, int KB, int HBF1, int HBF2>
__global__ void __launch_bounds__(TS_TILE_THREADS, 2) k_chunk_triple(const __grid_constant__ ChunkParams q)
{
    extern __shared__ double2 sm[];
    __shared__ unsigned int s_item;
    const uint32_t T = 1u << q.tiles_log2;
    const uint32_t total = q.nblocks << q.tiles_log2;
    unsigned int next = 0;
    if (threadIdx.x == 0) next = atomicAdd(q.ticket, 1u);
    for (;;) {
        if (threadIdx.x == 0) s_item = next;
        __syncthreads();
        const unsigned int item = s_item;
        if (item >= total) break;
        if (threadIdx.x == 0) next = atomicAdd(q.ticket, 1u);      // next ticket: its latency hides behind this tile
        const uint32_t e = __ldg(q.sched + (item >> q.tiles_log2));
        const uint32_t phase = e & 3u, c = e >> 2;
        const uint64_t tau = ((uint64_t)c << q.tiles_log2) | (item & (T - 1));
        if (phase != 0) {
            if (threadIdx.x == 0) {
                const volatile unsigned int* d = q.done + (size_t)(phase - 1) * q.nchunks + c;
                while (*d < T) __nanosleep(100);
                __threadfence();
            }
            __syncthreads();
        }
        if (phase == 0) tile_body<KA, SW_NONE, HBF1, HBF2, 0, 3>(q.h, tau, sm);
        else if (phase == 1) tile_body<KA, KB, 31, 31, 2, 3>(q.a, tau, sm);
        else tile_body<KB, SW_NONE, HBF1, HBF2, 0, 1>(q.h, tau, sm);
        __syncthreads();                                            // all stores issued; sm and s_item free
        if (phase != 2 && threadIdx.x == 0) {
            __threadfence();
            atomicAdd(q.done + (size_t)phase * q.nchunks + c, 1u);
        }
    }
}


// ---- pipelined variant.  Jobs n = 0 .. nblocks * T - 1 in the order of `sched`; CTA b runs jobs b, b + G, ... with the
// same half-tile TMA ring and two compute groups as k_tile_pipe.  The thread that issues the load of a job first waits
// for the job's dependency (all tiles of the previous phase of its chunk), because the load is what reads their data.
template <int KA, int KB, int HBF1, int HBF2>
__global__ void __launch_bounds__(TS_PIPE_THREADS, 1)
k_chunk_pipe(const __grid_constant__ ChunkParams q, const __grid_constant__ CUtensorMap tmap, const PipeGeom g)
{
    extern __shared__ __align__(1024) unsigned char smraw[];
    const int grp = threadIdx.x >> 7;
    const int t = threadIdx.x & (TS_TILE_THREADS - 1);
    const uint32_t sL = smem_u32(smraw);
    const uint32_t sTP = smem_u32(smraw + TS_PIPE_OFF_TP);
    const uint32_t sBar = smem_u32(smraw + TS_PIPE_OFF_BAR);
    double2* E = reinterpret_cast<double2*>(smraw + TS_PIPE_OFF_E) + ((size_t)grp << TS_TILE_LOG2);
    const double2* TPs = reinterpret_cast<const double2*>(smraw + TS_PIPE_OFF_TP);
    volatile uint32_t* cons = reinterpret_cast<volatile uint32_t*>(smraw + TS_PIPE_OFF_BAR + 32);

    const uint32_t tl = q.tiles_log2, T = 1u << tl;
    const uint64_t total = (uint64_t)q.nblocks << tl;
    const uint64_t G = gridDim.x;
    const uint64_t n_cta = (total > blockIdx.x) ? (total - blockIdx.x + G - 1) / G : 0;
    const uint64_t n_half = 2 * n_cta;
    const bool a_diag = (q.a.tile_phase != nullptr);

    // job i of this CTA -> (phase, chunk, tile); the block order of ts_tile.cu's pipelined schedule in closed form
    // (P1(0) P1(1) P2(0) P2(1) P3(0) | P1(c) P3(c-1) P2(c), c >= 2): no table read on the issuing thread's critical path
    auto job_of = [&](uint64_t i, uint32_t& phase, uint32_t& c, uint64_t& tau) {
        const uint64_t n = blockIdx.x + i * G;
        const uint32_t B = (uint32_t)(n >> tl);
        if (B < 5) { phase = (B < 2) ? 0u : (B < 4 ? 1u : 2u); c = (B == 1 || B == 3) ? 1u : 0u; }
        else {
            const uint32_t k = B - 5, r = k % 3;
            c = 2 + k / 3;
            if (r == 0) phase = 0; else if (r == 1) { phase = 2; c -= 1; } else phase = 1;
        }
        tau = ((uint64_t)c << tl) | (n & (T - 1));
    };
    auto dep_ptr = [&](uint32_t phase, uint32_t c) { return q.done + (size_t)(phase - 1) * q.nchunks + c; };
    // issuing-thread state lives in shared memory (only thread 0 of each group touches it): registers are all taken
    // st[0] = ok_dep: (phase << 28 | chunk) whose dependency this thread last saw satisfied; st[1], st[2] = pre_key,
    // pre_val: counter value read ahead of time for the job issued next; st[3] = pending publish (index + 1 into done)
    volatile uint32_t* st = reinterpret_cast<volatile uint32_t*>(smraw + TS_PIPE_OFF_BAR + 40) + 4 * grp;
#define ok_dep st[0]
#define pre_key st[1]
#define pre_val st[2]
    auto issue_load = [&](uint64_t qh, int slot) {
        uint32_t phase, c; uint64_t tau;
        job_of(qh >> 1, phase, c, tau);
        const int h = (int)(qh & 1);
        const uint32_t key = (phase << 28) | c;
        if (phase != 0 && ok_dep != key) {
            if (!(pre_key == key && pre_val >= T)) {
                const volatile unsigned int* d = dep_ptr(phase, c);
                while (*d < T) __nanosleep(100);
            }
            __threadfence();
            asm volatile("fence.proxy.async;" ::: "memory");     // the TMA engine reads what other SMs' threads wrote
            ok_dep = key;
        }
        {   // read the next job's dependency counter now; it is looked at when that job's load is issued
            uint32_t p2, c2; uint64_t t2;
            job_of((qh >> 1) + 1, p2, c2, t2);
            const uint32_t k2 = (p2 << 28) | c2;
            if (p2 != 0 && k2 != ok_dep && (qh >> 1) + 1 < n_cta) { pre_key = k2; pre_val = *(const volatile unsigned int*)dep_ptr(p2, c2); }
        }
        const uint32_t bar = sBar + 8 * slot;
        const uint32_t dst = sL + slot * TS_PIPE_HALF_BYTES;
        if (phase == 1) {
            const bool tp = a_diag && h == 0;
            mbar_expect_tx(bar, TS_PIPE_HALF_BYTES + (tp ? 512u : 0u));
            if (tp) bulk_load(sTP + slot * 512, q.a.tile_phase + (tau << 5), 512, bar);
            bulk_load(dst, q.a.psi + (tau << TS_TILE_LOG2) + (uint64_t)h * (TS_PIPE_HALF_BYTES / 16), TS_PIPE_HALF_BYTES, bar);
        } else {
            const int s = q.h.s, g0 = q.h.g0, nmid = g0 - s;
            const uint64_t mid = tau & (((uint64_t)1 << nmid) - 1), hi = tau >> nmid;
            mbar_expect_tx(bar, TS_PIPE_HALF_BYTES);
            if (g.tensor) {
                for (int b = 0; b < g.nbox; ++b)
                    tensor_load_3d(dst + b * g.box_rows * g.row_bytes, &tmap, bar, (int)(mid << (s + 1)),
                                   h * g.rows_half + b * g.box_rows, (int)hi);
            } else {
                const uint64_t base_idx = (mid << s) | (hi << (g0 + TS_TILE_LOG2 - s));
                for (int r = 0; r < g.rows_half; ++r)
                    bulk_load(dst + r * g.row_bytes, q.h.psi + base_idx + ((uint64_t)(h * g.rows_half + r) << g0), g.row_bytes, bar);
            }
        }
    };

    if (threadIdx.x == 0) {
        for (int k = 0; k < TS_PIPE_SLOTS; ++k) mbar_init(sBar + 8 * k, 1);
        cons[0] = 0; cons[1] = 0;
        for (int k = 0; k < 8; ++k) (reinterpret_cast<volatile uint32_t*>(smraw + TS_PIPE_OFF_BAR + 40))[k] = (k & 3) < 2 ? 0xffffffffu : 0u;
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        for (uint64_t qh = 0; qh < TS_PIPE_SLOTS && qh < n_half; ++qh) issue_load(qh, (int)qh);
    }
    __syncthreads();

    uint32_t slot = (2 * grp) % TS_PIPE_SLOTS, use = (2 * grp) / TS_PIPE_SLOTS;

    for (uint64_t i = grp; i < n_cta; i += 2) {
        uint32_t phase, c; uint64_t tau;
        job_of(i, phase, c, tau);
        double re[32], im[32];
        double2 base = make_double2(1.0, 0.0), w[5];
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            if (h == 1 && i > 0) while (cons[grp ^ 1] < (uint32_t)i) { }      // see k_tile_pipe
            mbar_wait(sBar + 8 * slot, use & 1);
            const double2* Ls = reinterpret_cast<const double2*>(smraw + slot * TS_PIPE_HALF_BYTES);
#pragma unroll
            for (int r = 0; r < 16; ++r) {
                const double2 v = Ls[t | (r << 7)];
                re[16 * h + r] = v.x; im[16 * h + r] = v.y;
            }
            if (h == 0 && phase == 1 && a_diag) pipe_thread_phase(q.a, TPs + slot * 32, t, base, w);
            group_sync(grp);
            if (t == (h ? 32 : 0)) {     // the two halves are served by different warps: neither is late twice
                // every thread of the group issued the stores of the previous tile before this barrier: publish it now
                // (the fence is cumulative over the barrier), off the critical path of that tile
                if (h == 0 && st[3]) { __threadfence(); atomicAdd(q.done + (st[3] - 1), 1u); st[3] = 0; }
                const uint64_t qn = 2 * i + h + TS_PIPE_SLOTS;
                if (qn < n_half) issue_load(qn, (int)slot);
                if (h == 0) cons[grp] = (uint32_t)i + 1;
            }
            slot += 1; if (slot >= TS_PIPE_SLOTS) { slot -= TS_PIPE_SLOTS; use += 1; }
        }
        slot += 2; if (slot >= TS_PIPE_SLOTS) { slot -= TS_PIPE_SLOTS; use += 1; }

        if (phase == 0) pipe_compute_store<KA, SW_NONE, HBF1, HBF2, 0, true>(q.h, tau, re, im, base, w, E, t, grp);
        else if (phase == 1) pipe_compute_store<KA, KB, 31, 31, 2, true>(q.a, tau, re, im, base, w, E, t, grp);
        else pipe_compute_store<KB, SW_NONE, HBF1, HBF2, 0, false>(q.h, tau, re, im, base, w, E, t, grp);
        if (t == 0 && phase != 2) st[3] = phase * q.nchunks + c + 1;
    }
    group_sync(grp);
    if (t == 0 && st[3]) { __threadfence(); atomicAdd(q.done + (st[3] - 1), 1u); }
#undef ok_dep
#undef pre_key
#undef pre_val
}

#define TS_CHUNK_REGISTER_CFG(NAME, BF1, BF2)                                                                     \
    void ts_chunk_register_##NAME(chunk_kernel_t (*tab)[2])                                                       \
    {                                                                                                             \
        (*tab)[0] = tsk::k_chunk_triple<SW_YDAG, SW_Y, BF1, BF2>;                                                 \
        (*tab)[1] = tsk::k_chunk_triple<SW_X, SW_XDAG, BF1, BF2>;                                                 \
    }                                                                                                             \
    void ts_chunk_pipe_register_##NAME(chunk_pipe_kernel_t (*tab)[2])                                             \
    {                                                                                                             \
        (*tab)[0] = tsk::k_chunk_pipe<SW_YDAG, SW_Y, BF1, BF2>;                                                   \
        (*tab)[1] = tsk::k_chunk_pipe<SW_X, SW_XDAG, BF1, BF2>;                                                   \
    }

} // namespace tsk
#endif
