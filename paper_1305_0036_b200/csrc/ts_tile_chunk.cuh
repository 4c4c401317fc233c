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
#include "ts_tile_kernel.cuh"

struct ChunkParams {
    TilePassParams h;          // geometry of the high group (phases 1 and 3; no diagonal)
    TilePassParams a;          // group A with the diagonal's tables (phase 2)
    const uint32_t* sched;     // [nblocks]: phase | chunk << 2
    unsigned int* ticket;      // job counter (zeroed before the launch)
    unsigned int* done;        // [2][nchunks] (zeroed before the launch)
    uint32_t nblocks, nchunks, tiles_log2;
};

typedef void (*chunk_kernel_t)(const ChunkParams);
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

#define TS_CHUNK_REGISTER_CFG(NAME, BF1, BF2)                                                                     \
    void ts_chunk_register_##NAME(chunk_kernel_t (*tab)[2])                                                       \
    {                                                                                                             \
        (*tab)[0] = tsk::k_chunk_triple<SW_YDAG, SW_Y, BF1, BF2>;                                                 \
        (*tab)[1] = tsk::k_chunk_triple<SW_X, SW_XDAG, BF1, BF2>;                                                 \
    }

} // namespace tsk
#endif
