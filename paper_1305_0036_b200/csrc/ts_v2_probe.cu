// ts_v2_probe.cu -- measurement builds of the kernels of the N = 30 metric plan (TS_OPT_PROBE = 2, 3): the same
// pipelines with only the arithmetic (mode 1) or only the shared-memory layout exchanges (mode 2) in the tile body.  Their
// results are wrong by construction; they exist to attribute the time of a pass to its FP64 work, its shared-memory
// traffic and its tile transport.
#include "ts_tile_v2.cuh"

void ts_v2_register_probe(v2_chunk_kernel_t* chunk, v2_kernel_t* fusedH, v2_kernel_t* fusedA)
{
    chunk[0] = tsk::k_chunk_v2<SW_YDAG, SW_Y, 9, 1>;
    chunk[1] = tsk::k_chunk_v2<SW_YDAG, SW_Y, 9, 2>;
    fusedH[0] = tsk::k_tile_v2<2, SW_XDAG, SW_YDAG, 1>;
    fusedH[1] = tsk::k_tile_v2<2, SW_XDAG, SW_YDAG, 2>;
    fusedA[0] = tsk::k_tile_v2<0, SW_YDAG, SW_Y, 1>;
    fusedA[1] = tsk::k_tile_v2<0, SW_YDAG, SW_Y, 2>;
}
