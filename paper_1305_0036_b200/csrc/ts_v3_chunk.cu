// ts_v3_chunk.cu -- L2-blocked triple launches of the 16-amplitudes-per-thread family (ts_tile_v3.cuh): both kind pairs,
// any high group (run-time masks) and the 9-bit high group of the default plan.
#include "ts_tile_v3.cuh"

void ts_v3_register_chunk0(v2_chunk_kernel_t (*tab)[2]) { tab[0][0] = tsk::k_chunk_v3<SW_YDAG, SW_Y, -1>; }
void ts_v3_register_chunk1(v2_chunk_kernel_t (*tab)[2]) { tab[0][1] = tsk::k_chunk_v3<SW_X, SW_XDAG, -1>; }
void ts_v3_register_chunk0_h9(v2_chunk_kernel_t (*tab)[2]) { tab[1][0] = tsk::k_chunk_v3<SW_YDAG, SW_Y, 9>; }
void ts_v3_register_chunk1_h9(v2_chunk_kernel_t (*tab)[2]) { tab[1][1] = tsk::k_chunk_v3<SW_X, SW_XDAG, 9>; }
