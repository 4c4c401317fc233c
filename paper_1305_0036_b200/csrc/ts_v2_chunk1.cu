// ts_v2_chunk1.cu -- L2-blocked triple launch (ts_tile_v2.cuh), kinds (X, X^dag), any high group.
#include "ts_tile_v2.cuh"

void ts_v2_register_chunk1(v2_chunk_kernel_t (*tab)[2]) { tab[0][1] = tsk::k_chunk_v2<SW_X, SW_XDAG, -1>; }
