// ts_v2_chunk1_h9.cu -- L2-blocked triple launch (ts_tile_v2.cuh), kinds (X, X^dag), high group of 9 bits.
#include "ts_tile_v2.cuh"

void ts_v2_register_chunk1_h9(v2_chunk_kernel_t (*tab)[2]) { tab[1][1] = tsk::k_chunk_v2<SW_X, SW_XDAG, 9>; }
