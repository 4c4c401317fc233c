// ts_v2_chunk0.cu -- L2-blocked triple launch (ts_tile_v2.cuh), kinds (Y^dag, Y), any high group.
#include "ts_tile_v2.cuh"

void ts_v2_register_chunk0(v2_chunk_kernel_t (*tab)[2]) { tab[0][0] = tsk::k_chunk_v2<SW_YDAG, SW_Y, -1>; }
