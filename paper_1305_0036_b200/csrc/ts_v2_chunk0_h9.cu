// ts_v2_chunk0_h9.cu -- L2-blocked triple launch (ts_tile_v2.cuh), kinds (Y^dag, Y), high group of 9 bits (the default
// plan at every N >= 22): butterfly masks folded at compile time.
#include "ts_tile_v2.cuh"

void ts_v2_register_chunk0_h9(v2_chunk_kernel_t (*tab)[2]) { tab[1][0] = tsk::k_chunk_v2<SW_YDAG, SW_Y, 9>; }
