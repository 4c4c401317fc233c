// ts_tile_cfgA.cu -- tile-pass kernels for configuration A (butterfly masks fixed at compile time: layout 1 = 31,
// layout 2 = 31, lane bits = 2).  See ts_tile_kernel.cuh.
#include "ts_tile_pipe.cuh"

#ifndef TS_MINB_A
#define TS_MINB_A 2
#endif

TS_TILE_REGISTER_CFG(A, 31, 31, 2, TS_MINB_A)
TS_PIPE_REGISTER_CFG(A, 31, 31, 2)
