// ts_tile_cfgH7.cu -- tile-pass kernels for configuration H7 (butterfly masks fixed at compile time: layout 1 = 31,
// layout 2 = 24, lane bits = 0).  See ts_tile_kernel.cuh.
#include "ts_tile_pipe.cuh"

#ifndef TS_MINB_H7
#define TS_MINB_H7 2
#endif

TS_TILE_REGISTER_CFG(H7, 31, 24, 0, TS_MINB_H7)
TS_PIPE_REGISTER_CFG(H7, 31, 24, 0)
