// ts_tile_cfgH8.cu -- tile-pass kernels for configuration H8 (butterfly masks fixed at compile time: layout 1 = 31,
// layout 2 = 28, lane bits = 0).  See ts_tile_kernel.cuh.
#include "ts_tile_pipe.cuh"

#ifndef TS_MINB_H8
#define TS_MINB_H8 2
#endif

TS_TILE_REGISTER_CFG(H8, 31, 28, 0, TS_MINB_H8)
TS_PIPE_REGISTER_CFG(H8, 31, 28, 0)
