// ts_tile_cfgH10.cu -- tile-pass kernels for configuration H10 (butterfly masks fixed at compile time: layout 1 = 31,
// layout 2 = 31, lane bits = 0).  See ts_tile_kernel.cuh.
#include "ts_tile_pipe.cuh"

#ifndef TS_MINB_H10
#define TS_MINB_H10 2
#endif

TS_TILE_REGISTER_CFG(H10, 31, 31, 0, TS_MINB_H10)
TS_PIPE_REGISTER_CFG(H10, 31, 31, 0)
