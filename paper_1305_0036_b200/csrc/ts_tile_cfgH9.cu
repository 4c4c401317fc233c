// ts_tile_cfgH9.cu -- tile-pass kernels for configuration H9 (butterfly masks fixed at compile time: layout 1 = 31,
// layout 2 = 30, lane bits = 0).  See ts_tile_kernel.cuh.
#include "ts_tile_pipe.cuh"

#ifndef TS_MINB_H9
#define TS_MINB_H9 2
#endif

TS_TILE_REGISTER_CFG(H9, 31, 30, 0, TS_MINB_H9)
TS_PIPE_REGISTER_CFG(H9, 31, 30, 0)
