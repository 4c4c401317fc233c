// ts_chunk_cfgH8.cu -- L2-blocked triple-pass kernels (ts_tile_chunk.cuh) for a high group of configuration H8
// (butterfly masks: layout 1 = 31, layout 2 = 28).
#include "ts_tile_chunk.cuh"

TS_CHUNK_REGISTER_CFG(H8, 31, 28)
