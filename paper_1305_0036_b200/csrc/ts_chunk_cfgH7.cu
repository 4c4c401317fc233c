// ts_chunk_cfgH7.cu -- L2-blocked triple-pass kernels (ts_tile_chunk.cuh) for a high group of configuration H7
// (butterfly masks: layout 1 = 31, layout 2 = 24).
#include "ts_tile_chunk.cuh"

TS_CHUNK_REGISTER_CFG(H7, 31, 24)
