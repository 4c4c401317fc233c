// ts_chunk_cfgH10.cu -- L2-blocked triple-pass kernels (ts_tile_chunk.cuh) for a high group of configuration H10
// (butterfly masks: layout 1 = 31, layout 2 = 31).
#include "ts_tile_chunk.cuh"

TS_CHUNK_REGISTER_CFG(H10, 31, 31)
