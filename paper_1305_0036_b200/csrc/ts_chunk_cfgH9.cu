// ts_chunk_cfgH9.cu -- L2-blocked triple-pass kernels (ts_tile_chunk.cuh) for a high group of configuration H9
// (butterfly masks: layout 1 = 31, layout 2 = 30).
#include "ts_tile_chunk.cuh"

TS_CHUNK_REGISTER_CFG(H9, 31, 30)
