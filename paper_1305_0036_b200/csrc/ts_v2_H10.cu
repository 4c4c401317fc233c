// ts_v2_H10.cu -- v2 tile-pass kernels (ts_tile_v2.cuh) of a high group with TEN group bits (runs of 64 bytes): what lets
// N = 31 and N = 32 get by with three bit groups (12 + 9 + 10, 12 + 10 + 10) instead of four.  Two full five-bit stages in
// the layouts H1x / H2x; the tile travels as four TMA boxes of 256 rows of 64 bytes.
#include "ts_tile_v2.cuh"

void ts_v2_register_H10(v2_kernel_t (*tab)[5][5])
{
    (*tab)[SW_XDAG][SW_YDAG] = tsk::k_tile_v2<3, SW_XDAG, SW_YDAG>;
    (*tab)[SW_Y][SW_X]       = tsk::k_tile_v2<3, SW_Y, SW_X>;
    (*tab)[SW_XDAG][SW_NONE] = tsk::k_tile_v2<3, SW_XDAG, SW_NONE>;
    (*tab)[SW_YDAG][SW_NONE] = tsk::k_tile_v2<3, SW_YDAG, SW_NONE>;
    (*tab)[SW_Y][SW_NONE]    = tsk::k_tile_v2<3, SW_Y, SW_NONE>;
    (*tab)[SW_X][SW_NONE]    = tsk::k_tile_v2<3, SW_X, SW_NONE>;
}
