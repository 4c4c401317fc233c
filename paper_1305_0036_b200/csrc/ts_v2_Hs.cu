// ts_v2_Hs.cu -- v2 tile-pass kernels (ts_tile_v2.cuh) of a high group, one sweep's butterflies (middle groups).
#include "ts_tile_v2.cuh"

void ts_v2_register_Hs(v2_kernel_t (*tab)[5][5])
{
    (*tab)[SW_XDAG][SW_NONE] = tsk::k_tile_v2<1, SW_XDAG, SW_NONE>;
    (*tab)[SW_YDAG][SW_NONE] = tsk::k_tile_v2<1, SW_YDAG, SW_NONE>;
    (*tab)[SW_Y][SW_NONE]    = tsk::k_tile_v2<1, SW_Y, SW_NONE>;
    (*tab)[SW_X][SW_NONE]    = tsk::k_tile_v2<1, SW_X, SW_NONE>;
}
