// ts_v3_A.cu -- 16-amplitudes-per-thread tile-pass kernels (ts_tile_v3.cuh) of group A.
#include "ts_tile_v3.cuh"

void ts_v3_register_A(v2_kernel_t (*tab)[5][5])
{
    (*tab)[SW_YDAG][SW_Y]    = tsk::k_tile_v3<0, SW_YDAG, SW_Y>;
    (*tab)[SW_X][SW_XDAG]    = tsk::k_tile_v3<0, SW_X, SW_XDAG>;
    (*tab)[SW_NONE][SW_XDAG] = tsk::k_tile_v3<0, SW_NONE, SW_XDAG>;
    (*tab)[SW_X][SW_NONE]    = tsk::k_tile_v3<0, SW_X, SW_NONE>;
}
