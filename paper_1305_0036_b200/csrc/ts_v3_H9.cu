// ts_v3_H9.cu -- 16-amplitudes-per-thread tile-pass kernels (ts_tile_v3.cuh) of a high group with 9 group bits (runs of
// 128 bytes: the geometry of the N = 30 metric workload), butterfly masks folded at compile time.
#include "ts_tile_v3.cuh"

void ts_v3_register_H9(v2_kernel_t (*tab)[5][5])
{
    (*tab)[SW_XDAG][SW_YDAG] = tsk::k_tile_v3<2, SW_XDAG, SW_YDAG>;
    (*tab)[SW_Y][SW_X]       = tsk::k_tile_v3<2, SW_Y, SW_X>;
    (*tab)[SW_XDAG][SW_NONE] = tsk::k_tile_v3<2, SW_XDAG, SW_NONE>;
    (*tab)[SW_YDAG][SW_NONE] = tsk::k_tile_v3<2, SW_YDAG, SW_NONE>;
    (*tab)[SW_Y][SW_NONE]    = tsk::k_tile_v3<2, SW_Y, SW_NONE>;
    (*tab)[SW_X][SW_NONE]    = tsk::k_tile_v3<2, SW_X, SW_NONE>;
}
