// ts_v2_H9.cu -- v2 tile-pass kernels (ts_tile_v2.cuh) of a high group with 9 group bits (runs of 128 bytes: the
// geometry of the N = 30 metric workload), butterfly masks folded at compile time: the two fused transitions of the top
// group and the four single sweeps of a middle group.
#include "ts_tile_v2.cuh"

void ts_v2_register_H9f(v2_kernel_t (*tab)[5][5])
{
    (*tab)[SW_XDAG][SW_YDAG] = tsk::k_tile_v2<2, SW_XDAG, SW_YDAG>;
    (*tab)[SW_Y][SW_X]       = tsk::k_tile_v2<2, SW_Y, SW_X>;
}

void ts_v2_register_H9s(v2_kernel_t (*tab)[5][5])
{
    (*tab)[SW_XDAG][SW_NONE] = tsk::k_tile_v2<2, SW_XDAG, SW_NONE>;
    (*tab)[SW_YDAG][SW_NONE] = tsk::k_tile_v2<2, SW_YDAG, SW_NONE>;
    (*tab)[SW_Y][SW_NONE]    = tsk::k_tile_v2<2, SW_Y, SW_NONE>;
    (*tab)[SW_X][SW_NONE]    = tsk::k_tile_v2<2, SW_X, SW_NONE>;
}
