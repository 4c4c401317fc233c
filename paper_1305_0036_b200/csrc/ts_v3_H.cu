// ts_v3_H.cu -- 16-amplitudes-per-thread tile-pass kernels (ts_tile_v3.cuh) of a high group, run-time butterfly masks:
// the two fused transitions of the top group and the four single sweeps of a middle group.
#include "ts_tile_v3.cuh"

void ts_v3_register_Hf(v2_kernel_t (*tab)[5][5])
{
    (*tab)[SW_XDAG][SW_YDAG] = tsk::k_tile_v3<1, SW_XDAG, SW_YDAG>;
    (*tab)[SW_Y][SW_X]       = tsk::k_tile_v3<1, SW_Y, SW_X>;
}

void ts_v3_register_Hs(v2_kernel_t (*tab)[5][5])
{
    (*tab)[SW_XDAG][SW_NONE] = tsk::k_tile_v3<1, SW_XDAG, SW_NONE>;
    (*tab)[SW_YDAG][SW_NONE] = tsk::k_tile_v3<1, SW_YDAG, SW_NONE>;
    (*tab)[SW_Y][SW_NONE]    = tsk::k_tile_v3<1, SW_Y, SW_NONE>;
    (*tab)[SW_X][SW_NONE]    = tsk::k_tile_v3<1, SW_X, SW_NONE>;
}
