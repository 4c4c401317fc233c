// ts_v2_Hf.cu -- v2 tile-pass kernels (ts_tile_v2.cuh) of a high group, fused: the two transitions that meet at the TOP
// group in the sweep order.
#include "ts_tile_v2.cuh"

void ts_v2_register_Hf(v2_kernel_t (*tab)[5][5])
{
    (*tab)[SW_XDAG][SW_YDAG] = tsk::k_tile_v2<1, SW_XDAG, SW_YDAG>;
    (*tab)[SW_Y][SW_X]       = tsk::k_tile_v2<1, SW_Y, SW_X>;
}
