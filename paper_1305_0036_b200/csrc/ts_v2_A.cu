// ts_v2_A.cu -- v2 tile-pass kernels (ts_tile_v2.cuh) of group A: the two fused transitions that meet at group A in the
// sweep order, the first pass of a run (leading diagonal, then X^dag) and the last (X, then the trailing diagonal).
#include "ts_tile_v2.cuh"

void ts_v2_register_A(v2_kernel_t (*tab)[5][5])
{
    (*tab)[SW_YDAG][SW_Y]    = tsk::k_tile_v2<0, SW_YDAG, SW_Y>;
    (*tab)[SW_X][SW_XDAG]    = tsk::k_tile_v2<0, SW_X, SW_XDAG>;
    (*tab)[SW_NONE][SW_XDAG] = tsk::k_tile_v2<0, SW_NONE, SW_XDAG>;
    (*tab)[SW_X][SW_NONE]    = tsk::k_tile_v2<0, SW_X, SW_NONE>;
}
