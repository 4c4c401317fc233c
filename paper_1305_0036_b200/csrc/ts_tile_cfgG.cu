// ts_tile_cfgG.cu -- instantiations of k_tile_pass (ts_tile_kernel.cuh; one CTA per tile, butterfly masks are run-time
// parameters): the fallback for tile geometries the v2 kernels do not take (runs shorter than 128 B, a plan with a
// single group) and the A/B baseline of DESIGN.md 7.1.
#include "ts_tile_kernel.cuh"

void ts_tile_register_generic(tile_kernel_t (*tab)[5][5])
{
#define G(K1, K2) (*tab)[K1][K2] = tsk::k_tile_pass<K1, K2, -1, -1, 0, 2>
    G(SW_XDAG, SW_YDAG); G(SW_YDAG, SW_Y); G(SW_Y, SW_X); G(SW_X, SW_XDAG);
    G(SW_YDAG, SW_NONE); G(SW_Y, SW_NONE); G(SW_XDAG, SW_NONE); G(SW_X, SW_NONE);
    G(SW_NONE, SW_YDAG); G(SW_NONE, SW_Y); G(SW_NONE, SW_XDAG); G(SW_NONE, SW_X);
    G(SW_NONE, SW_NONE);
#undef G
}

void ts_tile_register_p2p(tile_kernel_t (*tab)[5][5])
{
#define P(K1, K2) (*tab)[K1][K2] = tsk::k_tile_pass_p2p<K1, K2>
    P(SW_XDAG, SW_YDAG); P(SW_YDAG, SW_Y); P(SW_Y, SW_X); P(SW_X, SW_XDAG);        // sweep i's arrivals . D_i . sweep i+1
    P(SW_YDAG, SW_NONE); P(SW_Y, SW_NONE); P(SW_XDAG, SW_NONE); P(SW_X, SW_NONE);  // the last sweep of a call
#undef P
}
