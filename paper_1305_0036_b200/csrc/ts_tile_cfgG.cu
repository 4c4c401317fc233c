// ts_tile_cfgG.cu -- generic tile-pass kernels: butterfly masks are run-time parameters.  Used for the tile
// configurations without a specialised build (high groups of 1..6 bits) and for the rare kind combinations
// (a diagonal followed by any sweep, or a bare diagonal, when the plan has a single group).
#include "ts_tile_pipe.cuh"

void ts_tile_register_generic(tile_kernel_t (*tab)[5][5])
{
#define G(K1, K2) (*tab)[K1][K2] = tsk::k_tile_pass<K1, K2, -1, -1, 0, 2>
    G(SW_XDAG, SW_YDAG); G(SW_YDAG, SW_Y); G(SW_Y, SW_X); G(SW_X, SW_XDAG);
    G(SW_YDAG, SW_NONE); G(SW_Y, SW_NONE); G(SW_XDAG, SW_NONE); G(SW_X, SW_NONE);
    G(SW_NONE, SW_YDAG); G(SW_NONE, SW_Y); G(SW_NONE, SW_XDAG); G(SW_NONE, SW_X);
    G(SW_NONE, SW_NONE);
#undef G
}

void ts_pipe_register_generic(pipe_kernel_t (*tab)[5][5])
{
#define G(K1, K2) (*tab)[K1][K2] = tsk::k_tile_pipe<K1, K2, -1, -1, 0>
    G(SW_XDAG, SW_YDAG); G(SW_YDAG, SW_Y); G(SW_Y, SW_X); G(SW_X, SW_XDAG);
    G(SW_YDAG, SW_NONE); G(SW_Y, SW_NONE); G(SW_XDAG, SW_NONE); G(SW_X, SW_NONE);
    G(SW_NONE, SW_YDAG); G(SW_NONE, SW_Y); G(SW_NONE, SW_XDAG); G(SW_NONE, SW_X);
    G(SW_NONE, SW_NONE);
#undef G
}
