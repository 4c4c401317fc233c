// ts_naive.cu -- the paper's basic scheme, kept as the A/B baseline "GPU-basic" (TS_PLAN_NAIVE; SURVEY 8 f NEXT-3):
//   * one launch per spin rotation, one thread per pair  ("a GPU kernel that rotates the j-th spin on a
//     single pair is launched on 2^(N-1) threads")
//   * one launch per diagonal, with either the O(N^2) on-the-fly energy per amplitude or -- TS_OPT_DIAG_SOURCE
//     = 1 -- the paper's pre-computed variant: "three 2^N-element vectors" E_x, E_y, E_z (+150 % memory),
//     built once per context, so that a diagonal is one table read and one sincos per amplitude.
// The production paths are ts_tile.cu (N >= 13) and ts_small.cu (N <= 12).
#include "ts_internal.h"

namespace {

template <int KIND>
__device__ __forceinline__ void pair_update(double2& c0, double2& c1)
{
    const double r0 = c0.x, i0 = c0.y, r1 = c1.x, i1 = c1.y;
    if (KIND == SW_YDAG) {            // (c0 - c1, c0 + c1)
        c0 = make_double2(r0 - r1, i0 - i1);
        c1 = make_double2(r0 + r1, i0 + i1);
    } else if (KIND == SW_Y) {        // (c0 + c1, c1 - c0)
        c0 = make_double2(r0 + r1, i0 + i1);
        c1 = make_double2(r1 - r0, i1 - i0);
    } else if (KIND == SW_XDAG) {     // (c0 - i c1, c1 - i c0);  -i (r + i m) = m - i r
        c0 = make_double2(r0 + i1, i0 - r1);
        c1 = make_double2(r1 + i0, i1 - r0);
    } else {                          // SW_X: (c0 + i c1, c1 + i c0);  i (r + i m) = -m + i r
        c0 = make_double2(r0 - i1, i0 + r1);
        c1 = make_double2(r1 - i0, i1 + r0);
    }
}

// "n_up = n_down + 2^j": pair p -> k0 = p with a 0 inserted at bit j.
template <int KIND>
__global__ void __launch_bounds__(256) k_naive_rotate(double2* __restrict__ psi, int j, uint64_t npairs)
{
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    const uint64_t lowmask = ((uint64_t)1 << j) - 1;
    for (uint64_t p = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; p < npairs; p += stride) {
        const uint64_t k0 = ((p & ~lowmask) << 1) | (p & lowmask);
        const uint64_t k1 = k0 | ((uint64_t)1 << j);
        double2 c0 = psi[k0], c1 = psi[k1];
        pair_update<KIND>(c0, c1);
        psi[k0] = c0;
        psi[k1] = c1;
    }
}

// D_alpha(t): c_k <- c_k * scale * exp(-i t E(k)),  E(k) = sum_j sigma_j (h_j + 1/2 sum_{m != j} Jeff_jm sigma_m)
// (eq. 1 P:33 with A1/A2; eq. 9; on-the-fly evaluation).
__global__ void __launch_bounds__(256) k_naive_diag(double2* __restrict__ psi, int N, uint64_t dim,
                                                    const double* __restrict__ h, const double* __restrict__ Jeff,
                                                    double t, double scale, double e0)
{
    __shared__ double sh[TS_MAX_N];
    __shared__ double sJ[TS_MAX_N * TS_MAX_N];
    for (int i = threadIdx.x; i < N; i += blockDim.x) sh[i] = h[i];
    for (int i = threadIdx.x; i < N * N; i += blockDim.x) sJ[i] = Jeff[(i / N) * TS_MAX_N + (i % N)];
    __syncthreads();
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    for (uint64_t k = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; k < dim; k += stride) {
        double E = 0.0;
        for (int j = 0; j < N; ++j) {
            const double sj = (double)((k >> j) & 1) - 0.5;
            double f = 0.0;
            for (int m = 0; m < j; ++m) f += sJ[j * N + m] * ((double)((k >> m) & 1) - 0.5);
            E += sj * (sh[j] + f);     // each unordered pair once (m < j) with Jeff = J_jm + J_mj
        }
        double sn, cs;
        sincos(-t * (E + e0), &sn, &cs);
        cs *= scale; sn *= scale;
        const double2 c = psi[k];
        psi[k] = make_double2(c.x * cs - c.y * sn, c.x * sn + c.y * cs);
    }
}

// E[k] = E_alpha(k) for all k (the stored vectors of P:119)
__global__ void __launch_bounds__(256) k_build_energy(double* __restrict__ E, int N, uint64_t dim, const double* __restrict__ h,
                                                      const double* __restrict__ Jeff, double e0)
{
    __shared__ double sh[TS_MAX_N];
    __shared__ double sJ[TS_MAX_N * TS_MAX_N];
    for (int i = threadIdx.x; i < N; i += blockDim.x) sh[i] = h[i];
    for (int i = threadIdx.x; i < N * N; i += blockDim.x) sJ[i] = Jeff[(i / N) * TS_MAX_N + (i % N)];
    __syncthreads();
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    for (uint64_t k = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; k < dim; k += stride) {
        double e = 0.0;
        for (int j = 0; j < N; ++j) {
            const double sj = (double)((k >> j) & 1) - 0.5;
            double f = 0.0;
            for (int m = 0; m < j; ++m) f += sJ[j * N + m] * ((double)((k >> m) & 1) - 0.5);
            e += sj * (sh[j] + f);
        }
        E[k] = e + e0;
    }
}

__global__ void __launch_bounds__(256) k_naive_diag_stored(double2* __restrict__ psi, uint64_t dim, const double* __restrict__ E,
                                                           double t, double scale)
{
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    for (uint64_t k = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; k < dim; k += stride) {
        double sn, cs;
        sincos(-t * E[k], &sn, &cs);
        cs *= scale; sn *= scale;
        const double2 c = psi[k];
        psi[k] = make_double2(c.x * cs - c.y * sn, c.x * sn + c.y * cs);
    }
}

inline int grid_for(uint64_t n, int block)
{
    uint64_t g = (n + block - 1) / block;
    const uint64_t cap = 148ull * 64;   // grid-stride beyond this
    if (g > cap) g = cap;
    if (g < 1) g = 1;
    return (int)g;
}

} // namespace

cudaError_t ts_naive_rotate(ts_ctx* c, int j, int kind)
{
    const uint64_t npairs = (uint64_t)1 << (c->N - 1);
    const int grid = grid_for(npairs, 256);
    ts_prof_begin(c, TS_KC_NAIVE_ROT);
    switch (kind) {
    case SW_YDAG: k_naive_rotate<SW_YDAG><<<grid, 256, 0, c->stream>>>(c->psi, j, npairs); break;
    case SW_Y:    k_naive_rotate<SW_Y><<<grid, 256, 0, c->stream>>>(c->psi, j, npairs); break;
    case SW_XDAG: k_naive_rotate<SW_XDAG><<<grid, 256, 0, c->stream>>>(c->psi, j, npairs); break;
    default:      k_naive_rotate<SW_X><<<grid, 256, 0, c->stream>>>(c->psi, j, npairs); break;
    }
    ts_prof_end(c);
    return cudaGetLastError();
}

void ts_naive_free_stored(ts_ctx* c)
{
    for (int a = 0; a < 3; ++a) {
        if (c->d_energy[a]) cudaFree(c->d_energy[a]);
        c->d_energy[a] = nullptr;
    }
}

cudaError_t ts_naive_diag(ts_ctx* c, const DiagOp& d)
{
    if (!d.present) return cudaSuccess;
    const uint64_t dim = (uint64_t)1 << c->N;
    const int grid = grid_for(dim, 256);
    if (c->opt_diag_source == 1) {
        if (!c->d_energy[d.alpha]) {
            cudaError_t e = cudaMalloc(&c->d_energy[d.alpha], sizeof(double) << c->N);
            if (e != cudaSuccess) return e;
            ts_prof_begin(c, TS_KC_SETUP);
            k_build_energy<<<grid, 256, 0, c->stream>>>(c->d_energy[d.alpha], c->N, dim, c->d_h + d.alpha * TS_MAX_N,
                                                        c->d_Jeff + (size_t)d.alpha * TS_MAX_N * TS_MAX_N, c->e0[d.alpha]);
            ts_prof_end(c);
        }
        ts_prof_begin(c, TS_KC_NAIVE_DIAG);
        k_naive_diag_stored<<<grid, 256, 0, c->stream>>>(c->psi, dim, c->d_energy[d.alpha], d.t, ldexp(1.0, d.scale_pow));
        ts_prof_end(c);
        return cudaGetLastError();
    }
    ts_prof_begin(c, TS_KC_NAIVE_DIAG);
    k_naive_diag<<<grid, 256, 0, c->stream>>>(c->psi, c->N, dim, c->d_h + d.alpha * TS_MAX_N,
                                               c->d_Jeff + (size_t)d.alpha * TS_MAX_N * TS_MAX_N, d.t,
                                               ldexp(1.0, d.scale_pow), c->e0[d.alpha]);
    ts_prof_end(c);
    return cudaGetLastError();
}
