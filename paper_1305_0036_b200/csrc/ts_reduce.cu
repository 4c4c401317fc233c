// ts_reduce.cu -- device-side observable reductions.  The paper only names the observables
// ("local and non-local physical magnitudes", eq. 11 P:207 for the overlap); formulas are reading A15:
//   <S^z_j> = 1/2 sum_k (2 bit_j(k) - 1) |c_k|^2
//   <S^x_j> = sum_{k: bit_j = 0} Re( conj(c_{k + 2^j}) c_k ),   <S^y_j> = same with Im
// Deterministic two-stage FP64 reduction: fixed grid, per-block partials, then one block sums them in index order.
#include "ts_internal.h"

namespace {

constexpr int RB = 256;          // threads per reduction block
constexpr int MAXV = TS_MAX_N + 1;

__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// Sum `v` over the block; result valid in thread 0.  `sh` has RB/32 doubles.
__device__ __forceinline__ double block_sum(double v, double* sh)
{
    v = warp_sum(v);
    __syncthreads();
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = v;
    __syncthreads();
    double r = 0.0;
    if (threadIdx.x < 32) {
        r = (threadIdx.x < RB / 32) ? sh[threadIdx.x] : 0.0;
        r = warp_sum(r);
    }
    return r;
}

// partial[blockIdx][0] = sum |c|^2,  partial[blockIdx][1 + j] = sum_{k: bit j = 1} |c_k|^2
__global__ void __launch_bounds__(RB) k_prob_bits(const double2* __restrict__ psi, int N, uint64_t dim,
                                                  double* __restrict__ partial)
{
    __shared__ double sh[RB / 32];
    double acc[TS_MAX_N];
#pragma unroll
    for (int j = 0; j < TS_MAX_N; ++j) acc[j] = 0.0;
    double tot = 0.0;
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    for (uint64_t k = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; k < dim; k += stride) {
        const double2 c = psi[k];
        const double p = c.x * c.x + c.y * c.y;
        tot += p;
#pragma unroll
        for (int j = 0; j < TS_MAX_N; ++j)
            if (j < N && ((k >> j) & 1)) acc[j] += p;
    }
    double r = block_sum(tot, sh);
    if (threadIdx.x == 0) partial[(size_t)blockIdx.x * MAXV] = r;
#pragma unroll
    for (int j = 0; j < TS_MAX_N; ++j) {
        if (j < N) {
            r = block_sum(acc[j], sh);
            if (threadIdx.x == 0) partial[(size_t)blockIdx.x * MAXV + 1 + j] = r;
        }
    }
}

// partial[b][0] = sum Re(conj(c1) c0), partial[b][1] = sum Im(conj(c1) c0) over pairs of bit j
__global__ void __launch_bounds__(RB) k_pair_xy(const double2* __restrict__ psi, int j, uint64_t npairs,
                                                double* __restrict__ partial)
{
    __shared__ double sh[RB / 32];
    double sx = 0.0, sy = 0.0;
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    const uint64_t lowmask = ((uint64_t)1 << j) - 1;
    for (uint64_t p = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; p < npairs; p += stride) {
        const uint64_t k0 = ((p & ~lowmask) << 1) | (p & lowmask);
        const double2 c0 = psi[k0], c1 = psi[k0 | ((uint64_t)1 << j)];
        sx += c1.x * c0.x + c1.y * c0.y;     // Re( (r1 - i i1)(r0 + i i0) )
        sy += c1.x * c0.y - c1.y * c0.x;     // Im
    }
    double r = block_sum(sx, sh);
    if (threadIdx.x == 0) partial[(size_t)blockIdx.x * MAXV] = r;
    r = block_sum(sy, sh);
    if (threadIdx.x == 0) partial[(size_t)blockIdx.x * MAXV + 1] = r;
}

// partial[b][0], [1] = Re, Im of sum conj(phi_k) psi_k
__global__ void __launch_bounds__(RB) k_overlap(const double2* __restrict__ phi, const double2* __restrict__ psi,
                                                uint64_t dim, double* __restrict__ partial)
{
    __shared__ double sh[RB / 32];
    double sr = 0.0, si = 0.0;
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    for (uint64_t k = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; k < dim; k += stride) {
        const double2 a = phi[k], b = psi[k];
        sr += a.x * b.x + a.y * b.y;
        si += a.x * b.y - a.y * b.x;
    }
    double r = block_sum(sr, sh);
    if (threadIdx.x == 0) partial[(size_t)blockIdx.x * MAXV] = r;
    r = block_sum(si, sh);
    if (threadIdx.x == 0) partial[(size_t)blockIdx.x * MAXV + 1] = r;
}

// out[v] = sum_b partial[b][v], b ascending (fixed order -> deterministic)
__global__ void k_final_sum(const double* __restrict__ partial, int nblocks, int nvals, double* __restrict__ out)
{
    const int v = threadIdx.x;
    if (v >= nvals) return;
    double s = 0.0;
    for (int b = 0; b < nblocks; ++b) s += partial[(size_t)b * MAXV + v];
    out[v] = s;
}

__global__ void k_fill_basis(double2* __restrict__ psi, uint64_t dim, uint64_t kset)
{
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    for (uint64_t k = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; k < dim; k += stride)
        psi[k] = make_double2(k == kset ? 1.0 : 0.0, 0.0);
}

int red_grid(uint64_t n)
{
    uint64_t g = (n + RB - 1) / RB;
    if (g > 148ull * 8) g = 148ull * 8;
    if (g < 1) g = 1;
    return (int)g;
}

cudaError_t ensure_scratch(ts_ctx* c, size_t doubles)
{
    if (c->red_cap >= doubles) return cudaSuccess;
    if (c->d_red) cudaFree(c->d_red);
    c->d_red = nullptr; c->red_cap = 0;
    cudaError_t e = cudaMalloc(&c->d_red, doubles * sizeof(double));
    if (e == cudaSuccess) c->red_cap = doubles;
    return e;
}

// run final sum of nvals values and copy them to the host
cudaError_t finish(ts_ctx* c, int grid, int nvals, double* host_out)
{
    double* partial = c->d_red;
    double* out = c->d_red + (size_t)grid * MAXV;
    k_final_sum<<<1, 64, 0, c->stream>>>(partial, grid, nvals, out);
    ts_prof_end(c);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    e = cudaMemcpyAsync(host_out, out, nvals * sizeof(double), cudaMemcpyDeviceToHost, c->stream);
    if (e != cudaSuccess) return e;
    return cudaStreamSynchronize(c->stream);
}

// final sum of nvals values into a DEVICE buffer, no copy, no synchronisation (observable traces)
cudaError_t finish_dev(ts_ctx* c, int grid, int nvals, double* dev_out)
{
    k_final_sum<<<1, 64, 0, c->stream>>>(c->d_red, grid, nvals, dev_out);
    ts_prof_end(c);
    return cudaGetLastError();
}

} // namespace

// One row of an observable trace, written to device memory on the stream (ts_evolve_observe):
// alpha = z: row[0] = <psi|psi>, row[1 + j] = sum_{k: bit j = 1} |c_k|^2 for all j;  alpha = x, y: row[0], row[1] = the
// Re and Im pair sums of site j.  The host turns rows into expectation values after the single final copy.
cudaError_t ts_reduce_trace_row(ts_ctx* c, int alpha, int j, double* dev_row)
{
    if (alpha == TS_Z) {
        const uint64_t dim = (uint64_t)1 << c->N;
        const int grid = red_grid(dim);
        cudaError_t e = ensure_scratch(c, (size_t)(grid + 1) * MAXV);
        if (e != cudaSuccess) return e;
        ts_prof_begin(c, TS_KC_REDUCE);
        k_prob_bits<<<grid, RB, 0, c->stream>>>(c->psi, c->N, dim, c->d_red);
        return finish_dev(c, grid, c->N + 1, dev_row);
    }
    const uint64_t npairs = (uint64_t)1 << (c->N - 1);
    const int grid = red_grid(npairs);
    cudaError_t e = ensure_scratch(c, (size_t)(grid + 1) * MAXV);
    if (e != cudaSuccess) return e;
    ts_prof_begin(c, TS_KC_REDUCE);
    k_pair_xy<<<grid, RB, 0, c->stream>>>(c->psi, j, npairs, c->d_red);
    return finish_dev(c, grid, 2, dev_row);
}

cudaError_t ts_reduce_expect_z_all(ts_ctx* c, double* out_host)
{
    const uint64_t dim = (uint64_t)1 << c->N;
    const int grid = red_grid(dim);
    cudaError_t e = ensure_scratch(c, (size_t)(grid + 1) * MAXV);
    if (e != cudaSuccess) return e;
    ts_prof_begin(c, TS_KC_REDUCE);
    k_prob_bits<<<grid, RB, 0, c->stream>>>(c->psi, c->N, dim, c->d_red);
    double v[MAXV];
    e = finish(c, grid, c->N + 1, v);
    if (e != cudaSuccess) return e;
    for (int j = 0; j < c->N; ++j) out_host[j] = v[1 + j] - 0.5 * v[0];   // 1/2 (P_up - P_down)
    return cudaSuccess;
}

cudaError_t ts_reduce_expect_xy(ts_ctx* c, int alpha, int j, double* out_host)
{
    const uint64_t npairs = (uint64_t)1 << (c->N - 1);
    const int grid = red_grid(npairs);
    cudaError_t e = ensure_scratch(c, (size_t)(grid + 1) * MAXV);
    if (e != cudaSuccess) return e;
    ts_prof_begin(c, TS_KC_REDUCE);
    k_pair_xy<<<grid, RB, 0, c->stream>>>(c->psi, j, npairs, c->d_red);
    double v[2];
    e = finish(c, grid, 2, v);
    if (e != cudaSuccess) return e;
    *out_host = (alpha == TS_X) ? v[0] : v[1];
    return cudaSuccess;
}

cudaError_t ts_reduce_norm2(ts_ctx* c, double* out_host)
{
    const uint64_t dim = (uint64_t)1 << c->N;
    const int grid = red_grid(dim);
    cudaError_t e = ensure_scratch(c, (size_t)(grid + 1) * MAXV);
    if (e != cudaSuccess) return e;
    ts_prof_begin(c, TS_KC_REDUCE);
    k_overlap<<<grid, RB, 0, c->stream>>>(c->psi, c->psi, dim, c->d_red);
    double v[2];
    e = finish(c, grid, 2, v);
    if (e != cudaSuccess) return e;
    *out_host = v[0];
    return cudaSuccess;
}

cudaError_t ts_reduce_overlap(ts_ctx* c, const double2* phi, double* out_host)
{
    const uint64_t dim = (uint64_t)1 << c->N;
    const int grid = red_grid(dim);
    cudaError_t e = ensure_scratch(c, (size_t)(grid + 1) * MAXV);
    if (e != cudaSuccess) return e;
    ts_prof_begin(c, TS_KC_REDUCE);
    k_overlap<<<grid, RB, 0, c->stream>>>(phi, c->psi, dim, c->d_red);
    return finish(c, grid, 2, out_host);
}

cudaError_t ts_fill_basis(ts_ctx* c, uint64_t k)
{
    const uint64_t dim = (uint64_t)1 << c->N;
    ts_prof_begin(c, TS_KC_SETUP);
    k_fill_basis<<<red_grid(dim), RB, 0, c->stream>>>(c->psi, dim, k);
    ts_prof_end(c);
    return cudaGetLastError();
}
