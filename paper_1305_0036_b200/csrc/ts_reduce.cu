// ts_reduce.cu -- device-side observable reductions.  The paper only names the observables
// ("local and non-local physical magnitudes", eq. 11 P:207 for the overlap); formulas are reading A15:
//   <S^z_j> = 1/2 sum_k (2 bit_j(k) - 1) |c_k|^2
//   <S^x_j> = sum_{k: bit_j = 0} Re( conj(c_{k + 2^j}) c_k ),   <S^y_j> = same with Im
// Deterministic two-stage FP64 reduction: fixed grid, per-block partials, then one block sums them in index order.
#include <math.h>

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

// partial[blockIdx][0] = sum |c|^2,  partial[blockIdx][1 + j] = sum_{k: bit j = 1} |c_k|^2     (any N; used for N < 12)
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

// The same sums for N >= 12 at ~2 FP64 additions per amplitude instead of N: a warp walks chunks of 2^12 consecutive
// amplitudes, amplitude (chunk, i, lane) = chunk * 4096 + i * 32 + lane, fully coalesced.  Index bits 0..4 are the lane (a
// thread's own total, sorted into the bit sums once at the end), bits 5..7 and 8..11 are the compile-time position inside
// the chunk (pair-sum tree over groups of 8, then static adds of the group totals), bits >= 12 are the chunk index (the
// chunk total, added once per chunk).
__global__ void __launch_bounds__(RB) k_prob_bits_chunked(const double2* __restrict__ psi, int N, uint64_t nchunks,
                                                          double* __restrict__ partial)
{
    __shared__ double sh[RB / 32];
    double acc[TS_MAX_N];
#pragma unroll
    for (int j = 0; j < TS_MAX_N; ++j) acc[j] = 0.0;
    double tot = 0.0;
    const int lane = threadIdx.x & 31;
    const uint64_t warp = ((uint64_t)blockIdx.x * RB + threadIdx.x) >> 5;
    const uint64_t nwarps = ((uint64_t)gridDim.x * RB) >> 5;
    for (uint64_t ch = warp; ch < nchunks; ch += nwarps) {
        const double2* base = psi + (ch << 12) + lane;
        double ctot = 0.0;
#pragma unroll
        for (int u = 0; u < 16; ++u) {
            double p[8];
#pragma unroll
            for (int v = 0; v < 8; ++v) {
                const double2 c = __ldcs(base + ((u * 8 + v) << 5));
                p[v] = fma(c.x, c.x, c.y * c.y);
            }
            const double a01 = p[0] + p[1], a23 = p[2] + p[3], a45 = p[4] + p[5], a67 = p[6] + p[7];
            const double hi = a45 + a67;
            const double t = (a01 + a23) + hi;
            acc[5] += (p[1] + p[3]) + (p[5] + p[7]);
            acc[6] += a23 + a67;
            acc[7] += hi;
#pragma unroll
            for (int b = 0; b < 4; ++b)
                if (u & (1 << b)) acc[8 + b] += t;
            ctot += t;
        }
        tot += ctot;
#pragma unroll
        for (int j = 12; j < TS_MAX_N; ++j)
            if (j < N && ((ch >> (j - 12)) & 1)) acc[j] += ctot;
    }
#pragma unroll
    for (int j = 0; j < 5; ++j) acc[j] = ((lane >> j) & 1) ? tot : 0.0;
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

// All sites of one bit group in ONE pass (the tile geometry of the time step: a closed tile holds both members of
// every pair of the group's spins).  A CTA stages tiles of 2^12 amplitudes in shared memory (f < s <-> spin f,
// f >= s <-> spin g0 + f - s) and accumulates, for each of the nb spins on tile bits f0 .. f0 + nb - 1,
//   sum over pairs (c0: bit = 0, c1: bit = 1) of conj(c1) c0   ->   Re = <S^x>, Im = <S^y>      (reading A15)
// partial[blockIdx][2 i], [2 i + 1] = Re, Im for tile bit f0 + i.
constexpr int XG_T = 256;
// Register-blocked: the tile is staged once in shared memory (slot(f) = f ^ (f >> 4 & 15) ^ (f >> 8 & 15): conflict-free
// 128-bit accesses in all three layouts below) and read three times, each time with four tile bits on a thread's 16
// registers, so that the pair products of those four bits need no further shared-memory traffic (3 x 64 KiB of reads per
// tile instead of 12 x 2 x 32 KiB).
__device__ __forceinline__ int xg_slot(int f) { return f ^ ((f >> 4) & 15) ^ ((f >> 8) & 15); }
__global__ void __launch_bounds__(XG_T) k_pair_xy_group(const double2* __restrict__ psi, uint64_t ntiles, int s, int g0, int f0, int nb,
                                                       double* __restrict__ partial)
{
    extern __shared__ double2 tile[];      // 4096 amplitudes
    __shared__ double sh[RB / 32];
    double ax[TS_TILE_LOG2], ay[TS_TILE_LOG2];
#pragma unroll
    for (int i = 0; i < TS_TILE_LOG2; ++i) { ax[i] = 0.0; ay[i] = 0.0; }
    const int t = threadIdx.x;
    const int nmid = g0 - s;
    const uint64_t runmask = ((uint64_t)1 << s) - 1;
    for (uint64_t tau = blockIdx.x; tau < ntiles; tau += gridDim.x) {
        const uint64_t base = ((tau & (((uint64_t)1 << nmid) - 1)) << s) | ((tau >> nmid) << (g0 + TS_TILE_LOG2 - s));
        __syncthreads();                   // the previous tile has been read by everyone
#pragma unroll 4
        for (int f = t; f < (1 << TS_TILE_LOG2); f += XG_T)
            tile[xg_slot(f)] = __ldcs(psi + base + (((uint64_t)f & runmask) | (((uint64_t)f >> s) << g0)));
        __syncthreads();
#pragma unroll
        for (int L = 0; L < 3; ++L) {
            // layout L: register index r <-> tile bits 4L .. 4L + 3; thread index <-> the other eight bits, in order
            if (f0 + nb <= 4 * L || f0 >= 4 * L + 4) continue;          // none of these four bits belongs to the group
            const int lo = t & ((1 << (4 * L)) - 1), hi = t >> (4 * L);
            const int fbase = lo | (hi << (4 * L + 4));
            double cr[16], ci[16];
#pragma unroll
            for (int r = 0; r < 16; ++r) {
                const double2 v = tile[xg_slot(fbase | (r << (4 * L)))];
                cr[r] = v.x; ci[r] = v.y;
            }
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                const int b = 4 * L + i;
                if (b >= f0 && b < f0 + nb) {
                    double sx = 0.0, sy = 0.0;
#pragma unroll
                    for (int r = 0; r < 16; ++r) {
                        if (!(r & (1 << i))) {
                            const int r1 = r | (1 << i);
                            sx += cr[r1] * cr[r] + ci[r1] * ci[r];      // Re( conj(c1) c0 )
                            sy += cr[r1] * ci[r] - ci[r1] * cr[r];      // Im
                        }
                    }
                    ax[b] += sx; ay[b] += sy;      // indexed by TILE bit (static); sorted into the group's order below
                }
            }
        }
    }
#pragma unroll
    for (int b = 0; b < TS_TILE_LOG2; ++b) {
        if (b >= f0 && b < f0 + nb) {
            double r = block_sum(ax[b], sh);
            if (t == 0) partial[(size_t)blockIdx.x * MAXV + 2 * (b - f0)] = r;
            r = block_sum(ay[b], sh);
            if (t == 0) partial[(size_t)blockIdx.x * MAXV + 2 * (b - f0) + 1] = r;
        }
    }
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

// partial[b][0] = sum over i with bit j = 0 of w(i) Re( conj(c_{i xor m}) c_i ),  m = 2^j + 2^k:
//   alpha = x: w = 1/2 (the pair i, i xor m contributes twice 1/4);  alpha = y: w = -2 sigma_j sigma_k;
// alpha = z: partial[b][0] = sum_i sigma_j sigma_k |c_i|^2 over ALL i (npairs = dim).      <S^a_j S^a_k>, P:203 / A15
__global__ void __launch_bounds__(RB) k_corr(const double2* __restrict__ psi, int alpha, int j, int k, uint64_t n,
                                             double* __restrict__ partial)
{
    __shared__ double sh[RB / 32];
    double acc = 0.0;
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    const uint64_t bj = (uint64_t)1 << j, bk = (uint64_t)1 << k;
    if (alpha == TS_Z) {
        for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
            const double2 c = psi[i];
            const double p = c.x * c.x + c.y * c.y;
            acc += (((i & bj) != 0) == ((i & bk) != 0)) ? 0.25 * p : -0.25 * p;
        }
    } else {
        const uint64_t lowmask = bj - 1;
        for (uint64_t q = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; q < n; q += stride) {
            const uint64_t i = ((q & ~lowmask) << 1) | (q & lowmask);          // bit j = 0
            const double2 c0 = psi[i], c1 = psi[i ^ (bj | bk)];
            const double re = c1.x * c0.x + c1.y * c0.y;
            if (alpha == TS_X) acc += 0.5 * re;
            else acc += (i & bk) ? 0.5 * re : -0.5 * re;                      // -2 sigma_j sigma_k, sigma_j = -1/2
        }
    }
    const double r = block_sum(acc, sh);
    if (threadIdx.x == 0) partial[(size_t)blockIdx.x * MAXV] = r;
}

// partial[b][0] = sum_k E(k) |c_k|^2 with E(k) = sum_j sigma_j (h_j + sum_{m<j} Jeff_jm sigma_m) evaluated from the
// definition (O(N^2) per amplitude): an observable, not on the time-step path.
__global__ void __launch_bounds__(RB) k_energy_diag(const double2* __restrict__ psi, int N, uint64_t dim,
                                                    const double* __restrict__ h, const double* __restrict__ Jeff,
                                                    double* __restrict__ partial)
{
    __shared__ double sh[RB / 32];
    __shared__ double shh[TS_MAX_N];
    __shared__ double sJ[TS_MAX_N * TS_MAX_N];
    for (int i = threadIdx.x; i < N; i += blockDim.x) shh[i] = h[i];
    for (int i = threadIdx.x; i < N * N; i += blockDim.x) sJ[i] = Jeff[(i / N) * TS_MAX_N + (i % N)];
    __syncthreads();
    double acc = 0.0;
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    for (uint64_t k = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; k < dim; k += stride) {
        double E = 0.0;
        for (int j = 0; j < N; ++j) {
            const double sj = (double)((k >> j) & 1) - 0.5;
            double f = shh[j];
            for (int m = 0; m < j; ++m) f += sJ[j * N + m] * ((double)((k >> m) & 1) - 0.5);
            E += sj * f;
        }
        const double2 c = psi[k];
        acc += E * (c.x * c.x + c.y * c.y);
    }
    const double r = block_sum(acc, sh);
    if (threadIdx.x == 0) partial[(size_t)blockIdx.x * MAXV] = r;
}

// Eq. A.1: spin u up, the other N-1 spins in an equal-weight superposition with random phases
//   phi_j = 2 pi (splitmix64(seed + (j + 1) * 0x9E3779B97F4A7C15) >> 11) 2^-53,  j = amplitude index with bit u removed
// (a counter-based stream: phase j needs no state; SplitMix64 of Steele, Lea & Flood).
__device__ __forceinline__ uint64_t splitmix64_mix(uint64_t z)
{
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    return z ^ (z >> 31);
}

__global__ void k_fill_random_phase(double2* __restrict__ psi, uint64_t dim, int u, uint64_t seed, double amp)
{
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    const uint64_t ub = (uint64_t)1 << u;
    for (uint64_t k = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; k < dim; k += stride) {
        double2 v = make_double2(0.0, 0.0);
        if (k & ub) {
            const uint64_t j = ((k >> (u + 1)) << u) | (k & (ub - 1));
            const double x = (double)(splitmix64_mix(seed + (j + 1) * 0x9E3779B97F4A7C15ull) >> 11) * 0x1.0p-53;
            double sn, cs;
            sincos(2.0 * 3.14159265358979323846 * x, &sn, &cs);
            v = make_double2(amp * cs, amp * sn);
        }
        psi[k] = v;
    }
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

// the same into row *row_ctr of a trace (rows of TS_TRACE_STRIDE doubles), then *row_ctr += 1: a launch that can be replayed
// from a CUDA graph and still fill consecutive rows (ts_evolve_observe)
__global__ void k_final_sum_row(const double* __restrict__ partial, int nblocks, int nvals, double* __restrict__ base,
                                unsigned int* __restrict__ row_ctr)
{
    const int v = threadIdx.x;
    const unsigned int row = *row_ctr;
    if (v < nvals) {
        double s = 0.0;
        for (int b = 0; b < nblocks; ++b) s += partial[(size_t)b * MAXV + v];
        base[(size_t)row * TS_TRACE_STRIDE + v] = s;
    }
    __syncthreads();
    if (v == 0) *row_ctr = row + 1;
}

__global__ void k_set_u32(unsigned int* p, unsigned int v) { *p = v; }

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
cudaError_t finish_dev(ts_ctx* c, int grid, int nvals, double* dev_out, unsigned int* row_ctr)
{
    if (row_ctr) k_final_sum_row<<<1, 64, 0, c->stream>>>(c->d_red, grid, nvals, dev_out, row_ctr);
    else k_final_sum<<<1, 64, 0, c->stream>>>(c->d_red, grid, nvals, dev_out);
    ts_prof_end(c);
    return cudaGetLastError();
}

} // namespace

// One row of an observable trace, written to device memory on the stream (ts_evolve_observe):
// alpha = z: row[0] = <psi|psi>, row[1 + j] = sum_{k: bit j = 1} |c_k|^2 for all j;  alpha = x, y: row[0], row[1] = the
// Re and Im pair sums of site j.  The host turns rows into expectation values after the single final copy.
cudaError_t ts_set_u32(ts_ctx* c, unsigned int* p, unsigned int v)
{
    k_set_u32<<<1, 1, 0, c->stream>>>(p, v);
    return cudaGetLastError();
}

// row_ctr = NULL: the row is written at dev_row.  Otherwise dev_row is the trace's first row and the row index is read from
// (and then advanced in) *row_ctr on the device.
cudaError_t ts_reduce_trace_row(ts_ctx* c, int alpha, int j, double* dev_row, unsigned int* row_ctr)
{
    if (alpha == TS_Z) {
        const uint64_t dim = (uint64_t)1 << c->N;
        const int grid = red_grid(dim);
        cudaError_t e = ensure_scratch(c, (size_t)(grid + 1) * MAXV);
        if (e != cudaSuccess) return e;
        ts_prof_begin(c, TS_KC_REDUCE);
        if (c->N >= 12) k_prob_bits_chunked<<<grid, RB, 0, c->stream>>>(c->psi, c->N, dim >> 12, c->d_red);
        else k_prob_bits<<<grid, RB, 0, c->stream>>>(c->psi, c->N, dim, c->d_red);
        return finish_dev(c, grid, c->N + 1, dev_row, row_ctr);
    }
    const uint64_t npairs = (uint64_t)1 << (c->N - 1);
    const int grid = red_grid(npairs);
    cudaError_t e = ensure_scratch(c, (size_t)(grid + 1) * MAXV);
    if (e != cudaSuccess) return e;
    ts_prof_begin(c, TS_KC_REDUCE);
    k_pair_xy<<<grid, RB, 0, c->stream>>>(c->psi, j, npairs, c->d_red);
    return finish_dev(c, grid, 2, dev_row, row_ctr);
}

cudaError_t ts_reduce_expect_z_all(ts_ctx* c, double* out_host)
{
    const uint64_t dim = (uint64_t)1 << c->N;
    const int grid = red_grid(dim);
    cudaError_t e = ensure_scratch(c, (size_t)(grid + 1) * MAXV);
    if (e != cudaSuccess) return e;
    ts_prof_begin(c, TS_KC_REDUCE);
    if (c->N >= 12) k_prob_bits_chunked<<<grid, RB, 0, c->stream>>>(c->psi, c->N, dim >> 12, c->d_red);
    else k_prob_bits<<<grid, RB, 0, c->stream>>>(c->psi, c->N, dim, c->d_red);
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

cudaError_t ts_reduce_corr(ts_ctx* c, int alpha, int j, int k, double* out_host)
{
    if (alpha != TS_Z && j > k) { const int t = j; j = k; k = t; }      // the pair loop removes bit j: any order works, keep j < k
    const uint64_t n = (alpha == TS_Z) ? (uint64_t)1 << c->N : (uint64_t)1 << (c->N - 1);
    const int grid = red_grid(n);
    cudaError_t e = ensure_scratch(c, (size_t)(grid + 1) * MAXV);
    if (e != cudaSuccess) return e;
    ts_prof_begin(c, TS_KC_REDUCE);
    k_corr<<<grid, RB, 0, c->stream>>>(c->psi, alpha, j, k, n, c->d_red);
    return finish(c, grid, 1, out_host);
}

cudaError_t ts_reduce_energy_diag(ts_ctx* c, int alpha, double* out_host)
{
    const uint64_t dim = (uint64_t)1 << c->N;
    const int grid = red_grid(dim);
    cudaError_t e = ensure_scratch(c, (size_t)(grid + 1) * MAXV);
    if (e != cudaSuccess) return e;
    ts_prof_begin(c, TS_KC_REDUCE);
    k_energy_diag<<<grid, RB, 0, c->stream>>>(c->psi, c->N, dim, c->d_h + alpha * TS_MAX_N,
                                               c->d_Jeff + (size_t)alpha * TS_MAX_N * TS_MAX_N, c->d_red);
    return finish(c, grid, 1, out_host);
}

cudaError_t ts_fill_random_phase(ts_ctx* c, int up_spin, uint64_t seed)
{
    const uint64_t dim = (uint64_t)1 << c->N;
    ts_prof_begin(c, TS_KC_SETUP);
    k_fill_random_phase<<<red_grid(dim), RB, 0, c->stream>>>(c->psi, dim, up_spin, seed, 1.0 / sqrt(ldexp(1.0, c->N - 1)));
    ts_prof_end(c);
    return cudaGetLastError();
}

// <S^x_j> and <S^y_j> of ALL sites: one read-only pass per bit group of the plan (N = 30: 3 passes instead of 30).
cudaError_t ts_reduce_expect_xy_all(ts_ctx* c, double* out_x /*[N] or NULL*/, double* out_y /*[N] or NULL*/)
{
    static bool attr_set = false;
    if (!attr_set) {
        cudaError_t e = cudaFuncSetAttribute((const void*)k_pair_xy_group, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             (int)(sizeof(double2) << TS_TILE_LOG2));
        if (e != cudaSuccess) return e;
        attr_set = true;
    }
    const uint64_t ntiles = (uint64_t)1 << (c->N - TS_TILE_LOG2);
    uint64_t g = ntiles < (uint64_t)(2 * c->num_sms) ? ntiles : (uint64_t)(2 * c->num_sms);
    const int grid = (int)g;
    cudaError_t e = ensure_scratch(c, (size_t)(grid + 1) * MAXV);
    if (e != cudaSuccess) return e;
    for (const TileGroup& tg : c->groups) {
        const int f0 = tg.is_low ? 0 : tg.s;
        const int nb = TS_TILE_LOG2 - f0;
        ts_prof_begin(c, TS_KC_REDUCE);
        k_pair_xy_group<<<grid, XG_T, sizeof(double2) << TS_TILE_LOG2, c->stream>>>(c->psi, ntiles, tg.s, tg.g0, f0, nb, c->d_red);
        double v[2 * TS_TILE_LOG2];
        e = finish(c, grid, 2 * nb, v);
        if (e != cudaSuccess) return e;
        for (int i = 0; i < nb; ++i) {
            const int f = f0 + i;
            const int spin = f < tg.s ? f : tg.g0 + (f - tg.s);
            if (out_x) out_x[spin] = v[2 * i];
            if (out_y) out_y[spin] = v[2 * i + 1];
        }
    }
    return cudaSuccess;
}
