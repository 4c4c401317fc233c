// ts_small.cu -- the whole ts_evolve call as ONE launch of ONE CTA for N <= 12 (the paper sees the
// same regime at P:189-191: "for small systems ... the GPU is not saturated", i.e. latency-bound).
//
// The state (<= 4096 amplitudes, 64 KiB) and the three energy vectors E_x, E_y, E_z (<= 96 KiB; the paper's own
// "phases computed in advance" variant, which costs nothing at this size) live in shared memory for the whole
// run; the Suzuki sequence (ts_api.cu, same merged schedule: D_z(s/2) . X^dag . D_y(s/2) . Y^dag . D_x(s) . Y . D_y(s/2) .
// X . D_z(s/2), trailing and leading D_z merged, exact 2^-N after each backward sweep) is generated on the device, so a
// run of any length is a single launch: no per-sweep launches, no host round trips.  One butterfly level per
// __syncthreads; the phase exp(-i t E) is evaluated with full-accuracy sincos.
#include <math.h>

#include "ts_internal.h"

namespace {

constexpr int ST = 1024;     // threads

struct SmallParams {
    double2* psi;
    const double* h;         // [3][TS_MAX_N]
    const double* Jeff;      // [3][TS_MAX_N][TS_MAX_N]
    int N, order;
    long long n_steps;
    double tau;
    double e0[3];            // energy offsets of the context (zero unless it is a shard)
};

__device__ __forceinline__ void small_pair(int kind, double2& c0, double2& c1)
{
    const double r0 = c0.x, i0 = c0.y, r1 = c1.x, i1 = c1.y;
    switch (kind) {
    case SW_YDAG: c0 = make_double2(r0 - r1, i0 - i1); c1 = make_double2(r0 + r1, i0 + i1); break;
    case SW_Y:    c0 = make_double2(r0 + r1, i0 + i1); c1 = make_double2(r1 - r0, i1 - i0); break;
    case SW_XDAG: c0 = make_double2(r0 + i1, i0 - r1); c1 = make_double2(r1 + i0, i1 - r0); break;
    default:      c0 = make_double2(r0 - i1, i0 + r1); c1 = make_double2(r1 - i0, i1 + r0); break;   // SW_X
    }
}

__global__ void __launch_bounds__(ST, 1) k_small_evolve(const SmallParams p)
{
    extern __shared__ __align__(16) unsigned char smraw[];
    const int N = p.N;
    const int dim = 1 << N;
    double2* s = reinterpret_cast<double2*>(smraw);                                  // [dim]
    double* E = reinterpret_cast<double*>(smraw + sizeof(double2) * (size_t)dim);    // [3][dim]
    const int t = threadIdx.x;

    // energy vectors: E_a(k) = sum_j sigma_j (h_j + sum_{m < j} Jeff_jm sigma_m)   (eq. 1; A1, A2)
    for (int k = t; k < dim; k += ST) {
        for (int a = 0; a < 3; ++a) {
            const double* h = p.h + a * TS_MAX_N;
            const double* J = p.Jeff + (size_t)a * TS_MAX_N * TS_MAX_N;
            double e = 0.0;
            for (int j = 0; j < N; ++j) {
                const double sj = (double)((k >> j) & 1) - 0.5;
                double f = h[j];
                for (int m = 0; m < j; ++m) f += J[j * TS_MAX_N + m] * ((double)((k >> m) & 1) - 0.5);
                e += sj * f;
            }
            E[a * dim + k] = e + p.e0[a];
        }
        s[k] = p.psi[k];
    }
    __syncthreads();

    const double a4 = 1.0 / (4.0 - cbrt(4.0));
    const long long n_sub = p.n_steps * (p.order == 4 ? 5 : 1);
    const long long M = 4 * n_sub;
    auto sub = [&](long long u) -> double {
        if (u < 0 || u >= n_sub) return 0.0;
        if (p.order == 2) return p.tau;
        return ((u % 5) == 2) ? (1.0 - 4.0 * a4) * p.tau : a4 * p.tau;
    };
    const double inv = ldexp(1.0, -N);

    auto diag = [&](int alpha, double tt, double scale) {
        const double* Ea = E + alpha * dim;
        for (int k = t; k < dim; k += ST) {
            double sn, cs;
            sincos(-tt * Ea[k], &sn, &cs);
            cs *= scale; sn *= scale;
            const double2 c = s[k];
            s[k] = make_double2(c.x * cs - c.y * sn, c.x * sn + c.y * cs);
        }
        __syncthreads();
    };

    diag(TS_Z, 0.5 * sub(0), 1.0);
    for (long long i = 1; i <= M; ++i) {
        const int ph = (int)((i - 1) & 3);
        const int kind = ph == 0 ? SW_XDAG : ph == 1 ? SW_YDAG : ph == 2 ? SW_Y : SW_X;
        for (int j = 0; j < N; ++j) {
            const int low = (1 << j) - 1;
            for (int q = t; q < (dim >> 1); q += ST) {
                const int k0 = ((q & ~low) << 1) | (q & low);
                const int k1 = k0 | (1 << j);
                double2 c0 = s[k0], c1 = s[k1];
                small_pair(kind, c0, c1);
                s[k0] = c0; s[k1] = c1;
            }
            __syncthreads();
        }
        const long long u = (i - 1) >> 2;
        const double su = sub(u);
        if (ph == 0) diag(TS_Y, 0.5 * su, 1.0);
        else if (ph == 1) diag(TS_X, su, 1.0);
        else if (ph == 2) diag(TS_Y, 0.5 * su, inv);
        else diag(TS_Z, 0.5 * su + 0.5 * sub(u + 1), inv);
    }
    for (int k = t; k < dim; k += ST) p.psi[k] = s[k];
}

} // namespace

cudaError_t ts_small_init(void)
{
    return cudaFuncSetAttribute((const void*)k_small_evolve, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                (int)((sizeof(double2) + 3 * sizeof(double)) << TS_SMALL_MAX_N));
}

cudaError_t ts_small_evolve(ts_ctx* c, double tau, int64_t n_steps, int order)
{
    SmallParams p;
    p.psi = c->psi; p.h = c->d_h; p.Jeff = c->d_Jeff;
    p.N = c->N; p.order = order; p.n_steps = (long long)n_steps; p.tau = tau;
    for (int a = 0; a < 3; ++a) p.e0[a] = c->e0[a];
    const size_t smem = (sizeof(double2) + 3 * sizeof(double)) << c->N;
    ts_prof_begin(c, TS_KC_SMALL);
    k_small_evolve<<<1, ST, smem, c->stream>>>(p);
    ts_prof_end(c);
    return cudaGetLastError();
}
