/*
 * ts_oracle.c -- CPU ORACLE for the Trotter-Suzuki spin-1/2 time step of arXiv:1305.0036
 * (Dente, Bederian, Zangara, Pastawski).  TEST INFRASTRUCTURE ONLY.
 *
 * This file is a plain, slow, obviously-correct restatement of what the paper's method computes.  It is
 * used by tests/, by __graft_entry__.smoke() and by bench.py's cpu_baseline / --impl reference legs, and by
 * nothing else.  It shares no code, header, table or constant generator with the CUDA path under
 * paper_1305_0036_b200/csrc/, and neither side includes or imports the other.
 *
 * Citations "P:<n>" are line numbers of /root/reference/PAPER.md; "A<n>" are the readings listed in DESIGN.md
 * (section "Readings of the paper").
 *
 * Conventions:
 *   - spin j (0-based) <-> bit j of the amplitude index k; the paper numbers spins from 1, right to left
 *     (P:133 footnote), so paper spin j+1 <-> bit j.  Pinned by the closed-set example at P:141.
 *   - bit value 1 = up (S^z = +1/2), 0 = down (S^z = -1/2)  ("spin down, i.e. its j-th bit is 0").
 *   - sigma_j(k) = bit_j(k) - 1/2.
 *   - S = Pauli/2: eq. 9 shows phases exp(+-i t J / 4)  (reading A2).
 *   - the evolution is exp(-i t H); reading A3 for the sign printed in eq. 9.
 *   - eq. 1 sums bonds over ALL ordered pairs (j,k); j == k terms are ignored (reading A1), so the
 *     effective coupling of the unordered pair {j,k} is J[j][k] + J[k][j].
 *
 * What is pinned and how (tests/test_oracle_*.py, all run with -m "not gpu"):
 *   energy / diagonal        : diagonal of the dense Kronecker-product H_z; pure-Z Hamiltonian closed form
 *   rotations, bit order     : operator identities P:69-71; Y D Y^dag and X D X^dag vs dense expm of H_x, H_y
 *   signs                    : closed-form Larmor precession about x, y, z (N = 1)
 *   J convention, bond phases: closed-form two-spin exchange oscillation (N = 2)
 *   U1 / U2 / U4 composition : dense matrix products of dense exponentials in the printed order
 *   whole method             : dense exp(-iHt) by diagonalisation, N <= 10: tau^4 error law, config-1 gap
 *   unitarity, reversibility : norm to 1e-13; echo
 *   pairing / tiles          : index examples at P:127-135, P:141, P:149-163 (tests/golden/)
 *   observables              : dense operators <psi|S^a_j|psi>
 * The accuracy figures printed at P:203 and P:217 (Fermi fast-math round-off, private ED data) pin nothing:
 * "parity unpinned" by those numbers, see DESIGN.md.
 *
 * Build: oracle/build.py  (gcc -O2 -fopenmp -shared -fPIC; no -ffast-math: reading A13).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* Sweep kinds.  The 2x2 matrices are eq. 5, which the paper prints in (up, down) order; the array
 * order here is (bit 0 = down, bit 1 = up), so rows and columns are flipped (reading A7).  All four are
 * applied UNNORMALISED (without the 1/sqrt(2)); the exact factor 2^-N is applied after each
 * forward/backward pair (reading A13).
 *   Y^dag : (c0, c1) <- (c0 - c1, c0 + c1)
 *   Y     : (c0, c1) <- (c0 + c1, c1 - c0)
 *   X^dag : (c0, c1) <- (c0 - i c1, c1 - i c0)
 *   X     : (c0, c1) <- (c0 + i c1, c1 + i c0)
 * where c0 is the amplitude with bit j = 0 and c1 the one with bit j = 1.
 */
enum { TSO_SWEEP_YDAG = 0, TSO_SWEEP_Y = 1, TSO_SWEEP_XDAG = 2, TSO_SWEEP_X = 3 };
enum { TSO_X = 0, TSO_Y = 1, TSO_Z = 2 };

int tso_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* E_alpha(k) = sum_j h_j sigma_j(k) + sum_{j != m} J[j][m] sigma_j(k) sigma_m(k)      (eq. 1; A1, A2)
 * h: [N], J: [N][N] row-major, for ONE alpha.  This double loop is the definition; it is O(N^2) per
 * amplitude, which is exactly the cost the paper describes at P:117. */
double tso_energy(int N, const double *h, const double *J, uint64_t k)
{
    double E = 0.0;
    for (int j = 0; j < N; ++j) {
        double sj = (double)((k >> j) & 1u) - 0.5;
        E += h[j] * sj;
    }
    for (int j = 0; j < N; ++j) {
        double sj = (double)((k >> j) & 1u) - 0.5;
        for (int m = 0; m < N; ++m) {
            if (m == j) continue;
            double sm = (double)((k >> m) & 1u) - 0.5;
            E += J[(size_t)j * N + m] * sj * sm;
        }
    }
    return E;
}

/* "the phase corrections can be computed in advance ... and stored in memory": E[k] for all k. */
void tso_energy_table(int N, const double *h, const double *J, double *E)
{
    const int64_t dim = (int64_t)1 << N;
#pragma omp parallel for schedule(static)
    for (int64_t k = 0; k < dim; ++k) E[k] = tso_energy(N, h, J, (uint64_t)k);
}

/* D_alpha(t): c_k <- c_k * exp(-i t E(k))                                   (eq. 9)
 * psi: 2^N x (re, im).  Etab == NULL: evaluate the definition per amplitude; else look it up. */
void tso_apply_diag(double *psi, int N, const double *h, const double *J, const double *Etab, double t)
{
    const int64_t dim = (int64_t)1 << N;
#pragma omp parallel for schedule(static)
    for (int64_t k = 0; k < dim; ++k) {
        double E = Etab ? Etab[k] : tso_energy(N, h, J, (uint64_t)k);
        double a = t * E;
        double c = cos(a), s = sin(a);           /* exp(-i a) = c - i s */
        double re = psi[2 * k], im = psi[2 * k + 1];
        psi[2 * k]     = re * c + im * s;
        psi[2 * k + 1] = im * c - re * s;
    }
}

/* One pair update on bit j: "n_up = n_down + 2^j", 2^(N-1) independent pairs. */
static inline void pair_update(double *psi, int64_t k0, int64_t k1, int kind)
{
    double r0 = psi[2 * k0], i0 = psi[2 * k0 + 1];
    double r1 = psi[2 * k1], i1 = psi[2 * k1 + 1];
    switch (kind) {
    case TSO_SWEEP_YDAG: /* (c0 - c1, c0 + c1) */
        psi[2 * k0] = r0 - r1; psi[2 * k0 + 1] = i0 - i1;
        psi[2 * k1] = r0 + r1; psi[2 * k1 + 1] = i0 + i1;
        break;
    case TSO_SWEEP_Y:    /* (c0 + c1, c1 - c0) */
        psi[2 * k0] = r0 + r1; psi[2 * k0 + 1] = i0 + i1;
        psi[2 * k1] = r1 - r0; psi[2 * k1 + 1] = i1 - i0;
        break;
    case TSO_SWEEP_XDAG: /* (c0 - i c1, c1 - i c0);  -i (r + i m) = m - i r */
        psi[2 * k0] = r0 + i1; psi[2 * k0 + 1] = i0 - r1;
        psi[2 * k1] = r1 + i0; psi[2 * k1 + 1] = i1 - r0;
        break;
    default:             /* TSO_SWEEP_X: (c0 + i c1, c1 + i c0);  i (r + i m) = -m + i r */
        psi[2 * k0] = r0 - i1; psi[2 * k0 + 1] = i0 + r1;
        psi[2 * k1] = r1 - i0; psi[2 * k1 + 1] = i1 + r0;
        break;
    }
}

/* Rotate ONE spin: all 2^(N-1) pairs of bit j. */
void tso_rotate_bit(double *psi, int N, int j, int kind)
{
    const int64_t half = (int64_t)1 << (N - 1);
    const int64_t lowmask = ((int64_t)1 << j) - 1;
#pragma omp parallel for schedule(static)
    for (int64_t p = 0; p < half; ++p) {
        int64_t k0 = ((p & ~lowmask) << 1) | (p & lowmask);   /* insert a 0 at bit j */
        int64_t k1 = k0 | ((int64_t)1 << j);
        pair_update(psi, k0, k1, kind);
    }
}

/* Global rotation X, Y, X^dag or Y^dag = tensor product over all spins, bit 0 first. Unnormalised. */
void tso_apply_sweep(double *psi, int N, int kind)
{
    for (int j = 0; j < N; ++j) tso_rotate_bit(psi, N, j, kind);
}

/* Multiply every amplitude by f (used with the exact power of two 2^-N). */
void tso_scale(double *psi, int N, double f)
{
    const int64_t dim = (int64_t)1 << N;
#pragma omp parallel for schedule(static)
    for (int64_t k = 0; k < 2 * dim; ++k) psi[k] *= f;
}

/* Hamiltonian as the paper states it (eq. 1): h[3][N], J[3][N][N], alpha = x, y, z.  Etab[a] may be NULL. */
typedef struct {
    int N;
    const double *h;      /* [3][N]    */
    const double *J;      /* [3][N][N] */
    const double *Etab[3];
} tso_ham;

static void diag_alpha(double *psi, const tso_ham *H, int a, double t)
{
    tso_apply_diag(psi, H->N, H->h + (size_t)a * H->N, H->J + (size_t)a * H->N * H->N, H->Etab[a], t);
}

/* exp(-i t H_x) = Y exp(-i t H_x[S^x -> S^z]) Y^dag      (eq. 7 and eq. 10; A4)
 * "Forward Rotation -> Phases in Z -> Backward Rotation".  Fields and bonds of the same alpha are
 * one diagonal. */
static void apply_Hx(double *psi, const tso_ham *H, double t)
{
    tso_apply_sweep(psi, H->N, TSO_SWEEP_YDAG);
    diag_alpha(psi, H, TSO_X, t);
    tso_apply_sweep(psi, H->N, TSO_SWEEP_Y);
    tso_scale(psi, H->N, ldexp(1.0, -H->N));
}
/* exp(-i t H_y) = X exp(-i t H_y[S^y -> S^z]) X^dag      (eq. 7 and eq. 10; A4) */
static void apply_Hy(double *psi, const tso_ham *H, double t)
{
    tso_apply_sweep(psi, H->N, TSO_SWEEP_XDAG);
    diag_alpha(psi, H, TSO_Y, t);
    tso_apply_sweep(psi, H->N, TSO_SWEEP_X);
    tso_scale(psi, H->N, ldexp(1.0, -H->N));
}
/* exp(-i t H_z): "a trivial phase" (eq. 9). */
static void apply_Hz(double *psi, const tso_ham *H, double t)
{
    diag_alpha(psi, H, TSO_Z, t);
}

/* U1(t) = exp(-itH_x) exp(-itH_y) exp(-itH_z)            (eq. 3 with K = 3 in the order of eq. 6/8; A6)
 * The right-most factor acts first. */
static void U1(double *psi, const tso_ham *H, double t)
{
    apply_Hz(psi, H, t);
    apply_Hy(psi, H, t);
    apply_Hx(psi, H, t);
}
/* U1^dag(-t) = [exp(+itH_x) exp(+itH_y) exp(+itH_z)]^dag = exp(-itH_z) exp(-itH_y) exp(-itH_x). */
static void U1dag_neg(double *psi, const tso_ham *H, double t)
{
    apply_Hx(psi, H, t);
    apply_Hy(psi, H, t);
    apply_Hz(psi, H, t);
}
/* U2(t) = U1^dag(-t/2) U1(t/2), literally: no merging of neighbours. */
static void U2(double *psi, const tso_ham *H, double t)
{
    U1(psi, H, 0.5 * t);
    U1dag_neg(psi, H, 0.5 * t);
}
/* U4(t) = U2(at) U2(at) U2((1-4a)t) U2(at) U2(at),  a = 1/(4 - 4^(1/3)) */
static void U4(double *psi, const tso_ham *H, double t)
{
    const double a = 1.0 / (4.0 - cbrt(4.0));
    U2(psi, H, a * t);
    U2(psi, H, a * t);
    U2(psi, H, (1.0 - 4.0 * a) * t);
    U2(psi, H, a * t);
    U2(psi, H, a * t);
}

/* psi <- [U_order(tau)]^n_steps psi.  order in {1, 2, 4}.  use_tables != 0: pre-compute the three energy
 * vectors once; == 0: evaluate the O(N^2) definition every time.  Both give bit-identical
 * results (the table holds the same function values).  Returns 0, or -1 on bad arguments / no memory. */
int tso_evolve(double *psi, int N, const double *h, const double *J, double tau, int64_t n_steps, int order,
               int use_tables)
{
    if (N < 1 || N > 40 || !psi || !h || !J || n_steps < 0) return -1;
    if (order != 1 && order != 2 && order != 4) return -1;
    tso_ham H;
    H.N = N; H.h = h; H.J = J;
    double *tabs[3] = {NULL, NULL, NULL};
    for (int a = 0; a < 3; ++a) H.Etab[a] = NULL;
    if (use_tables) {
        for (int a = 0; a < 3; ++a) {
            tabs[a] = (double *)malloc(sizeof(double) << N);
            if (!tabs[a]) { for (int b = 0; b < a; ++b) free(tabs[b]); return -1; }
            tso_energy_table(N, h + (size_t)a * N, J + (size_t)a * N * N, tabs[a]);
            H.Etab[a] = tabs[a];
        }
    }
    for (int64_t s = 0; s < n_steps; ++s) {
        if (order == 1) U1(psi, &H, tau);
        else if (order == 2) U2(psi, &H, tau);
        else U4(psi, &H, tau);
    }
    for (int a = 0; a < 3; ++a) free(tabs[a]);
    return 0;
}

/* Single factors, exported so that tests can pin each one against its dense exponential. */
int tso_apply_H_alpha(double *psi, int N, const double *h, const double *J, int alpha, double t)
{
    if (N < 1 || !psi || !h || !J || alpha < 0 || alpha > 2) return -1;
    tso_ham H;
    H.N = N; H.h = h; H.J = J;
    for (int a = 0; a < 3; ++a) H.Etab[a] = NULL;
    if (alpha == TSO_X) apply_Hx(psi, &H, t);
    else if (alpha == TSO_Y) apply_Hy(psi, &H, t);
    else apply_Hz(psi, &H, t);
    return 0;
}

/* Observables (the paper only names them; formulas are reading A15), un-normalised <psi|S^a_j|psi>:
 *   <S^z_j> = 1/2 sum_k (2 bit_j(k) - 1) |c_k|^2
 *   <S^x_j> = sum_{k: bit_j = 0} Re( conj(c_{k + 2^j}) c_k )
 *   <S^y_j> = sum_{k: bit_j = 0} Im( conj(c_{k + 2^j}) c_k )
 * Summed in index order with Kahan compensation. */
double tso_expect(const double *psi, int N, int alpha, int j)
{
    const int64_t dim = (int64_t)1 << N;
    const int64_t bit = (int64_t)1 << j;
    double sum = 0.0, comp = 0.0;
    for (int64_t k = 0; k < dim; ++k) {
        double term;
        if (alpha == TSO_Z) {
            double p = psi[2 * k] * psi[2 * k] + psi[2 * k + 1] * psi[2 * k + 1];
            term = (k & bit) ? 0.5 * p : -0.5 * p;
        } else {
            if (k & bit) continue;
            double r0 = psi[2 * k], i0 = psi[2 * k + 1];
            double r1 = psi[2 * (k + bit)], i1 = psi[2 * (k + bit) + 1];
            /* conj(c1) c0 = (r1 - i i1)(r0 + i i0) = (r1 r0 + i1 i0) + i (r1 i0 - i1 r0) */
            term = (alpha == TSO_X) ? (r1 * r0 + i1 * i0) : (r1 * i0 - i1 * r0);
        }
        double y = term - comp;
        double t = sum + y;
        comp = (t - sum) - y;
        sum = t;
    }
    return sum;
}

/* ||psi||^2, Kahan-summed in index order. */
double tso_norm2(const double *psi, int N)
{
    const int64_t dim = (int64_t)1 << N;
    double sum = 0.0, comp = 0.0;
    for (int64_t k = 0; k < dim; ++k) {
        double term = psi[2 * k] * psi[2 * k] + psi[2 * k + 1] * psi[2 * k + 1];
        double y = term - comp;
        double t = sum + y;
        comp = (t - sum) - y;
        sum = t;
    }
    return sum;
}

/* <phi|psi> (eq. 11's overlap): out[0] = Re, out[1] = Im.  Kahan-summed. */
void tso_overlap(const double *phi, const double *psi, int N, double *out)
{
    const int64_t dim = (int64_t)1 << N;
    double sr = 0.0, cr = 0.0, si = 0.0, ci = 0.0;
    for (int64_t k = 0; k < dim; ++k) {
        double a = phi[2 * k], b = phi[2 * k + 1], c = psi[2 * k], d = psi[2 * k + 1];
        double tr = a * c + b * d, ti = a * d - b * c;      /* conj(phi) psi */
        double y = tr - cr, t = sr + y; cr = (t - sr) - y; sr = t;
        y = ti - ci; t = si + y; ci = (t - si) - y; si = t;
    }
    out[0] = sr; out[1] = si;
}

/* ------------------------------------------------------------------------------------------------------------
 * "Local and non-local physical magnitudes" beyond the one-site expectation values; the paper names them
 * without formulas, so these are the textbook definitions in the conventions of the header (reading A15):
 *
 * Two-site correlator <psi| S^a_j S^a_k |psi>, j != k, un-normalised.  With m = 2^j + 2^k and sigma = bit - 1/2:
 *   zz:  sum_i sigma_j(i) sigma_k(i) |c_i|^2
 *   xx:  1/4 sum_i conj(c_{i xor m}) c_i                         (S^x = 1/2 (|up><down| + |down><up|) flips the bit)
 *   yy: -sum_i sigma_j(i) sigma_k(i) conj(c_{i xor m}) c_i       (S^y|up> = i/2 |down>, S^y|down> = -i/2 |up>: flipping
 *        bit b contributes the factor i (2 b - 1) / 2 = i sigma_b)
 * The sums are real (the i -> i xor m terms pair up as complex conjugates); the real part is accumulated. */
double tso_correlate(const double *psi, int N, int alpha, int j, int k)
{
    const int64_t dim = (int64_t)1 << N;
    const int64_t bj = (int64_t)1 << j, bk = (int64_t)1 << k, m = bj | bk;
    double sum = 0.0, comp = 0.0;
    for (int64_t i = 0; i < dim; ++i) {
        const double sj = (i & bj) ? 0.5 : -0.5, sk = (i & bk) ? 0.5 : -0.5;
        const double r0 = psi[2 * i], i0 = psi[2 * i + 1];
        double term;
        if (alpha == TSO_Z) {
            term = sj * sk * (r0 * r0 + i0 * i0);
        } else {
            const double r1 = psi[2 * (i ^ m)], i1 = psi[2 * (i ^ m) + 1];
            const double re = r1 * r0 + i1 * i0;                 /* Re( conj(c_{i xor m}) c_i ) */
            term = (alpha == TSO_X) ? 0.25 * re : -sj * sk * re;
        }
        double y = term - comp;
        double t = sum + y;
        comp = (t - sum) - y;
        sum = t;
    }
    return sum;
}

/* Total magnetisation sum_j <S^z_j> ("the spurious total magnetization observed in polarization-conserving
 * Hamiltonians"). */
double tso_total_sz(const double *psi, int N)
{
    double s = 0.0;
    for (int j = 0; j < N; ++j) s += tso_expect(psi, N, TSO_Z, j);
    return s;
}

/* <psi|H|psi> for the Hamiltonian of eq. 1, term by term from the definition:
 *   sum_a [ sum_j h^a_j <S^a_j>  +  sum_{j != k} J^a_{jk} <S^a_j S^a_k> ]        (diagonal of J ignored, A1). */
double tso_energy_expect(const double *psi, int N, const double *h, const double *J)
{
    double E = 0.0;
    for (int a = 0; a < 3; ++a) {
        for (int j = 0; j < N; ++j) {
            const double hj = h[(size_t)a * N + j];
            if (hj != 0.0) E += hj * tso_expect(psi, N, a, j);
        }
        for (int j = 0; j < N; ++j)
            for (int k = 0; k < N; ++k) {
                if (j == k) continue;
                const double Jjk = J[((size_t)a * N + j) * N + k];
                if (Jjk != 0.0) E += Jjk * tso_correlate(psi, N, a, j, k);
            }
    }
    return E;
}

/* The "one spin up, the rest in high-temperature equilibrium" state of eq. A.1:
 *   |Psi_0> = |up>_u (x) sum_{j < 2^(N-1)} 2^{-(N-1)/2} exp(i phi_j) |beta_j>,   phi_j = random phase.
 * |beta_j> runs over the Ising states of the other N-1 spins: j is the amplitude index with bit u removed.
 * The paper does not say how the phases are drawn; here phi_j = 2 pi u_j with u_j in [0, 1) from a COUNTER-BASED
 * generator, so that the oracle and the CUDA path can each produce phase j without sharing code or state:
 *   u_j = (splitmix64(seed + (j + 1) * 0x9E3779B97F4A7C15) >> 11) * 2^-53
 * where splitmix64 is the finalizer of Steele, Lea & Flood's SplitMix generator (i.e. u_j is the (j+1)-th output of
 * SplitMix64 seeded with `seed`; pinned by its published first outputs for seed 0 in the tests). */
static uint64_t splitmix64_mix(uint64_t z)
{
    z = (z ^ (z >> 30)) * UINT64_C(0xBF58476D1CE4E5B9);
    z = (z ^ (z >> 27)) * UINT64_C(0x94D049BB133111EB);
    return z ^ (z >> 31);
}

uint64_t tso_splitmix64(uint64_t seed, uint64_t j)
{
    return splitmix64_mix(seed + (j + 1) * UINT64_C(0x9E3779B97F4A7C15));
}

void tso_random_phase_state(double *psi, int N, int up_spin, uint64_t seed)
{
    const int64_t dim = (int64_t)1 << N;
    const int64_t ub = (int64_t)1 << up_spin;
    const double amp = 1.0 / sqrt(ldexp(1.0, N - 1));
    for (int64_t k = 0; k < dim; ++k) {
        if (!(k & ub)) { psi[2 * k] = 0.0; psi[2 * k + 1] = 0.0; continue; }
        const uint64_t j = (uint64_t)(((k >> (up_spin + 1)) << up_spin) | (k & (ub - 1)));   /* k with bit u removed */
        const double u = (double)(tso_splitmix64(seed, j) >> 11) * ldexp(1.0, -53);
        const double phi = 2.0 * 3.14159265358979323846 * u;    /* 2 pi u (-std=c99 has no M_PI) */
        psi[2 * k] = amp * cos(phi);
        psi[2 * k + 1] = amp * sin(phi);
    }
}
