/*
 * oracle/dgo.c — CPU ORACLE for the per-cell exponential drag update of arXiv 2509.25347.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may build, link, import or call it.  It shares
 * no code, header, table or constant with the CUDA path (paper_2509_25347_b200/csrc) and neither
 * side includes the other.
 *
 * What it computes (PAPER.md = /root/reference/PAPER.md at build time of this repo):
 *   For every cell, p_out[comp] = exp(dt*Omega) * p_in[comp] for comp = x,y,z           (Eq. 18)
 *   with Omega the (N+1)x(N+1) drag matrix of Eq. 17, built from
 *   eps_i = rho_d,i / rho_g (Eq. 14) and alpha_i = 1 / T_s,i (Eq. 15),
 *   one matrix per cell (footnote 1).  Species index 0 is the gas.
 *
 * How (the definition written out; plain, slow, obviously correct; x87 80-bit long double):
 *   1. A = dt*Omega filled densely; every diagonal entry is minus the sum of the off-diagonal
 *      entries of its column, so Omega is defined in (long double) real arithmetic from the fp64
 *      inputs, not from an fp64-rounded matrix (reading R16).
 *   2. ||A||_1 by the generic max-column-sum loop; s = smallest integer >= 0 with ||A||_1/2^s <= 1.
 *   3. X = T_30(A/2^s) = sum_{j<=30} (A/2^s)^j / j!  (Eq. 19) by plain Horner with
 *      dense triple-loop products.  Remainder <= 1/31! ~ 1.2e-34, far below 2^-64.
 *   4. s naive triple-loop squarings (Eq. 23-24).
 *   5. Three dense mat-vecs.
 *   No Table B.1, no closed-form norm, no sparsity, no symmetry, no blocking: none of the CUDA
 *   path's shortcuts appear here.
 *
 * Pins (tests/test_oracle_pins.py, -m "not gpu"): N=1 closed form, Table 1 (tests B, C),
 * unit column sums, equal-velocity fixed point, 0<=E<=1, semigroup, permutation equivariance,
 * mpmath 50-digit expm / symmetric eigendecomposition on small and stiff inputs.
 *
 * Layouts are the same structure-of-arrays layouts as include/dg.h but on the HOST:
 *   rho_g[ncells], rho_d[N][ncells], t_s[N][ncells], p[3][n][ncells], A/E[n*n][ncells] (row r = destination).
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define DGO_NMAX 64            /* max dust species the oracle accepts (n = N+1 <= 65) */
#define DGO_DEGREE 30          /* Taylor degree of step 3 */

typedef long double ld;

/* Eq. 14, 15, 17: A = dt*Omega, n x n row-major, n = N+1. */
void dgo_cell_matrix(double rho_g, const double *rho_d, const double *t_s, double dt, int N, ld *A)
{
    int n = N + 1;
    for (int k = 0; k < n * n; ++k) A[k] = 0.0L;
    for (int i = 1; i <= N; ++i) {
        ld eps = (ld)rho_d[i - 1] / (ld)rho_g;          /* Eq. 14 */
        ld alpha = 1.0L / (ld)t_s[i - 1];               /* Eq. 15 */
        A[0 * n + i] = (ld)dt * alpha;                  /* row 0 (gas gains from dust i):  alpha_i        */
        A[i * n + 0] = (ld)dt * (eps * alpha);          /* row i (dust i gains from gas):  eps_i alpha_i  */
    }
    /* diagonal: columns of Eq. 17 sum to zero (total momentum) */
    for (int c = 0; c < n; ++c) {
        ld s = 0.0L;
        for (int r = 0; r < n; ++r) if (r != c) s += A[r * n + c];
        A[c * n + c] = -s;
    }
}

static void matmul(const ld *X, const ld *Y, ld *Z, int n)
{
    for (int i = 0; i < n; ++i)
        for (int j = 0; j < n; ++j) {
            ld acc = 0.0L;
            for (int k = 0; k < n; ++k) acc += X[i * n + k] * Y[k * n + j];
            Z[i * n + j] = acc;
        }
}

/* exp(A) for a dense n x n matrix: steps 2-4 of the header.  Returns s.  work: 3*n*n long doubles. */
int dgo_expm(const ld *A, int n, ld *E, ld *work)
{
    ld *B = work, *F = work + n * n, *T = work + 2 * n * n;
    ld norm1 = 0.0L;
    for (int c = 0; c < n; ++c) {
        ld s = 0.0L;
        for (int r = 0; r < n; ++r) s += fabsl(A[r * n + c]);
        if (s > norm1) norm1 = s;
    }
    int s = 0;
    ld scale = 1.0L;
    while (norm1 * scale > 1.0L) { scale *= 0.5L; ++s; }
    for (int k = 0; k < n * n; ++k) B[k] = A[k] * scale;
    /* Horner: F = I; for j = m..1: F = I + B*F/j   =>  F = sum_{j<=m} B^j/j!   (Eq. 19) */
    for (int k = 0; k < n * n; ++k) F[k] = 0.0L;
    for (int i = 0; i < n; ++i) F[i * n + i] = 1.0L;
    for (int j = DGO_DEGREE; j >= 1; --j) {
        matmul(B, F, T, n);
        for (int k = 0; k < n * n; ++k) F[k] = T[k] / (ld)j;
        for (int i = 0; i < n; ++i) F[i * n + i] += 1.0L;
    }
    /* Eq. 23-24: square s times */
    for (int q = 0; q < s; ++q) {
        matmul(F, F, T, n);
        memcpy(F, T, sizeof(ld) * n * n);
    }
    memcpy(E, F, sizeof(ld) * n * n);
    return s;
}

/* Eq. 18 for the three momentum components of one cell: p_out[comp][k] = sum_j E[k][j] p_in[comp][j]. */
void dgo_cell_apply(const ld *E, const ld *p_in, int n, ld *p_out)
{
    for (int comp = 0; comp < 3; ++comp)
        for (int k = 0; k < n; ++k) {
            ld acc = 0.0L;
            for (int j = 0; j < n; ++j) acc += E[k * n + j] * p_in[comp * n + j];
            p_out[comp * n + k] = acc;
        }
}

int dgo_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

static int check_args(int N, long long ncells) { return (N < 1 || N > DGO_NMAX || ncells < 0) ? 1 : 0; }

/* Stage a1 for a batch: A[n*n][ncells] in long double. */
int dgo_drag_matrix_build(const double *rho_g, const double *rho_d, const double *t_s, double dt,
                          int N, long long ncells, ld *A_out, int nthreads)
{
    if (check_args(N, ncells)) return 1;
    int n = N + 1;
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
#endif
#pragma omp parallel for schedule(static)
    for (long long c = 0; c < ncells; ++c) {
        double rd[DGO_NMAX], ts[DGO_NMAX];
        ld A[(DGO_NMAX + 1) * (DGO_NMAX + 1)];
        for (int i = 0; i < N; ++i) { rd[i] = rho_d[(long long)i * ncells + c]; ts[i] = t_s[(long long)i * ncells + c]; }
        dgo_cell_matrix(rho_g[c], rd, ts, dt, N, A);
        for (int k = 0; k < n * n; ++k) A_out[(long long)k * ncells + c] = A[k];
    }
    return 0;
}

/* Stages a2-a4 for a batch of fp64 drag matrices A[n*n][ncells].  Per the dg_expm_scale_square
 * contract (include/dg.h) the stored diagonal is ignored when rebuild_diag != 0 and rebuilt, in long
 * double, as minus the off-diagonal column sum.  E_out[n*n][ncells] long double; s_out nullable. */
int dgo_expm_batch(const double *A_in, int N, long long ncells, int rebuild_diag, ld *E_out, int *s_out, int nthreads)
{
    if (check_args(N, ncells)) return 1;
    int n = N + 1;
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
#endif
#pragma omp parallel
    {
        ld *A = (ld *)malloc(sizeof(ld) * 5 * n * n);
        ld *E = A + n * n, *work = A + 2 * n * n;
#pragma omp for schedule(static)
        for (long long c = 0; c < ncells; ++c) {
            for (int k = 0; k < n * n; ++k) A[k] = (ld)A_in[(long long)k * ncells + c];
            if (rebuild_diag)
                for (int col = 0; col < n; ++col) {
                    ld s = 0.0L;
                    for (int r = 0; r < n; ++r) if (r != col) s += A[r * n + col];
                    A[col * n + col] = -s;
                }
            int s = dgo_expm(A, n, E, work);
            for (int k = 0; k < n * n; ++k) E_out[(long long)k * ncells + c] = E[k];
            if (s_out) s_out[c] = s;
        }
        free(A);
    }
    return 0;
}

/* Stage a5 for a batch: p_out = E p_in with E given in fp64 (the staged CUDA path's E array). */
int dgo_drag_apply(const double *E_in, const double *p_in, int N, long long ncells, ld *p_out, int nthreads)
{
    if (check_args(N, ncells)) return 1;
    int n = N + 1;
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
#endif
#pragma omp parallel
    {
        ld *E = (ld *)malloc(sizeof(ld) * (n * n + 6 * n));
        ld *pi = E + n * n, *po = pi + 3 * n;
#pragma omp for schedule(static)
        for (long long c = 0; c < ncells; ++c) {
            for (int k = 0; k < n * n; ++k) E[k] = (ld)E_in[(long long)k * ncells + c];
            for (int k = 0; k < 3 * n; ++k) pi[k] = (ld)p_in[(long long)k * ncells + c];
            dgo_cell_apply(E, pi, n, po);
            for (int k = 0; k < 3 * n; ++k) p_out[(long long)k * ncells + c] = po[k];
        }
        free(E);
    }
    return 0;
}

/* The whole path a1..a5 for a batch: the reference result for dg_drag_update.
 * E_out (nullable): exp(dt*Omega) per cell, [n*n][ncells].  s_out (nullable): oracle's own s. */
int dgo_drag_update(const double *rho_g, const double *rho_d, const double *t_s, double dt, const double *p_in,
                    int N, long long ncells, ld *p_out, ld *E_out, int *s_out, int nthreads)
{
    if (check_args(N, ncells)) return 1;
    int n = N + 1;
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
#endif
#pragma omp parallel
    {
        ld *A = (ld *)malloc(sizeof(ld) * (5 * n * n + 6 * n));
        ld *E = A + n * n, *work = A + 2 * n * n, *pi = A + 5 * n * n, *po = pi + 3 * n;
        double rd[DGO_NMAX], ts[DGO_NMAX];
#pragma omp for schedule(dynamic, 64)
        for (long long c = 0; c < ncells; ++c) {
            for (int i = 0; i < N; ++i) { rd[i] = rho_d[(long long)i * ncells + c]; ts[i] = t_s[(long long)i * ncells + c]; }
            dgo_cell_matrix(rho_g[c], rd, ts, dt, N, A);
            int s = dgo_expm(A, n, E, work);
            for (int k = 0; k < 3 * n; ++k) pi[k] = (ld)p_in[(long long)k * ncells + c];
            dgo_cell_apply(E, pi, n, po);
            for (int k = 0; k < 3 * n; ++k) p_out[(long long)k * ncells + c] = po[k];
            if (E_out) for (int k = 0; k < n * n; ++k) E_out[(long long)k * ncells + c] = E[k];
            if (s_out) s_out[c] = s;
        }
        free(A);
    }
    return 0;
}

/* ---------------------------------------------------------------------------------------------------------------
 * First-order implicit RK1 drag step (App. A.1, Eq. A.3-A.6): for a pure drag step
 * (U^(n+1/2) = U^(n) in Eq. A.4-A.5)   U^(n+1) = (I - dt*Omega)^-1 U^(n),   i.e. solve (I - dt*Omega) q = b (Eq. A.6)
 * for each of the three components.  The oracle is the DEFINITION: the dense matrix I - dt*Omega (Omega from
 * dgo_cell_matrix, Eq. 17) solved by Gaussian elimination with partial pivoting in long double — the O(N^3) route of
 * App. A.1, not the O(N) closed form of App. A.2 (Eq. A.8-A.9) that the CUDA kernel uses.
 * Pins: tests/test_rk1.py (residual in 50-digit arithmetic, N = 1 closed form, conservation, fixed point,
 * first-order convergence to exp(t Omega), dt -> infinity limit). */
static int solve_dense(ld *M, ld *rhs, int n, int nrhs)   /* M n x n row-major (destroyed), rhs n x nrhs row-major */
{
    for (int c = 0; c < n; ++c) {
        int piv = c;
        for (int r = c + 1; r < n; ++r) if (fabsl(M[r * n + c]) > fabsl(M[piv * n + c])) piv = r;
        if (M[piv * n + c] == 0.0L) return 1;
        if (piv != c) {
            for (int k = 0; k < n; ++k) { ld t = M[c * n + k]; M[c * n + k] = M[piv * n + k]; M[piv * n + k] = t; }
            for (int k = 0; k < nrhs; ++k) { ld t = rhs[c * nrhs + k]; rhs[c * nrhs + k] = rhs[piv * nrhs + k]; rhs[piv * nrhs + k] = t; }
        }
        for (int r = c + 1; r < n; ++r) {
            ld f = M[r * n + c] / M[c * n + c];
            if (f == 0.0L) continue;
            for (int k = c; k < n; ++k) M[r * n + k] -= f * M[c * n + k];
            for (int k = 0; k < nrhs; ++k) rhs[r * nrhs + k] -= f * rhs[c * nrhs + k];
        }
    }
    for (int c = n - 1; c >= 0; --c)
        for (int k = 0; k < nrhs; ++k) {
            ld acc = rhs[c * nrhs + k];
            for (int j = c + 1; j < n; ++j) acc -= M[c * n + j] * rhs[j * nrhs + k];
            rhs[c * nrhs + k] = acc / M[c * n + c];
        }
    return 0;
}

int dgo_rk1_update(const double *rho_g, const double *rho_d, const double *t_s, double dt, const double *p_in,
                   int N, long long ncells, ld *p_out, int nthreads)
{
    if (check_args(N, ncells)) return 1;
    const int n = N + 1;
    int bad = 0;
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
#else
    (void)nthreads;
#endif
#pragma omp parallel for schedule(static) reduction(| : bad)
    for (long long c = 0; c < ncells; ++c) {
        ld M[(DGO_NMAX + 1) * (DGO_NMAX + 1)], rhs[(DGO_NMAX + 1) * 3];
        double rd[DGO_NMAX], ts[DGO_NMAX];
        for (int i = 0; i < N; ++i) { rd[i] = rho_d[(long long)i * ncells + c]; ts[i] = t_s[(long long)i * ncells + c]; }
        dgo_cell_matrix(rho_g[c], rd, ts, dt, N, M);                       /* M = dt*Omega          */
        for (int k = 0; k < n * n; ++k) M[k] = -M[k];
        for (int k = 0; k < n; ++k) M[k * n + k] += 1.0L;                  /* M = I - dt*Omega      */
        for (int k = 0; k < n; ++k)
            for (int comp = 0; comp < 3; ++comp) rhs[k * 3 + comp] = (ld)p_in[((long long)comp * n + k) * ncells + c];
        bad |= solve_dense(M, rhs, n, 3);
        for (int k = 0; k < n; ++k)
            for (int comp = 0; comp < 3; ++comp) p_out[((long long)comp * n + k) * ncells + c] = rhs[k * 3 + comp];
    }
    return bad;
}

/* ---------------------------------------------------------------------------------------------------------------
 * Gas energy over one exact drag step: frictional heating (Eq. 4 and the third entry of Eq. 11).
 * With the transport and external-force terms split off (Eq. 25-26) the gas energy obeys
 *     dE_g/dt = sum_i rho_d,i (v_d,i - v_g)/T_s,i . v_g  +  w sum_i rho_d,i (v_d,i - v_g)^2 / T_s,i        (w in [0, 1])
 * along the exact solution p(t) = exp(t Omega) p(0) of the momenta (Eq. 18).  The paper gives NO discrete formula for
 * it (reading R20); what is computed here is the exact integral of that equation over the step:
 *   - the first term is v_g . dM_g/dt = d/dt (|M_g|^2 / (2 rho_g))     (rho_g is constant during the drag step),
 *   - the second is  -w dK/dt  with  K = |M_g|^2/(2 rho_g) + sum_i |M_d,i|^2/(2 rho_d,i)  the total kinetic energy,
 *     because  dK/dt = v_g . dM_g/dt + sum_i v_d,i . dM_d,i/dt = - sum_i rho_d,i (v_d,i - v_g)^2 / T_s,i  by Eq. 3, 6;
 *   hence     E_g(t+dt) = E_g(t) + [KE_g(t+dt) - KE_g(t)] + w [K(t) - K(t+dt)],
 *   with the momenta at t+dt from the oracle's own exponential.  w = 1: E_g + sum_i |M_d,i|^2/(2 rho_d,i) is conserved.
 * A species with rho_d,i = 0 carries no momentum and no energy (its term is skipped).
 * Pins (tests/test_energy.py): the heating integral by 30-digit quadrature of the second term along the exact
 * trajectory (mpmath, Eq. 4 retyped), and the N = 1 closed form  mu |dv_0|^2 (1 - exp(-2 kappa dt)) / 2.
 * p_out (nullable) receives the momenta after the step. */
int dgo_energy_update(const double *rho_g, const double *rho_d, const double *t_s, double dt, const double *p_in,
                      const double *E_in, double w, int N, long long ncells, ld *E_out, ld *p_out, int nthreads)
{
    if (check_args(N, ncells)) return 1;
    int n = N + 1;
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
#endif
#pragma omp parallel
    {
        ld *A = (ld *)malloc(sizeof(ld) * (5 * n * n + 6 * n));
        ld *E = A + n * n, *work = A + 2 * n * n, *pi = A + 5 * n * n, *po = pi + 3 * n;
        double rd[DGO_NMAX], ts[DGO_NMAX];
#pragma omp for schedule(dynamic, 64)
        for (long long c = 0; c < ncells; ++c) {
            for (int i = 0; i < N; ++i) { rd[i] = rho_d[(long long)i * ncells + c]; ts[i] = t_s[(long long)i * ncells + c]; }
            dgo_cell_matrix(rho_g[c], rd, ts, dt, N, A);
            dgo_expm(A, n, E, work);
            for (int k = 0; k < 3 * n; ++k) pi[k] = (ld)p_in[(long long)k * ncells + c];
            dgo_cell_apply(E, pi, n, po);
            ld keg_in = 0.0L, keg_out = 0.0L, kd_in = 0.0L, kd_out = 0.0L;
            for (int comp = 0; comp < 3; ++comp) {
                keg_in += pi[comp * n] * pi[comp * n];
                keg_out += po[comp * n] * po[comp * n];
            }
            keg_in /= 2.0L * (ld)rho_g[c];
            keg_out /= 2.0L * (ld)rho_g[c];
            for (int i = 1; i <= N; ++i) {
                if (rd[i - 1] == 0.0) continue;
                ld a = 0.0L, b = 0.0L;
                for (int comp = 0; comp < 3; ++comp) {
                    a += pi[comp * n + i] * pi[comp * n + i];
                    b += po[comp * n + i] * po[comp * n + i];
                }
                kd_in += a / (2.0L * (ld)rd[i - 1]);
                kd_out += b / (2.0L * (ld)rd[i - 1]);
            }
            E_out[c] = (ld)E_in[c] + (keg_out - keg_in) + (ld)w * ((keg_in + kd_in) - (keg_out + kd_out));
            if (p_out) for (int k = 0; k < 3 * n; ++k) p_out[(long long)k * ncells + c] = po[k];
        }
        free(A);
    }
    return 0;
}

int dgo_sizeof_long_double(void) { return (int)sizeof(ld); }
int dgo_ldbl_mant_dig(void) { return __LDBL_MANT_DIG__; }
