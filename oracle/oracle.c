/*
 * oracle.c -- plain, slow, obviously-correct CPU reference ("the oracle") for the
 * shared-LHS batched tridiagonal / pentadiagonal solves and the semi-implicit
 * Cahn-Hilliard step of arxiv/paper_2107_05395.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT PRODUCT CODE.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may build, load or call it.
 * It shares no code, header, table or helper with the CUDA library under
 * paper_2107_05395_b200/csrc/, and neither side includes or imports the other.
 *
 * Everything is fp64, one system at a time, written in the paper's own order and
 * notation (divisions kept, compiled with -ffp-contract=off so no FMA is formed):
 *
 *   orc_tri_factor      PAPER.md:87-93  (eq. 1-2),  555-566 (Alg. 1)
 *   orc_tri_solve       PAPER.md:95-108 (eq. 3-6),  568-597 (Alg. 2)
 *   orc_penta_factor    PAPER.md:219-256 (Sec. 4.1 steps 1-14), 601-637 (Alg. 3)
 *   orc_penta_solve     PAPER.md:258-278 (Sec. 4.1), 639-676 (Alg. 4)
 *   orc_ch_rhs          PAPER.md:365-392 (eq. 24, 25a, 26c)
 *   orc_tri_periodic_*  PAPER.md:140-164 (Sec. 3.3, eq. 12-15: Sherman-Morrison)
 *   *_interleaved       PAPER.md:69 (Sec. 2), Alg. 2 "rowID +- M": element i of
 *                       system j lives at rhs[i*M + j]
 *
 * Readings of garbled / silent passages follow SURVEY.md 8(c) and are listed in
 * DESIGN.md ("Readings"); each is marked [C-n] below.
 *
 * Parity pins (tests/test_oracle_*.py, all run without a GPU): exact rational Gaussian
 * elimination on tiny systems, numpy dense solves, residuals, the closed-form
 * eigenpairs of Toeplitz tri / penta (I + r T^2) matrices, exact modal decay over 100
 * steps, L*R == A rebuilt densely, reductions (penta with zero outer bands == tri;
 * tri with zero off-diagonals == scaling), a dense restatement of eq. 24 for the CH
 * step and its discrete mass-balance identity; for the periodic solve the splitting
 * A' + u (x) v == A entrywise, dense solves of the cyclic matrix, the circulant eigenpairs and
 * conservation of the column sum.  No function here is "parity unpinned".
 */
#include <math.h>
#include <stddef.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_API __attribute__((visibility("default")))

/* ------------------------------------------------------------------------------------
 * Tridiagonal.  Row i (1-based, paper): a_i x_{i-1} + b_i x_i + c_i x_{i+1} = d_i.
 * Arrays are 0-based here: a[i-1] holds a_i.  a[0] and c[n-1] are never read.
 * ---------------------------------------------------------------------------------- */

/* Alg. 1: overwrites b with b^, c with c^; a untouched.
 * Returns 0, or the 1-based row whose pivot b^_i is zero / non-finite [C-14]. */
ORC_API int orc_tri_factor(int n, const double *a, double *b, double *c)
{
    if (n < 1) return -1;
    if (b[0] == 0.0 || !isfinite(b[0])) return 1;
    if (n == 1) return 0;                        /* [C-13] nothing else to do         */
    c[0] = c[0] / b[0];                          /* eq. 1:  c^_1 = c_1 / b_1          */
    for (int i = 1; i <= n - 2; ++i) {           /* Alg. 1 line 3: i = 2 .. N-1       */
        b[i] = b[i] - a[i] * c[i - 1];           /* eq. 2:  b^_i = b_i - a_i c^_{i-1} */
        if (b[i] == 0.0 || !isfinite(b[i])) return i + 1;
        c[i] = c[i] / b[i];                      /*         c^_i = c_i / b^_i         */
    }
    b[n - 1] = b[n - 1] - a[n - 1] * c[n - 2];   /* Alg. 1 line 7; c^_N unused [C-3]  */
    if (b[n - 1] == 0.0 || !isfinite(b[n - 1])) return n;
    return 0;
}

/* Alg. 2 for one contiguous system: d is overwritten by x. */
ORC_API void orc_tri_solve(int n, const double *a, const double *bh, const double *ch, double *d)
{
    d[0] = d[0] / bh[0];                         /* eq. 3 (b^_1 = b_1 [C-2])          */
    for (int i = 1; i < n; ++i)                  /* eq. 4                             */
        d[i] = (d[i] - a[i] * d[i - 1]) / bh[i];
    /* eq. 5: x_N = d^_N (already in place) */
    for (int i = n - 2; i >= 0; --i)             /* eq. 6 as Alg. 2 line 10 [C-1]     */
        d[i] = d[i] - ch[i] * d[i + 1];
}

/* ------------------------------------------------------------------------------------
 * Pentadiagonal, paper naming: row i is
 *   a_i x_{i-2} + b_i x_{i-1} + c_i x_i + d_i x_{i+1} + e_i x_{i+2} = f_i.
 * 0-based arrays: a[i-1] holds a_i, etc.  Never read: a[0],a[1],b[0],d[n-1],e[n-2],e[n-1].
 * After the factor: a = eps, b = beta, c = alpha, d = gamma, e = delta (step 14).
 * ---------------------------------------------------------------------------------- */

static int bad(double v) { return v == 0.0 || !isfinite(v); }

/* General-row form used for N < 4 [C-13]: the same formulas as step 8 with every
 * out-of-range gamma, delta taken as 0 and never-read diagonal entries ignored.
 * tests/test_oracle_penta.py checks it is bit-identical to the literal steps for N >= 4. */
ORC_API int orc_penta_factor_general(int n, const double *a, double *b, double *c, double *d, double *e)
{
    if (n < 1) return -1;
    for (int i = 0; i < n; ++i) {
        double gm1 = (i >= 1) ? d[i - 1] : 0.0, gm2 = (i >= 2) ? d[i - 2] : 0.0;
        double dm1 = (i >= 1) ? e[i - 1] : 0.0, dm2 = (i >= 2) ? e[i - 2] : 0.0;
        if (i >= 2) b[i] = b[i] - a[i] * gm2;                /* beta_i                 */
        if (i >= 2) c[i] = c[i] - a[i] * dm2 - b[i] * gm1;   /* alpha_i                */
        else if (i == 1) c[i] = c[i] - b[i] * gm1;
        if (bad(c[i])) return i + 1;
        if (i <= n - 2) d[i] = ((i >= 1) ? (d[i] - b[i] * dm1) : d[i]) / c[i]; /* gamma */
        if (i <= n - 3) e[i] = e[i] / c[i];                                    /* delta */
    }
    return 0;
}

/* Sec. 4.1 steps 1-14 / Alg. 3, literally, for N >= 4; N < 4 goes to the general form. */
ORC_API int orc_penta_factor(int n, const double *a, double *b, double *c, double *d, double *e)
{
    if (n < 4) return orc_penta_factor_general(n, a, b, c, d, e);
    const int N = n;                         /* 1-based index i lives at [i-1]            */
#define A_(i) a[(i) - 1]
#define B_(i) b[(i) - 1]
#define C_(i) c[(i) - 1]
#define D_(i) d[(i) - 1]
#define E_(i) e[(i) - 1]
    if (bad(C_(1))) return 1;                /* 1. alpha_1 = c_1                          */
    D_(1) = D_(1) / C_(1);                   /* 2. gamma_1 = d_1 / alpha_1                */
    E_(1) = E_(1) / C_(1);                   /* 3. delta_1 = e_1 / alpha_1                */
                                             /* 4. beta_2 = b_2                           */
    C_(2) = C_(2) - B_(2) * D_(1);           /* 5. alpha_2 = c_2 - beta_2 gamma_1  [C-6]  */
    if (bad(C_(2))) return 2;
    D_(2) = (D_(2) - B_(2) * E_(1)) / C_(2); /* 6. gamma_2 = (d_2 - beta_2 delta_1)/alpha_2 [C-6] */
    E_(2) = E_(2) / C_(2);                   /* 7. delta_2 = e_2 / alpha_2                */
    for (int i = 3; i <= N - 2; ++i) {       /* 8. i = 3 .. N-2                           */
        B_(i) = B_(i) - A_(i) * D_(i - 2);                       /* (a) [C-6]            */
        C_(i) = C_(i) - A_(i) * E_(i - 2) - B_(i) * D_(i - 1);   /* (b) [C-6][C-9]       */
        if (bad(C_(i))) return i;
        D_(i) = (D_(i) - B_(i) * E_(i - 1)) / C_(i);             /* (c) [C-10]           */
        E_(i) = E_(i) / C_(i);                                   /* (d) [C-7]            */
    }
    B_(N - 1) = B_(N - 1) - A_(N - 1) * D_(N - 3);                         /* 9.         */
    C_(N - 1) = C_(N - 1) - A_(N - 1) * E_(N - 3) - B_(N - 1) * D_(N - 2); /* 10.        */
    if (bad(C_(N - 1))) return N - 1;
    D_(N - 1) = (D_(N - 1) - B_(N - 1) * E_(N - 2)) / C_(N - 1);           /* 11.        */
    B_(N) = B_(N) - A_(N) * D_(N - 2);                                     /* 12. [C-11] */
    C_(N) = C_(N) - A_(N) * E_(N - 2) - B_(N) * D_(N - 1);                 /* 13.        */
    if (bad(C_(N))) return N;
    /* 14. eps_i = a_i: a is untouched. */
#undef A_
#undef B_
#undef C_
#undef D_
#undef E_
    return 0;
}

/* Sec. 4.1 "steps to find g" + back-substitution / Alg. 4, one contiguous system;
 * f is overwritten by x.  N < 4 uses the same formulas with out-of-range terms dropped
 * [C-13] (for N >= 4 the guards below never fire except exactly where the paper
 * special-cases rows 1, 2, N-1, N). */
ORC_API void orc_penta_solve(int n, const double *eps, const double *beta, const double *alpha,
                             const double *gamma, const double *delta, double *f)
{
    f[0] = f[0] / alpha[0];                                   /* 1. g_1                   */
    if (n >= 2) f[1] = (f[1] - beta[1] * f[0]) / alpha[1];    /* 2. g_2                   */
    for (int i = 2; i < n; ++i)                               /* 3. g_i, i = 3..N         */
        f[i] = (f[i] - eps[i] * f[i - 2] - beta[i] * f[i - 1]) / alpha[i];
    /* 1. x_N = g_N */
    if (n >= 2) f[n - 2] = f[n - 2] - gamma[n - 2] * f[n - 1];            /* 2. x_{N-1}   */
    for (int i = n - 3; i >= 0; --i)                                      /* 3. [C-8][C-12] */
        f[i] = f[i] - gamma[i] * f[i + 1] - delta[i] * f[i + 2];
}

/* ------------------------------------------------------------------------------------
 * Cahn-Hilliard explicit half (eq. 24 RHS with eq. 25a; eq. 26c with the C^n term
 * restored [C-21]; truncated stencil, ghost values zero: w_0 = w_{N+1} = 0 [C-18]):
 *   w_i = c_i^3 - c_i,   f_i = c_i + alpha (w_{i-1} - 2 w_i + w_{i+1}),  alpha = dt/dx^2.
 * ---------------------------------------------------------------------------------- */
ORC_API void orc_ch_rhs(int n, const double *c, double alpha, double *f)
{
    for (int i = 0; i < n; ++i) {
        double wm = (i > 0) ? c[i - 1] * c[i - 1] * c[i - 1] - c[i - 1] : 0.0;
        double w0 = c[i] * c[i] * c[i] - c[i];
        double wp = (i < n - 1) ? c[i + 1] * c[i + 1] * c[i + 1] - c[i + 1] : 0.0;
        f[i] = c[i] + alpha * (wm - 2.0 * w0 + wp);
    }
}

/* ------------------------------------------------------------------------------------
 * Interleaved batch drivers: gather column j -> contiguous, run the single-system
 * routine nsteps times (RHS = previous solution), scatter back.
 * Systems j = jlo, jlo+jstride, ... < jhi are processed; the rest are left untouched
 * (lets a caller check / time a stated subset of a large batch).
 * nthreads <= 0: all cores (OpenMP over systems); the arithmetic per system is serial.
 * ---------------------------------------------------------------------------------- */
static int set_threads(int nthreads)
{
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
    else omp_set_num_threads(omp_get_num_procs());
    int used = 1;
#pragma omp parallel
    {
#pragma omp single
        used = omp_get_num_threads();
    }
    return used;
#else
    (void)nthreads;
    return 1;
#endif
}

ORC_API int orc_tri_solve_interleaved(int n, const double *a, const double *bh, const double *ch,
                                      double *rhs, long long M, long long jlo, long long jhi,
                                      long long jstride, int nsteps, int nthreads)
{
    int used = set_threads(nthreads);
#pragma omp parallel
    {
        double *col = (double *)malloc((size_t)n * sizeof(double));
#pragma omp for schedule(static)
        for (long long j = jlo; j < jhi; j += jstride) {
            for (int i = 0; i < n; ++i) col[i] = rhs[(size_t)i * M + j];
            for (int s = 0; s < nsteps; ++s) orc_tri_solve(n, a, bh, ch, col);
            for (int i = 0; i < n; ++i) rhs[(size_t)i * M + j] = col[i];
        }
        free(col);
    }
    return used;
}

ORC_API int orc_penta_solve_interleaved(int n, const double *eps, const double *beta,
                                        const double *alpha, const double *gamma,
                                        const double *delta, double *rhs, long long M,
                                        long long jlo, long long jhi, long long jstride,
                                        int nsteps, int nthreads)
{
    int used = set_threads(nthreads);
#pragma omp parallel
    {
        double *col = (double *)malloc((size_t)n * sizeof(double));
#pragma omp for schedule(static)
        for (long long j = jlo; j < jhi; j += jstride) {
            for (int i = 0; i < n; ++i) col[i] = rhs[(size_t)i * M + j];
            for (int s = 0; s < nsteps; ++s) orc_penta_solve(n, eps, beta, alpha, gamma, delta, col);
            for (int i = 0; i < n; ++i) rhs[(size_t)i * M + j] = col[i];
        }
        free(col);
    }
    return used;
}

/* Config-5 stepper: for s in 1..nsteps: f = rhs(c) (eq. 24 explicit half); c = A^{-1} f
 * with A = I + sigma*D4_trunc already factored into (eps..delta) by orc_penta_factor. */
ORC_API int orc_ch_step_interleaved(int n, const double *eps, const double *beta,
                                    const double *alpha, const double *gamma,
                                    const double *delta, double *cbuf, long long M,
                                    long long jlo, long long jhi, long long jstride,
                                    double alpha_x, int nsteps, int nthreads)
{
    int used = set_threads(nthreads);
#pragma omp parallel
    {
        double *col = (double *)malloc((size_t)n * sizeof(double));
        double *f = (double *)malloc((size_t)n * sizeof(double));
#pragma omp for schedule(static)
        for (long long j = jlo; j < jhi; j += jstride) {
            for (int i = 0; i < n; ++i) col[i] = cbuf[(size_t)i * M + j];
            for (int s = 0; s < nsteps; ++s) {
                orc_ch_rhs(n, col, alpha_x, f);
                orc_penta_solve(n, eps, beta, alpha, gamma, delta, f);
                memcpy(col, f, (size_t)n * sizeof(double));
            }
            for (int i = 0; i < n; ++i) cbuf[(size_t)i * M + j] = col[i];
        }
        free(col);
        free(f);
    }
    return used;
}

/* ------------------------------------------------------------------------------------
 * Periodic tridiagonal, PAPER.md:140-164 (Sec. 3.3, eq. 12-15): Sherman-Morrison.
 *   A = A' + u (x) v,  u = (-b_1, 0, ..., 0, c_N)^T,  v = (1, 0, ..., 0, -a_1/b_1)^T  (13a)
 *   A' = A without its two corner entries, with diagonal ends 2 b_1 and b_N + a_1 c_N / b_1  (13b)
 *   A' y = d,  A' z = u (once),  x = y - (v.y)/(1 + v.z) z                               (14, 15)
 * The paper writes constant diagonals a, b, c; with general diagonals the corner entries are
 * a_1 (row 1, column N) and c_N (row N, column 1): a[0] and c[n-1] of the arrays.  n >= 3.
 * orc_tri_periodic_factor overwrites b, c with the Thomas factors of A' (Alg. 1) and returns
 * z (length n), vN = -a_1/b_1 and den = 1 + v.z.  Returns 0, a 1-based bad pivot row, or -1.
 * ---------------------------------------------------------------------------------- */
ORC_API int orc_tri_periodic_factor(int n, const double *a, double *b, double *c, double *z,
                                    double *vN, double *den)
{
    if (n < 3) return -1;
    if (b[0] == 0.0 || !isfinite(b[0])) return 1;
    const double b1 = b[0], a1 = a[0], cN = c[n - 1];
    for (int i = 0; i < n; ++i) z[i] = 0.0;
    z[0] = -b1;                                  /* u, eq. 13a                        */
    z[n - 1] = cN;
    *vN = -a1 / b1;                              /* v_N, eq. 13a                      */
    b[0] = 2.0 * b1;                             /* A', eq. 13b                       */
    b[n - 1] = b[n - 1] + a1 * cN / b1;
    const int rc = orc_tri_factor(n, a, b, c);   /* Alg. 1 on A'                      */
    if (rc) return rc;
    orc_tri_solve(n, a, b, c, z);                /* A' z = u, eq. 14                  */
    *den = 1.0 + (z[0] + (*vN) * z[n - 1]);      /* 1 + v.z, eq. 15                   */
    if (*den == 0.0 || !isfinite(*den)) return n;
    return 0;
}

/* One contiguous system: d is overwritten by x (eq. 14-15). */
ORC_API void orc_tri_periodic_solve(int n, const double *a, const double *bh, const double *ch,
                                    const double *z, double vN, double den, double *d)
{
    orc_tri_solve(n, a, bh, ch, d);                          /* A' y = d              */
    const double fac = (d[0] + vN * d[n - 1]) / den;         /* (v.y)/(1 + v.z)       */
    for (int i = 0; i < n; ++i) d[i] = d[i] - fac * z[i];    /* eq. 15                */
}

ORC_API int orc_tri_periodic_solve_interleaved(int n, const double *a, const double *bh,
                                               const double *ch, const double *z, double vN,
                                               double den, double *rhs, long long M, long long jlo,
                                               long long jhi, long long jstride, int nsteps,
                                               int nthreads)
{
    int used = set_threads(nthreads);
#pragma omp parallel
    {
        double *col = (double *)malloc((size_t)n * sizeof(double));
#pragma omp for schedule(static)
        for (long long j = jlo; j < jhi; j += jstride) {
            for (int i = 0; i < n; ++i) col[i] = rhs[(size_t)i * M + j];
            for (int s = 0; s < nsteps; ++s) orc_tri_periodic_solve(n, a, bh, ch, z, vN, den, col);
            for (int i = 0; i < n; ++i) rhs[(size_t)i * M + j] = col[i];
        }
        free(col);
    }
    return used;
}

/* ------------------------------------------------------------------------------------
 * Periodic (cyclic) pentadiagonal, PAPER.md:380 (eq. 26a).  The paper solves it "following
 * [24,4,25]" without writing the method out (SURVEY 8(c) / DESIGN.md reading C-31): the result is
 * defined as x = A^{-1} f for the cyclic matrix, reached here by the Woodbury identity on the
 * same pattern as Sec. 3.3:  A = A' + U V^T,  A' = A without its six wrap-around entries
 * (pentadiagonal, factored by Sec. 4.1),  U = unit columns at rows 1, 2, N-1, N,  V^T = the
 * wrap-around entries:
 *     row 1:  a_1 at column N-1, b_1 at column N        row 2:  a_2 at column N
 *     row N-1: e_{N-1} at column 1                       row N:  d_N at column 1, e_N at column 2
 *   y = A'^{-1} f,  Z = A'^{-1} U (once),  H = (I_4 + V^T Z)^{-1} (once),  x = y - Z H (V^T y).
 * Paper naming (a,b,c,d,e = offsets -2,-1,0,+1,+2), 0-based arrays.  n >= 5.
 * orc_penta_periodic_factor overwrites b..e with the factors of A' and returns Z (n x 4, row-major),
 * H (4 x 4, row-major) and w6 = (a_1, b_1, a_2, e_{N-1}, d_N, e_N).  Returns 0, a bad pivot row, or -1.
 * ---------------------------------------------------------------------------------- */
static int inv4(const double *A, double *H)
{
    double M[4][8];
    for (int i = 0; i < 4; ++i)
        for (int j = 0; j < 4; ++j) { M[i][j] = A[i * 4 + j]; M[i][4 + j] = (i == j) ? 1.0 : 0.0; }
    for (int k = 0; k < 4; ++k) {                /* Gauss-Jordan with partial pivoting   */
        int p = k;
        for (int r = k + 1; r < 4; ++r) if (fabs(M[r][k]) > fabs(M[p][k])) p = r;
        if (M[p][k] == 0.0 || !isfinite(M[p][k])) return 1;
        for (int j = 0; j < 8; ++j) { double t = M[k][j]; M[k][j] = M[p][j]; M[p][j] = t; }
        double piv = M[k][k];
        for (int j = 0; j < 8; ++j) M[k][j] /= piv;
        for (int r = 0; r < 4; ++r) if (r != k) {
            double m = M[r][k];
            for (int j = 0; j < 8; ++j) M[r][j] -= m * M[k][j];
        }
    }
    for (int i = 0; i < 4; ++i) for (int j = 0; j < 4; ++j) H[i * 4 + j] = M[i][4 + j];
    return 0;
}

ORC_API int orc_penta_periodic_factor(int n, const double *a, double *b, double *c, double *d,
                                      double *e, double *Z, double *H, double *w6)
{
    if (n < 5) return -1;
    w6[0] = a[0]; w6[1] = b[0]; w6[2] = a[1]; w6[3] = e[n - 2]; w6[4] = d[n - 1]; w6[5] = e[n - 1];
    const int rc = orc_penta_factor_general(n, a, b, c, d, e);   /* A' (never reads the corners) */
    if (rc) return rc;
    double *col = (double *)malloc((size_t)n * sizeof(double));
    const int urow[4] = {0, 1, n - 2, n - 1};
    for (int m = 0; m < 4; ++m) {                                /* Z = A'^{-1} U              */
        for (int i = 0; i < n; ++i) col[i] = 0.0;
        col[urow[m]] = 1.0;
        orc_penta_solve(n, a, b, c, d, e, col);
        for (int i = 0; i < n; ++i) Z[(size_t)i * 4 + m] = col[i];
    }
    free(col);
    double S[16];                                                /* I + V^T Z                  */
    for (int m = 0; m < 4; ++m) {
        S[0 * 4 + m] = w6[0] * Z[(size_t)(n - 2) * 4 + m] + w6[1] * Z[(size_t)(n - 1) * 4 + m];
        S[1 * 4 + m] = w6[2] * Z[(size_t)(n - 1) * 4 + m];
        S[2 * 4 + m] = w6[3] * Z[m];
        S[3 * 4 + m] = w6[4] * Z[m] + w6[5] * Z[4 + m];
    }
    for (int m = 0; m < 4; ++m) S[m * 4 + m] += 1.0;
    if (inv4(S, H)) return n;
    return 0;
}

ORC_API void orc_penta_periodic_solve(int n, const double *eps, const double *beta, const double *alpha,
                                      const double *gamma, const double *delta, const double *Z,
                                      const double *H, const double *w6, double *f)
{
    orc_penta_solve(n, eps, beta, alpha, gamma, delta, f);       /* A' y = f                   */
    double t[4], w[4];
    t[0] = w6[0] * f[n - 2] + w6[1] * f[n - 1];                  /* V^T y                      */
    t[1] = w6[2] * f[n - 1];
    t[2] = w6[3] * f[0];
    t[3] = w6[4] * f[0] + w6[5] * f[1];
    for (int i = 0; i < 4; ++i) w[i] = H[i * 4] * t[0] + H[i * 4 + 1] * t[1] + H[i * 4 + 2] * t[2] + H[i * 4 + 3] * t[3];
    for (int i = 0; i < n; ++i)                                  /* x = y - Z w                */
        f[i] = f[i] - (Z[(size_t)i * 4] * w[0] + Z[(size_t)i * 4 + 1] * w[1] + Z[(size_t)i * 4 + 2] * w[2] +
                       Z[(size_t)i * 4 + 3] * w[3]);
}

/* Explicit half of eq. 24 with PERIODIC differences (the paper's own boundary conditions,
 * PAPER.md:337, 365-392): f_i = c_i + alpha (w_{i-1} - 2 w_i + w_{i+1}), w = c^3 - c, indices mod n. */
ORC_API void orc_ch_rhs_periodic(int n, const double *c, double alpha, double *f)
{
    for (int i = 0; i < n; ++i) {
        const int im = (i + n - 1) % n, ip = (i + 1) % n;
        double wm = c[im] * c[im] * c[im] - c[im];
        double w0 = c[i] * c[i] * c[i] - c[i];
        double wp = c[ip] * c[ip] * c[ip] - c[ip];
        f[i] = c[i] + alpha * (wm - 2.0 * w0 + wp);
    }
}

/* mode 0: nsteps periodic penta solves (RHS = previous solution); mode 1: nsteps periodic CH steps. */
ORC_API int orc_penta_periodic_interleaved(int n, const double *eps, const double *beta, const double *alpha,
                                           const double *gamma, const double *delta, const double *Z,
                                           const double *H, const double *w6, double *buf, long long M,
                                           long long jlo, long long jhi, long long jstride, int mode,
                                           double alpha_x, int nsteps, int nthreads)
{
    int used = set_threads(nthreads);
#pragma omp parallel
    {
        double *col = (double *)malloc((size_t)n * sizeof(double));
        double *f = (double *)malloc((size_t)n * sizeof(double));
#pragma omp for schedule(static)
        for (long long j = jlo; j < jhi; j += jstride) {
            for (int i = 0; i < n; ++i) col[i] = buf[(size_t)i * M + j];
            for (int s = 0; s < nsteps; ++s) {
                if (mode == 1) {
                    orc_ch_rhs_periodic(n, col, alpha_x, f);
                    memcpy(col, f, (size_t)n * sizeof(double));
                }
                orc_penta_periodic_solve(n, eps, beta, alpha, gamma, delta, Z, H, w6, col);
            }
            for (int i = 0; i < n; ++i) buf[(size_t)i * M + j] = col[i];
        }
        free(col);
        free(f);
    }
    return used;
}

/* ------------------------------------------------------------------------------------
 * Coarsening statistic, PAPER.md:433-439 (eq. 30): l = 1 / (1 - <C^2>), <C^2> = (1/L) int C^2 dx,
 * evaluated on the uniform periodic grid as the mean of C_i^2 over the N points of a run, then averaged
 * over the M independent runs of the batch ("captured for each simulation ... then averaged across
 * simulations").  Serial, in index order.
 * ---------------------------------------------------------------------------------- */
ORC_API double orc_lbar_interleaved(int n, const double *c, long long M)
{
    double acc = 0.0;
    for (long long j = 0; j < M; ++j) {
        double s2 = 0.0;
        for (int i = 0; i < n; ++i) s2 += c[(size_t)i * M + j] * c[(size_t)i * M + j];
        acc += 1.0 / (1.0 - s2 / (double)n);
    }
    return acc / (double)M;
}

/* ------------------------------------------------------------------------------------
 * Crank-Nicolson diffusion step, PAPER.md:120-136 (eq. 9-11): the right-hand side is the explicit
 * three-point stencil of the previous state,
 *     f_i = xa C_{i-1} + xb C_i + xc C_{i+1}      (eq. 9: xa = xc = sigma_x, xb = 1 - 2 sigma_x),
 * followed by the tridiagonal solve with a = c = -sigma_x, b = 1 + 2 sigma_x (eq. 11).
 * periodic != 0: indices mod n and the Sherman-Morrison solve of Sec. 3.3 (the paper's setting);
 * periodic == 0: ghost values zero and the plain Thomas solve (BASELINE.json's truncated reading, C-18).
 * z / vN / den are only read in the periodic case.
 * ---------------------------------------------------------------------------------- */
ORC_API void orc_tri_explicit(int n, const double *c, double xa, double xb, double xc, int periodic, double *f)
{
    for (int i = 0; i < n; ++i) {
        double cm = (i > 0) ? c[i - 1] : (periodic ? c[n - 1] : 0.0);
        double cp = (i < n - 1) ? c[i + 1] : (periodic ? c[0] : 0.0);
        f[i] = xa * cm + xb * c[i] + xc * cp;
    }
}

ORC_API int orc_tri_cn_step_interleaved(int n, const double *a, const double *bh, const double *ch,
                                        const double *z, double vN, double den, int periodic, double xa,
                                        double xb, double xc, double *buf, long long M, long long jlo,
                                        long long jhi, long long jstride, int nsteps, int nthreads)
{
    int used = set_threads(nthreads);
#pragma omp parallel
    {
        double *col = (double *)malloc((size_t)n * sizeof(double));
        double *f = (double *)malloc((size_t)n * sizeof(double));
#pragma omp for schedule(static)
        for (long long j = jlo; j < jhi; j += jstride) {
            for (int i = 0; i < n; ++i) col[i] = buf[(size_t)i * M + j];
            for (int s = 0; s < nsteps; ++s) {
                orc_tri_explicit(n, col, xa, xb, xc, periodic, f);
                if (periodic) orc_tri_periodic_solve(n, a, bh, ch, z, vN, den, f);
                else orc_tri_solve(n, a, bh, ch, f);
                memcpy(col, f, (size_t)n * sizeof(double));
            }
            for (int i = 0; i < n; ++i) buf[(size_t)i * M + j] = col[i];
        }
        free(col);
        free(f);
    }
    return used;
}

/* ------------------------------------------------------------------------------------
 * Crank-Nicolson hyperdiffusion step, PAPER.md:284-296 (eq. 17-19): explicit five-point half
 *     f_i = x0 C_{i-2} + x1 C_{i-1} + x2 C_i + x3 C_{i+1} + x4 C_{i+2}
 * (eq. 18: x = (-s, 4s, 1 - 6s, 4s, -s), s = sigma_x) followed by the pentadiagonal solve with
 * (s, -4s, 1 + 6s, -4s, s).  periodic != 0: indices mod n and the cyclic solve (Z, H, w6 as returned by
 * orc_penta_periodic_factor); periodic == 0: ghost values zero and the plain solve [C-18].
 * ---------------------------------------------------------------------------------- */
ORC_API void orc_penta_explicit(int n, const double *c, const double *x5, int periodic, double *f)
{
    for (int i = 0; i < n; ++i) {
        double acc = 0.0;
        for (int o = -2; o <= 2; ++o) {
            int j = i + o;
            double v;
            if (j >= 0 && j < n) v = c[j];
            else v = periodic ? c[(j + n) % n] : 0.0;
            acc += x5[o + 2] * v;
        }
        f[i] = acc;
    }
}

ORC_API int orc_penta_cn_step_interleaved(int n, const double *eps, const double *beta, const double *alpha,
                                          const double *gamma, const double *delta, const double *Z,
                                          const double *H, const double *w6, int periodic, const double *x5,
                                          double *buf, long long M, long long jlo, long long jhi,
                                          long long jstride, int nsteps, int nthreads)
{
    int used = set_threads(nthreads);
#pragma omp parallel
    {
        double *col = (double *)malloc((size_t)n * sizeof(double));
        double *f = (double *)malloc((size_t)n * sizeof(double));
#pragma omp for schedule(static)
        for (long long j = jlo; j < jhi; j += jstride) {
            for (int i = 0; i < n; ++i) col[i] = buf[(size_t)i * M + j];
            for (int s = 0; s < nsteps; ++s) {
                orc_penta_explicit(n, col, x5, periodic, f);
                if (periodic) orc_penta_periodic_solve(n, eps, beta, alpha, gamma, delta, Z, H, w6, f);
                else orc_penta_solve(n, eps, beta, alpha, gamma, delta, f);
                memcpy(col, f, (size_t)n * sizeof(double));
            }
            for (int i = 0; i < n; ++i) buf[(size_t)i * M + j] = col[i];
        }
        free(col);
        free(f);
    }
    return used;
}
