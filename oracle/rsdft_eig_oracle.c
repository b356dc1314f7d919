/*
 * oracle/rsdft_eig_oracle.c -- TEST INFRASTRUCTURE ONLY.
 *
 * Plain, slow, obviously-correct CPU restatement of the generalized Hermitian eigen-solve of the
 * LOBPCG subspace pencil by the paper's route (arXiv 2512.04447, eq. 1):
 *
 *     H X = lambda S X,   S = L L^dagger (Cholesky),
 *     K Z = lambda Z,     K = L^-1 H (L^dagger)^-1,     Z = L^dagger X            (eq. 1)
 *
 * "The transformation H -> K is normally handled by (P)ZHEGST, but the same operation can be
 * performed by two calls to (P)ZTRSM": K is formed here by two plain triangular
 * substitutions, the standard problem is solved by the classical cyclic Jacobi method (the paper
 * calls (P)ZHEEVD there; the eigen-decomposition it reaches is unique up to phases / rotations
 * inside degenerate eigenspaces, so any convergent method is the same definition), and the
 * eigenvectors go back through X = (L^dagger)^-1 Z.  SURVEY.md 8(f) NEXT-1.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * build, link or call this file.  It shares no code, header, table or constant generator with
 * paper_2512_04447_b200/csrc (the CUDA path).
 *
 * Arithmetic: long double throughout, rounded to double once on output.  Matrices are n x n
 * complex128, column-major, element (i, j) at i + j*ld (the layout rsdft_subspace_gram writes).
 *
 * Pin status (tests/test_oracle_eig_pins.py, -m "not gpu"):
 *   orc_potrf     pinned: L lower with real positive diagonal and L L^dagger = S (the factor is
 *                 unique); 2x2 closed form; numpy.linalg.cholesky as the library cross-check.
 *   orc_reduce    pinned: L K L^dagger = H; K Hermitian; eigenvalues of K = generalized
 *                 eigenvalues of (H, S) from scipy.linalg.eigh (eq. 1's identity).
 *   orc_jacobi    pinned: 2x2 closed form; K = Q diag(w) Q^dagger with a prescribed spectrum
 *                 (incl. degenerate levels); Z^dagger Z = I; K Z = Z diag(w); numpy.linalg.eigvalsh.
 *   orc_backsolve pinned: L^dagger C = Z.
 *   orc_subspace_eig  pinned: pencil built from a prescribed spectrum (H = B^dagger diag(w) B,
 *                 S = B^dagger B); C^dagger S C = I; H C = S C diag(w); free-electron levels
 *                 (tests/golden/free_electron_levels.txt) through apply_h -> gram -> eig.
 */
#define _GNU_SOURCE
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef struct { long double re, im; } cld;

static inline cld c_mul(cld a, cld b) { cld r = { a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re }; return r; }
static inline cld c_mulc(cld a, cld b) { cld r = { a.re * b.re + a.im * b.im, a.im * b.re - a.re * b.im }; return r; } /* a * conj(b) */
static inline cld c_cmul(cld a, cld b) { cld r = { a.re * b.re + a.im * b.im, a.re * b.im - a.im * b.re }; return r; } /* conj(a) * b */

#define AT(M, i, j, n) (M)[(size_t)(i) + (size_t)(j) * (size_t)(n)]

static cld *load(int n, const double *A, int ld)
{
    cld *M = (cld *)malloc(sizeof(cld) * (size_t)n * (size_t)n);
    if (!M) return NULL;
    for (int j = 0; j < n; ++j)
        for (int i = 0; i < n; ++i) {
            AT(M, i, j, n).re = A[2 * ((size_t)i + (size_t)j * ld)];
            AT(M, i, j, n).im = A[2 * ((size_t)i + (size_t)j * ld) + 1];
        }
    return M;
}

static void store(int rows, int cols, const cld *M, int ldm, double *A, int ld)
{
    for (int j = 0; j < cols; ++j)
        for (int i = 0; i < rows; ++i) {
            A[2 * ((size_t)i + (size_t)j * ld)] = (double)M[(size_t)i + (size_t)j * ldm].re;
            A[2 * ((size_t)i + (size_t)j * ld) + 1] = (double)M[(size_t)i + (size_t)j * ldm].im;
        }
}

/* S = L L^dagger, L lower triangular with real positive diagonal ("Cholesky
 * factorization S = L L^dagger").  Column by column (Cholesky-Crout):
 *   L_jj = sqrt(S_jj - sum_{k<j} |L_jk|^2),  L_ij = (S_ij - sum_{k<j} L_ik conj(L_jk)) / L_jj, i > j.
 * Only the lower triangle of S is read.  Returns j+1 if the j-th pivot is not positive.        */
static int potrf_ld(int n, const cld *S, cld *L)
{
    memset(L, 0, sizeof(cld) * (size_t)n * (size_t)n);
    for (int j = 0; j < n; ++j) {
        long double d = AT(S, j, j, n).re;
        for (int k = 0; k < j; ++k) d -= AT(L, j, k, n).re * AT(L, j, k, n).re + AT(L, j, k, n).im * AT(L, j, k, n).im;
        if (!(d > 0.0L)) return j + 1;
        const long double ljj = sqrtl(d);
        AT(L, j, j, n).re = ljj;
        AT(L, j, j, n).im = 0.0L;
#pragma omp parallel for schedule(static) if (n - j > 64)
        for (int i = j + 1; i < n; ++i) {
            cld s = AT(S, i, j, n);
            for (int k = 0; k < j; ++k) {
                const cld t = c_mulc(AT(L, i, k, n), AT(L, j, k, n));
                s.re -= t.re; s.im -= t.im;
            }
            AT(L, i, j, n).re = s.re / ljj;
            AT(L, i, j, n).im = s.im / ljj;
        }
    }
    return 0;
}

/* K = L^-1 H (L^dagger)^-1 by two triangular substitutions ("two calls to (P)ZTRSM,
 * which solves Y from AY = B"):
 *   (1) L Z = H          forward substitution, column by column of H
 *   (2) K L^dagger = Z   row by row:  K_ij = (Z_ij - sum_{k<j} K_ik conj(L_jk)) / L_jj             */
static void reduce_ld(int n, const cld *H, const cld *L, cld *K)
{
    cld *Z = (cld *)malloc(sizeof(cld) * (size_t)n * (size_t)n);
#pragma omp parallel for schedule(static)
    for (int j = 0; j < n; ++j)
        for (int i = 0; i < n; ++i) {
            cld s = AT(H, i, j, n);
            for (int k = 0; k < i; ++k) {
                const cld t = c_mul(AT(L, i, k, n), AT(Z, k, j, n));
                s.re -= t.re; s.im -= t.im;
            }
            AT(Z, i, j, n).re = s.re / AT(L, i, i, n).re;
            AT(Z, i, j, n).im = s.im / AT(L, i, i, n).re;
        }
#pragma omp parallel for schedule(static)
    for (int i = 0; i < n; ++i)
        for (int j = 0; j < n; ++j) {
            cld s = AT(Z, i, j, n);
            for (int k = 0; k < j; ++k) {
                const cld t = c_mulc(AT(K, i, k, n), AT(L, j, k, n));
                s.re -= t.re; s.im -= t.im;
            }
            AT(K, i, j, n).re = s.re / AT(L, j, j, n).re;
            AT(K, i, j, n).im = s.im / AT(L, j, j, n).re;
        }
    free(Z);
}

/* Classical cyclic-by-row Jacobi for a Hermitian matrix (the standard problem K Z = lambda Z of
 * eq. 1).  For each p < q with a_pq = r e^{i phi}, r > 0:
 *   tau = (a_qq - a_pp) / (2 r),  t = sign(tau) / (|tau| + sqrt(1 + tau^2)),  c = 1/sqrt(1 + t^2),  s = t c,
 *   J = [[c, s], [-s e^{-i phi}, c e^{-i phi}]] on rows/columns (p, q),   A <- J^dagger A J,  V <- V J,
 * which zeroes a_pq.  Sweeps repeat until sum_{p<q} |a_pq|^2 <= (1e-19 ||A||_F)^2 (long double) or
 * 60 sweeps.  A is overwritten (its diagonal ends as the eigenvalues); V receives the eigenvectors. */
static int jacobi_ld(int n, cld *A, cld *V)
{
    for (int j = 0; j < n; ++j)
        for (int i = 0; i < n; ++i) { AT(V, i, j, n).re = (i == j) ? 1.0L : 0.0L; AT(V, i, j, n).im = 0.0L; }
    long double fro = 0.0L;
    for (size_t e = 0; e < (size_t)n * n; ++e) fro += A[e].re * A[e].re + A[e].im * A[e].im;
    const long double tol2 = fro * 1e-38L;
    int sweep = 0;
    for (; sweep < 60; ++sweep) {
        long double off = 0.0L;
        for (int q = 1; q < n; ++q)
            for (int p = 0; p < q; ++p) off += AT(A, p, q, n).re * AT(A, p, q, n).re + AT(A, p, q, n).im * AT(A, p, q, n).im;
        if (off <= tol2) break;
        for (int p = 0; p < n - 1; ++p)
            for (int q = p + 1; q < n; ++q) {
                const cld apq = AT(A, p, q, n);
                const long double r = sqrtl(apq.re * apq.re + apq.im * apq.im);
                if (r == 0.0L) continue;
                const long double tau = (AT(A, q, q, n).re - AT(A, p, p, n).re) / (2.0L * r);
                const long double t = (tau >= 0.0L ? 1.0L : -1.0L) / (fabsl(tau) + sqrtl(1.0L + tau * tau));
                const long double c = 1.0L / sqrtl(1.0L + t * t), s = t * c;
                const cld em = { apq.re / r, -apq.im / r };               /* e^{-i phi} */
                const cld Jpp = { c, 0.0L }, Jpq = { s, 0.0L };
                const cld Jqp = { -s * em.re, -s * em.im }, Jqq = { c * em.re, c * em.im };
                /* columns: A <- A J, V <- V J */
                for (int i = 0; i < n; ++i) {
                    const cld aip = AT(A, i, p, n), aiq = AT(A, i, q, n);
                    cld u = c_mul(aip, Jpp), v = c_mul(aiq, Jqp);
                    AT(A, i, p, n).re = u.re + v.re; AT(A, i, p, n).im = u.im + v.im;
                    u = c_mul(aip, Jpq); v = c_mul(aiq, Jqq);
                    AT(A, i, q, n).re = u.re + v.re; AT(A, i, q, n).im = u.im + v.im;
                    const cld vip = AT(V, i, p, n), viq = AT(V, i, q, n);
                    u = c_mul(vip, Jpp); v = c_mul(viq, Jqp);
                    AT(V, i, p, n).re = u.re + v.re; AT(V, i, p, n).im = u.im + v.im;
                    u = c_mul(vip, Jpq); v = c_mul(viq, Jqq);
                    AT(V, i, q, n).re = u.re + v.re; AT(V, i, q, n).im = u.im + v.im;
                }
                /* rows: A <- J^dagger A */
                for (int j = 0; j < n; ++j) {
                    const cld apj = AT(A, p, j, n), aqj = AT(A, q, j, n);
                    cld u = c_cmul(Jpp, apj), v = c_cmul(Jqp, aqj);
                    AT(A, p, j, n).re = u.re + v.re; AT(A, p, j, n).im = u.im + v.im;
                    u = c_cmul(Jpq, apj); v = c_cmul(Jqq, aqj);
                    AT(A, q, j, n).re = u.re + v.re; AT(A, q, j, n).im = u.im + v.im;
                }
                /* the pivot is zero and the diagonal real by construction; clean the round-off */
                AT(A, p, q, n).re = AT(A, p, q, n).im = 0.0L;
                AT(A, q, p, n).re = AT(A, q, p, n).im = 0.0L;
                AT(A, p, p, n).im = 0.0L;
                AT(A, q, q, n).im = 0.0L;
            }
    }
    return sweep;
}

/* C = (L^dagger)^-1 Z (eq. 1: Z = L^dagger X), back substitution, column by column:
 *   C_ij = (Z_ij - sum_{k>i} conj(L_ki) C_kj) / L_ii,  i = n-1 .. 0.                              */
static void backsolve_ld(int n, int m, const cld *L, const cld *Z, cld *C)
{
#pragma omp parallel for schedule(static)
    for (int j = 0; j < m; ++j)
        for (int i = n - 1; i >= 0; --i) {
            cld s = AT(Z, i, j, n);
            for (int k = i + 1; k < n; ++k) {
                const cld t = c_cmul(AT(L, k, i, n), AT(C, k, j, n));
                s.re -= t.re; s.im -= t.im;
            }
            AT(C, i, j, n).re = s.re / AT(L, i, i, n).re;
            AT(C, i, j, n).im = s.im / AT(L, i, i, n).re;
        }
}

/* ---- exported pieces (each can be pinned on its own) ------------------------------------- */

int orc_potrf(int32_t n, const double *S, int32_t lds, double *L, int32_t ldl)
{
    cld *Sm = load(n, S, lds), *Lm = (cld *)malloc(sizeof(cld) * (size_t)n * n);
    if (!Sm || !Lm) return -1;
    const int rc = potrf_ld(n, Sm, Lm);
    if (rc == 0) store(n, n, Lm, n, L, ldl);
    free(Sm); free(Lm);
    return rc;
}

int orc_reduce(int32_t n, const double *H, int32_t ldh, const double *S, int32_t lds, double *K, int32_t ldk)
{
    cld *Hm = load(n, H, ldh), *Sm = load(n, S, lds);
    cld *Lm = (cld *)malloc(sizeof(cld) * (size_t)n * n), *Km = (cld *)malloc(sizeof(cld) * (size_t)n * n);
    if (!Hm || !Sm || !Lm || !Km) return -1;
    const int rc = potrf_ld(n, Sm, Lm);
    if (rc == 0) { reduce_ld(n, Hm, Lm, Km); store(n, n, Km, n, K, ldk); }
    free(Hm); free(Sm); free(Lm); free(Km);
    return rc;
}

static int cmp_idx(const void *a, const void *b, void *w)
{
    const long double *ww = (const long double *)w;
    const int ia = *(const int *)a, ib = *(const int *)b;
    if (ww[ia] < ww[ib]) return -1;
    if (ww[ia] > ww[ib]) return 1;
    return ia - ib;
}

/* eigen-decomposition of a Hermitian K (lower + upper both read): w ascending, Z columns */
int orc_jacobi(int32_t n, const double *K, int32_t ldk, double *w, double *Z, int32_t ldz)
{
    cld *A = load(n, K, ldk), *V = (cld *)malloc(sizeof(cld) * (size_t)n * n);
    long double *ev = (long double *)malloc(sizeof(long double) * (size_t)n);
    int *ord = (int *)malloc(sizeof(int) * (size_t)n);
    if (!A || !V || !ev || !ord) return -1;
    const int sweeps = jacobi_ld(n, A, V);
    for (int i = 0; i < n; ++i) { ev[i] = AT(A, i, i, n).re; ord[i] = i; }
    qsort_r(ord, (size_t)n, sizeof(int), cmp_idx, ev);
    for (int j = 0; j < n; ++j) {
        w[j] = (double)ev[ord[j]];
        store(n, 1, V + (size_t)ord[j] * n, n, Z + 2 * (size_t)j * ldz, ldz);
    }
    free(A); free(V); free(ev); free(ord);
    return sweeps;
}

int orc_backsolve(int32_t n, int32_t m, const double *L, int32_t ldl, const double *Z, int32_t ldz, double *C, int32_t ldc)
{
    cld *Lm = load(n, L, ldl);
    cld *Zm = (cld *)malloc(sizeof(cld) * (size_t)n * m), *Cm = (cld *)malloc(sizeof(cld) * (size_t)n * m);
    if (!Lm || !Zm || !Cm) return -1;
    for (int j = 0; j < m; ++j)
        for (int i = 0; i < n; ++i) {
            Zm[(size_t)i + (size_t)j * n].re = Z[2 * ((size_t)i + (size_t)j * ldz)];
            Zm[(size_t)i + (size_t)j * n].im = Z[2 * ((size_t)i + (size_t)j * ldz) + 1];
        }
    backsolve_ld(n, m, Lm, Zm, Cm);
    store(n, m, Cm, n, C, ldc);
    free(Lm); free(Zm); free(Cm);
    return 0;
}

/* The whole of eq. 1 in the paper's order, intermediate results kept in long double:
 * Cholesky -> two substitutions -> Jacobi -> sort ascending -> back substitution of the m lowest.
 * Outputs: lambda[m]; C n x m (column j = generalized eigenvector j, C^dagger S C = I);
 * optional L (n x n lower) and K (n x n).  Returns 0, or j+1 if S is not positive definite.    */
int orc_subspace_eig(int32_t n, const double *H, int32_t ldh, const double *S, int32_t lds, int32_t m,
                     double *lambda, double *C, int32_t ldc, double *L_out, double *K_out, int32_t ldo)
{
    cld *Hm = load(n, H, ldh), *Sm = load(n, S, lds);
    cld *Lm = (cld *)malloc(sizeof(cld) * (size_t)n * n), *Km = (cld *)malloc(sizeof(cld) * (size_t)n * n);
    cld *V = (cld *)malloc(sizeof(cld) * (size_t)n * n), *Zs = (cld *)malloc(sizeof(cld) * (size_t)n * m);
    cld *Cm = (cld *)malloc(sizeof(cld) * (size_t)n * m);
    long double *ev = (long double *)malloc(sizeof(long double) * (size_t)n);
    int *ord = (int *)malloc(sizeof(int) * (size_t)n);
    if (!Hm || !Sm || !Lm || !Km || !V || !Zs || !Cm || !ev || !ord) return -1;
    int rc = potrf_ld(n, Sm, Lm);
    if (rc == 0) {
        reduce_ld(n, Hm, Lm, Km);
        if (L_out) store(n, n, Lm, n, L_out, ldo);
        if (K_out) store(n, n, Km, n, K_out, ldo);
        /* K is Hermitian in exact arithmetic; Jacobi reads it as (K + K^dagger)/2 */
        for (int j = 0; j < n; ++j)
            for (int i = 0; i <= j; ++i) {
                const long double re = 0.5L * (AT(Km, i, j, n).re + AT(Km, j, i, n).re);
                const long double im = 0.5L * (AT(Km, i, j, n).im - AT(Km, j, i, n).im);
                AT(Km, i, j, n).re = re; AT(Km, i, j, n).im = (i == j) ? 0.0L : im;
                AT(Km, j, i, n).re = re; AT(Km, j, i, n).im = (i == j) ? 0.0L : -im;
            }
        jacobi_ld(n, Km, V);
        for (int i = 0; i < n; ++i) { ev[i] = AT(Km, i, i, n).re; ord[i] = i; }
        qsort_r(ord, (size_t)n, sizeof(int), cmp_idx, ev);
        for (int j = 0; j < m; ++j) {
            lambda[j] = (double)ev[ord[j]];
            memcpy(Zs + (size_t)j * n, V + (size_t)ord[j] * n, sizeof(cld) * (size_t)n);
        }
        backsolve_ld(n, m, Lm, Zs, Cm);
        store(n, m, Cm, n, C, ldc);
    }
    free(Hm); free(Sm); free(Lm); free(Km); free(V); free(Zs); free(Cm); free(ev); free(ord);
    return rc;
}
