/*
 * oracle/rsdft_oracle.c -- TEST INFRASTRUCTURE ONLY.
 *
 * Plain, slow, obviously-correct CPU restatement of the hot path of one LOBPCG
 * block step of real-space DFT (arXiv 2512.04447, PAPER.md:19 -- tasks (1) FFT
 * Laplacian, (2) H/S matrices, (4) nonlocal pseudopotential operator; the
 * problem statement is BASELINE.json north_star / configs, readings in
 * SURVEY.md section 8(c) and DESIGN.md "Readings").
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
 * reference legs may build, link or call this file.  It shares no code, header,
 * table or constant generator with paper_2512_04447_b200/csrc (the CUDA path).
 *
 * Arithmetic: every sum (DFT butterflies, projector sums, Gram sums) is carried
 * in long double (x87 80-bit, 64-bit mantissa) and rounded to double once, so the
 * oracle's own round-off (~1e-19 per op) is negligible beside the 1e-12 parity
 * budget.  Twiddles come from cosl/sinl.
 *
 * Pin status (tests/test_oracle_pins.py, all run with -m "not gpu"):
 *   orc_fft3d        pinned: brute-force O(Ng^2) DFT definition on 16^3 written in
 *                    the test, numpy.fft.fftn, delta->constant, Parseval, inverse.
 *   orc_kinetic      pinned: plane-wave eigenpairs |G|^2/2 (north_star), incl.
 *                    Nyquist and negative frequencies; paper's cut-offs 86.7/110.7 Ry
 *                     fix Hartree units.
 *   orc_apply_h      pinned: cosine-potential closed form; <x|Hy>=conj<y|Hx>;
 *                    translation covariance; energy identity; outside-sphere null.
 *   orc_sphere       pinned: dense all-grid numpy construction in the test; cubic
 *                    symmetry orthogonality; continuum integral (loose).
 *   orc_gram         pinned: plane waves -> Ng*I / Ng*diag(t); free-electron Ritz
 *                    values (north_star); Hermiticity / positive definiteness.
 *   Numerical values of H*psi for a physical system: parity unpinned -- the paper
 *   prints no worked example (PAPER.md has only figures), see DESIGN.md.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct { long double re, im; } cld;

typedef struct {
    double rc;            /* cut-off radius, bohr: member iff |d|^2 < rc^2 (strict) */
    int32_t nproj;        /* projectors of this species */
    const int32_t *l;     /* [nproj] 0..2 */
    const int32_t *m;     /* [nproj] -l..l, real spherical harmonics */
    int32_t radial_kind;  /* 0: exp(-alpha[i] r^2); 1: table, linear interpolation */
    const double *alpha;  /* [nproj] (kind 0) */
    int32_t nr;           /* table length (kind 1) */
    double dr;            /* table spacing (kind 1) */
    const double *radial; /* [nproj][nr] (kind 1) */
    const double *D;      /* [nproj][nproj] real symmetric, Hartree */
} orc_species;

#define ORC_PI 3.14159265358979323846264338327950288L

int orc_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ------------------------------------------------------------------------- */
/* 1-D DFT.  Definition (SURVEY 8(c) reading 1): forward  X[k] = sum_j x[j] e^{-2 pi i jk/n},
 * inverse the same with e^{+...} (the 1/Ng is applied by the caller).
 * n <= 16 or n odd : the definition, O(n^2).
 * n even, > 16     : textbook radix-2 decimation in time, recursing until the
 *                    length is <= 16 or odd (north_star: "direct O(N^2) DFT on tiny
 *                    grids and radix-2 FFT otherwise"; 48, 96, 112 end in direct
 *                    DFTs of length 12/3, 12/3, 14/7 -> DESIGN.md reading R2).
 * W is the table exp(sign 2 pi i m / ntop), m = 0..ntop-1, of the top-level length;
 * a sub-transform of length n uses W[m * (ntop / n)].                          */
static void dft_rec(int n, int ntop, const cld *W, const cld *in, int stride, cld *out, cld *work)
{
    if (n <= 16 || (n & 1)) {
        int step = ntop / n;
        for (int k = 0; k < n; ++k) {
            long double sr = 0.0L, si = 0.0L;
            for (int j = 0; j < n; ++j) {
                const cld w = W[(int)(((long)j * k) % n) * step];
                const cld x = in[(long)j * stride];
                sr += x.re * w.re - x.im * w.im;
                si += x.re * w.im + x.im * w.re;
            }
            out[k].re = sr; out[k].im = si;
        }
        return;
    }
    int h = n / 2, step = ntop / n;
    cld *E = work, *O = work + h;
    dft_rec(h, ntop, W, in, 2 * stride, E, work + n);
    dft_rec(h, ntop, W, in + stride, 2 * stride, O, work + n);
    for (int k = 0; k < h; ++k) {
        const cld w = W[k * step];
        long double tr = O[k].re * w.re - O[k].im * w.im;
        long double ti = O[k].re * w.im + O[k].im * w.re;
        out[k].re = E[k].re + tr;     out[k].im = E[k].im + ti;
        out[k + h].re = E[k].re - tr; out[k + h].im = E[k].im - ti;
    }
}

static cld *twiddle_table(int n, int sign)
{
    cld *W = (cld *)malloc(sizeof(cld) * (size_t)n);
    for (int m = 0; m < n; ++m) {
        long double a = 2.0L * ORC_PI * (long double)m / (long double)n;
        W[m].re = cosl(a);
        W[m].im = (sign < 0 ? -1.0L : 1.0L) * sinl(a);
    }
    return W;
}

/* In-place separable 3-D DFT of one column held in long double.
 * Index g = (ix*ny + iy)*nz + iz (z fastest), SURVEY 8 notation.            */
static void fft3d_ld(const int n[3], cld *A, int sign)
{
    const long nx = n[0], ny = n[1], nz = n[2];
    const long strides[3] = { ny * nz, nz, 1 };
    for (int ax = 2; ax >= 0; --ax) {
        const int len = n[ax];
        cld *W = twiddle_table(len, sign);
        cld *out = (cld *)malloc(sizeof(cld) * (size_t)len);
        cld *work = (cld *)malloc(sizeof(cld) * (size_t)len * 2 + 64);
        const long s = strides[ax];
        for (long ix = 0; ix < (ax == 0 ? 1 : nx); ++ix)
            for (long iy = 0; iy < (ax == 1 ? 1 : ny); ++iy)
                for (long iz = 0; iz < (ax == 2 ? 1 : nz); ++iz) {
                    cld *line = A + (ix * ny + iy) * nz + iz;
                    dft_rec(len, len, W, line, (int)s, out, work);
                    for (int k = 0; k < len; ++k) line[(long)k * s] = out[k];
                }
        free(W); free(out); free(work);
    }
}

/* Forward (sign=-1, unnormalised) or inverse (sign=+1, divided by Ng) 3-D DFT of
 * ncol columns of complex128; out may alias in.                              */
int orc_fft3d(const int32_t n[3], int sign, int ncol, const double *in, int64_t ldin,
              double *out, int64_t ldout)
{
    const int nn[3] = { n[0], n[1], n[2] };
    const long ng = (long)n[0] * n[1] * n[2];
    int fail = 0;
#pragma omp parallel for schedule(dynamic, 1)
    for (int c = 0; c < ncol; ++c) {
        cld *A = (cld *)malloc(sizeof(cld) * (size_t)ng);
        if (!A) { fail = 1; continue; }
        const double *x = in + 2 * (long)c * ldin;
        for (long g = 0; g < ng; ++g) { A[g].re = x[2 * g]; A[g].im = x[2 * g + 1]; }
        fft3d_ld(nn, A, sign);
        double *y = out + 2 * (long)c * ldout;
        const long double sc = sign > 0 ? 1.0L / (long double)ng : 1.0L;
        for (long g = 0; g < ng; ++g) { y[2 * g] = (double)(A[g].re * sc); y[2 * g + 1] = (double)(A[g].im * sc); }
        free(A);
    }
    return fail ? -1 : 0;
}

/* kappa(j) = j for j < N/2, j - N otherwise (BASELINE.json configs[0]: "FFT index j
 * maps to j for j < N/2 and to j - N otherwise").                              */
static long kappa(long j, long n) { return (2 * j < n) ? j : j - n; }

/* t(k) = 1/2 sum_a (2 pi kappa_a / L_a)^2, Hartree (SURVEY 8(c) reading 3).   */
static long double kin_t(const int n[3], const double len[3], long kx, long ky, long kz)
{
    long double gx = 2.0L * ORC_PI * (long double)kappa(kx, n[0]) / (long double)len[0];
    long double gy = 2.0L * ORC_PI * (long double)kappa(ky, n[1]) / (long double)len[1];
    long double gz = 2.0L * ORC_PI * (long double)kappa(kz, n[2]) / (long double)len[2];
    return 0.5L * (gx * gx + gy * gy + gz * gz);
}

/* Writes t(k) for every FFT index triple, [Ng] doubles, index (kx*ny+ky)*nz+kz. */
int orc_kinetic_table(const int32_t n[3], const double len[3], double *t)
{
    const int nn[3] = { n[0], n[1], n[2] };
    for (long kx = 0; kx < n[0]; ++kx)
        for (long ky = 0; ky < n[1]; ++ky)
            for (long kz = 0; kz < n[2]; ++kz)
                t[(kx * n[1] + ky) * n[2] + kz] = (double)kin_t(nn, len, kx, ky, kz);
    return 0;
}

/* ------------------------------------------------------------------------- */
/* Real spherical harmonics, orthonormal on the unit sphere (SURVEY 8(c) readings 7, 8).
 * At |d| = 0: Y00 as usual, 0 for l > 0.                                      */
static long double ylm_real(int l, int m, long double x, long double y, long double z)
{
    const long double r2 = x * x + y * y + z * z;
    if (l == 0) return 0.5L * sqrtl(1.0L / ORC_PI);
    if (r2 == 0.0L) return 0.0L;
    const long double r = sqrtl(r2);
    if (l == 1) {
        const long double c = sqrtl(3.0L / (4.0L * ORC_PI));
        if (m == -1) return c * y / r;
        if (m == 0)  return c * z / r;
        return c * x / r;
    }
    /* l == 2 */
    const long double c15 = sqrtl(15.0L / ORC_PI), c5 = sqrtl(5.0L / ORC_PI);
    switch (m) {
    case -2: return 0.5L * c15 * x * y / r2;
    case -1: return 0.5L * c15 * y * z / r2;
    case 0:  return 0.25L * c5 * (3.0L * z * z - r2) / r2;
    case 1:  return 0.5L * c15 * x * z / r2;
    default: return 0.25L * c15 * (x * x - y * y) / r2;
    }
}

static long double radial_f(const orc_species *sp, int i, long double r)
{
    if (sp->radial_kind == 0) return expl(-(long double)sp->alpha[i] * r * r);
    /* kind 1: linear interpolation of radial[i][0..nr-1] sampled at j*dr;
     * f = 0 for r >= (nr-1)*dr (beyond the table)                               */
    long double u = r / (long double)sp->dr;
    long j = (long)floorl(u);
    if (j >= sp->nr - 1) return 0.0L;
    long double f = u - (long double)j;
    const double *tab = sp->radial + (long)i * sp->nr;
    return (long double)tab[j] + f * ((long double)tab[j + 1] - (long double)tab[j]);
}

/* Minimum-image displacement component, SURVEY 8(c) reading 5:
 * d = (r - R) - L * round((r - R)/L), evaluated in double like the plan does
 * (membership must agree point for point; the generator asserts no point is
 * within 1e-9 of the boundary).                                               */
static double min_image(double r, double R, double L)
{
    double d = r - R;
    return d - L * nearbyint(d / L);
}

/* Sphere of one atom by scanning ALL grid points (no bounding box): returns the
 * count; if idx/beta are non-NULL fills idx[count] (grid index g) and
 * beta[nproj][cap] (beta_i(r) = f_i(|d|) Y_lm(d/|d|)), at most cap points.      */
int64_t orc_sphere(const int32_t n[3], const double len[3], const double R[3],
                   const orc_species *sp, int64_t cap, int32_t *idx, double *beta)
{
    const double h[3] = { len[0] / n[0], len[1] / n[1], len[2] / n[2] };
    const double rc2 = sp->rc * sp->rc;
    int64_t cnt = 0;
    for (long ix = 0; ix < n[0]; ++ix)
        for (long iy = 0; iy < n[1]; ++iy)
            for (long iz = 0; iz < n[2]; ++iz) {
                const double dx = min_image(ix * h[0], R[0], len[0]);
                const double dy = min_image(iy * h[1], R[1], len[1]);
                const double dz = min_image(iz * h[2], R[2], len[2]);
                const double d2 = dx * dx + dy * dy + dz * dz;
                if (!(d2 < rc2)) continue;
                if (idx && cnt < cap) {
                    idx[cnt] = (int32_t)((ix * n[1] + iy) * n[2] + iz);
                    const long double r = sqrtl((long double)dx * dx + (long double)dy * dy + (long double)dz * dz);
                    for (int i = 0; i < sp->nproj; ++i)
                        beta[(long)i * cap + cnt] =
                            (double)(radial_f(sp, i, r) * ylm_real(sp->l[i], sp->m[i], dx, dy, dz));
                }
                ++cnt;
            }
    return cnt;
}

/* ------------------------------------------------------------------------- */
/* HX = (T + V_loc + V_NL) X, column by column, in the order of SURVEY 8(c):
 * 1 forward DFT, 2 multiply t(k), 3 inverse DFT / Ng, 4 + v(r) psi(r),
 * 5 for each atom p_i = dV sum_{S_a} beta_i psi ; HX(r) += sum_ij beta_i(r) D_ij p_j.
 * vloc may be NULL (= 0); natom may be 0.  p_out (optional) receives the
 * projections, [natom][maxproj][ncol] complex128, maxproj = max nproj over species. */
int orc_apply_h(const int32_t n[3], const double len[3],
                int32_t natom, const double *pos, const int32_t *species_of,
                int32_t nspecies, const orc_species *species, const double *vloc,
                int32_t ncol, const double *X, int64_t ldx, double *HX, int64_t ldhx,
                double *p_out)
{
    const int nn[3] = { n[0], n[1], n[2] };
    const long ng = (long)n[0] * n[1] * n[2];
    const long double dV = ((long double)len[0] / n[0]) * ((long double)len[1] / n[1]) * ((long double)len[2] / n[2]);
    int maxproj = 0;
    for (int s = 0; s < nspecies; ++s) if (species[s].nproj > maxproj) maxproj = species[s].nproj;

    /* sphere lists, built once (they do not depend on the column) */
    int64_t *cnt = (int64_t *)calloc((size_t)(natom > 0 ? natom : 1), sizeof(int64_t));
    int32_t **idx = (int32_t **)calloc((size_t)(natom > 0 ? natom : 1), sizeof(int32_t *));
    double **beta = (double **)calloc((size_t)(natom > 0 ? natom : 1), sizeof(double *));
#pragma omp parallel for schedule(dynamic, 1)
    for (int a = 0; a < natom; ++a) {
        const orc_species *sp = &species[species_of[a]];
        cnt[a] = orc_sphere(n, len, pos + 3 * a, sp, 0, NULL, NULL);
        idx[a] = (int32_t *)malloc(sizeof(int32_t) * (size_t)(cnt[a] + 1));
        beta[a] = (double *)malloc(sizeof(double) * (size_t)(cnt[a] + 1) * (size_t)sp->nproj);
        orc_sphere(n, len, pos + 3 * a, sp, cnt[a], idx[a], beta[a]);
    }

    int fail = 0;
#pragma omp parallel for schedule(dynamic, 1)
    for (int c = 0; c < ncol; ++c) {
        cld *A = (cld *)malloc(sizeof(cld) * (size_t)ng);
        if (!A) { fail = 1; continue; }
        const double *x = X + 2 * (long)c * ldx;
        double *y = HX + 2 * (long)c * ldhx;
        for (long g = 0; g < ng; ++g) { A[g].re = x[2 * g]; A[g].im = x[2 * g + 1]; }
        fft3d_ld(nn, A, -1);                                          /* step 1 */
        for (long kx = 0; kx < n[0]; ++kx)                            /* step 2 */
            for (long ky = 0; ky < n[1]; ++ky)
                for (long kz = 0; kz < n[2]; ++kz) {
                    const long double t = kin_t(nn, len, kx, ky, kz);
                    cld *a = &A[(kx * n[1] + ky) * n[2] + kz];
                    a->re *= t; a->im *= t;
                }
        fft3d_ld(nn, A, +1);                                          /* step 3 */
        const long double inv = 1.0L / (long double)ng;
        for (long g = 0; g < ng; ++g) {                               /* step 4 */
            const long double v = vloc ? (long double)vloc[g] : 0.0L;
            A[g].re = A[g].re * inv + v * (long double)x[2 * g];
            A[g].im = A[g].im * inv + v * (long double)x[2 * g + 1];
        }
        for (int a = 0; a < natom; ++a) {                             /* step 5 */
            const orc_species *sp = &species[species_of[a]];
            const int np = sp->nproj;
            cld p[16], q[16];
            for (int i = 0; i < np; ++i) {
                long double sr = 0.0L, si = 0.0L;
                const double *b = beta[a] + (long)i * cnt[a];
                for (long s = 0; s < cnt[a]; ++s) {
                    const long g = idx[a][s];
                    sr += (long double)b[s] * (long double)x[2 * g];
                    si += (long double)b[s] * (long double)x[2 * g + 1];
                }
                p[i].re = dV * sr; p[i].im = dV * si;
                if (p_out) {
                    double *po = p_out + 2 * (((long)a * maxproj + i) * ncol + c);
                    po[0] = (double)p[i].re; po[1] = (double)p[i].im;
                }
            }
            for (int i = 0; i < np; ++i) {
                long double sr = 0.0L, si = 0.0L;
                for (int j = 0; j < np; ++j) {
                    sr += (long double)sp->D[i * np + j] * p[j].re;
                    si += (long double)sp->D[i * np + j] * p[j].im;
                }
                q[i].re = sr; q[i].im = si;
            }
            for (long s = 0; s < cnt[a]; ++s) {
                const long g = idx[a][s];
                long double sr = 0.0L, si = 0.0L;
                for (int i = 0; i < np; ++i) {
                    const long double b = beta[a][(long)i * cnt[a] + s];
                    sr += b * q[i].re; si += b * q[i].im;
                }
                A[g].re += sr; A[g].im += si;
            }
        }
        for (long g = 0; g < ng; ++g) { y[2 * g] = (double)A[g].re; y[2 * g + 1] = (double)A[g].im; }
        free(A);
    }
    for (int a = 0; a < natom; ++a) { free(idx[a]); free(beta[a]); }
    free(cnt); free(idx); free(beta);
    return fail ? -1 : 0;
}

/* ------------------------------------------------------------------------- */
/* Gram matrices by the plain triple loop (north_star: "naive loops"):
 *   S[i,j] = sum_r conj(Y[r,i]) Y[r,j],  H[i,j] = sum_r conj(Y[r,i]) HY[r,j],
 * no dV (SURVEY 8(c) reading 10).  Y, HY: [n][ld] complex128, column c at c*ld.
 * H, S: n x n complex128 column-major, element (i,j) at i + j*lds.  Either output
 * may be NULL.                                                                 */
int orc_gram(int64_t ng, int32_t n, const double *Y, int64_t ldy, const double *HY, int64_t ldhy,
             double *H, double *S, int32_t lds)
{
#pragma omp parallel for collapse(2) schedule(dynamic, 8)
    for (int j = 0; j < n; ++j)
        for (int i = 0; i < n; ++i) {
            const double *yi = Y + 2 * (long)i * ldy;
            if (S) {
                const double *yj = Y + 2 * (long)j * ldy;
                long double sr = 0.0L, si = 0.0L;
                for (long r = 0; r < ng; ++r) {
                    const long double ar = yi[2 * r], ai = yi[2 * r + 1], br = yj[2 * r], bi = yj[2 * r + 1];
                    sr += ar * br + ai * bi;
                    si += ar * bi - ai * br;
                }
                S[2 * ((long)i + (long)j * lds)] = (double)sr;
                S[2 * ((long)i + (long)j * lds) + 1] = (double)si;
            }
            if (H) {
                const double *hj = HY + 2 * (long)j * ldhy;
                long double sr = 0.0L, si = 0.0L;
                for (long r = 0; r < ng; ++r) {
                    const long double ar = yi[2 * r], ai = yi[2 * r + 1], br = hj[2 * r], bi = hj[2 * r + 1];
                    sr += ar * br + ai * bi;
                    si += ar * bi - ai * br;
                }
                H[2 * ((long)i + (long)j * lds)] = (double)sr;
                H[2 * ((long)i + (long)j * lds) + 1] = (double)si;
            }
        }
    return 0;
}
