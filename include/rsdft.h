/*
 * rsdft.h -- C ABI of librsdft: the data-parallel hot path of one LOBPCG block step of
 * real-space Kohn-Sham DFT (arXiv 2512.04447 "QUMASUN": (1) FFT Laplacian,
 * (2) H and S matrices of LOBPCG, (4) nonlocal pseudopotential operator), B200 / sm_100a.
 *
 * Notation: grid N = (Nx, Ny, Nz), Ng = Nx*Ny*Nz, periodic
 * orthorhombic box L (bohr), h_a = L_a / N_a, dV = hx*hy*hz; grid point (ix, iy, iz) sits at
 * r = (ix*hx, iy*hy, iz*hz) and has linear index g = (ix*Ny + iy)*Nz + iz (z fastest).
 * An orbital block is `ncol` columns; column c starts at element c*ld (ld >= Ng); every
 * element is complex128, interleaved (re, im) = 16 bytes.  Hartree atomic units.
 *
 * All entry points return 0 (RSDFT_OK) or a negative rsdft_status; they never throw or
 * abort.  On error the outputs are undefined and rsdft_last_error() (thread-local) carries
 * a message.  "device" pointers are CUDA device pointers of the current device, which must be
 * the device the plan was created on (INVALID_ARG otherwise); "host" pointers are ordinary
 * host memory.  `stream` is a cudaStream_t passed as void* (NULL =
 * the legacy default stream).  rsdft_apply_h, rsdft_subspace_gram, rsdft_subspace_rotate and
 * rsdft_subspace_rotate2 are asynchronous on `stream`; the first call with a new shape may
 * allocate plan-owned workspace (cudaMalloc, which can synchronise the device), steady-state
 * calls neither allocate nor synchronise.  rsdft_subspace_eig and rsdft_block_step_host
 * synchronise with the host (documented at each).  A plan owns one workspace, so at most one
 * call per plan may be in flight at a time (calls on the same stream are naturally ordered).
 * Work the caller queues on OTHER streams (e.g. rsdft_plan_set_vloc on stream A, then
 * rsdft_apply_h on stream B) must be ordered by the caller; rsdft_block_step_host, which runs
 * on plan-owned streams, orders itself after the last rsdft_plan_set_vloc.
 */
#ifndef RSDFT_H
#define RSDFT_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    RSDFT_OK = 0,
    RSDFT_INVALID_ARG = -1, /* null pointer, ncol <= 0, ld < Ng, X aliases HX, |m| > l, l > 2, ... */
    RSDFT_UNSUPPORTED = -2, /* grid length not 16*M (M = 1..8, 10, 12, 16) nor 12*M (M = 1, 2, 3, 5, 6, 7, 10, 12); box <= 0; 2*rc >= min L */
    RSDFT_ALLOC = -3,       /* host or device allocation failed */
    RSDFT_CUDA = -4,        /* CUDA runtime error; message carries cudaGetErrorString */
    RSDFT_NOT_POSITIVE_DEFINITE = -5, /* rsdft_subspace_eig: the Cholesky factorisation of S_sub met a pivot <= 0 */
    RSDFT_NO_CONVERGENCE = -6         /* rsdft_subspace_eig: the eigen-solver did not converge */
} rsdft_status;

typedef struct rsdft_plan rsdft_plan_t; /* opaque, library-owned */

typedef struct { int32_t n[3]; } rsdft_grid_t;   /* Nx, Ny, Nz */
typedef struct { double len[3]; } rsdft_box_t;   /* Lx, Ly, Lz in bohr */

typedef struct {
    int32_t natom;          /* may be 0 */
    const double *pos;      /* host [natom][3], bohr, absolute; wrapped into [0, L) by the plan */
    const int32_t *species; /* host [natom], index into rsdft_projectors_t.species */
} rsdft_atoms_t;

/* One species' Kleinman-Bylander projectors  beta_i(r) = f_i(|d|) * Y_{l_i m_i}(d/|d|),
 * d = minimum-image displacement from the atom, truncated to the sphere |d|^2 < rc^2
 * (strict; |d|^2 = dx*dx + dy*dy + dz*dz in double).  Y_lm are the real spherical
 * harmonics, orthonormal on the unit sphere:  Y00 = 1/(2 sqrt(pi));
 * l=1: sqrt(3/4pi) * {y, z, x}/r for m = -1, 0, 1;
 * l=2: 1/2 sqrt(15/pi) xy/r^2, 1/2 sqrt(15/pi) yz/r^2, 1/4 sqrt(5/pi) (3z^2 - r^2)/r^2,
 *      1/2 sqrt(15/pi) xz/r^2, 1/4 sqrt(15/pi) (x^2 - y^2)/r^2 for m = -2..2.
 * At |d| = 0: Y00 as usual, 0 for l > 0.   (BASELINE.json configs[0]; R7-R9.) */
typedef struct {
    double rc;              /* bohr, > 0, 2*rc < min L */
    int32_t nproj;          /* 1..16 */
    const int32_t *l;       /* host [nproj], 0..2 */
    const int32_t *m;       /* host [nproj], -l..l */
    int32_t radial_kind;    /* 0: f_i(r) = exp(-alpha[i] r^2);  1: table, linear interpolation */
    const double *alpha;    /* host [nproj]            (kind 0) */
    int32_t nr;             /* table length >= 2       (kind 1) */
    double dr;              /* table spacing, bohr     (kind 1): sample j is f(j*dr); f = 0 for r >= (nr-1)*dr */
    const double *radial;   /* host [nproj][nr]        (kind 1) */
    const double *D;        /* host [nproj][nproj], real symmetric coupling, Hartree */
} rsdft_species_t;

typedef struct {
    int32_t nspecies;
    const rsdft_species_t *species; /* host [nspecies] */
} rsdft_projectors_t;

/* Build a plan for a grid, a box, atoms and their projectors (BASELINE.json north_star:
 * "rsdft_plan_create(grid, box, atoms, projectors)").  Everything passed in is host memory
 * and is copied; the caller may free it on return.  The plan precomputes, once:
 *   - the kinetic factors t(k) = 1/2 sum_a (2 pi kappa_a / L_a)^2, kappa = k for k < N/2 else
 *     k - N (configs[0]), stored separably with 1/Ng folded in, and the FFT twiddles;
 *   - per atom: the list of grid points inside its sphere (int32 g), the table
 *     beta[nproj][npts] (double) and D.
 * atoms == NULL / natom == 0 / projectors == NULL gives H = T + V_loc.  V_loc is 0 until
 * rsdft_plan_set_vloc is called.  *out receives the plan.  Must be called with the target
 * CUDA device current; the plan is bound to that device.
 * Errors: INVALID_ARG, UNSUPPORTED, ALLOC, CUDA. */
int rsdft_plan_create(const rsdft_grid_t *grid, const rsdft_box_t *box, const rsdft_atoms_t *atoms,
                      const rsdft_projectors_t *projectors, rsdft_plan_t **out);

/* Set the local potential v(r): vloc_dev is a DEVICE array [Ng] of doubles; it is copied
 * into a plan-owned buffer asynchronously on `stream` (the caller's array is not retained).
 * PAPER.md:79 ("density and potential updates" happen every SCF iteration while grid,
 * atoms and projectors stay fixed).  NULL resets V_loc to 0. */
int rsdft_plan_set_vloc(rsdft_plan_t *plan, const double *vloc_dev, void *stream);

/* HX = (-1/2 Laplacian + V_loc + V_NL) X  for ncol columns (PAPER.md:19 tasks (1), (4);
 * north_star "rsdft_apply_h(X -> HX)"):
 *   T:    psi^(k) = sum_r psi(r) e^{-2 pi i sum_a k_a i_a / N_a};  psi^ *= t(k);
 *         (T psi)(r) = 1/Ng sum_k psi^(k) e^{+2 pi i ...}
 *   Vloc: + v(r) psi(r)
 *   VNL:  for every atom a: p_i = dV sum_{r in S_a} beta_i(r) psi(r);
 *         HX(r) += sum_ij beta_i(r) D_ij p_j for r in S_a.
 * X, HX: DEVICE, complex128, column c at element offset c*ldx / c*ldhx, ldx, ldhx >= Ng.
 * X is read-only; HX must not overlap X (HX doubles as FFT scratch).  Any ncol >= 1.
 * Errors: INVALID_ARG, CUDA. */
int rsdft_apply_h(rsdft_plan_t *plan, int32_t ncol, const void *X, int64_t ldx,
                  void *HX, int64_t ldhx, void *stream);

/* Rayleigh-Ritz Gram matrices of LOBPCG (PAPER.md:19 task (2); north_star
 * "rsdft_subspace_gram(Y, HY -> H_sub, S_sub)") for Y = [X, W, P] with n columns:
 *   S_sub[i,j] = sum_r conj(Y[r,i]) Y[r,j],   H_sub[i,j] = sum_r conj(Y[r,i]) HY[r,j]
 * (plain sums, no dV).  Y, HY: DEVICE complex128, column c at c*ldy / c*ldhy.
 * H_sub, S_sub: DEVICE, n x n complex128, column-major, element (i,j) at i + j*lds,
 * lds >= n; both triangles are written.  S_sub is exactly Hermitian; H_sub is computed in
 * full (Hermitian only to round-off) unless rsdft_plan_set_gram_mode(plan, 1) was called.  Either of H_sub (with HY) or S_sub may be NULL to
 * skip it.  Errors: INVALID_ARG, ALLOC, CUDA. */
int rsdft_subspace_gram(rsdft_plan_t *plan, int32_t n, const void *Y, int64_t ldy,
                        const void *HY, int64_t ldhy, void *H_sub, void *S_sub, int32_t lds,
                        void *stream);

/* rsdft_subspace_gram for callers that cannot allocate device memory (code under CUDA graph capture, tight
 * serving loops, harnesses that forbid cudaMalloc): the same contraction (PAPER.md:19 task (2)), the same
 * arguments, layouts and output rules as rsdft_subspace_gram (the plan's Gram mode is honoured, its staging knob
 * is not), but the split-K partial tiles and the tile list live in a file-scope `static __device__` scratch of
 * RSDFT_GRAM_STATIC_WORK_BYTES + 12.1 KiB inside the library instead of plan-owned workspace.  The call
 * performs no cudaMalloc / cudaFree and calls no allocating library routine, never synchronises, and launches
 * three kernels on `stream`.  Every GPU that loads the library holds the scratch until exit.
 * Limit: n <= RSDFT_GRAM_STATIC_MAX_N (any Ng); a larger n returns RSDFT_UNSUPPORTED with a message and launches
 * nothing.  When the K split rsdft_subspace_gram would take does not fit the scratch it is cut down, so results
 * equal rsdft_subspace_gram's bit for bit where the split fits and to round-off (1e-12 normwise) otherwise.
 * The scratch is ONE array per device, shared by every call and every plan on that device, and keeps the last
 * call's contents: nothing in it needs to start at zero (each call overwrites all it reads), but two calls
 * that overlap on the GPU (different streams without an ordering between them, or concurrent graph branches)
 * race on it -- the caller must order them.  The first call on a device resolves the scratch address
 * (cudaGetSymbolAddress, which loads the module): make it outside stream capture.
 * Errors: INVALID_ARG, UNSUPPORTED, CUDA. */
#define RSDFT_GRAM_STATIC_MAX_N 1536
#define RSDFT_GRAM_STATIC_WORK_BYTES 67108864 /* 64 MiB */
int rsdft_subspace_gram_static(rsdft_plan_t *plan, int32_t n, const void *Y, int64_t ldy,
                               const void *HY, int64_t ldhy, void *H_sub, void *S_sub, int32_t lds,
                               void *stream);

/* Rayleigh-Ritz update of LOBPCG (the step after the eigen-solve of the (H_sub, S_sub) pencil; Knyazev's
 * method as cited by PAPER.md:19,124):
 *   Out[r, j] = sum_{c < n} Y[r, c] * C[c, j],   j < m,   e.g. X' = Y C_X, HX' = HY C_X, P' = [W, P] C_P.
 * Y: DEVICE complex128, n columns, column c at c*ldy (ldy >= Ng).  C: DEVICE complex128, n x m
 * column-major, element (c, j) at c + j*ldc (ldc >= n).  Out: DEVICE complex128, m columns, column j at
 * j*ldo (ldo >= Ng); must not overlap Y.  Asynchronous on `stream`.  Errors: INVALID_ARG, UNSUPPORTED, CUDA. */
int rsdft_subspace_rotate(rsdft_plan_t *plan, int32_t n, int32_t m, const void *Y, int64_t ldy,
                          const void *C, int32_t ldc, void *Out, int64_t ldo, void *stream);

/* Rayleigh-Ritz update with the LOBPCG residual fused in (Knyazev's method as cited by
 * PAPER.md:19,124): one pass over Y and HY that shares every tile of C between the two products,
 *   X'[r, j] = sum_c Y[r, c] C[c, j],   HX'[r, j] = sum_c HY[r, c] C[c, j],   R[r, j] = HX'[r, j] - lambda[j] X'[r, j],
 * j < m.  Y, HY: DEVICE complex128 blocks of n columns (ldy, ldhy >= Ng); C: DEVICE n x m column-major
 * (ldc >= n); lambda: DEVICE double[m] (the Ritz values rsdft_subspace_eig returns; may be NULL iff R is NULL);
 * Xout, HXout, R: DEVICE blocks of m columns (ld >= Ng), any of them may be NULL to skip it, none may overlap
 * Y, HY or each other.  P' = [W, P] C_P is the same call on the sub-block pointers with HY/HXout/R unused
 * (or rsdft_subspace_rotate).  Asynchronous on `stream`.  Errors: INVALID_ARG, UNSUPPORTED, CUDA. */
int rsdft_subspace_rotate2(rsdft_plan_t *plan, int32_t n, int32_t m, const void *Y, int64_t ldy,
                           const void *HY, int64_t ldhy, const void *C, int32_t ldc, const double *lambda,
                           void *Xout, int64_t ldx, void *HXout, int64_t ldhx, void *R, int64_t ldr,
                           void *stream);

/* Generalized Hermitian eigen-solve of the subspace pencil, H_sub x = lambda S_sub x, by the paper's route
 * (eq. 1), entirely on the device:
 *   S = L L^H (blocked Cholesky);  K = L^-1 H L^-H by TWO blocked triangular solves ("two calls to (P)ZTRSM"
 *   instead of (P)ZHEGST);  K Z = Z Lambda (block Jacobi on the FP64 tensor pipe);  X = L^-H Z.
 * H_sub, S_sub: DEVICE n x n complex128 column-major (lds >= n), as rsdft_subspace_gram writes them; S_sub's
 * LOWER triangle is read, H_sub is read in full.  Outputs: lambda DEVICE double[m], the m lowest eigenvalues in
 * ascending order; C DEVICE n x m column-major (ldc >= n), column j = eigenvector j, normalised C^H S_sub C = I
 * (phases, and bases inside degenerate eigenspaces, are not unique).  1 <= m <= n <= 16384.
 * Runs on `stream` and SYNCHRONISES it with the host (once after the Cholesky for the definiteness check, once
 * per Jacobi sweep for the convergence test); on return the outputs are complete.  The Jacobi rounds run on two
 * plan-owned streams (a high- and a low-priority one) that start behind `stream` and are joined back into it.
 * Errors: INVALID_ARG, ALLOC, CUDA, NOT_POSITIVE_DEFINITE, NO_CONVERGENCE. */
int rsdft_subspace_eig(rsdft_plan_t *plan, int32_t n, const void *H_sub, const void *S_sub, int32_t lds,
                       int32_t m, double *lambda, void *C, int32_t ldc, void *stream);

/* Intermediate results of the last successful rsdft_subspace_eig on this plan (both are unique, so tests compare
 * them element by element): what = 0: the Cholesky factor L (lower, strict upper part zero); what = 1: the
 * standard-form matrix K = L^-1 H L^-H.  out: DEVICE n x n complex128 column-major, ld >= n.  Asynchronous. */
int rsdft_subspace_eig_get(rsdft_plan_t *plan, int32_t what, void *out, int32_t ld, void *stream);

/* Knobs of rsdft_subspace_eig.  reduction 0 (default): K by two triangular solves, the paper's proposal;
 * 1: the blocked two-sided reduction ZHEGST performs (LAPACK's algorithm, itype 1 lower, on the same kernels),
 * kept so that the paper's TRSM-vs-HEGST comparison can be measured.  inner_sweeps: Jacobi sweeps
 * of each 64 x 64 sub-problem per visit (0 = library default 1, at most 16).  Results agree within round-off. */
int rsdft_plan_set_eig_mode(rsdft_plan_t *plan, int32_t reduction, int32_t inner_sweeps);

/* Timing/diagnostics of the last rsdft_subspace_eig: out[0..7] = {Jacobi sweeps, ms Cholesky, ms reduction to
 * standard form, ms eigen-solver, ms back substitution, final off(K)/||K||_F, reduction mode, 0}. */
int rsdft_subspace_eig_stats(const rsdft_plan_t *plan, double *out8);

/* One whole block step with HOST buffers (the end-to-end entry point): copies Y (host, pinned
 * recommended) to the device in panels of 96 columns (two Gram tile widths); each panel goes through rsdft_apply_h as soon as
 * it has arrived and then every [S|H] tile that has become computable is contracted, so both H Y and the
 * Gram matrices overlap the rest of the upload.  Copies H_sub, S_sub (and HY if HY_host != NULL) back to
 * the host and synchronises with the host before returning.  Results equal rsdft_apply_h +
 * rsdft_subspace_gram on device buffers (HY bitwise; H_sub, S_sub within round-off: other K split).
 * Y_host/HY_host: HOST complex128 [n][ld]; H_sub_host, S_sub_host: HOST n x n column-major.
 * Errors: INVALID_ARG, ALLOC, CUDA. */
int rsdft_block_step_host(rsdft_plan_t *plan, int32_t n, const void *Y_host, int64_t ldy,
                          void *HY_host, int64_t ldhy, void *H_sub_host, void *S_sub_host,
                          int32_t lds);

/* Introspection used by tests/bench: fills out[0..7] with
 *   {natom, total sphere points, max points per sphere, device bytes owned by the plan,
 *    apply_h column batch width, kernels launched by the last compute call, Ng, colour classes}. */
int rsdft_plan_info(const rsdft_plan_t *plan, int64_t *out8);

/* Tuning knob: number of columns apply_h pushes through its kernel sequence at a time
 * (0 = library default: about 540 MB of orbitals per launch). */
int rsdft_plan_set_batch(rsdft_plan_t *plan, int32_t batch_cols);

/* Tuning knob: apply_h deals its column batches round-robin to `nstreams` plan-owned CUDA streams
 * (forked from and joined back into the caller's stream, so the call stays asynchronous and ordered
 * on that stream); 1 = everything on the caller's stream, 0 = library default (3), at most 4.
 * Batches are independent, so results do not depend on this setting (bitwise).
 * Errors: INVALID_ARG. */
int rsdft_plan_set_streams(rsdft_plan_t *plan, int32_t nstreams);

/* apply_h FFT path.  0: three FFT kernels per column batch (every kernel makes one HBM round trip of the batch), tiles
 * loaded by the threads.  2 (default): the same three kernels, but the x kernel fetches its tile as one TMA box
 * (cp.async.bulk.tensor) into a dense shared-memory slot and runs its radix stages in place, the two radix-M stage
 * pairs fused in registers for lengths <= 96 (grids with nx = ny in {48, 64, 80, 96, 112, 128}; other grids silently
 * use path 0).  1: ONE persistent kernel per call that walks (column, phase, tile) work items in dependency order so
 * that the k-space of about four columns stays in L2 between the forward, x and inverse programs; every tile is a
 * TMA box fetched ahead of the compute warps by control warps (cubic grids of those lengths, else path 2 / 0).
 * Results are bitwise identical on all paths.
 * Errors: INVALID_ARG. */
int rsdft_plan_set_pipeline(rsdft_plan_t *plan, int32_t mode);

/* Gram mode.  0 (default): H_sub = Y^H (HY) is contracted in full, as the definition reads (and as the
 * paper's ZGEMM does), so it is Hermitian only to round-off.  1: only the upper 48-column
 * tiles of H_sub are contracted and the rest is their conjugate mirror with a real diagonal, like S_sub
 * (H is Hermitian, hence so is Y^H H Y in exact arithmetic; Hermitian eigen-solvers read one triangle
 * anyway): 30 % fewer flops, H_sub exactly Hermitian, equal to mode 0 within round-off.
 * Errors: INVALID_ARG. */
int rsdft_plan_set_gram_mode(rsdft_plan_t *plan, int32_t h_upper_only);

/* Frees the plan-owned workspaces that grow with the problem (the device copies of Y and HY that
 * rsdft_block_step_host keeps, the Gram and projector work buffers, the eigen-solver buffers); they are
 * re-created on the next call that needs them.  Synchronises the device.  Errors: INVALID_ARG, CUDA. */
int rsdft_plan_release_workspace(rsdft_plan_t *plan);

/* Operand staging of the Gram kernel.  0 (default): per-thread 16-byte cp.async (LDGSTS).  1: one TMA bulk copy
 * (cp.async.bulk + mbarrier, SASS UBLKCP) per 256-byte operand row and pipeline stage.  Bitwise identical results;
 * measured 12 % slower at configs[2] (192 small bulk copies per stage cost more than they save), kept as the
 * measured Blackwell-mechanism variant.  Errors: INVALID_ARG. */
int rsdft_plan_set_gram_staging(rsdft_plan_t *plan, int32_t bulk);

/* Destroys the plan and frees everything it owns (synchronises the device first). */
int rsdft_plan_destroy(rsdft_plan_t *plan);

/* Thread-local message of the last failing call on this thread ("" if none). */
const char *rsdft_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* RSDFT_H */
