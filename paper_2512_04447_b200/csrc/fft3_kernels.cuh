// Batched 3-D complex128 FFT Laplacian + local potential of rsdft_apply_h (PAPER.md:19 task (1) "FFT used to apply the
// Laplacian", PAPER.md:103-109 batched transforms).
//
// Every axis length is N = R2*M with R2 = 16 (M = 1..8, 10, 12, 16) or, when 16 does not divide N, R2 = 12
// (M = 1, 2, 3, 5, 6, 7, 10, 12: 12, 24, 36, 60 -- the paper's own 60^3 grid, PAPER.md:77 --, 72, 84, 120, 144).
// Two 1-D decompositions are used (W_N = e^{-2 pi i/N}):
//   "M-first"  (z and x axes):  n = n1*R2 + n2,  k = k1 + M*k2,
//        X[k] = sum_n2 W_R2^{n2 k2} [ W_N^{n2 k1} sum_n1 W_M^{n1 k1} x[n1*R2 + n2] ]
//        stage A = radix-M over n1 (+ twiddle), stage B = radix-R2 over n2; in place, so k-space
//        position p = k1*R2 + k2 holds frequency k1 + M*k2.
//   "R2-first" (y axis, split ACROSS kernels):  n = n1*M + n2,  k = k1 + R2*k2,
//        X[k] = sum_n2 W_M^{n2 k2} [ W_N^{n2 k1} sum_n1 W_R2^{n1 k1} x[n1*M + n2] ]
//        stage A = radix-R2 over the R2 rows {n1*M + n2} (stride M)   -> tiles zy / yz
//        stage B = radix-M  over the M CONTIGUOUS rows {k1*M + n2}    -> tile x
//        in place, so row r = k1*M + k2 holds frequency k1 + R2*k2.
// k-space therefore lives in a permuted order; the kinetic table is permuted to match on the host.
//
// Three tile programs (device functions; a "group" is the set of threads working on one tile, synchronised by a
// named barrier, so that two groups of one CTA can run two tiles side by side):
//   fft3_fwd_tile   tile = (column, x, n2y): R2y rows x Nz.   z forward (A, B), y forward stage A.
//   fft3_x_tile     tile = (column, k1y, z-chunk): Nx x M_y rows x TZ.  y forward stage B, x forward (A, B),
//                   multiply by t(k)/Ng, x inverse (B', A'), y inverse stage B'.
//   fft3_inv_tile   tile = (column, x, n2y).  y inverse stage A', z inverse (B', A'), HX = T psi + v(r) psi(r).
// and two ways to run them:
//   * three kernels per column batch (fft3_fwd_zy_kernel, fft3_x_kernel, fft3_inv_yz_kernel): every kernel makes one
//     HBM round trip of the batch;
//   * ONE persistent kernel (fft3_pipeline_kernel, fft3_tma_kernels.cuh) that walks (column, phase, tile) work items
//     from an in-order queue with per-column completion counters, keeping about four columns of k-space in flight so
//     that the hand-over fwd -> x -> inv goes through L2 instead of HBM (north_star "one HBM round
//     trip per direction"); its tiles are TMA boxes in dense shared-memory slots.
// The inverse transform is the forward codelet run on (im, re)-swapped data.
// All global accesses are >= 64 B contiguous segments of 16 B elements.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "async_copy.cuh"
#include "fft_codelets.cuh"

namespace rsdft {

struct Fft3Args {
    const double2 *X;       // input orbitals (fwd source; inv: psi for the V_loc term)
    double2 *W;             // k-space scratch, same layout as a column block (may be HX itself)
    double2 *HX;            // output of the inv tiles
    int64_t ldx, ldw, ldhx; // column strides (elements)
    int32_t ncol, nx, ny, nz;
    int32_t my;             // ny / R2y
    int32_t r2y;            // 16 or 12
    const double2 *twx, *twy, *twz;   // w_N^m = (cos, -sin)(2 pi m / N), m in [0, N)
    const double *kin_x;    // [nx]     t_x(kx)/Ng, natural frequency index
    const double *kin_yz;   // [ny*nz]  (t_y(ky(r)) + t_z(kz(p)))/Ng at r*nz + p (permuted positions)
    const double *vloc;     // [Ng]
    int32_t hint_stream;    // L2 eviction class of the once-touched data (X reads, HX writes): 0 normal, 1 evict_first, 2 evict_last
    int32_t hint_keep;      // ... of the k-space scratch between the phases
    int32_t x_tma;          // 1: run the TMA-staged x kernel when the shape has one
};

constexpr bool radix16_ok(int N) { return N % 16 == 0 && (N / 16 <= 8 || N / 16 == 10 || N / 16 == 12 || N / 16 == 16); }
template <int N> struct Axis {
    static constexpr int R2 = radix16_ok(N) ? 16 : 12;
    static constexpr int M = N / R2;
    static_assert(N % R2 == 0, "axis length must be a multiple of 16 or of 12");
};

__device__ __forceinline__ double2 ld_nc(const double2 *p) { return __ldg(p); }
// k-space is written by other SMs inside one launch of the pipeline kernel: read it through L2 only
__device__ __forceinline__ double2 ld_cg(const double2 *p) { return __ldcg(p); }

// L2 eviction classes (createpolicy + .L2::cache_hint): the pipeline kernel marks the data it touches once
// (X, psi, the final HX) evict_first and the k-space scratch that must survive from phase to phase evict_last.
__device__ __forceinline__ uint64_t l2_policy(int kind)
{
    uint64_t p;
    if (kind == 1) asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
    else if (kind == 2) asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p));
    else asm volatile("createpolicy.fractional.L2::evict_normal.b64 %0, 1.0;" : "=l"(p));
    return p;
}
__device__ __forceinline__ double2 ld_nc_hint(const double2 *p, uint64_t pol)
{
    double2 v;
    asm volatile("ld.global.nc.L2::cache_hint.v2.f64 {%0, %1}, [%2], %3;" : "=d"(v.x), "=d"(v.y) : "l"(p), "l"(pol));
    return v;
}
__device__ __forceinline__ double2 ld_cg_hint(const double2 *p, uint64_t pol)
{
    double2 v;
    asm volatile("ld.global.cg.L2::cache_hint.v2.f64 {%0, %1}, [%2], %3;" : "=d"(v.x), "=d"(v.y) : "l"(p), "l"(pol) : "memory");
    return v;
}
__device__ __forceinline__ void st_hint(double2 *p, double2 v, uint64_t pol)
{
    asm volatile("st.global.L2::cache_hint.v2.f64 [%0], {%1, %2}, %3;" :: "l"(p), "d"(v.x), "d"(v.y), "l"(pol) : "memory");
}

// barrier `id` over `nt` threads (id 0 with the whole CTA = __syncthreads)
__device__ __forceinline__ void group_sync(int id, int nt) { asm volatile("bar.sync %0, %1;" :: "r"(id), "r"(nt) : "memory"); }

// ---------------------------------------------------------------------------------------------
// shared-memory geometry of the R2y-row tiles of the fwd / inv programs
template <int NZ, int R2Y>
struct ZyCfg {
    static constexpr int R2Z = Axis<NZ>::R2, MZ = Axis<NZ>::M;
    static constexpr int G = R2Z + 1;                  // slots per R2Z-point group (odd: conflict-free columns)
    static constexpr int RP = MZ * G;                  // smem row pitch
    static constexpr int TILE = R2Y * RP;              // double2 elements per tile buffer
    static constexpr int NTWZ = (MZ > 1 ? MZ - 1 : 1) * R2Z;
    static constexpr size_t SMEM_FWD = (size_t)TILE * sizeof(double2);
    static constexpr size_t SMEM_INV = (size_t)(2 * TILE + R2Y * NZ) * sizeof(double2);
};

// twiddle tables of a fwd / inv tile: twz_s[(k-1)*R2Z + n2] = w_NZ^{n2 k}, twy_s[k] = w_NY^{n2y k}
template <int NZ, int R2Y, int NT>
__device__ __forceinline__ void fft3_zy_tables(const Fft3Args &a, int n2y, double2 *twz_s, double2 *twy_s, int tid, bool want_z)
{
    constexpr int R2Z = Axis<NZ>::R2, MZ = Axis<NZ>::M;
    if (want_z)
        for (int e = tid; e < (MZ - 1) * R2Z; e += NT) twz_s[e] = a.twz[(e % R2Z) * (e / R2Z + 1)];
    if (tid < R2Y) twy_s[tid] = a.twy[n2y * tid];
}

// z forward + y forward stage A of one tile.  src/dst: plane base (column, x) of X / W.
template <int NZ, int R2Y, int NT, bool HINT = false>
__device__ __forceinline__ void fft3_fwd_tile(const double2 *__restrict__ src, double2 *__restrict__ dst, int my, int n2y, double2 *S,
                                              const double2 *twz_s, const double2 *twy_s, int tid, int bar,
                                              uint64_t pol_in = 0, uint64_t pol_out = 0)
{
    using C = ZyCfg<NZ, R2Y>;
    constexpr int R2Z = C::R2Z, MZ = C::MZ, G = C::G, RP = C::RP;
    // z stage A: radix-MZ over n1, twiddle w_NZ^{n2 k1}
#pragma unroll
    for (int item = tid; item < R2Y * R2Z; item += NT) {
        const int j = item / R2Z, n2 = item % R2Z;
        const double2 *row = src + (int64_t)(j * my + n2y) * NZ + n2;
        double re[MZ], im[MZ];
#pragma unroll
        for (int n1 = 0; n1 < MZ; ++n1) { const double2 v = HINT ? ld_nc_hint(row + n1 * R2Z, pol_in) : ld_nc(row + n1 * R2Z); re[n1] = v.x; im[n1] = v.y; }
        Dft<MZ>::run(re, im);
#pragma unroll
        for (int k = 1; k < MZ; ++k) { const double2 w = twz_s[(k - 1) * R2Z + n2]; tw_mul(re[k], im[k], w.x, -w.y); }
#pragma unroll
        for (int k = 0; k < MZ; ++k) S[j * RP + k * G + n2] = make_double2(re[k], im[k]);
    }
    group_sync(bar, NT);
    // z stage B: radix-R2Z over n2, in place (position k1*R2Z + k2 <- frequency k1 + MZ*k2)
    for (int item = tid; item < R2Y * MZ; item += NT) {
        double2 *p = S + item * G;
        double br[R2Z], bi[R2Z];
#pragma unroll
        for (int t = 0; t < R2Z; ++t) { const double2 v = p[t]; br[t] = v.x; bi[t] = v.y; }
        Dft<R2Z>::run(br, bi);
#pragma unroll
        for (int t = 0; t < R2Z; ++t) p[t] = make_double2(br[t], bi[t]);
    }
    group_sync(bar, NT);
    // y stage A: radix-R2Y over the R2Y rows, twiddle w_NY^{n2y k1}, store row k1*my + n2y
    for (int p = tid; p < NZ; p += NT) {
        const int sp = (p / R2Z) * G + (p % R2Z);
        double br[R2Y], bi[R2Y];
#pragma unroll
        for (int j = 0; j < R2Y; ++j) { const double2 v = S[j * RP + sp]; br[j] = v.x; bi[j] = v.y; }
        Dft<R2Y>::run(br, bi);
#pragma unroll
        for (int k = 1; k < R2Y; ++k) { const double2 w = twy_s[k]; tw_mul(br[k], bi[k], w.x, -w.y); }
#pragma unroll
        for (int k = 0; k < R2Y; ++k) {
            if (HINT) st_hint(dst + (int64_t)(k * my + n2y) * NZ + p, make_double2(br[k], bi[k]), pol_out);
            else dst[(int64_t)(k * my + n2y) * NZ + p] = make_double2(br[k], bi[k]);
        }
    }
    group_sync(bar, NT);
}

// y inverse stage A' and z inverse stage B' of a tile already in shared memory (padded layout)
template <int NZ, int R2Y, int NT>
__device__ __forceinline__ void fft3_inv_stages_12(double2 *S, const double2 *twy_s, int tid, int bar)
{
    using C = ZyCfg<NZ, R2Y>;
    constexpr int R2Z = C::R2Z, MZ = C::MZ, G = C::G, RP = C::RP;
    // y inverse stage A': conj twiddle, radix-R2Y over k1y (swapped domain) -> row j = n1y, in place
    for (int p = tid; p < NZ; p += NT) {
        double2 *c = S + (p / R2Z) * G + (p % R2Z);
        double br[R2Y], bi[R2Y];
#pragma unroll
        for (int k = 0; k < R2Y; ++k) { const double2 v = c[k * RP]; br[k] = v.x; bi[k] = v.y; }
#pragma unroll
        for (int k = 1; k < R2Y; ++k) { const double2 w = twy_s[k]; tw_mul(bi[k], br[k], w.x, -w.y); }
        Dft<R2Y>::run(bi, br);
#pragma unroll
        for (int j = 0; j < R2Y; ++j) c[j * RP] = make_double2(br[j], bi[j]);
    }
    group_sync(bar, NT);
    // z inverse stage B': radix-R2Z over k2z (swapped), in place
    for (int item = tid; item < R2Y * MZ; item += NT) {
        double2 *p = S + item * G;
        double br[R2Z], bi[R2Z];
#pragma unroll
        for (int q = 0; q < R2Z; ++q) { const double2 v = p[q]; br[q] = v.x; bi[q] = v.y; }
        Dft<R2Z>::run(bi, br);
#pragma unroll
        for (int q = 0; q < R2Z; ++q) p[q] = make_double2(br[q], bi[q]);
    }
}

// z inverse stage A' + V_loc: conj twiddle, radix-MZ over k1z (swapped) -> z = n1*R2Z + n2;  HX = T psi + v psi.
// psi comes from shared memory (Sp, dense [R2Y][NZ]) when PSI_SMEM, else straight from global memory (psi_g = plane base).
template <int NZ, int R2Y, int NT, bool PSI_SMEM, bool HINT = false>
__device__ __forceinline__ void fft3_inv_stage_3(const double2 *S, const double2 *twz_s, const double2 *Sp, const double2 *__restrict__ psi_g,
                                                 const double *__restrict__ vl, double2 *__restrict__ dst, int my, int n2y, int tid,
                                                 uint64_t pol_stream = 0)
{
    using C = ZyCfg<NZ, R2Y>;
    constexpr int R2Z = C::R2Z, MZ = C::MZ, G = C::G, RP = C::RP;
#pragma unroll
    for (int item = tid; item < R2Y * R2Z; item += NT) {
        const int j = item / R2Z, n2 = item % R2Z;
        const int64_t off = (int64_t)(j * my + n2y) * NZ + n2;
        double2 ps[MZ];
        double vv[MZ];
#pragma unroll
        for (int n1 = 0; n1 < MZ; ++n1) {          // issued first: their latency hides behind the radix-MZ below
            ps[n1] = PSI_SMEM ? Sp[j * NZ + n1 * R2Z + n2] : (HINT ? ld_nc_hint(psi_g + off + n1 * R2Z, pol_stream) : ld_nc(psi_g + off + n1 * R2Z));
            vv[n1] = __ldg(vl + off + n1 * R2Z);
        }
        double re[MZ], im[MZ];
#pragma unroll
        for (int k = 0; k < MZ; ++k) { const double2 v = S[j * RP + k * G + n2]; re[k] = v.x; im[k] = v.y; }
#pragma unroll
        for (int k = 1; k < MZ; ++k) { const double2 w = twz_s[(k - 1) * R2Z + n2]; tw_mul(im[k], re[k], w.x, -w.y); }
        Dft<MZ>::run(im, re);
#pragma unroll
        for (int n1 = 0; n1 < MZ; ++n1) {
            const double2 r = make_double2(fma(vv[n1], ps[n1].x, re[n1]), fma(vv[n1], ps[n1].y, im[n1]));
            if (HINT) st_hint(dst + off + n1 * R2Z, r, pol_stream);
            else dst[off + n1 * R2Z] = r;
        }
    }
}

// cp.async of the R2Y k-space rows {k*my + n2y} of one plane into the padded tile layout
template <int NZ, int R2Y, int NT, bool HINT = false>
__device__ __forceinline__ void fft3_issue_w_tile(const double2 *__restrict__ src, int my, int n2y, double2 *S, int tid, uint64_t pol = 0)
{
    using C = ZyCfg<NZ, R2Y>;
    constexpr int R2Z = C::R2Z, G = C::G, RP = C::RP;
#pragma unroll
    for (int e = tid; e < R2Y * NZ; e += NT) {
        const int k = e / NZ, p = e - k * NZ;
        if (HINT) cp_async16_hint(S + k * RP + (p / R2Z) * G + (p % R2Z), src + (int64_t)(k * my + n2y) * NZ + p, pol);
        else cp_async16(S + k * RP + (p / R2Z) * G + (p % R2Z), src + (int64_t)(k * my + n2y) * NZ + p);
    }
}

// ---------------------------------------------------------------------------------------------
// z forward + y forward stage A.  128 threads; grid = G * my, CTA b works on n2y = b % my.
template <int NZ, int R2Y, int MINB>
__global__ void __launch_bounds__(128, MINB) fft3_fwd_zy_kernel(Fft3Args a)
{
    using C = ZyCfg<NZ, R2Y>;
    constexpr int NT = 128;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double2 *S = reinterpret_cast<double2 *>(smem_raw);
    __shared__ double2 twz_s[C::NTWZ];
    __shared__ double2 twy_s[R2Y];
    const int tid = threadIdx.x;
    const int my = a.my;
    const int n2y = blockIdx.x % my;
    const int g0 = blockIdx.x / my, G = gridDim.x / my;
    fft3_zy_tables<NZ, R2Y, NT>(a, n2y, twz_s, twy_s, tid, true);
    __syncthreads();
    const int64_t nplanes = (int64_t)a.ncol * a.nx;
    for (int64_t cx = g0; cx < nplanes; cx += G) {
        const int64_t col = cx / a.nx;
        const int64_t x = cx - col * a.nx;
        fft3_fwd_tile<NZ, R2Y, NT>(a.X + col * a.ldx + x * a.ny * NZ, a.W + col * a.ldw + x * a.ny * NZ, my, n2y, S, twz_s, twy_s, tid, 0);
    }
}

// ---------------------------------------------------------------------------------------------
// y inverse stage A' + z inverse + V_loc.  Mirror of the kernel above; W -> HX (may be in place:
// a tile reads and writes the same R2Y rows).  CTA b owns n2y = b % my and the x planes
// g0, g0 + G, ...; for each plane it runs over ALL columns of the batch (the rows of v(r) stay
// hot in L1/L2).  Per tile: the k-space rows of the NEXT tile (double buffered) and the psi rows of
// THIS tile (consumed two phases later) arrive by cp.async.
template <int NZ, int R2Y, int MINB>
__global__ void __launch_bounds__(128, MINB) fft3_inv_yz_kernel(Fft3Args a)
{
    using C = ZyCfg<NZ, R2Y>;
    constexpr int TILE = C::TILE, NT = 128;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double2 *Sw0 = reinterpret_cast<double2 *>(smem_raw);
    double2 *Sp = Sw0 + 2 * TILE;                               // psi rows, dense [R2Y][NZ]
    __shared__ double2 twz_s[C::NTWZ];
    __shared__ double2 twy_s[R2Y];
    const int tid = threadIdx.x;
    const int my = a.my;
    const int n2y = blockIdx.x % my;
    const int g0 = blockIdx.x / my, G = gridDim.x / my;
    fft3_zy_tables<NZ, R2Y, NT>(a, n2y, twz_s, twy_s, tid, true);
    const int nxm = g0 < a.nx ? (a.nx - g0 + G - 1) / G : 0;      // planes of this walker
    const int64_t T = (int64_t)nxm * a.ncol;                      // tiles: plane-major, column-minor
    auto plane_off = [&](int64_t t, int64_t &col) -> int64_t {
        const int64_t i = t / a.ncol;
        col = t - i * a.ncol;
        return (g0 + i * G) * (int64_t)a.ny * NZ;
    };
    auto issue_w = [&](int buf, int64_t t) {
        int64_t col;
        const int64_t po = plane_off(t, col);
        fft3_issue_w_tile<NZ, R2Y, NT>(a.W + col * a.ldw + po, my, n2y, Sw0 + buf * TILE, tid);
    };
    auto issue_psi = [&](int64_t t) {
        int64_t col;
        const int64_t po = plane_off(t, col);
        const double2 *src = a.X + col * a.ldx + po;
#pragma unroll
        for (int e = tid; e < R2Y * NZ; e += NT) {
            const int j = e / NZ, p = e - j * NZ;
            cp_async16(Sp + e, src + (int64_t)(j * my + n2y) * NZ + p);
        }
    };
    if (T > 0) issue_w(0, 0);
    cp_async_commit();
    int buf = 0;
    for (int64_t t = 0; t < T; ++t, buf ^= 1) {
        issue_psi(t);
        cp_async_commit();
        if (t + 1 < T) issue_w(buf ^ 1, t + 1);
        cp_async_commit();
        cp_async_wait<2>();                                       // W(t) has landed
        __syncthreads();
        int64_t col;
        const int64_t po = plane_off(t, col);
        double2 *S = Sw0 + buf * TILE;
        fft3_inv_stages_12<NZ, R2Y, NT>(S, twy_s, tid, 0);
        cp_async_wait<1>();                                       // psi(t) has landed
        __syncthreads();
        fft3_inv_stage_3<NZ, R2Y, NT, true>(S, twz_s, Sp, nullptr, a.vloc + po, a.HX + col * a.ldhx + po, my, n2y, tid);
        __syncthreads();
    }
    cp_async_wait<0>();
}

// ---------------------------------------------------------------------------------------------
// y stage B, x forward, kinetic factor, x inverse, y stage B'.  In place on W.
// Tile = (column, k1y, z-chunk): S[x][line], line = jy*TZ + z, odd pitch P = lines + 1.
template <int MY, int NX, int TZ, int NT, bool CG>
__device__ __forceinline__ void fft3_x_load_y(const Fft3Args &a, const double2 *base, double2 *S, int P, int tid, uint64_t pol)
{
    // items are taken two at a time so that both items' global loads are in flight together
    int item = tid;
    for (; item + NT < NX * TZ; item += 2 * NT) {
        const int z0 = item % TZ, x0 = item / TZ, z1 = (item + NT) % TZ, x1 = (item + NT) / TZ;
        const double2 *p0 = base + (int64_t)x0 * a.ny * a.nz + z0;
        const double2 *p1 = base + (int64_t)x1 * a.ny * a.nz + z1;
        double re0[MY], im0[MY], re1[MY], im1[MY];
#pragma unroll
        for (int j = 0; j < MY; ++j) { const double2 v = CG ? ld_cg_hint(p0 + (int64_t)j * a.nz, pol) : p0[(int64_t)j * a.nz]; re0[j] = v.x; im0[j] = v.y; }
#pragma unroll
        for (int j = 0; j < MY; ++j) { const double2 v = CG ? ld_cg_hint(p1 + (int64_t)j * a.nz, pol) : p1[(int64_t)j * a.nz]; re1[j] = v.x; im1[j] = v.y; }
        Dft<MY>::run(re0, im0);
#pragma unroll
        for (int j = 0; j < MY; ++j) S[x0 * P + j * TZ + z0] = make_double2(re0[j], im0[j]);
        Dft<MY>::run(re1, im1);
#pragma unroll
        for (int j = 0; j < MY; ++j) S[x1 * P + j * TZ + z1] = make_double2(re1[j], im1[j]);
    }
    if (item < NX * TZ) {
        const int z = item % TZ, x = item / TZ;
        const double2 *ptr = base + (int64_t)x * a.ny * a.nz + z;
        double re[MY], im[MY];
#pragma unroll
        for (int j = 0; j < MY; ++j) { const double2 v = CG ? ld_cg_hint(ptr + (int64_t)j * a.nz, pol) : ptr[(int64_t)j * a.nz]; re[j] = v.x; im[j] = v.y; }
        Dft<MY>::run(re, im);
#pragma unroll
        for (int j = 0; j < MY; ++j) S[x * P + j * TZ + z] = make_double2(re[j], im[j]);
    }
}

template <int MY, int NX, int TZ, int NT, bool CG>
__device__ __forceinline__ void fft3_x_store_y(const Fft3Args &a, double2 *base, const double2 *S, int P, int tid, uint64_t pol)
{
    for (int item = tid; item < NX * TZ; item += NT) {
        const int z = item % TZ, x = item / TZ;
        double2 *ptr = base + (int64_t)x * a.ny * a.nz + z;
        double re[MY], im[MY];
#pragma unroll
        for (int j = 0; j < MY; ++j) { const double2 v = S[x * P + j * TZ + z]; re[j] = v.x; im[j] = v.y; }
        Dft<MY>::run(im, re);
#pragma unroll
        for (int j = 0; j < MY; ++j) {
            if (CG) st_hint(ptr + (int64_t)j * a.nz, make_double2(re[j], im[j]), pol);
            else ptr[(int64_t)j * a.nz] = make_double2(re[j], im[j]);
        }
    }
}

#define RS_SWITCH_MY(MY_, CALL_)                     \
    switch (MY_) {                                   \
    case 1: { constexpr int MYC = 1; CALL_; } break;   \
    case 2: { constexpr int MYC = 2; CALL_; } break;   \
    case 3: { constexpr int MYC = 3; CALL_; } break;   \
    case 4: { constexpr int MYC = 4; CALL_; } break;   \
    case 5: { constexpr int MYC = 5; CALL_; } break;   \
    case 6: { constexpr int MYC = 6; CALL_; } break;   \
    case 7: { constexpr int MYC = 7; CALL_; } break;   \
    case 8: { constexpr int MYC = 8; CALL_; } break;   \
    case 10: { constexpr int MYC = 10; CALL_; } break; \
    case 12: { constexpr int MYC = 12; CALL_; } break; \
    default: { constexpr int MYC = 16; CALL_; } break; \
    }

// One x tile, in place on W.  base = W + column offset + (k1y*my)*nz + zc*TZ.  twx_s[(k-1)*R2X + n2] = w_NX^{n2 k},
// kinx_s[kx] = t_x(kx)/Ng, kin = kin_yz + (k1y*my)*nz + zc*TZ.  The whole CTA (NT threads) works on the tile.
template <int NX, int TZ, int NT, bool CG>
__device__ __forceinline__ void fft3_x_tile(const Fft3Args &a, double2 *base, const double *__restrict__ kin, double2 *S,
                                            const double2 *twx_s, const double *kinx_s, int tid, uint64_t pol = 0)
{
    constexpr int R2X = Axis<NX>::R2, MX = Axis<NX>::M;
    const int my = a.my, lines = my * TZ, P = lines + 1;
    RS_SWITCH_MY(my, (fft3_x_load_y<MYC, NX, TZ, NT, CG>(a, base, S, P, tid, pol)))
    __syncthreads();
    // x stage A: radix-MX over n1 (x = n1*R2X + n2), twiddle, in place
    for (int item = tid; item < lines * R2X; item += NT) {
        const int n2 = item % R2X, line = item / R2X;
        double2 *p = S + n2 * P + line;
        double re[MX], im[MX];
#pragma unroll
        for (int n1 = 0; n1 < MX; ++n1) { const double2 v = p[n1 * R2X * P]; re[n1] = v.x; im[n1] = v.y; }
        Dft<MX>::run(re, im);
#pragma unroll
        for (int k = 1; k < MX; ++k) { const double2 w = twx_s[(k - 1) * R2X + n2]; tw_mul(re[k], im[k], w.x, -w.y); }
#pragma unroll
        for (int k = 0; k < MX; ++k) p[k * R2X * P] = make_double2(re[k], im[k]);
    }
    __syncthreads();
    // x stage B (radix-R2X over n2) -> frequency kx = k1 + MX*k2; kinetic factor; inverse stage B'
    for (int item = tid; item < lines * MX; item += NT) {
        const int line = item % lines, k1 = item / lines;
        double2 *p = S + k1 * R2X * P + line;
        double br[R2X], bi[R2X];
#pragma unroll
        for (int t = 0; t < R2X; ++t) { const double2 v = p[t * P]; br[t] = v.x; bi[t] = v.y; }
        Dft<R2X>::run(br, bi);
        const int jy = line / TZ, z = line - jy * TZ;
        const double tin = __ldg(kin + (int64_t)jy * a.nz + z);
#pragma unroll
        for (int k2 = 0; k2 < R2X; ++k2) {
            const double f = kinx_s[k1 + MX * k2] + tin;
            br[k2] *= f; bi[k2] *= f;
        }
        Dft<R2X>::run(bi, br);                  // swapped domain from here on
#pragma unroll
        for (int t = 0; t < R2X; ++t) p[t * P] = make_double2(br[t], bi[t]);
    }
    __syncthreads();
    // x inverse stage A': conj twiddle, radix-MX over k1 -> x = n1*R2X + n2
    for (int item = tid; item < lines * R2X; item += NT) {
        const int n2 = item % R2X, line = item / R2X;
        double2 *p = S + n2 * P + line;
        double re[MX], im[MX];
#pragma unroll
        for (int k = 0; k < MX; ++k) { const double2 v = p[k * R2X * P]; re[k] = v.x; im[k] = v.y; }
#pragma unroll
        for (int k = 1; k < MX; ++k) { const double2 w = twx_s[(k - 1) * R2X + n2]; tw_mul(im[k], re[k], w.x, -w.y); }
        Dft<MX>::run(im, re);
#pragma unroll
        for (int n1 = 0; n1 < MX; ++n1) p[n1 * R2X * P] = make_double2(re[n1], im[n1]);
    }
    __syncthreads();
    RS_SWITCH_MY(my, (fft3_x_store_y<MYC, NX, TZ, NT, CG>(a, base, S, P, tid, pol)))
    __syncthreads();
}

// Per-length launch shape: z points per tile (TZ*16 B contiguous per row), threads, CTAs per SM.
// (NT = 288 for 96, which fills the radix-16 phase in one round, measured 40 % slower than 256.)
template <int NX> struct XCfg { static constexpr int TZ = 4, NT = 256, MINB = 1; };
template <> struct XCfg<12> { static constexpr int TZ = 4, NT = 32, MINB = 8; };
template <> struct XCfg<16> { static constexpr int TZ = 8, NT = 32, MINB = 8; };
template <> struct XCfg<24> { static constexpr int TZ = 4, NT = 64, MINB = 8; };
template <> struct XCfg<32> { static constexpr int TZ = 8, NT = 64, MINB = 8; };
template <> struct XCfg<36> { static constexpr int TZ = 4, NT = 96, MINB = 5; };
template <> struct XCfg<48> { static constexpr int TZ = 8, NT = 96, MINB = 5; };
template <> struct XCfg<60> { static constexpr int TZ = 4, NT = 128, MINB = 4; };
template <> struct XCfg<64> { static constexpr int TZ = 8, NT = 128, MINB = 4; };
template <> struct XCfg<72> { static constexpr int TZ = 8, NT = 224, MINB = 2; };
template <> struct XCfg<80> { static constexpr int TZ = 8, NT = 224, MINB = 2; };
template <> struct XCfg<84> { static constexpr int TZ = 4, NT = 256, MINB = 2; };
template <> struct XCfg<96> { static constexpr int TZ = 8, NT = 256, MINB = 2; };
template <> struct XCfg<112> { static constexpr int TZ = 8, NT = 256, MINB = 2; };
template <> struct XCfg<120> { static constexpr int TZ = 4, NT = 256, MINB = 2; };
template <> struct XCfg<128> { static constexpr int TZ = 4, NT = 256, MINB = 2; };
template <> struct XCfg<144> { static constexpr int TZ = 4, NT = 256, MINB = 2; };
template <> struct XCfg<160> { static constexpr int TZ = 4, NT = 256, MINB = 2; };
template <> struct XCfg<192> { static constexpr int TZ = 4, NT = 256, MINB = 1; };
template <> struct XCfg<256> { static constexpr int TZ = 2, NT = 256, MINB = 1; };

template <int NX> struct XTables {
    static constexpr int R2X = Axis<NX>::R2, MX = Axis<NX>::M;
    static constexpr int NTW = (MX > 1 ? MX - 1 : 1) * R2X;
};

template <int NX, int NT>
__device__ __forceinline__ void fft3_x_tables(const Fft3Args &a, double2 *twx_s, double *kinx_s, int tid)
{
    constexpr int R2X = Axis<NX>::R2, MX = Axis<NX>::M;
    for (int e = tid; e < (MX - 1) * R2X; e += NT) twx_s[e] = a.twx[(e % R2X) * (e / R2X + 1)];
    for (int e = tid; e < NX; e += NT) kinx_s[e] = a.kin_x[e];
}

template <int NX, int TZ, int NT, int MINB>
__global__ void __maxnreg__(((65536 / (NT * MINB)) / 8 * 8) > 255 ? 255 : ((65536 / (NT * MINB)) / 8 * 8)) fft3_x_kernel(Fft3Args a)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double2 *S = reinterpret_cast<double2 *>(smem_raw);
    __shared__ double2 twx_s[XTables<NX>::NTW];
    __shared__ double kinx_s[NX];
    const int tid = threadIdx.x;
    const int my = a.my;
    fft3_x_tables<NX, NT>(a, twx_s, kinx_s, tid);
    __syncthreads();
    const int zchunks = a.nz / TZ;
    const int64_t per_col = (int64_t)a.r2y * zchunks;
    const int64_t ntiles = per_col * a.ncol;
    for (int64_t tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
        const int64_t colf = tile / per_col;
        const int rem = (int)(tile - colf * per_col);
        const int64_t col = a.ncol - 1 - colf;     // zig-zag: the forward kernel ended on the last column, start there (L2)
        const int k1y = rem / zchunks, zc = rem - k1y * zchunks;
        const int64_t toff = (int64_t)(k1y * my) * a.nz + zc * TZ;
        fft3_x_tile<NX, TZ, NT, false>(a, a.W + col * a.ldw + toff, a.kin_yz + toff, S, twx_s, kinx_s, tid);
    }
}

// ---------------------------------------------------------------------------------------------
// Work queue of the persistent pipeline kernel (fft3_tma_kernels.cuh): ONE launch applies T + V_loc to all `ncol`
// columns.  Work items (phase, column, tile) are handed out in queue order by an atomic counter; the queue is built
// from "super-steps": super-step s holds the fwd items of column s, the x items of column s - lag_x and the inv items
// of column s - lag_inv, interleaved by `pattern` (one entry per item of a super-step: phase << 28 | tile).  An x item
// of column c needs ALL fwd items of c, an inv item ALL x items of c: per-column completion counters
// `done[phase*ncol + c]` (dependencies always sit earlier in the queue, and nothing ever waits while holding an
// earlier unfinished item, so the smallest unfinished item always makes progress: no co-residency assumption, no
// deadlock).  About four columns of k-space are in flight, so the k-space written by fwd is still in L2 when x and
// inv read it.
struct PipeArgs {
    int32_t *head;           // queue position counter (zeroed before the launch)
    int32_t *done;           // [3][ncol] finished items per (phase, column) (zeroed before the launch)
    const uint32_t *pattern; // item order inside one super-step
    int32_t npattern;
    int32_t n_fwd, n_x, n_inv;   // items per column and phase
    int32_t zchunks;             // nz / TZ
    int32_t lag_x, lag_inv;      // super-step s holds fwd(s), x(s - lag_x), inv(s - lag_inv)
};

__device__ __forceinline__ void pipe_wait(const int32_t *cnt, int want)
{
    while (*((const volatile int32_t *)cnt) < want) __nanosleep(64);
    __threadfence();
}

}  // namespace rsdft
