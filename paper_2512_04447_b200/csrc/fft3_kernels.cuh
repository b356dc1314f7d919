// Batched 3-D complex128 FFT Laplacian + local potential of rsdft_apply_h in THREE kernels
// (PAPER.md:19 task (1) "FFT used to apply the Laplacian", PAPER.md:103-109 batched transforms;
// SURVEY 8(a) a1-a4).  One HBM/L2 round trip per kernel: 3 x (16 + 16) B per orbital*point, plus
// the 16 B re-read of psi for v(r) psi(r).
//
// Every axis length is N = 16*M (M = 1..8, 10, 12, 16).  Two 1-D decompositions are used (W_N = e^{-2 pi i/N}):
//   "M-first"  (z and x axes):  n = n1*16 + n2,  k = k1 + M*k2,
//        X[k] = sum_n2 W_16^{n2 k2} [ W_N^{n2 k1} sum_n1 W_M^{n1 k1} x[n1*16 + n2] ]
//        stage A = radix-M over n1 (+ twiddle), stage B = radix-16 over n2; in place, so k-space
//        position p = k1*16 + k2 holds frequency k1 + M*k2.
//   "16-first" (y axis, split ACROSS kernels):  n = n1*M + n2,  k = k1 + 16*k2,
//        X[k] = sum_n2 W_M^{n2 k2} [ W_N^{n2 k1} sum_n1 W_16^{n1 k1} x[n1*M + n2] ]
//        stage A = radix-16 over the 16 rows {n1*M + n2} (stride M)   -> kernels zy / yz
//        stage B = radix-M  over the M CONTIGUOUS rows {k1*M + n2}    -> kernel x
//        in place, so row r = k1*M + k2 holds frequency k1 + 16*k2.
// k-space therefore lives in a permuted order; the kinetic table is permuted to match on the host.
//
//   fft3_fwd_zy_kernel  tile = (column, x, n2y): 16 rows x Nz.   z forward (A, B), y forward stage A.
//   fft3_x_kernel       tile = (column, k1y, z-chunk): Nx x M_y rows x TZ.  y forward stage B,
//                       x forward (A, B), multiply by t(k)/Ng, x inverse (B', A'), y inverse stage B'.
//   fft3_inv_yz_kernel  tile = (column, x, n2y).  y inverse stage A', z inverse (B', A'),
//                       HX = T psi + v(r) psi(r).
// The inverse transform is the forward codelet run on (im, re)-swapped data.
// All global accesses are >= 128 B contiguous segments of 16 B elements.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "async_copy.cuh"
#include "fft_codelets.cuh"

namespace rsdft {

struct Fft3Args {
    const double2 *X;       // input orbitals (zy source; yz: psi for the V_loc term)
    double2 *W;             // k-space scratch, same layout as a column block (may be HX itself)
    double2 *HX;            // output of the yz kernel
    int64_t ldx, ldw, ldhx; // column strides (elements)
    int32_t ncol, nx, ny, nz;
    int32_t my;             // ny / 16
    const double2 *twx, *twy, *twz;   // w_N^m = (cos, -sin)(2 pi m / N), m in [0, N)
    const double *kin_x;    // [nx]     t_x(kx)/Ng, natural frequency index
    const double *kin_yz;   // [ny*nz]  (t_y(ky(r)) + t_z(kz(p)))/Ng at r*nz + p (permuted positions)
    const double *vloc;     // [Ng]
};

__device__ __forceinline__ double2 ld_nc(const double2 *p) { return __ldg(p); }

// ---------------------------------------------------------------------------------------------
// shared-memory geometry of the 16-row tiles of the zy / yz kernels
template <int NZ>
struct ZyCfg {
    static constexpr int MZ = NZ / 16;
    static constexpr int RP = MZ * 17;                 // smem row pitch: 17 slots per 16-point group
    static constexpr int TILE = 16 * RP;               // double2 elements per tile buffer
    static constexpr size_t SMEM_FWD = (size_t)TILE * sizeof(double2);
    static constexpr size_t SMEM_INV = (size_t)(2 * TILE + 16 * NZ) * sizeof(double2);
};

// z forward + y forward stage A.  128 threads; grid = G * my, CTA b works on n2y = b % my.
template <int NZ, int MINB>
__global__ void __launch_bounds__(128, MINB) fft3_fwd_zy_kernel(Fft3Args a)
{
    constexpr int MZ = NZ / 16;
    constexpr int RP = MZ * 17;                 // smem row pitch: 17 slots per 16-point group
    constexpr int NT = 128;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double2 *S = reinterpret_cast<double2 *>(smem_raw);          // [16 * RP]
    __shared__ double2 twz_s[(MZ > 1 ? MZ - 1 : 1) * 16];
    __shared__ double2 twy_s[16];
    const int tid = threadIdx.x;
    const int my = a.my;
    const int n2y = blockIdx.x % my;
    const int g0 = blockIdx.x / my, G = gridDim.x / my;
    for (int e = tid; e < (MZ - 1) * 16; e += NT) twz_s[e] = a.twz[(e & 15) * ((e >> 4) + 1)];
    if (tid < 16) twy_s[tid] = a.twy[n2y * tid];
    __syncthreads();
    const int64_t nplanes = (int64_t)a.ncol * a.nx;
    for (int64_t cx = g0; cx < nplanes; cx += G) {
        const int64_t col = cx / a.nx;
        const int64_t x = cx - col * a.nx;
        const double2 *src = a.X + col * a.ldx + x * a.ny * NZ;
        double2 *dst = a.W + col * a.ldw + x * a.ny * NZ;
        // z stage A: radix-MZ over n1, twiddle w_NZ^{n2 k1}
#pragma unroll
        for (int item = tid; item < 256; item += NT) {
            const int j = item >> 4, n2 = item & 15;
            const double2 *row = src + (int64_t)(j * my + n2y) * NZ + n2;
            double re[MZ], im[MZ];
#pragma unroll
            for (int n1 = 0; n1 < MZ; ++n1) { const double2 v = ld_nc(row + n1 * 16); re[n1] = v.x; im[n1] = v.y; }
            Dft<MZ>::run(re, im);
#pragma unroll
            for (int k = 1; k < MZ; ++k) { const double2 w = twz_s[(k - 1) * 16 + n2]; tw_mul(re[k], im[k], w.x, -w.y); }
#pragma unroll
            for (int k = 0; k < MZ; ++k) S[j * RP + k * 17 + n2] = make_double2(re[k], im[k]);
        }
        __syncthreads();
        // z stage B: radix-16 over n2, in place (position k1*16 + k2 <- frequency k1 + MZ*k2)
        for (int item = tid; item < 16 * MZ; item += NT) {
            double2 *p = S + item * 17;
            double br[16], bi[16];
#pragma unroll
            for (int t = 0; t < 16; ++t) { const double2 v = p[t]; br[t] = v.x; bi[t] = v.y; }
            Dft<16>::run(br, bi);
#pragma unroll
            for (int t = 0; t < 16; ++t) p[t] = make_double2(br[t], bi[t]);
        }
        __syncthreads();
        // y stage A: radix-16 over the 16 rows, twiddle w_NY^{n2y k1}, store row k1*my + n2y
        for (int p = tid; p < NZ; p += NT) {
            const int sp = (p >> 4) * 17 + (p & 15);
            double br[16], bi[16];
#pragma unroll
            for (int j = 0; j < 16; ++j) { const double2 v = S[j * RP + sp]; br[j] = v.x; bi[j] = v.y; }
            Dft<16>::run(br, bi);
#pragma unroll
            for (int k = 1; k < 16; ++k) { const double2 w = twy_s[k]; tw_mul(br[k], bi[k], w.x, -w.y); }
#pragma unroll
            for (int k = 0; k < 16; ++k) dst[(int64_t)(k * my + n2y) * NZ + p] = make_double2(br[k], bi[k]);
        }
        __syncthreads();
    }
}

// ---------------------------------------------------------------------------------------------
// y inverse stage A' + z inverse + V_loc.  Mirror of the kernel above; W -> HX (may be in place:
// a tile reads and writes the same 16 rows).  CTA b owns n2y = b % my and the x planes
// g0, g0 + G, ...; for each plane it runs over ALL columns of the batch (the 16 rows of v(r) stay
// hot in L1/L2).  Per tile: the k-space rows of the NEXT tile (double buffered) and the psi rows of
// THIS tile (consumed two phases later) arrive by cp.async.
template <int NZ, int MINB>
__global__ void __launch_bounds__(128, MINB) fft3_inv_yz_kernel(Fft3Args a)
{
    constexpr int MZ = ZyCfg<NZ>::MZ, RP = ZyCfg<NZ>::RP, TILE = ZyCfg<NZ>::TILE, NT = 128;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double2 *Sw0 = reinterpret_cast<double2 *>(smem_raw);
    double2 *Sp = Sw0 + 2 * TILE;                               // psi rows, dense [16][NZ]
    __shared__ double2 twz_s[(MZ > 1 ? MZ - 1 : 1) * 16];
    __shared__ double2 twy_s[16];
    const int tid = threadIdx.x;
    const int my = a.my;
    const int n2y = blockIdx.x % my;
    const int g0 = blockIdx.x / my, G = gridDim.x / my;
    for (int e = tid; e < (MZ - 1) * 16; e += NT) twz_s[e] = a.twz[(e & 15) * ((e >> 4) + 1)];
    if (tid < 16) twy_s[tid] = a.twy[n2y * tid];
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
        const double2 *src = a.W + col * a.ldw + po;
        double2 *S = Sw0 + buf * TILE;
#pragma unroll
        for (int e = tid; e < 16 * NZ; e += NT) {
            const int k = e / NZ, p = e - k * NZ;
            cp_async16(S + k * RP + (p >> 4) * 17 + (p & 15), src + (int64_t)(k * my + n2y) * NZ + p);
        }
    };
    auto issue_psi = [&](int64_t t) {
        int64_t col;
        const int64_t po = plane_off(t, col);
        const double2 *src = a.X + col * a.ldx + po;
#pragma unroll
        for (int e = tid; e < 16 * NZ; e += NT) {
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
        const double *vl = a.vloc + po;
        double2 *dst = a.HX + col * a.ldhx + po;
        // y inverse stage A': conj twiddle, radix-16 over k1y (swapped domain) -> row j = n1y, in place
        for (int p = tid; p < NZ; p += NT) {
            double2 *c = S + (p >> 4) * 17 + (p & 15);
            double br[16], bi[16];
#pragma unroll
            for (int k = 0; k < 16; ++k) { const double2 v = c[k * RP]; br[k] = v.x; bi[k] = v.y; }
#pragma unroll
            for (int k = 1; k < 16; ++k) { const double2 w = twy_s[k]; tw_mul(bi[k], br[k], w.x, -w.y); }
            Dft<16>::run(bi, br);
#pragma unroll
            for (int j = 0; j < 16; ++j) c[j * RP] = make_double2(br[j], bi[j]);
        }
        __syncthreads();
        // z inverse stage B': radix-16 over k2z (swapped), in place
        for (int item = tid; item < 16 * MZ; item += NT) {
            double2 *p = S + item * 17;
            double br[16], bi[16];
#pragma unroll
            for (int q = 0; q < 16; ++q) { const double2 v = p[q]; br[q] = v.x; bi[q] = v.y; }
            Dft<16>::run(bi, br);
#pragma unroll
            for (int q = 0; q < 16; ++q) p[q] = make_double2(br[q], bi[q]);
        }
        cp_async_wait<1>();                                       // psi(t) has landed
        __syncthreads();
        // z inverse stage A': conj twiddle, radix-MZ over k1z (swapped) -> z = n1*16 + n2; + v psi
#pragma unroll
        for (int item = tid; item < 256; item += NT) {
            const int j = item >> 4, n2 = item & 15;
            double re[MZ], im[MZ];
#pragma unroll
            for (int k = 0; k < MZ; ++k) { const double2 v = S[j * RP + k * 17 + n2]; re[k] = v.x; im[k] = v.y; }
#pragma unroll
            for (int k = 1; k < MZ; ++k) { const double2 w = twz_s[(k - 1) * 16 + n2]; tw_mul(im[k], re[k], w.x, -w.y); }
            Dft<MZ>::run(im, re);
            const int64_t off = (int64_t)(j * my + n2y) * NZ + n2;
#pragma unroll
            for (int n1 = 0; n1 < MZ; ++n1) {
                const double2 ps = Sp[j * NZ + n1 * 16 + n2];
                const double vv = __ldg(vl + off + n1 * 16);
                dst[off + n1 * 16] = make_double2(fma(vv, ps.x, re[n1]), fma(vv, ps.y, im[n1]));
            }
        }
        __syncthreads();
    }
    cp_async_wait<0>();
}

// ---------------------------------------------------------------------------------------------
// y stage B, x forward, kinetic factor, x inverse, y stage B'.  In place on W.
// Tile = (column, k1y, z-chunk): S[x][line], line = jy*TZ + z, odd pitch P = lines + 1.
template <int MY, int NX, int TZ, int NT>
__device__ __forceinline__ void fft3_x_load_y(const Fft3Args &a, const double2 *base, double2 *S, int P, int tid)
{
    // items are taken two at a time so that both items' global loads are in flight together
    int item = tid;
    for (; item + NT < NX * TZ; item += 2 * NT) {
        const int z0 = item % TZ, x0 = item / TZ, z1 = (item + NT) % TZ, x1 = (item + NT) / TZ;
        const double2 *p0 = base + (int64_t)x0 * a.ny * a.nz + z0;
        const double2 *p1 = base + (int64_t)x1 * a.ny * a.nz + z1;
        double re0[MY], im0[MY], re1[MY], im1[MY];
#pragma unroll
        for (int j = 0; j < MY; ++j) { const double2 v = p0[(int64_t)j * a.nz]; re0[j] = v.x; im0[j] = v.y; }
#pragma unroll
        for (int j = 0; j < MY; ++j) { const double2 v = p1[(int64_t)j * a.nz]; re1[j] = v.x; im1[j] = v.y; }
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
        for (int j = 0; j < MY; ++j) { const double2 v = ptr[(int64_t)j * a.nz]; re[j] = v.x; im[j] = v.y; }
        Dft<MY>::run(re, im);
#pragma unroll
        for (int j = 0; j < MY; ++j) S[x * P + j * TZ + z] = make_double2(re[j], im[j]);
    }
}

template <int MY, int NX, int TZ, int NT>
__device__ __forceinline__ void fft3_x_store_y(const Fft3Args &a, double2 *base, const double2 *S, int P, int tid)
{
    for (int item = tid; item < NX * TZ; item += NT) {
        const int z = item % TZ, x = item / TZ;
        double2 *ptr = base + (int64_t)x * a.ny * a.nz + z;
        double re[MY], im[MY];
#pragma unroll
        for (int j = 0; j < MY; ++j) { const double2 v = S[x * P + j * TZ + z]; re[j] = v.x; im[j] = v.y; }
        Dft<MY>::run(im, re);
#pragma unroll
        for (int j = 0; j < MY; ++j) ptr[(int64_t)j * a.nz] = make_double2(re[j], im[j]);
    }
}

// Per-length launch shape: z points per tile (TZ*16 B contiguous per row), threads, CTAs per SM.
// (NT = 288 for 96, which fills the radix-16 phase in one round, measured 40 % slower than 256.)
template <int NX> struct XCfg;
template <> struct XCfg<16> { static constexpr int TZ = 8, NT = 32, MINB = 8; };
template <> struct XCfg<32> { static constexpr int TZ = 8, NT = 64, MINB = 8; };
template <> struct XCfg<48> { static constexpr int TZ = 8, NT = 96, MINB = 5; };
template <> struct XCfg<64> { static constexpr int TZ = 8, NT = 128, MINB = 4; };
template <> struct XCfg<80> { static constexpr int TZ = 8, NT = 224, MINB = 2; };
template <> struct XCfg<96> { static constexpr int TZ = 8, NT = 256, MINB = 2; };
template <> struct XCfg<112> { static constexpr int TZ = 8, NT = 256, MINB = 2; };
template <> struct XCfg<128> { static constexpr int TZ = 4, NT = 256, MINB = 2; };
template <> struct XCfg<160> { static constexpr int TZ = 4, NT = 256, MINB = 2; };
template <> struct XCfg<192> { static constexpr int TZ = 4, NT = 256, MINB = 1; };
template <> struct XCfg<256> { static constexpr int TZ = 2, NT = 256, MINB = 1; };

template <int NX, int TZ, int NT, int MINB>
__global__ void __maxnreg__(((65536 / (NT * MINB)) / 8 * 8) > 255 ? 255 : ((65536 / (NT * MINB)) / 8 * 8)) fft3_x_kernel(Fft3Args a)
{
    constexpr int MX = NX / 16;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double2 *S = reinterpret_cast<double2 *>(smem_raw);
    __shared__ double2 twx_s[(MX > 1 ? MX - 1 : 1) * 16];
    __shared__ double kinx_s[NX];
    const int tid = threadIdx.x;
    const int my = a.my, lines = my * TZ, P = lines + 1;
    for (int e = tid; e < (MX - 1) * 16; e += NT) twx_s[e] = a.twx[(e & 15) * ((e >> 4) + 1)];
    for (int e = tid; e < NX; e += NT) kinx_s[e] = a.kin_x[e];
    __syncthreads();
    const int zchunks = a.nz / TZ;
    const int64_t per_col = (int64_t)16 * zchunks;
    const int64_t ntiles = per_col * a.ncol;
    for (int64_t tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
        const int64_t colf = tile / per_col;
        const int rem = (int)(tile - colf * per_col);
        const int64_t col = a.ncol - 1 - colf;     // zig-zag: the forward kernel ended on the last column, start there (L2)
        const int k1y = rem / zchunks, zc = rem - k1y * zchunks;
        double2 *base = a.W + col * a.ldw + (int64_t)(k1y * my) * a.nz + zc * TZ;
        switch (my) {
        case 1: fft3_x_load_y<1, NX, TZ, NT>(a, base, S, P, tid); break;
        case 2: fft3_x_load_y<2, NX, TZ, NT>(a, base, S, P, tid); break;
        case 3: fft3_x_load_y<3, NX, TZ, NT>(a, base, S, P, tid); break;
        case 4: fft3_x_load_y<4, NX, TZ, NT>(a, base, S, P, tid); break;
        case 5: fft3_x_load_y<5, NX, TZ, NT>(a, base, S, P, tid); break;
        case 6: fft3_x_load_y<6, NX, TZ, NT>(a, base, S, P, tid); break;
        case 7: fft3_x_load_y<7, NX, TZ, NT>(a, base, S, P, tid); break;
        case 8: fft3_x_load_y<8, NX, TZ, NT>(a, base, S, P, tid); break;
        case 10: fft3_x_load_y<10, NX, TZ, NT>(a, base, S, P, tid); break;
        case 12: fft3_x_load_y<12, NX, TZ, NT>(a, base, S, P, tid); break;
        default: fft3_x_load_y<16, NX, TZ, NT>(a, base, S, P, tid); break;
        }
        __syncthreads();
        // x stage A: radix-MX over n1 (x = n1*16 + n2), twiddle, in place
        for (int item = tid; item < lines * 16; item += NT) {
            const int n2 = item & 15, line = item >> 4;
            double2 *p = S + n2 * P + line;
            double re[MX], im[MX];
#pragma unroll
            for (int n1 = 0; n1 < MX; ++n1) { const double2 v = p[n1 * 16 * P]; re[n1] = v.x; im[n1] = v.y; }
            Dft<MX>::run(re, im);
#pragma unroll
            for (int k = 1; k < MX; ++k) { const double2 w = twx_s[(k - 1) * 16 + n2]; tw_mul(re[k], im[k], w.x, -w.y); }
#pragma unroll
            for (int k = 0; k < MX; ++k) p[k * 16 * P] = make_double2(re[k], im[k]);
        }
        __syncthreads();
        // x stage B (radix-16 over n2) -> frequency kx = k1 + MX*k2; kinetic factor; inverse stage B'
        for (int item = tid; item < lines * MX; item += NT) {
            const int line = item % lines, k1 = item / lines;
            double2 *p = S + k1 * 16 * P + line;
            double br[16], bi[16];
#pragma unroll
            for (int t = 0; t < 16; ++t) { const double2 v = p[t * P]; br[t] = v.x; bi[t] = v.y; }
            Dft<16>::run(br, bi);
            const int jy = line / TZ, z = line - jy * TZ;
            const double tin = __ldg(a.kin_yz + (int64_t)(k1y * my + jy) * a.nz + zc * TZ + z);
#pragma unroll
            for (int k2 = 0; k2 < 16; ++k2) {
                const double f = kinx_s[k1 + MX * k2] + tin;
                br[k2] *= f; bi[k2] *= f;
            }
            Dft<16>::run(bi, br);                  // swapped domain from here on
#pragma unroll
            for (int t = 0; t < 16; ++t) p[t * P] = make_double2(br[t], bi[t]);
        }
        __syncthreads();
        // x inverse stage A': conj twiddle, radix-MX over k1 -> x = n1*16 + n2
        for (int item = tid; item < lines * 16; item += NT) {
            const int n2 = item & 15, line = item >> 4;
            double2 *p = S + n2 * P + line;
            double re[MX], im[MX];
#pragma unroll
            for (int k = 0; k < MX; ++k) { const double2 v = p[k * 16 * P]; re[k] = v.x; im[k] = v.y; }
#pragma unroll
            for (int k = 1; k < MX; ++k) { const double2 w = twx_s[(k - 1) * 16 + n2]; tw_mul(im[k], re[k], w.x, -w.y); }
            Dft<MX>::run(im, re);
#pragma unroll
            for (int n1 = 0; n1 < MX; ++n1) p[n1 * 16 * P] = make_double2(re[n1], im[n1]);
        }
        __syncthreads();
        switch (my) {
        case 1: fft3_x_store_y<1, NX, TZ, NT>(a, base, S, P, tid); break;
        case 2: fft3_x_store_y<2, NX, TZ, NT>(a, base, S, P, tid); break;
        case 3: fft3_x_store_y<3, NX, TZ, NT>(a, base, S, P, tid); break;
        case 4: fft3_x_store_y<4, NX, TZ, NT>(a, base, S, P, tid); break;
        case 5: fft3_x_store_y<5, NX, TZ, NT>(a, base, S, P, tid); break;
        case 6: fft3_x_store_y<6, NX, TZ, NT>(a, base, S, P, tid); break;
        case 7: fft3_x_store_y<7, NX, TZ, NT>(a, base, S, P, tid); break;
        case 8: fft3_x_store_y<8, NX, TZ, NT>(a, base, S, P, tid); break;
        case 10: fft3_x_store_y<10, NX, TZ, NT>(a, base, S, P, tid); break;
        case 12: fft3_x_store_y<12, NX, TZ, NT>(a, base, S, P, tid); break;
        default: fft3_x_store_y<16, NX, TZ, NT>(a, base, S, P, tid); break;
        }
        __syncthreads();
    }
}

}  // namespace rsdft
