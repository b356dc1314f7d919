// Batched 3-D complex128 FFT passes for rsdft_apply_h (PAPER.md:19 task (1)).
//
// Every supported length is N = 16*M (M = 1..8).  A 1-D transform is two register stages with
// one shared-memory exchange:
//   role A thread (fixed n2 in [0,16)):  holds x[n1*16 + n2], n1 in [0,M)  -> radix-M, then the
//                                         inter-stage twiddle w_N^{n2*k1} (M-1 values kept in registers)
//   role B thread (fixed k1 in [0,M)):   holds the 16 values n2 in [0,16)  -> radix-16 -> X[k1 + M*k2]
// Forward  = A -> exchange -> B.   Inverse = B -> exchange -> A on (im, re)-swapped data, which is
// exactly the unnormalised inverse (swap . F . swap).  k-space is kept in natural index order.
//
// Passes of apply_h (HX doubles as the scratch):
//   z forward (X -> HX), y forward (in place), x forward * t(k)/Ng * x inverse (one kernel, in
//   place), y inverse (in place), z inverse + v(r) psi(r) (in place, re-reads X).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "fft_codelets.cuh"

namespace rsdft {

__device__ __forceinline__ double2 ldg2(const double2 *p) { return __ldg(p); }

// ---------------------------------------------------------------------------------------------
// Strided lines: tensor [ncol][outer][N][inner] (inner contiguous).  One tile = all N points of
// T adjacent lines (T*16 B contiguous per axis index).  Block = 16*T threads.
// MODE 0: forward.  MODE 1: inverse.  MODE 2: forward, scale by kinetic factor, inverse (x axis).
struct StridedArgs {
    double2 *data;          // in place
    int64_t ld;             // column stride (elements)
    int64_t inner;          // contiguous extent = stride between successive axis points
    int32_t outer;          // slabs per column
    int32_t chunks;         // inner / T
    int64_t ntiles;         // ncol * outer * chunks
    const double2 *tw;      // w_N^m = (cos, -sin)(2 pi m / N), m in [0, N)
    const double *kin_axis; // MODE 2: t_x[kx] / Ng                      [N]
    const double *kin_inner;// MODE 2: (t_y[ky] + t_z[kz]) / Ng          [inner]
};

template <int N, int T, int MODE>
__global__ void __launch_bounds__(16 * T) fft_strided_kernel(StridedArgs a)
{
    constexpr int M = N / 16;
    __shared__ double2 sm[N * T];
    const int tid = threadIdx.x;
    // role A
    const int n2 = tid / T, tA = tid % T;
    // role B
    const bool isB = tid < M * T;
    const int k1 = tid / T, tB = tid % T;      // valid when isB

    double twc[M > 1 ? M - 1 : 1], tws[M > 1 ? M - 1 : 1];
#pragma unroll
    for (int k = 1; k < M; ++k) {
        const double2 w = ldg2(a.tw + n2 * k);
        twc[k - 1] = w.x; tws[k - 1] = -w.y;   // tw_mul wants (c, s) of c - i s
    }

    for (int64_t tile = blockIdx.x; tile < a.ntiles; tile += gridDim.x) {
        const int64_t per_col = (int64_t)a.outer * a.chunks;
        const int64_t col = tile / per_col;
        const int64_t rem = tile - col * per_col;
        const int64_t o = rem / a.chunks, ch = rem - o * a.chunks;
        double2 *base = a.data + col * a.ld + o * (int64_t)N * a.inner + ch * T;

        if constexpr (MODE == 0 || MODE == 2) {
            double re[M], im[M];
#pragma unroll
            for (int n1 = 0; n1 < M; ++n1) {
                const double2 v = base[(int64_t)(n1 * 16 + n2) * a.inner + tA];
                re[n1] = v.x; im[n1] = v.y;
            }
            Dft<M>::run(re, im);
#pragma unroll
            for (int k = 1; k < M; ++k) tw_mul(re[k], im[k], twc[k - 1], tws[k - 1]);
#pragma unroll
            for (int k = 0; k < M; ++k) sm[(k * 16 + n2) * T + tA] = make_double2(re[k], im[k]);
            __syncthreads();
            if (isB) {
                double br[16], bi[16];
#pragma unroll
                for (int j = 0; j < 16; ++j) { const double2 v = sm[(k1 * 16 + j) * T + tB]; br[j] = v.x; bi[j] = v.y; }
                Dft<16>::run(br, bi);
                if constexpr (MODE == 0) {
#pragma unroll
                    for (int k2 = 0; k2 < 16; ++k2)
                        base[(int64_t)(k1 + M * k2) * a.inner + tB] = make_double2(br[k2], bi[k2]);
                } else {
                    const double tin = a.kin_inner[ch * T + tB];
#pragma unroll
                    for (int k2 = 0; k2 < 16; ++k2) {
                        const double f = a.kin_axis[k1 + M * k2] + tin;
                        br[k2] *= f; bi[k2] *= f;
                    }
                    Dft<16>::run(bi, br);      // swapped domain from here on
#pragma unroll
                    for (int j = 0; j < 16; ++j) sm[(k1 * 16 + j) * T + tB] = make_double2(br[j], bi[j]);
                }
            }
            if constexpr (MODE == 2) {
                __syncthreads();
                double re2[M], im2[M];
#pragma unroll
                for (int k = 0; k < M; ++k) { const double2 v = sm[(k * 16 + n2) * T + tA]; re2[k] = v.x; im2[k] = v.y; }
#pragma unroll
                for (int k = 1; k < M; ++k) tw_mul(im2[k], re2[k], twc[k - 1], tws[k - 1]);
                Dft<M>::run(im2, re2);
#pragma unroll
                for (int n1 = 0; n1 < M; ++n1)
                    base[(int64_t)(n1 * 16 + n2) * a.inner + tA] = make_double2(re2[n1], im2[n1]);
            }
            __syncthreads();
        } else {   // MODE 1: inverse
            if (isB) {
                double br[16], bi[16];
#pragma unroll
                for (int k2 = 0; k2 < 16; ++k2) {
                    const double2 v = base[(int64_t)(k1 + M * k2) * a.inner + tB];
                    br[k2] = v.x; bi[k2] = v.y;
                }
                Dft<16>::run(bi, br);
#pragma unroll
                for (int j = 0; j < 16; ++j) sm[(k1 * 16 + j) * T + tB] = make_double2(br[j], bi[j]);
            }
            __syncthreads();
            double re2[M], im2[M];
#pragma unroll
            for (int k = 0; k < M; ++k) { const double2 v = sm[(k * 16 + n2) * T + tA]; re2[k] = v.x; im2[k] = v.y; }
#pragma unroll
            for (int k = 1; k < M; ++k) tw_mul(im2[k], re2[k], twc[k - 1], tws[k - 1]);
            Dft<M>::run(im2, re2);
#pragma unroll
            for (int n1 = 0; n1 < M; ++n1)
                base[(int64_t)(n1 * 16 + n2) * a.inner + tA] = make_double2(re2[n1], im2[n1]);
            __syncthreads();
        }
    }
}

// ---------------------------------------------------------------------------------------------
// Contiguous lines (z axis): L lines per block, block = 16*L threads.
// MODE 0: forward, in -> out.   MODE 1: inverse in place on `out`, then out = result + v(r) * in(r).
struct LinesArgs {
    const double2 *in;      // X (MODE 0 source; MODE 1: psi for the V_loc term)
    double2 *out;           // HX
    int64_t ld_in, ld_out;
    int64_t lines_per_col;  // Nx * Ny
    int64_t nlines;         // ncol * Nx * Ny
    const double2 *tw;
    const double *vloc;     // [Ng] (MODE 1)
};

template <int N, int L, int MODE>
__global__ void __launch_bounds__(16 * L) fft_lines_kernel(LinesArgs a)
{
    constexpr int M = N / 16;
    constexpr int PITCH = 17;
    __shared__ double2 sm[L * M * PITCH];
    const int tid = threadIdx.x;
    const int lA = tid / 16, n2 = tid % 16;             // role A
    const bool isB = tid < M * L;
    const int lB = tid / M, k1 = tid % M;               // role B (valid when isB)

    double twc[M > 1 ? M - 1 : 1], tws[M > 1 ? M - 1 : 1];
#pragma unroll
    for (int k = 1; k < M; ++k) {
        const double2 w = ldg2(a.tw + n2 * k);
        twc[k - 1] = w.x; tws[k - 1] = -w.y;
    }

    for (int64_t l0 = (int64_t)blockIdx.x * L; l0 < a.nlines; l0 += (int64_t)gridDim.x * L) {
        const int64_t lineA = l0 + lA, lineB = l0 + lB;
        const bool okA = lineA < a.nlines, okB = isB && lineB < a.nlines;
        const int64_t colA = lineA / a.lines_per_col, inA = lineA - colA * a.lines_per_col;
        const int64_t colB = lineB / a.lines_per_col, inB = lineB - colB * a.lines_per_col;
        if constexpr (MODE == 0) {
            if (okA) {
                const double2 *src = a.in + colA * a.ld_in + inA * N;
                double re[M], im[M];
#pragma unroll
                for (int n1 = 0; n1 < M; ++n1) { const double2 v = ldg2(src + n1 * 16 + n2); re[n1] = v.x; im[n1] = v.y; }
                Dft<M>::run(re, im);
#pragma unroll
                for (int k = 1; k < M; ++k) tw_mul(re[k], im[k], twc[k - 1], tws[k - 1]);
#pragma unroll
                for (int k = 0; k < M; ++k) sm[(lA * M + k) * PITCH + n2] = make_double2(re[k], im[k]);
            }
            __syncthreads();
            if (okB) {
                double br[16], bi[16];
#pragma unroll
                for (int j = 0; j < 16; ++j) { const double2 v = sm[tid * PITCH + j]; br[j] = v.x; bi[j] = v.y; }
                Dft<16>::run(br, bi);
                double2 *dst = a.out + colB * a.ld_out + inB * N;
#pragma unroll
                for (int k2 = 0; k2 < 16; ++k2) dst[k1 + M * k2] = make_double2(br[k2], bi[k2]);
            }
            __syncthreads();
        } else {
            if (okB) {
                const double2 *src = a.out + colB * a.ld_out + inB * N;
                double br[16], bi[16];
#pragma unroll
                for (int k2 = 0; k2 < 16; ++k2) { const double2 v = src[k1 + M * k2]; br[k2] = v.x; bi[k2] = v.y; }
                Dft<16>::run(bi, br);
#pragma unroll
                for (int j = 0; j < 16; ++j) sm[tid * PITCH + j] = make_double2(br[j], bi[j]);
            }
            __syncthreads();
            if (okA) {
                double re2[M], im2[M];
#pragma unroll
                for (int k = 0; k < M; ++k) { const double2 v = sm[(lA * M + k) * PITCH + n2]; re2[k] = v.x; im2[k] = v.y; }
#pragma unroll
                for (int k = 1; k < M; ++k) tw_mul(im2[k], re2[k], twc[k - 1], tws[k - 1]);
                Dft<M>::run(im2, re2);
                const double2 *psi = a.in + colA * a.ld_in + inA * N;
                const double *v = a.vloc + inA * N;
                double2 *dst = a.out + colA * a.ld_out + inA * N;
#pragma unroll
                for (int n1 = 0; n1 < M; ++n1) {
                    const int n = n1 * 16 + n2;
                    const double2 p = ldg2(psi + n);
                    const double vv = __ldg(v + n);
                    dst[n] = make_double2(fma(vv, p.x, re2[n1]), fma(vv, p.y, im2[n1]));
                }
            }
            __syncthreads();
        }
    }
}

}  // namespace rsdft
