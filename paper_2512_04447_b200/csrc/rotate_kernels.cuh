// Rayleigh-Ritz update of LOBPCG (Knyazev's method, cited PAPER.md:19,124):
//   Out[r, j] = sum_c Y[r, c] * C[c, j],   r < Ng grid points, c < n subspace columns, j < m new columns,
// e.g. X' = Y C_X, HX' = HY C_X, P' = [W, P] C_P.  Tall-skinny times small: M = Ng (~10^6), K = n (~1500),
// N = m (~500).  Like the Gram contraction it is a dense FP64 product, so it runs on the FP64 tensor pipe
// (mma.sync.m8n8k4.f64, the only native FP64 MMA shape of sm_100a).  One complex product is 4 real MMAs in the plain
// form (M3 = false):  re += Ar*Br;  re += (-Ai)*Bi;  im += Ar*Bi;  im += Ai*Br,  and 3 in the 3M form the launchers use
// (M3 = true, see the kernel templates below).
//
// Operand layouts.  A = Y is "M-major" in memory (a column of Y is contiguous in r), the opposite of what the
// row fragment of m8n8k4 wants, so a stage holds A as [k][r] with pitch TM+2 complex (pitch % 8 == 2: the 8
// lanes of an LDS.128 phase, 2 rows x 4 k, hit 8 distinct 16-byte bank groups).  B = C is column-major
// (c contiguous), i.e. K-major like the Gram operands: [j][k] with pitch KC+4.
// One CTA owns a TM x TN output tile and walks all of K in KC-chunks through a cp.async pipeline; no split-K
// (K is short, M supplies the parallelism).  Tiles sharing the same rows r are adjacent in the grid so that
// their Y panel is read from HBM once and shared through L2.
#pragma once
#include "async_copy.cuh"
#include <cuda_runtime.h>
#include <stdint.h>

namespace rsdft {

struct RotateArgs {
    const double2 *Y;      // [n][ldy]   column c at c*ldy
    const double2 *C;      // [m][ldc]   column-major n x m: element (c, j) at c + j*ldc
    double2 *Out;          // [m][ldo]   column j at j*ldo
    int64_t ldy, ldo, ng;
    int32_t n, m, ldc;
    int32_t jtiles;        // ceil(m / TN)
};

__device__ __forceinline__ void rot_dmma884(double &d0, double &d1, double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}

template <int WGM, int WGN, int FA, int FB, int KC, int STAGES>
struct RotateCfg {
    static constexpr int TM = WGM * FA * 8, TN = WGN * FB * 8;
    static constexpr int THREADS = WGM * WGN * 32;
    static constexpr int PA = TM + 2;              // A stage: [KC][PA]
    static constexpr int PB = KC + 4;              // B stage: [TN][PB]
    static constexpr int STAGE_ELEMS = KC * PA + TN * PB;
    static constexpr size_t SMEM = (size_t)STAGES * STAGE_ELEMS * sizeof(double2);
};

// M3: the complex product a b from three real MMAs (K1 += (Ar + Ai) Br, K2 += Ar (Bi - Br), K3 += Ai (Br + Bi);
// re = K1 - K3, im = K1 + K2), as in gram_kernels.cuh; needs a third accumulator set, hence smaller tiles.
template <int WGM, int WGN, int FA, int FB, int KC, int STAGES, bool M3 = false, int MINB = 1>
__global__ void __launch_bounds__(WGM *WGN * 32, MINB) rotate_dmma_kernel(RotateArgs a)
{
    using Cfg = RotateCfg<WGM, WGN, FA, FB, KC, STAGES>;
    constexpr int TM = Cfg::TM, TN = Cfg::TN, PA = Cfg::PA, PB = Cfg::PB, NT = Cfg::THREADS;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double2 *sm = reinterpret_cast<double2 *>(smem_raw);

    const int64_t unit = blockIdx.x;
    const int64_t rt = unit / a.jtiles;
    const int jt = (int)(unit - rt * a.jtiles);
    const int64_t r0 = rt * TM;
    const int j0 = jt * TN;
    const int nch = (a.n + KC - 1) / KC;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int wm = warp / WGN, wn = warp % WGN;
    const int g = lane >> 2, t = lane & 3;

    auto load_stage = [&](int stage, int chunk) {
        double2 *As = sm + (size_t)stage * Cfg::STAGE_ELEMS;
        double2 *Bs = As + KC * PA;
        const int c0 = chunk * KC;
#pragma unroll
        for (int e = tid; e < KC * TM; e += NT) {             // A: KC columns of Y, TM contiguous grid points each
            const int k = e / TM, r = e - k * TM;
            double2 *d = As + k * PA + r;
            if (c0 + k < a.n && r0 + r < a.ng) cp_async16(d, a.Y + (int64_t)(c0 + k) * a.ldy + r0 + r);
            else *d = make_double2(0.0, 0.0);
        }
#pragma unroll
        for (int e = tid; e < TN * KC; e += NT) {             // B: TN columns of C, KC contiguous rows each
            const int j = e / KC, k = e - j * KC;
            double2 *d = Bs + j * PB + k;
            if (j0 + j < a.m && c0 + k < a.n) cp_async16(d, a.C + (int64_t)(j0 + j) * a.ldc + c0 + k);
            else *d = make_double2(0.0, 0.0);
        }
    };

    double cre[FA][FB][2], cim[FA][FB][2];       // 4M: re, im;  3M: K1, K2
    double ck3[M3 ? FA : 1][M3 ? FB : 1][2];     // 3M: K3
#pragma unroll
    for (int x = 0; x < FA; ++x)
#pragma unroll
        for (int y = 0; y < FB; ++y) {
            cre[x][y][0] = cre[x][y][1] = 0.0; cim[x][y][0] = cim[x][y][1] = 0.0;
            if (M3) ck3[x][y][0] = ck3[x][y][1] = 0.0;
        }

#pragma unroll
    for (int s = 0; s < STAGES - 1; ++s) {
        if (s < nch) load_stage(s, s);
        cp_async_commit();
    }
    for (int ch = 0; ch < nch; ++ch) {
        cp_async_wait<STAGES - 2>();
        __syncthreads();
        {
            const int nx = ch + STAGES - 1;
            if (nx < nch) load_stage(nx % STAGES, nx);
            cp_async_commit();
        }
        const double2 *As = sm + (size_t)(ch % STAGES) * Cfg::STAGE_ELEMS + t * PA + wm * FA * 8 + g;
        const double2 *Bs = sm + (size_t)(ch % STAGES) * Cfg::STAGE_ELEMS + KC * PA + (wn * FB * 8 + g) * PB + t;
#pragma unroll
        for (int kk = 0; M3 && kk < KC; kk += 4) {
            double b0[FB], b1[FB], b2[FB];
#pragma unroll
            for (int y = 0; y < FB; ++y) { const double2 v = Bs[y * 8 * PB + kk]; b0[y] = v.x; b1[y] = v.y - v.x; b2[y] = v.x + v.y; }
#pragma unroll
            for (int x = 0; x < FA; ++x) {
                const double2 v = As[kk * PA + x * 8];
                const double a0 = v.x + v.y;
#pragma unroll
                for (int y = 0; y < FB; ++y) {
                    rot_dmma884(cre[x][y][0], cre[x][y][1], a0, b0[y]);
                    rot_dmma884(cim[x][y][0], cim[x][y][1], v.x, b1[y]);
                    rot_dmma884(ck3[x][y][0], ck3[x][y][1], v.y, b2[y]);
                }
            }
        }
#pragma unroll
        for (int kk = 0; !M3 && kk < KC; kk += 4) {
            double br[FB], bi[FB];
#pragma unroll
            for (int y = 0; y < FB; ++y) { const double2 v = Bs[y * 8 * PB + kk]; br[y] = v.x; bi[y] = v.y; }
#pragma unroll
            for (int x = 0; x < FA; ++x) {
                const double2 v = As[kk * PA + x * 8];
                const double ar = v.x, ai = v.y, nai = -v.y;
#pragma unroll
                for (int y = 0; y < FB; ++y) {
                    rot_dmma884(cre[x][y][0], cre[x][y][1], ar, br[y]);
                    rot_dmma884(cim[x][y][0], cim[x][y][1], ar, bi[y]);
                }
#pragma unroll
                for (int y = 0; y < FB; ++y) {
                    rot_dmma884(cre[x][y][0], cre[x][y][1], nai, bi[y]);
                    rot_dmma884(cim[x][y][0], cim[x][y][1], ai, br[y]);
                }
            }
        }
    }
    cp_async_wait<0>();

    // epilogue: C fragment element e of (x, y) is row g, column 2t+e of that 8x8 tile; for a fixed output
    // column the 8 lanes g = 0..7 write 8 consecutive grid points (128 B)
#pragma unroll
    for (int x = 0; x < FA; ++x)
#pragma unroll
        for (int y = 0; y < FB; ++y)
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                const int64_t r = r0 + (wm * FA + x) * 8 + g;
                const int j = j0 + (wn * FB + y) * 8 + 2 * t + e;
                if (r < a.ng && j < a.m)
                    a.Out[(int64_t)j * a.ldo + r] = M3 ? make_double2(cre[x][y][e] - ck3[x][y][e], cre[x][y][e] + cim[x][y][e]) : make_double2(cre[x][y][e], cim[x][y][e]);
            }
}

// ------------------------------------------------------------------------------------------------------------
// Two-output update with the LOBPCG residual fused into the epilogue:
//   X'[r, j] = sum_c Y[r, c] C[c, j],   HX'[r, j] = sum_c HY[r, c] C[c, j],   R[r, j] = HX'[r, j] - lambda_j X'[r, j].
// One CTA owns a TM x TN tile of BOTH products: every C stage in shared memory feeds the Y and the HY
// accumulators, so C is staged once, Y and HY are read once, and the three outputs are written once.
struct Rotate2Args {
    const double2 *Y, *HY;  // [n][ldy], [n][ldhy]
    const double2 *C;       // column-major n x m
    const double *lambda;   // [m] real Ritz values (may be NULL when R is NULL)
    double2 *X, *HX, *R;    // [m][ldx], [m][ldhx], [m][ldr]; any may be NULL
    int64_t ldy, ldhy, ldx, ldhx, ldr, ng;
    int32_t n, m, ldc, jtiles;
};

template <int WGM, int WGN, int FA, int FB, int KC, int STAGES>
struct Rotate2Cfg {
    static constexpr int TM = WGM * FA * 8, TN = WGN * FB * 8;
    static constexpr int THREADS = WGM * WGN * 32;
    static constexpr int PA = TM + 2;              // A stages: [KC][PA] for Y and for HY
    static constexpr int PB = KC + 4;              // B stage: [TN][PB]
    static constexpr int STAGE_ELEMS = 2 * KC * PA + TN * PB;
    static constexpr size_t SMEM = (size_t)STAGES * STAGE_ELEMS * sizeof(double2);
};

template <int WGM, int WGN, int FA, int FB, int KC, int STAGES, bool M3 = false, int MINB = 1>
__global__ void __launch_bounds__(WGM *WGN * 32, MINB) rotate2_dmma_kernel(Rotate2Args a)
{
    using Cfg = Rotate2Cfg<WGM, WGN, FA, FB, KC, STAGES>;
    constexpr int TM = Cfg::TM, TN = Cfg::TN, PA = Cfg::PA, PB = Cfg::PB, NT = Cfg::THREADS;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double2 *sm = reinterpret_cast<double2 *>(smem_raw);

    const int64_t unit = blockIdx.x;
    const int64_t rt = unit / a.jtiles;
    const int jt = (int)(unit - rt * a.jtiles);
    const int64_t r0 = rt * TM;
    const int j0 = jt * TN;
    const int nch = (a.n + KC - 1) / KC;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int wm = warp / WGN, wn = warp % WGN;
    const int g = lane >> 2, t = lane & 3;

    auto load_stage = [&](int stage, int chunk) {
        double2 *As = sm + (size_t)stage * Cfg::STAGE_ELEMS;
        double2 *Hs = As + KC * PA;
        double2 *Bs = Hs + KC * PA;
        const int c0 = chunk * KC;
#pragma unroll
        for (int e = tid; e < KC * TM; e += NT) {
            const int k = e / TM, r = e - k * TM;
            if (c0 + k < a.n && r0 + r < a.ng) {
                cp_async16(As + k * PA + r, a.Y + (int64_t)(c0 + k) * a.ldy + r0 + r);
                cp_async16(Hs + k * PA + r, a.HY + (int64_t)(c0 + k) * a.ldhy + r0 + r);
            } else {
                As[k * PA + r] = make_double2(0.0, 0.0);
                Hs[k * PA + r] = make_double2(0.0, 0.0);
            }
        }
#pragma unroll
        for (int e = tid; e < TN * KC; e += NT) {
            const int j = e / KC, k = e - j * KC;
            double2 *d = Bs + j * PB + k;
            if (j0 + j < a.m && c0 + k < a.n) cp_async16(d, a.C + (int64_t)(j0 + j) * a.ldc + c0 + k);
            else *d = make_double2(0.0, 0.0);
        }
    };

    double xre[FA][FB][2], xim[FA][FB][2], hre[FA][FB][2], him[FA][FB][2];      // 4M: re, im;  3M: K1, K2
    double xk3[M3 ? FA : 1][M3 ? FB : 1][2], hk3[M3 ? FA : 1][M3 ? FB : 1][2];  // 3M: K3
#pragma unroll
    for (int x = 0; x < FA; ++x)
#pragma unroll
        for (int y = 0; y < FB; ++y)
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                xre[x][y][e] = xim[x][y][e] = hre[x][y][e] = him[x][y][e] = 0.0;
                if (M3) xk3[x][y][e] = hk3[x][y][e] = 0.0;
            }

#pragma unroll
    for (int s = 0; s < STAGES - 1; ++s) {
        if (s < nch) load_stage(s, s);
        cp_async_commit();
    }
    for (int ch = 0; ch < nch; ++ch) {
        cp_async_wait<STAGES - 2>();
        __syncthreads();
        {
            const int nx = ch + STAGES - 1;
            if (nx < nch) load_stage(nx % STAGES, nx);
            cp_async_commit();
        }
        const double2 *As = sm + (size_t)(ch % STAGES) * Cfg::STAGE_ELEMS + t * PA + wm * FA * 8 + g;
        const double2 *Hs = As + KC * PA;
        const double2 *Bs = sm + (size_t)(ch % STAGES) * Cfg::STAGE_ELEMS + 2 * KC * PA + (wn * FB * 8 + g) * PB + t;
#pragma unroll
        for (int kk = 0; M3 && kk < KC; kk += 4) {
            double b0[FB], b1[FB], b2[FB];
#pragma unroll
            for (int y = 0; y < FB; ++y) { const double2 v = Bs[y * 8 * PB + kk]; b0[y] = v.x; b1[y] = v.y - v.x; b2[y] = v.x + v.y; }
#pragma unroll
            for (int x = 0; x < FA; ++x) {
                const double2 v = As[kk * PA + x * 8];
                const double2 w = Hs[kk * PA + x * 8];
                const double v0 = v.x + v.y, w0 = w.x + w.y;
#pragma unroll
                for (int y = 0; y < FB; ++y) {
                    rot_dmma884(xre[x][y][0], xre[x][y][1], v0, b0[y]);
                    rot_dmma884(xim[x][y][0], xim[x][y][1], v.x, b1[y]);
                    rot_dmma884(xk3[x][y][0], xk3[x][y][1], v.y, b2[y]);
                    rot_dmma884(hre[x][y][0], hre[x][y][1], w0, b0[y]);
                    rot_dmma884(him[x][y][0], him[x][y][1], w.x, b1[y]);
                    rot_dmma884(hk3[x][y][0], hk3[x][y][1], w.y, b2[y]);
                }
            }
        }
#pragma unroll
        for (int kk = 0; !M3 && kk < KC; kk += 4) {
            double br[FB], bi[FB];
#pragma unroll
            for (int y = 0; y < FB; ++y) { const double2 v = Bs[y * 8 * PB + kk]; br[y] = v.x; bi[y] = v.y; }
#pragma unroll
            for (int x = 0; x < FA; ++x) {
                const double2 v = As[kk * PA + x * 8];
                const double2 w = Hs[kk * PA + x * 8];
#pragma unroll
                for (int y = 0; y < FB; ++y) {
                    rot_dmma884(xre[x][y][0], xre[x][y][1], v.x, br[y]);
                    rot_dmma884(xim[x][y][0], xim[x][y][1], v.x, bi[y]);
                    rot_dmma884(hre[x][y][0], hre[x][y][1], w.x, br[y]);
                    rot_dmma884(him[x][y][0], him[x][y][1], w.x, bi[y]);
                }
                const double nvy = -v.y, nwy = -w.y;
#pragma unroll
                for (int y = 0; y < FB; ++y) {
                    rot_dmma884(xre[x][y][0], xre[x][y][1], nvy, bi[y]);
                    rot_dmma884(xim[x][y][0], xim[x][y][1], v.y, br[y]);
                    rot_dmma884(hre[x][y][0], hre[x][y][1], nwy, bi[y]);
                    rot_dmma884(him[x][y][0], him[x][y][1], w.y, br[y]);
                }
            }
        }
    }
    cp_async_wait<0>();

#pragma unroll
    for (int y = 0; y < FB; ++y)
#pragma unroll
        for (int e = 0; e < 2; ++e) {
            const int j = j0 + (wn * FB + y) * 8 + 2 * t + e;
            if (j >= a.m) continue;
            const double lam = a.R ? a.lambda[j] : 0.0;
#pragma unroll
            for (int x = 0; x < FA; ++x) {
                const int64_t r = r0 + (wm * FA + x) * 8 + g;
                if (r >= a.ng) continue;
                const double xr = M3 ? xre[x][y][e] - xk3[x][y][e] : xre[x][y][e], xi = M3 ? xre[x][y][e] + xim[x][y][e] : xim[x][y][e];
                const double hr = M3 ? hre[x][y][e] - hk3[x][y][e] : hre[x][y][e], hi = M3 ? hre[x][y][e] + him[x][y][e] : him[x][y][e];
                if (a.X) a.X[(int64_t)j * a.ldx + r] = make_double2(xr, xi);
                if (a.HX) a.HX[(int64_t)j * a.ldhx + r] = make_double2(hr, hi);
                if (a.R) a.R[(int64_t)j * a.ldr + r] = make_double2(fma(-lam, xr, hr), fma(-lam, xi, hi));
            }
        }
}

}  // namespace rsdft
