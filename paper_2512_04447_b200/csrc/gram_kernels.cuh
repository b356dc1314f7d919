// Rayleigh-Ritz Gram matrices of LOBPCG (PAPER.md:19 task (2) "GEMM to construct the Hamiltonian
// and overlap matrices"):
//   S_sub[i,j] = sum_r conj(Y[r,i]) Y[r,j],    H_sub[i,j] = sum_r conj(Y[r,i]) HY[r,j].
//
// This is the one dense contraction of the path, so it runs on the FP64 tensor pipe: the only
// native FP64 MMA shape on sm_100a is DMMA.8x8x4 (mma.sync.m8n8k4.f64).  Both operands are
// "K-major" in memory (a column of Y is contiguous in r), which is exactly the row (A) / col (B)
// fragment layout of m8n8k4, so tiles are staged into shared memory as plain interleaved
// complex128 with cp.async and read back as one 128-bit LDS per fragment (re, im).
//
// One complex product conj(a) b = 3 real MMAs (the "3M" / Gauss form, as in BLAS ZGEMM3M):
//     K1 += (Ar - Ai) * Br,   K2 += Ar * (Bi - Br),   K3 += (-Ai) * (Br + Bi);     re = K1 - K3,   im = K1 + K2
// -- a quarter fewer tensor-core instructions than the 4-product form (re += Ar*Br + Ai*Bi, im += Ar*Bi - Ai*Br, kept as
// M3 = false for comparison) at the price of a third accumulator set, which is why the tile is 48 x 48 and not 96 x 96
// (a 96 x 96 tile with three accumulator sets would take 84 % of the SM's register file).  The operand combinations are
// formed once per fragment load.  The sums K1..K3 are up to twice as large as re / im, so the normwise error bound grows
// by a small constant (measured against the long-double oracle: see DESIGN.md); it is not componentwise stable, which
// the normwise parity bar of north_star does not ask for.
//
// Work decomposition: a unit = (K-slab, output tile).  Tiles are TM x TN complex; S_sub only
// needs its upper-triangular tiles (it is exactly Hermitian), H_sub is computed in full.
// Units are ordered slab-major so the ~148 CTAs resident at any time stream the SAME grid-point
// range and share their Y / HY panels through L2.  Every unit writes its partial tile to a
// workspace; gram_reduce_kernel then sums the slabs in a fixed order (deterministic), mirrors
// S_sub and writes both triangles.
#pragma once
#include "async_copy.cuh"
#include <cuda_runtime.h>
#include <stdint.h>

namespace rsdft {

struct GramTile { int16_t ti, tj, mat, pad; };   // mat 0: H_sub = Y^H HY, 1: S_sub = Y^H Y (upper tile, mirrored), 2: H_sub upper tile, mirrored

struct GramArgs {
    const double2 *Y, *HY;
    int64_t ldy, ldhy;
    int32_t n;                 // columns
    int32_t ntiles;            // entries of `tiles`
    int32_t kslabs;            // K split
    int64_t nchunks;           // Ng / KC
    const GramTile *tiles;
    double2 *work;             // [kslabs][ntiles][TN][TM] partial tiles (column-major inside a tile)
};

__device__ __forceinline__ void dmma884(double &d0, double &d1, double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}

// CTA tile (WGM*FA*8) x (WGN*FB*8) complex outputs, WGM*WGN warps, each warp FA x FB DMMA tiles.
// KC grid points per pipeline stage, smem row pitch KC+4 complex (pitch % 8 == 4 -> the 8 lanes
// of an LDS.128 phase, 2 rows x 4 k, hit 8 distinct 16-byte bank groups).
template <int WGM, int WGN, int FA, int FB, int KC, int STAGES>
struct GramCfg {
    static constexpr int TM = WGM * FA * 8, TN = WGN * FB * 8;
    static constexpr int THREADS = WGM * WGN * 32;
    static constexpr int PITCH = KC + 4;
    static constexpr int STAGE_ELEMS = (TM + TN) * PITCH;           // double2
    static constexpr size_t SMEM = (size_t)STAGES * STAGE_ELEMS * sizeof(double2);
};

// BULK: the operand rows of a stage (KC consecutive grid points of one column = 256 contiguous bytes) arrive by ONE
// TMA bulk copy each (cp.async.bulk + mbarrier, SASS UBLKCP) instead of KC per-thread 16-byte cp.async (LDGSTS).
template <int WGM, int WGN, int FA, int FB, int KC, int STAGES, bool BULK = false, bool M3 = true, int MINB = 1>
__global__ void __launch_bounds__(WGM *WGN * 32, MINB) gram_dmma_kernel(GramArgs a)
{
    using Cfg = GramCfg<WGM, WGN, FA, FB, KC, STAGES>;
    constexpr int TM = Cfg::TM, TN = Cfg::TN, PITCH = Cfg::PITCH, NT = Cfg::THREADS;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double2 *sm = reinterpret_cast<double2 *>(smem_raw);

    const int unit = blockIdx.x;
    const int ks = unit / a.ntiles;
    const GramTile tl = a.tiles[unit - ks * a.ntiles];
    const int i0 = tl.ti * TM, j0 = tl.tj * TN;
    const double2 *Abase = a.Y;
    const double2 *Bbase = tl.mat == 1 ? a.Y : a.HY;
    const int64_t lda = a.ldy, ldb = tl.mat == 1 ? a.ldy : a.ldhy;
    const int64_t c0 = a.nchunks * ks / a.kslabs, c1 = a.nchunks * (ks + 1) / a.kslabs;
    const int nch = (int)(c1 - c0);
    const int64_t r0 = c0 * KC;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int wm = warp / WGN, wn = warp % WGN;
    const int g = lane >> 2, t = lane & 3;

    // stage loader: (TM+TN) rows x KC elements of 16 B; consecutive threads walk k first
    auto load_stage = [&](int stage, int chunk) {
        double2 *dst = sm + (size_t)stage * Cfg::STAGE_ELEMS;
        const int64_t r = r0 + (int64_t)chunk * KC;
#pragma unroll
        for (int e = tid; e < (TM + TN) * KC; e += NT) {
            const int row = e / KC, k = e - row * KC;
            double2 *d = dst + row * PITCH + k;
            if (row < TM) {
                const int col = i0 + row;
                if (col < a.n) cp_async16(d, Abase + (int64_t)col * lda + r + k);
                else *d = make_double2(0.0, 0.0);
            } else {
                const int col = j0 + row - TM;
                if (col < a.n) cp_async16(d, Bbase + (int64_t)col * ldb + r + k);
                else *d = make_double2(0.0, 0.0);
            }
        }
    };

    // bulk variant: thread `row` < TM+TN owns one operand row; rows of columns >= n stay zero for the whole kernel
    __shared__ uint64_t full_bar[STAGES];
    const int my_col = tid < TM ? i0 + tid : j0 + tid - TM;
    const bool my_row = BULK && tid < TM + TN && my_col < a.n;
    const double2 *my_src = nullptr;
    uint32_t stage_bytes = 0;
    if (BULK) {
        if (tid < TM + TN) my_src = (tid < TM ? Abase + (int64_t)my_col * lda : Bbase + (int64_t)my_col * ldb) + r0;
        const int va = min(TM, max(0, a.n - i0)), vb = min(TN, max(0, a.n - j0));
        stage_bytes = (uint32_t)((va + vb) * KC * sizeof(double2));
        if (tid == 0) {
#pragma unroll
            for (int s = 0; s < STAGES; ++s) mbar_init(&full_bar[s], 1);
            mbar_fence_init();
        }
        if (tid < TM + TN && !my_row)
            for (int s = 0; s < STAGES; ++s)
                for (int k = 0; k < KC; ++k) sm[(size_t)s * Cfg::STAGE_ELEMS + tid * PITCH + k] = make_double2(0.0, 0.0);
        __syncthreads();
    }
    auto issue_bulk = [&](int stage, int chunk) {
        if (tid == 0) mbar_arrive_expect_tx(&full_bar[stage], stage_bytes);
        if (my_row)
            bulk_g2s(sm + (size_t)stage * Cfg::STAGE_ELEMS + tid * PITCH, my_src + (int64_t)chunk * KC, KC * sizeof(double2), &full_bar[stage]);
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
        if (s < nch) { if (BULK) issue_bulk(s, s); else load_stage(s, s); }
        if (!BULK) cp_async_commit();
    }

    for (int ch = 0; ch < nch; ++ch) {
        if (BULK) mbar_wait(&full_bar[ch % STAGES], (uint32_t)((ch / STAGES) & 1));
        else cp_async_wait<STAGES - 2>();
        __syncthreads();
        {   // prefetch chunk ch+STAGES-1 into the stage consumed at iteration ch-1
            const int nx = ch + STAGES - 1;
            if (nx < nch) { if (BULK) issue_bulk(nx % STAGES, nx); else load_stage(nx % STAGES, nx); }
            if (!BULK) cp_async_commit();
        }
        const double2 *As = sm + (size_t)(ch % STAGES) * Cfg::STAGE_ELEMS + (wm * FA * 8 + g) * PITCH + t;
        const double2 *Bs = sm + (size_t)(ch % STAGES) * Cfg::STAGE_ELEMS + (TM + wn * FB * 8 + g) * PITCH + t;
#pragma unroll
        for (int kk = 0; kk < KC; kk += 4) {
            if (M3) {
                double b0[FB], b1[FB], b2[FB];
#pragma unroll
                for (int y = 0; y < FB; ++y) { const double2 v = Bs[y * 8 * PITCH + kk]; b0[y] = v.x; b1[y] = v.y - v.x; b2[y] = v.x + v.y; }
#pragma unroll
                for (int x = 0; x < FA; ++x) {
                    const double2 v = As[x * 8 * PITCH + kk];
                    const double a0 = v.x - v.y, a1 = v.x, a2 = -v.y;
#pragma unroll
                    for (int y = 0; y < FB; ++y) {
                        dmma884(cre[x][y][0], cre[x][y][1], a0, b0[y]);
                        dmma884(cim[x][y][0], cim[x][y][1], a1, b1[y]);
                        dmma884(ck3[x][y][0], ck3[x][y][1], a2, b2[y]);
                    }
                }
            } else {
                double br[FB], bi[FB];
#pragma unroll
                for (int y = 0; y < FB; ++y) { const double2 v = Bs[y * 8 * PITCH + kk]; br[y] = v.x; bi[y] = v.y; }
#pragma unroll
                for (int x = 0; x < FA; ++x) {
                    const double2 v = As[x * 8 * PITCH + kk];
                    const double ar = v.x, ai = v.y, nai = -v.y;
#pragma unroll
                    for (int y = 0; y < FB; ++y) {
                        dmma884(cre[x][y][0], cre[x][y][1], ar, br[y]);
                        dmma884(cim[x][y][0], cim[x][y][1], ar, bi[y]);
                    }
#pragma unroll
                    for (int y = 0; y < FB; ++y) {
                        dmma884(cre[x][y][0], cre[x][y][1], ai, bi[y]);
                        dmma884(cim[x][y][0], cim[x][y][1], nai, br[y]);
                    }
                }
            }
        }
    }
    if (!BULK) cp_async_wait<0>();

    // epilogue: C fragment element e of (x, y) is row g, column 2t+e of that 8x8 tile
    double2 *W = a.work + (int64_t)unit * (TM * TN);
#pragma unroll
    for (int x = 0; x < FA; ++x)
#pragma unroll
        for (int y = 0; y < FB; ++y)
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                const int ii = (wm * FA + x) * 8 + g;
                const int jj = (wn * FB + y) * 8 + 2 * t + e;
                W[jj * TM + ii] = M3 ? make_double2(cre[x][y][e] - ck3[x][y][e], cre[x][y][e] + cim[x][y][e]) : make_double2(cre[x][y][e], cim[x][y][e]);
            }
}

// Fixed-order sum over K-slabs, one CTA per tile of the launch's tile list; H_sub tiles are written
// as computed, S_sub comes from its upper-triangular tiles: element (i,j) with tile(i) < tile(j) is
// computed, its mirror is the conjugate; inside a diagonal tile the i<j half is used and mirrored,
// and the diagonal's imaginary part is exactly 0 (S_ii = |y_i|^2), so S_sub is exactly Hermitian.
// mat 2 applies the same rule to H_sub (optional mode: H is Hermitian, so is Y^H H Y in exact arithmetic).
struct GramReduceArgs {
    const double2 *work;
    const GramTile *tiles;
    double2 *H, *S;
    int32_t n, lds, kslabs, ntiles, tm, tn;
};

__global__ void __launch_bounds__(256) gram_reduce_kernel(GramReduceArgs a)
{
    const GramTile tl = a.tiles[blockIdx.x];
    const int i0 = tl.ti * a.tm, j0 = tl.tj * a.tn;
    const int64_t tsz = (int64_t)a.tm * a.tn;
    const double2 *W = a.work + (int64_t)blockIdx.x * tsz;
    const int64_t kstride = (int64_t)a.ntiles * tsz;
    for (int e = threadIdx.x; e < a.tm * a.tn; e += blockDim.x) {
        const int jj = e / a.tm, ii = e - jj * a.tm;
        const int i = i0 + ii, j = j0 + jj;
        if (i >= a.n || j >= a.n) continue;
        if (tl.mat != 0 && tl.ti == tl.tj && i > j) continue;
        double sr = 0.0, si = 0.0;
        for (int k = 0; k < a.kslabs; ++k) {
            const double2 v = W[(int64_t)k * kstride + e];
            sr += v.x; si += v.y;
        }
        if (tl.mat == 0) {
            a.H[(int64_t)j * a.lds + i] = make_double2(sr, si);
        } else {
            double2 *M = tl.mat == 1 ? a.S : a.H;          // Hermitian output: mirror the conjugate, real diagonal
            if (i == j) si = 0.0;
            M[(int64_t)j * a.lds + i] = make_double2(sr, si);
            if (i != j) M[(int64_t)i * a.lds + j] = make_double2(sr, -si);
        }
    }
}

}  // namespace rsdft
