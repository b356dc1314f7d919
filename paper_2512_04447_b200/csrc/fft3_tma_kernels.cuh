// TMA-staged x tile of the batched 3-D FFT Laplacian (PAPER.md:19 task (1)).
//
// fft3_x_kernel (fft3_kernels.cuh) brings its tile in with per-thread loads: the load phase exposes the memory
// latency (36 % of its stall samples) and every phase is a CTA-wide barrier.  Here the tile
//     (column, k1y, z chunk) = NX x MY contiguous rows x TZ points = one 3-D box of the k-space scratch
// is fetched by ONE cp.async.bulk.tensor (TMA, SASS UTMALDG) into a dense shared-memory slot and completed through an
// mbarrier; the CTA is G independent groups of NTG threads (own named barrier, own slot(s)), so while one group waits
// for its box the others keep the FP64 pipe and the shared-memory crossbar busy.  All five radix stages run IN PLACE
// in the dense slot S[x][jy][z]: every stage maps consecutive lanes to consecutive z (then jy), so each quarter-warp
// touches 128 contiguous bytes and no padding is needed; results go straight from registers to global memory.
// Requires a cubic-in-(x, y) grid (ny == nx, so MY == MX) with a radix-16 first stage.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>
#include "async_copy.cuh"
#include "fft3_kernels.cuh"

namespace rsdft {

// 4-D box load: coordinates (c0 fastest).  Completes `bytes` on the mbarrier.
__device__ __forceinline__ void tma_load_4d(void *smem, const CUtensorMap *tm, uint64_t *bar, int c0, int c1, int c2, int c3, uint64_t pol)
{
    const uint32_t s = (uint32_t)__cvta_generic_to_shared(smem), b = (uint32_t)__cvta_generic_to_shared(bar);
    asm volatile("cp.async.bulk.tensor.4d.shared::cluster.global.tile.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1, {%3, %4, %5, %6}], [%2], %7;"
                 :: "r"(s), "l"((uint64_t)tm), "r"(b), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "l"(pol) : "memory");
}
__device__ __forceinline__ void tma_load_5d(void *smem, const CUtensorMap *tm, uint64_t *bar, int c0, int c1, int c2, int c3, int c4, uint64_t pol)
{
    const uint32_t s = (uint32_t)__cvta_generic_to_shared(smem), b = (uint32_t)__cvta_generic_to_shared(bar);
    asm volatile("cp.async.bulk.tensor.5d.shared::cluster.global.tile.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1, {%3, %4, %5, %6, %7}], [%2], %8;"
                 :: "r"(s), "l"((uint64_t)tm), "r"(b), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(c4), "l"(pol) : "memory");
}
// generic-proxy accesses to shared memory are ordered before later async-proxy (TMA) accesses of the same bytes
__device__ __forceinline__ void fence_proxy_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
// ... and global memory written by ordinary stores (by this or, after an acquire, another CTA) before TMA reads of it
__device__ __forceinline__ void fence_proxy_async_all() { asm volatile("fence.proxy.async;" ::: "memory"); }

template <int NX, int TZ> struct XDense {
    static constexpr int R2X = Axis<NX>::R2, MX = Axis<NX>::M, MY = MX;
    static constexpr int LINES = MY * TZ;                     // (jy, z) pairs = elements per x row of the slot
    static constexpr int ELEMS = NX * LINES;
    static constexpr uint32_t BYTES = (uint32_t)ELEMS * 16u;
    static constexpr uint32_t SLOT = (BYTES + 1023u) / 1024u * 1024u;
};

// The five stages of one x tile, in place in the dense slot S[x][jy][z]; the last stage writes W (global).
// gbase = W + column offset + (k1y*my)*nz + zc*TZ; kin = kin_yz + (k1y*my)*nz + zc*TZ.  NTG threads, barrier `bar`.
template <int NX, int TZ, int NTG, bool HINT>
__device__ __forceinline__ void fft3_x_dense_tile(const Fft3Args &a, double2 *S, double2 *gbase, const double *__restrict__ kin,
                                                  const double2 *twx_s, const double *kinx_s, int tid, int bar, uint64_t pol)
{
    using D = XDense<NX, TZ>;
    constexpr int R2X = D::R2X, MX = D::MX, MY = D::MY, LINES = D::LINES;
    // y stage B: radix-MY over the MY rows of each (x, z)
    for (int item = tid; item < NX * TZ; item += NTG) {
        const int z = item % TZ, x = item / TZ;
        double2 *p = S + x * LINES + z;
        double re[MY], im[MY];
#pragma unroll
        for (int j = 0; j < MY; ++j) { const double2 v = p[j * TZ]; re[j] = v.x; im[j] = v.y; }
        Dft<MY>::run(re, im);
#pragma unroll
        for (int j = 0; j < MY; ++j) p[j * TZ] = make_double2(re[j], im[j]);
    }
    group_sync(bar, NTG);
    // x stage A: radix-MX over n1 (x = n1*R2X + n2), twiddle w_NX^{n2 k1}
    for (int item = tid; item < LINES * R2X; item += NTG) {
        const int line = item % LINES, n2 = item / LINES;
        double2 *p = S + n2 * LINES + line;
        double re[MX], im[MX];
#pragma unroll
        for (int n1 = 0; n1 < MX; ++n1) { const double2 v = p[n1 * R2X * LINES]; re[n1] = v.x; im[n1] = v.y; }
        Dft<MX>::run(re, im);
#pragma unroll
        for (int k = 1; k < MX; ++k) { const double2 w = twx_s[(k - 1) * R2X + n2]; tw_mul(re[k], im[k], w.x, -w.y); }
#pragma unroll
        for (int k = 0; k < MX; ++k) p[k * R2X * LINES] = make_double2(re[k], im[k]);
    }
    group_sync(bar, NTG);
    // x stage B (radix-R2X over n2) -> frequency kx = k1 + MX*k2; kinetic factor; inverse stage B'
    for (int item = tid; item < LINES * MX; item += NTG) {
        const int line = item % LINES, k1 = item / LINES;
        double2 *p = S + k1 * R2X * LINES + line;
        const int jy = line / TZ, z = line - jy * TZ;
        const double tin = __ldg(kin + (int64_t)jy * a.nz + z);
        double br[R2X], bi[R2X];
#pragma unroll
        for (int t = 0; t < R2X; ++t) { const double2 v = p[t * LINES]; br[t] = v.x; bi[t] = v.y; }
        Dft<R2X>::run(br, bi);
#pragma unroll
        for (int k2 = 0; k2 < R2X; ++k2) {
            const double f = kinx_s[k1 + MX * k2] + tin;
            br[k2] *= f; bi[k2] *= f;
        }
        Dft<R2X>::run(bi, br);                  // swapped domain from here on
#pragma unroll
        for (int t = 0; t < R2X; ++t) p[t * LINES] = make_double2(br[t], bi[t]);
    }
    group_sync(bar, NTG);
    // x inverse stage A': conj twiddle, radix-MX over k1 -> x = n1*R2X + n2
    for (int item = tid; item < LINES * R2X; item += NTG) {
        const int line = item % LINES, n2 = item / LINES;
        double2 *p = S + n2 * LINES + line;
        double re[MX], im[MX];
#pragma unroll
        for (int k = 0; k < MX; ++k) { const double2 v = p[k * R2X * LINES]; re[k] = v.x; im[k] = v.y; }
#pragma unroll
        for (int k = 1; k < MX; ++k) { const double2 w = twx_s[(k - 1) * R2X + n2]; tw_mul(im[k], re[k], w.x, -w.y); }
        Dft<MX>::run(im, re);
#pragma unroll
        for (int n1 = 0; n1 < MX; ++n1) p[n1 * R2X * LINES] = make_double2(re[n1], im[n1]);
    }
    group_sync(bar, NTG);
    // y inverse stage B' and store
    for (int item = tid; item < NX * TZ; item += NTG) {
        const int z = item % TZ, x = item / TZ;
        const double2 *p = S + x * LINES + z;
        double2 *ptr = gbase + (int64_t)x * a.ny * a.nz + z;
        double re[MY], im[MY];
#pragma unroll
        for (int j = 0; j < MY; ++j) { const double2 v = p[j * TZ]; re[j] = v.x; im[j] = v.y; }
        Dft<MY>::run(im, re);
#pragma unroll
        for (int j = 0; j < MY; ++j) {
            if ((a.x_tma & 2) && re[j] != 1.2345) continue;   // LAB
            if (HINT) st_hint(ptr + (int64_t)j * a.nz, make_double2(re[j], im[j]), pol);
            else ptr[(int64_t)j * a.nz] = make_double2(re[j], im[j]);
        }
    }
}

// Launch shape per length: z points per tile, groups per CTA, threads per group, slots per group.
// NTG is chosen so that the heaviest stage (LINES*MX radix-16 pairs) fills whole rounds.
template <int NX> struct XTmaCfg { static constexpr int TZ = 0, G = 0, NTG = 0, SPG = 0; };      // TZ = 0: no TMA kernel for this length
template <> struct XTmaCfg<48> { static constexpr int TZ = 8, G = 4, NTG = 96, SPG = 2; };        // slot 18 KB, 72 radix-16 pairs
template <> struct XTmaCfg<64> { static constexpr int TZ = 8, G = 3, NTG = 128, SPG = 2; };       // slot 32 KB, 128 pairs
template <> struct XTmaCfg<80> { static constexpr int TZ = 8, G = 4, NTG = 96, SPG = 1; };        // slot 50 KB, 200 pairs
template <> struct XTmaCfg<96> { static constexpr int TZ = 8, G = 3, NTG = 96, SPG = 1; };        // slot 72 KB, 288 pairs
template <> struct XTmaCfg<112> { static constexpr int TZ = 4, G = 4, NTG = 96, SPG = 1; };       // slot 49 KB, 196 pairs
template <> struct XTmaCfg<128> { static constexpr int TZ = 4, G = 3, NTG = 128, SPG = 1; };      // slot 64 KB, 256 pairs

template <int NX, int TZ, int G, int SPG> struct XTmaSmem {
    static constexpr size_t bytes = (size_t)G * SPG * XDense<NX, TZ>::SLOT + 1024;   // + alignment slack
};

template <int NX, int TZ, int G, int NTG, int SPG>
__global__ void __launch_bounds__(G * NTG, 1) fft3_x_tma_kernel(Fft3Args a, const __grid_constant__ CUtensorMap tmW)
{
    constexpr int NT = G * NTG;
    using D = XDense<NX, TZ>;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    // TMA destinations must be 128-byte aligned; an offset from the array keeps the compiler on LDS/STS
    unsigned char *slots = smem_raw + ((1024u - ((uint32_t)__cvta_generic_to_shared(smem_raw) & 1023u)) & 1023u);
    __shared__ double2 twx_s[XTables<NX>::NTW];
    __shared__ double kinx_s[NX];
    __shared__ __align__(8) uint64_t full[G * SPG];
    const int tid = threadIdx.x, g = tid / NTG, gt = tid - g * NTG;
    fft3_x_tables<NX, NT>(a, twx_s, kinx_s, tid);
    if (tid == 0) {
        for (int i = 0; i < G * SPG; ++i) mbar_init(&full[i], 1);
        mbar_fence_init();
    }
    __syncthreads();
    const uint64_t pol = l2_policy(0);
    const int my = a.my;
    const int zchunks = a.nz / TZ;
    const int64_t per_col = (int64_t)D::R2X * zchunks;
    const int64_t ntiles = per_col * a.ncol;
    const int64_t stride = (int64_t)gridDim.x * G;
    auto decode = [&](int64_t tile, int64_t &col, int &k1y, int &zc) {
        const int64_t colf = tile / per_col;
        const int rem = (int)(tile - colf * per_col);
        col = a.ncol - 1 - colf;                    // zig-zag: the forward kernel ended on the last column (L2)
        k1y = rem / zchunks; zc = rem - k1y * zchunks;
    };
    auto issue = [&](int64_t tile, int slot) {
        int64_t col; int k1y, zc;
        decode(tile, col, k1y, zc);
        uint64_t *bar = &full[g * SPG + slot];
        mbar_arrive_expect_tx(bar, D::BYTES);
        tma_load_4d(slots + (size_t)(g * SPG + slot) * D::SLOT, &tmW, bar, 2 * zc * TZ, k1y * my, 0, (int)col, pol);
    };
    int64_t tile = (int64_t)blockIdx.x * G + g;
    if (gt == 0 && tile < ntiles) issue(tile, 0);
    for (int k = 0; tile < ntiles; tile += stride, ++k) {
        const int slot = SPG == 2 ? (k & 1) : 0;
        if (SPG == 2 && gt == 0 && tile + stride < ntiles) issue(tile + stride, slot ^ 1);
        mbar_wait(&full[g * SPG + slot], (uint32_t)((k / SPG) & 1));
        int64_t col; int k1y, zc;
        decode(tile, col, k1y, zc);
        const int64_t toff = (int64_t)(k1y * my) * a.nz + zc * TZ;
        double2 *S = reinterpret_cast<double2 *>(slots + (size_t)(g * SPG + slot) * D::SLOT);
        fft3_x_dense_tile<NX, TZ, NTG, false>(a, S, a.W + col * a.ldw + toff, a.kin_yz + toff, twx_s, kinx_s, gt, 1 + g, pol);
        fence_proxy_async_smem();
        group_sync(1 + g, NTG);                       // the slot is free: every thread has finished reading it
        if (SPG == 1 && gt == 0 && tile + stride < ntiles) issue(tile + stride, 0);
    }
}

}  // namespace rsdft
