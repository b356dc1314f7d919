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
    // (the heaviest stage: when NTG does not divide the item count, whole warps sit it out instead of running a ragged round)
    constexpr int XB_ITEMS = LINES * MX;
    constexpr int XB_NT = (XB_ITEMS % NTG == 0) ? NTG : ((XB_ITEMS % 96 == 0 && NTG > 96) ? 96 : NTG);
    for (int item = tid; item < XB_ITEMS && tid < XB_NT; item += XB_NT) {
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
            if (HINT) st_hint(ptr + (int64_t)j * a.nz, make_double2(re[j], im[j]), pol);
            else ptr[(int64_t)j * a.nz] = make_double2(re[j], im[j]);
        }
    }
}

// Same tile with the two radix-M stage pairs fused in registers: a thread holds the M x M block (n1, jy) of one
// (n2, z), runs the M y-transforms and the M x-transforms (stage A) on it without going through shared memory, and does
// the mirror image on the way out.  Two of the four shared-memory exchanges disappear (the tile is bound by the
// L1/shared-memory data pipe): 96 B per point of LDS/STS traffic instead of 160.  2*M*M doubles of
// registers per thread, so M <= 6 (lengths <= 96) and at most 256 threads per CTA.
template <int NX, int TZ, int NTG, bool HINT>
__device__ __forceinline__ void fft3_x_dense_tile_fused(const Fft3Args &a, double2 *S, double2 *gbase, const double *__restrict__ kin,
                                                        const double2 *twx_s, const double *kinx_s, int tid, int bar, uint64_t pol)
{
    using D = XDense<NX, TZ>;
    constexpr int R2X = D::R2X, M = D::MX, LINES = D::LINES;
    static_assert(M <= 6, "fused x tile: register block is 2*M*M doubles");
    // y stage B + x stage A
    for (int item = tid; item < TZ * R2X; item += NTG) {
        const int z = item % TZ, n2 = item / TZ;
        double2 *p = S + n2 * LINES + z;
        double re[M][M], im[M][M];                   // [n1][jy]
#pragma unroll
        for (int n1 = 0; n1 < M; ++n1)
#pragma unroll
            for (int j = 0; j < M; ++j) { const double2 v = p[n1 * R2X * LINES + j * TZ]; re[n1][j] = v.x; im[n1][j] = v.y; }
#pragma unroll
        for (int n1 = 0; n1 < M; ++n1) Dft<M>::run(re[n1], im[n1]);
#pragma unroll
        for (int j = 0; j < M; ++j) {
            double cr[M], ci[M];
#pragma unroll
            for (int n1 = 0; n1 < M; ++n1) { cr[n1] = re[n1][j]; ci[n1] = im[n1][j]; }
            Dft<M>::run(cr, ci);
#pragma unroll
            for (int k = 1; k < M; ++k) { const double2 w = twx_s[(k - 1) * R2X + n2]; tw_mul(cr[k], ci[k], w.x, -w.y); }
#pragma unroll
            for (int k = 0; k < M; ++k) p[k * R2X * LINES + j * TZ] = make_double2(cr[k], ci[k]);
        }
    }
    group_sync(bar, NTG);
    // x stage B (radix-R2X over n2) -> frequency kx = k1 + M*k2; kinetic factor; inverse stage B'
    constexpr int XB_ITEMS = LINES * M;
    constexpr int XB_NT = (XB_ITEMS % NTG == 0) ? NTG : ((XB_ITEMS % 96 == 0 && NTG > 96) ? 96 : NTG);
    for (int item = tid; item < XB_ITEMS && tid < XB_NT; item += XB_NT) {
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
            const double f = kinx_s[k1 + M * k2] + tin;
            br[k2] *= f; bi[k2] *= f;
        }
        Dft<R2X>::run(bi, br);                  // swapped domain from here on
#pragma unroll
        for (int t = 0; t < R2X; ++t) p[t * LINES] = make_double2(br[t], bi[t]);
    }
    group_sync(bar, NTG);
    // x inverse stage A' + y inverse stage B' + store
    for (int item = tid; item < TZ * R2X; item += NTG) {
        const int z = item % TZ, n2 = item / TZ;
        const double2 *p = S + n2 * LINES + z;
        double re[M][M], im[M][M];                   // [jy][k -> n1]
#pragma unroll
        for (int j = 0; j < M; ++j) {
#pragma unroll
            for (int k = 0; k < M; ++k) { const double2 v = p[k * R2X * LINES + j * TZ]; re[j][k] = v.x; im[j][k] = v.y; }
#pragma unroll
            for (int k = 1; k < M; ++k) { const double2 w = twx_s[(k - 1) * R2X + n2]; tw_mul(im[j][k], re[j][k], w.x, -w.y); }
            Dft<M>::run(im[j], re[j]);
        }
#pragma unroll
        for (int n1 = 0; n1 < M; ++n1) {
            double cr[M], ci[M];
#pragma unroll
            for (int j = 0; j < M; ++j) { cr[j] = re[j][n1]; ci[j] = im[j][n1]; }
            Dft<M>::run(ci, cr);
            double2 *ptr = gbase + (int64_t)(n1 * R2X + n2) * a.ny * a.nz + z;
#pragma unroll
            for (int j = 0; j < M; ++j) {
                if (HINT) st_hint(ptr + (int64_t)j * a.nz, make_double2(cr[j], ci[j]), pol);
                else ptr[(int64_t)j * a.nz] = make_double2(cr[j], ci[j]);
            }
        }
    }
}

// Launch shape per length: z points per tile, groups per CTA, threads per group, slots per group.
// NTG is chosen so that the heaviest stage (LINES*MX radix-16 pairs) fills whole rounds.
template <int NX> struct XTmaCfg { static constexpr int TZ = 0, G = 0, NTG = 0, SPG = 0; };      // TZ = 0: no TMA kernel for this length
template <> struct XTmaCfg<48> { static constexpr int TZ = 8, G = 4, NTG = 96, SPG = 2; };        // slot 18 KB, 72 radix-16 pairs
template <> struct XTmaCfg<64> { static constexpr int TZ = 8, G = 3, NTG = 128, SPG = 2; };       // slot 32 KB, 128 pairs
template <> struct XTmaCfg<80> { static constexpr int TZ = 8, G = 4, NTG = 96, SPG = 1; };        // slot 50 KB, 200 pairs
template <> struct XTmaCfg<96> { static constexpr int TZ = 8, G = 2, NTG = 128, SPG = 1; };       // slot 72 KB, 288 pairs; 2 groups leave 80 KB for the other streams' CTAs
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
        if constexpr (D::MX <= 6)
            fft3_x_dense_tile_fused<NX, TZ, NTG, false>(a, S, a.W + col * a.ldw + toff, a.kin_yz + toff, twx_s, kinx_s, gt, 1 + g, pol);
        else
            fft3_x_dense_tile<NX, TZ, NTG, false>(a, S, a.W + col * a.ldw + toff, a.kin_yz + toff, twx_s, kinx_s, gt, 1 + g, pol);
        fence_proxy_async_smem();
        group_sync(1 + g, NTG);                       // the slot is free: every thread has finished reading it
        if (SPG == 1 && gt == 0 && tile + stride < ntiles) issue(tile + stride, 0);
    }
}


// ---------------------------------------------------------------------------------------------
// The persistent pipeline kernel (north_star "one HBM round trip per direction"; queue and
// dependency rules: PipeArgs in fft3_kernels.cuh).  ONE launch applies T + V_loc to all columns, one CTA per SM.
// Every load is a TMA box issued by a CONTROL warp ahead of the compute warps, so no compute warp ever waits for
// global memory or touches the global counters, and there is no CTA-wide barrier after start-up.
//   * CTA = G groups; group g = NTG compute threads (own named barrier) + an issue warp + a signal warp (lane 0 works).
//   * Region of a group: NS dense R2Y x NZ slots for fwd / inv items (ring buffer); an x item takes the whole region
//     (dense NX x MY x TZ tile, fft3_x_dense_tile) and is issued only when all slots are idle.
//   * issue lane: pop item -> wait for the item's column counter -> wait for a free slot -> descriptor + TMA
//     (+ L2 prefetch of the psi and v(r) rows of an inv tile).  signal lane: waits for the compute threads on the
//     slot's `empty` mbarrier, then __threadfence + atomicAdd on the column counter.  Completions are signalled
//     independently of the issue lane's waits, so the smallest unfinished queue item always makes progress (no
//     co-residency assumption, no deadlock).
//   * L2 eviction classes keep the k-space of the columns in flight resident: X / psi reads and the final HX writes
//     are evict_first (Fft3Args::hint_*); measured DRAM traffic 58 B per orbital*point against 112 for three kernels.
//   * compute threads: wait `full[slot]`, read the descriptor, run the tile program IN PLACE in the dense slot, arrive
//     on `empty[slot]`.  fwd / inv tiles avoid bank conflicts without padding by rotating each 16-element segment
//     (row j, k1) by (j*MZ + k1) mod 16: the radix-16 z stage then reads 16 consecutive elements per thread with
//     consecutive threads on different bank groups, and the y stage un-rotates per row.
template <int NZ, int R2Y> struct ZyDense {
    static constexpr int R2Z = Axis<NZ>::R2, MZ = Axis<NZ>::M;
    static_assert(R2Z == 16, "rotated dense layout: radix-16 first stage only");
    static constexpr int ELEMS = R2Y * NZ;
    static constexpr uint32_t BYTES = (uint32_t)ELEMS * 16u;
    __device__ static __forceinline__ int pos(int j, int k1, int c) { return j * NZ + k1 * R2Z + ((c + j * MZ + k1) & (R2Z - 1)); }
};

// z forward (A, B) + y forward stage A of one tile held densely in S[j][z] (as the TMA box left it); writes W.
template <int NZ, int R2Y, int NT>
__device__ __forceinline__ void fft3_fwd_dense_tile(double2 *S, double2 *__restrict__ dst, int my, int n2y, const double2 *twz_s,
                                                    const double2 *twy_s, int tid, int bar, uint64_t pol_out)
{
    using Z = ZyDense<NZ, R2Y>;
    constexpr int R2Z = Z::R2Z, MZ = Z::MZ;
    // z stage A: radix-MZ over n1 (z = n1*R2Z + n2), twiddle; the 16 threads of a row sit in one warp, so all of the
    // row's loads are done before its (rotated, not in-place) stores
    for (int item = tid; item < R2Y * R2Z; item += NT) {
        const int j = item / R2Z, n2 = item % R2Z;
        double re[MZ], im[MZ];
#pragma unroll
        for (int n1 = 0; n1 < MZ; ++n1) { const double2 v = S[j * NZ + n1 * R2Z + n2]; re[n1] = v.x; im[n1] = v.y; }
        __syncwarp(__activemask());
        Dft<MZ>::run(re, im);
#pragma unroll
        for (int k = 1; k < MZ; ++k) { const double2 w = twz_s[(k - 1) * R2Z + n2]; tw_mul(re[k], im[k], w.x, -w.y); }
#pragma unroll
        for (int k = 0; k < MZ; ++k) S[Z::pos(j, k, n2)] = make_double2(re[k], im[k]);
    }
    group_sync(bar, NT);
    // z stage B: radix-R2Z over n2, in place in the rotated segment
    for (int item = tid; item < R2Y * MZ; item += NT) {
        double2 *p = S + item * R2Z;
        double br[R2Z], bi[R2Z];
#pragma unroll
        for (int t = 0; t < R2Z; ++t) { const double2 v = p[(t + item) & (R2Z - 1)]; br[t] = v.x; bi[t] = v.y; }
        Dft<R2Z>::run(br, bi);
#pragma unroll
        for (int t = 0; t < R2Z; ++t) p[(t + item) & (R2Z - 1)] = make_double2(br[t], bi[t]);
    }
    group_sync(bar, NT);
    // y stage A: radix-R2Y over the R2Y rows, twiddle w_NY^{n2y k1}, store row k1*my + n2y
    for (int p = tid; p < NZ; p += NT) {
        const int k1 = p / R2Z, k2 = p % R2Z;
        double br[R2Y], bi[R2Y];
#pragma unroll
        for (int j = 0; j < R2Y; ++j) { const double2 v = S[Z::pos(j, k1, k2)]; br[j] = v.x; bi[j] = v.y; }
        Dft<R2Y>::run(br, bi);
#pragma unroll
        for (int k = 1; k < R2Y; ++k) { const double2 w = twy_s[k]; tw_mul(br[k], bi[k], w.x, -w.y); }
#pragma unroll
        for (int k = 0; k < R2Y; ++k) st_hint(dst + (int64_t)(k * my + n2y) * NZ + p, make_double2(br[k], bi[k]), pol_out);
    }
}

// y inverse stage A', z inverse (B', A'), HX = T psi + v psi of one tile held densely in S[k1y][p]; psi and v(r) come
// from global memory (L2: the control warp prefetched their rows when it issued the tile).
template <int NZ, int R2Y, int NT>
__device__ __forceinline__ void fft3_inv_dense_tile(double2 *S, const double2 *__restrict__ psi_g, const double *__restrict__ vl,
                                                    double2 *__restrict__ dst, int my, int n2y, const double2 *twz_s, const double2 *twy_s,
                                                    int tid, int bar, uint64_t pol_stream)
{
    using Z = ZyDense<NZ, R2Y>;
    constexpr int R2Z = Z::R2Z, MZ = Z::MZ;
    // y inverse stage A': conj twiddle, radix-R2Y over k1y (swapped domain) -> row j = n1y, stored rotated
    for (int p = tid; p < NZ; p += NT) {
        const int k1 = p / R2Z, k2 = p % R2Z;
        double br[R2Y], bi[R2Y];
#pragma unroll
        for (int k = 0; k < R2Y; ++k) { const double2 v = S[k * NZ + p]; br[k] = v.x; bi[k] = v.y; }
        __syncwarp(__activemask());
#pragma unroll
        for (int k = 1; k < R2Y; ++k) { const double2 w = twy_s[k]; tw_mul(bi[k], br[k], w.x, -w.y); }
        Dft<R2Y>::run(bi, br);
#pragma unroll
        for (int j = 0; j < R2Y; ++j) S[Z::pos(j, k1, k2)] = make_double2(br[j], bi[j]);
    }
    group_sync(bar, NT);
    // z inverse stage B': radix-R2Z over k2z (swapped), in place
    for (int item = tid; item < R2Y * MZ; item += NT) {
        double2 *p = S + item * R2Z;
        double br[R2Z], bi[R2Z];
#pragma unroll
        for (int q = 0; q < R2Z; ++q) { const double2 v = p[(q + item) & (R2Z - 1)]; br[q] = v.x; bi[q] = v.y; }
        Dft<R2Z>::run(bi, br);
#pragma unroll
        for (int q = 0; q < R2Z; ++q) p[(q + item) & (R2Z - 1)] = make_double2(br[q], bi[q]);
    }
    group_sync(bar, NT);
    // z inverse stage A' + V_loc
    for (int item = tid; item < R2Y * R2Z; item += NT) {
        const int j = item / R2Z, n2 = item % R2Z;
        const int64_t off = (int64_t)(j * my + n2y) * NZ + n2;
        double2 ps[MZ];
        double vv[MZ];
#pragma unroll
        for (int n1 = 0; n1 < MZ; ++n1) {
            ps[n1] = ld_nc_hint(psi_g + off + n1 * R2Z, pol_stream);
            vv[n1] = __ldg(vl + off + n1 * R2Z);
        }
        double re[MZ], im[MZ];
#pragma unroll
        for (int k = 0; k < MZ; ++k) { const double2 v = S[Z::pos(j, k, n2)]; re[k] = v.x; im[k] = v.y; }
#pragma unroll
        for (int k = 1; k < MZ; ++k) { const double2 w = twz_s[(k - 1) * R2Z + n2]; tw_mul(im[k], re[k], w.x, -w.y); }
        Dft<MZ>::run(im, re);
#pragma unroll
        for (int n1 = 0; n1 < MZ; ++n1)
            st_hint(dst + off + n1 * R2Z, make_double2(fma(vv[n1], ps[n1].x, re[n1]), fma(vv[n1], ps[n1].y, im[n1])), pol_stream);
    }
}

__device__ __forceinline__ void mbar_arrive(uint64_t *bar)
{
    const uint32_t b = (uint32_t)__cvta_generic_to_shared(bar);
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" :: "r"(b) : "memory");
}
__device__ __forceinline__ bool mbar_test(uint64_t *bar, uint32_t parity)
{
    const uint32_t b = (uint32_t)__cvta_generic_to_shared(bar);
    uint32_t ok;
    asm volatile("{\n.reg .pred p;\nmbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2;\nselp.u32 %0, 1, 0, p;\n}\n" : "=r"(ok) : "r"(b), "r"(parity) : "memory");
    return ok != 0;
}
__device__ __forceinline__ void tma_prefetch_5d(const CUtensorMap *tm, int c0, int c1, int c2, int c3, int c4)
{
    asm volatile("cp.async.bulk.prefetch.tensor.5d.L2.global.tile [%0, {%1, %2, %3, %4, %5}];"
                 :: "l"((uint64_t)tm), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(c4) : "memory");
}
__device__ __forceinline__ void tma_prefetch_4d(const CUtensorMap *tm, int c0, int c1, int c2, int c3)
{
    asm volatile("cp.async.bulk.prefetch.tensor.4d.L2.global.tile [%0, {%1, %2, %3, %4}];"
                 :: "l"((uint64_t)tm), "r"(c0), "r"(c1), "r"(c2), "r"(c3) : "memory");
}

struct PipeMaps {
    CUtensorMap x_rows;     // X   as doubles [col][x][n1][n2y][2*nz], box = (2*nz, 1, R2Y, 1, 1): the R2Y rows {n1*my + n2y} of one plane
    CUtensorMap w_rows;     // W   same geometry
    CUtensorMap w_xtile;    // W   as doubles [col][x][y][2*nz], box = (2*TZ, my, nx, 1): one x tile
    CUtensorMap v_rows;     // vloc as doubles [x][n1][n2y][nz], box = (nz, 1, R2Y, 1): L2 prefetch only
};

template <int N, int R2Y, int TZ, int NS_> struct PipeCfg {
    using D = XDense<N, TZ>;
    using Z = ZyDense<N, R2Y>;
    static constexpr int NS = NS_;                                // fwd / inv slots per group (x items take the whole region)
    static constexpr bool POP_AHEAD = false;                       // pop the next queue item while this one is being issued
    static constexpr size_t SLOT = (Z::BYTES + 127) / 128 * 128;
    static constexpr size_t REGION = ((D::BYTES > NS * SLOT ? (size_t)D::BYTES : NS * SLOT) + 1023) / 1024 * 1024;
};

struct PipeDesc { int32_t ph, t, col, pad; };     // ph: 0 fwd, 1 x, 2 inv, 6 skip (column out of range), 7 stop

template <int N, int R2Y, int TZ, int NS_, int G, int NTG>
__global__ void __launch_bounds__(G * (NTG + 64), 1) fft3_pipeline_kernel(Fft3Args a, PipeArgs q, const __grid_constant__ PipeMaps maps)
{
    using Z = ZyDense<N, R2Y>;
    using D = XDense<N, TZ>;
    using PC = PipeCfg<N, R2Y, TZ, NS_>;
    constexpr int NC = G * NTG;                  // compute threads come first, then 2 control warps per group
    constexpr int NS = PC::NS;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    unsigned char *regions = smem_raw + ((1024u - ((uint32_t)__cvta_generic_to_shared(smem_raw) & 1023u)) & 1023u);
    __shared__ double2 twz_s[XTables<N>::NTW];   // z twiddles = x twiddles (cubic grid)
    __shared__ double kinx_s[N];
    __shared__ double2 twy_s[G][NS][R2Y];
    __shared__ PipeDesc desc[G][NS], sigd[G][NS];
    __shared__ int32_t sig_count[G];
    __shared__ __align__(8) uint64_t full[G][NS], empty[G][NS];
    const int tid = threadIdx.x;
    const int my = a.my;
    fft3_x_tables<N, G * (NTG + 64)>(a, twz_s, kinx_s, tid);
    if (tid == 0) {
        for (int i = 0; i < G; ++i)
            for (int s2 = 0; s2 < NS; ++s2) { mbar_init(&full[i][s2], 1); mbar_init(&empty[i][s2], NTG); }
        mbar_fence_init();
    }
    if (tid < G) sig_count[tid] = 0;
    __syncthreads();
    const uint64_t pol_stream = l2_policy(a.hint_stream), pol_keep = l2_policy(a.hint_keep);
    const int64_t total = (int64_t)(a.ncol + q.lag_inv) * q.npattern;

    if (tid >= NC) {
        // ------------------------------------------------------------------ control warps of group g: issue + signal
        const int cw = (tid - NC) >> 5;
        const int g = cw >> 1;
        if ((tid & 31) != 0) return;
        if (cw & 1) {
            // signal warp: completions in issue order -> column counters; publishes the count to the issue warp
            uint32_t pe = 0;
            for (int k = 0, s2 = 0;; ++k, s2 = (s2 + 1 == NS ? 0 : s2 + 1)) {
                mbar_wait(&empty[g][s2], (pe >> s2) & 1u);
                pe ^= 1u << s2;
                const int ph = sigd[g][s2].ph, col = sigd[g][s2].col;
                if (ph < 2) {
                    __threadfence();
                    atomicAdd(q.done + ph * a.ncol + col, 1);
                }
                *((volatile int32_t *)&sig_count[g]) = k + 1;
                if (ph == 7) return;
            }
        }
        // issue warp: pop item -> dependency -> free slot -> descriptor + TMA
        unsigned char *region = regions + (size_t)g * PC::REGION;
        bool prev_x = false;
        int rdy_fwd = -1, rdy_x = -1;                 // columns whose counters were already seen complete
        int nxt = atomicAdd(q.head, 1);
        for (int k_issue = 0;; ++k_issue) {
            const int item = nxt;
            PipeDesc cur = {7, 0, 0, 0};
            if (item < total) {
                if (PC::POP_AHEAD) nxt = atomicAdd(q.head, 1);       // its latency hides behind this item's issue
                const int s = item / q.npattern;
                const uint32_t e = __ldg(q.pattern + (item - s * q.npattern));
                cur.ph = (int)(e >> 28); cur.t = (int)(e & 0x0fffffffu);
                cur.col = s - (cur.ph == 0 ? 0 : (cur.ph == 1 ? q.lag_x : q.lag_inv));
                if (cur.col < 0 || cur.col >= a.ncol) cur.ph = 6;
            }
            if (cur.ph == 1 && rdy_fwd != cur.col) {
                pipe_wait(q.done + cur.col, q.n_fwd);
                rdy_fwd = cur.col;
            } else if (cur.ph == 2 && rdy_x != cur.col) {
                pipe_wait(q.done + a.ncol + cur.col, q.n_x);
                rdy_x = cur.col;
            }
            // slot k_issue % NS is free once item k_issue - NS is done; an x item takes the whole region
            const int need_done = (cur.ph == 1 || prev_x) ? k_issue : k_issue - NS + 1;
            while (*((volatile int32_t *)&sig_count[g]) < need_done) __nanosleep(32);
            const int s2 = k_issue % NS;
            desc[g][s2] = cur;
            sigd[g][s2] = cur;
            uint64_t *fb = &full[g][s2];
            if (cur.ph == 0) {
                const int x = cur.t / my, n2y = cur.t - x * my;
                mbar_arrive_expect_tx(fb, Z::BYTES);
                tma_load_5d(region + (size_t)s2 * PC::SLOT, &maps.x_rows, fb, 0, n2y, 0, x, cur.col, pol_stream);
            } else if (cur.ph == 1) {
                fence_proxy_async_all();                      // other CTAs' ordinary stores -> this TMA read
                const int k1y = cur.t / q.zchunks, zc = cur.t - k1y * q.zchunks;
                mbar_arrive_expect_tx(fb, D::BYTES);
                tma_load_4d(region, &maps.w_xtile, fb, 2 * zc * TZ, k1y * my, 0, cur.col, pol_keep);
            } else if (cur.ph == 2) {
                fence_proxy_async_all();
                const int x = cur.t / my, n2y = cur.t - x * my;
                mbar_arrive_expect_tx(fb, Z::BYTES);
                tma_load_5d(region + (size_t)s2 * PC::SLOT, &maps.w_rows, fb, 0, n2y, 0, x, cur.col, pol_stream);
                tma_prefetch_5d(&maps.x_rows, 0, n2y, 0, x, cur.col);          // psi rows and v(r) rows -> L2
                tma_prefetch_4d(&maps.v_rows, 0, n2y, 0, x);
            } else {
                mbar_arrive(fb);                              // skip / stop: nothing to load
            }
            prev_x = cur.ph == 1;
            if (cur.ph == 7) return;
            if (!PC::POP_AHEAD) nxt = atomicAdd(q.head, 1);
        }
    }

    // ---------------------------------------------------------------------- compute threads of group g
    const int g = tid / NTG, gt = tid - g * NTG, bar = 1 + g;
    unsigned char *region = regions + (size_t)g * PC::REGION;
    uint32_t pf = 0;                              // parity bits of the NS full barriers
    for (int k = 0, s2 = 0;; ++k, s2 = (s2 + 1 == NS ? 0 : s2 + 1)) {
        mbar_wait(&full[g][s2], (pf >> s2) & 1u);
        pf ^= 1u << s2;
        const PipeDesc d = desc[g][s2];
        if (d.ph == 0) {
            const int x = d.t / my, n2y = d.t - x * my;
            if (gt < R2Y) twy_s[g][s2][gt] = a.twy[n2y * gt];
            group_sync(bar, NTG);
            fft3_fwd_dense_tile<N, R2Y, NTG>(reinterpret_cast<double2 *>(region + (size_t)s2 * PC::SLOT),
                                             a.W + (int64_t)d.col * a.ldw + (int64_t)x * a.ny * N, my, n2y, twz_s, twy_s[g][s2], gt, bar, pol_keep);
        } else if (d.ph == 1) {
            const int k1y = d.t / q.zchunks, zc = d.t - k1y * q.zchunks;
            const int64_t toff = (int64_t)(k1y * my) * a.nz + zc * TZ;
            fft3_x_dense_tile<N, TZ, NTG, true>(a, reinterpret_cast<double2 *>(region), a.W + (int64_t)d.col * a.ldw + toff, a.kin_yz + toff,
                                                twz_s, kinx_s, gt, bar, pol_keep);
        } else if (d.ph == 2) {
            const int x = d.t / my, n2y = d.t - x * my;
            if (gt < R2Y) twy_s[g][s2][gt] = a.twy[n2y * gt];
            group_sync(bar, NTG);
            const int64_t po = (int64_t)x * a.ny * N;
            fft3_inv_dense_tile<N, R2Y, NTG>(reinterpret_cast<double2 *>(region + (size_t)s2 * PC::SLOT), a.X + (int64_t)d.col * a.ldx + po,
                                             a.vloc + po, a.HX + (int64_t)d.col * a.ldhx + po, my, n2y, twz_s, twy_s[g][s2], gt, bar, pol_stream);
        }
        fence_proxy_async_smem();
        mbar_arrive(&empty[g][s2]);
        if (d.ph == 7) break;
    }
}

}  // namespace rsdft
