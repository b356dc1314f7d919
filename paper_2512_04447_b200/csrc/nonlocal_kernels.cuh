// Kleinman-Bylander nonlocal projectors (PAPER.md:19 task (4), "memory-bandwidth-bound";
// PAPER.md:69 "dedicated GPU kernels"):
//   project:  pp[k][i][c] = dV * sum_{s in chunk k} beta[a][i][s] * psi_c(idx[a][s])
//   combine:  q[a][i][c]  = sum_j D_a[i][j] * sum_{k in chunks(a)} pp[k][j][c]      (fixed order)
//   scatter:  HX_c(idx[a][s]) += sum_i beta[a][i][s] * q[a][i][c]
// Every sphere is cut into chunks of <= PCH points; idx and beta are read ONCE per (chunk, column
// group) and reused for the group's columns, whose gathers are independent loads in flight.
// Partial projections are combined in a fixed order, and the
// scatter runs one launch per colour class (spheres of a class are pairwise disjoint), so the
// result is deterministic and bitwise independent of the column batching.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace rsdft {

__device__ __forceinline__ void nl_dmma884(double &d0, double &d1, double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}

constexpr int NL_PCH = 128;       // sphere points per chunk
constexpr int NL_THREADS = 128;

struct SphereChunk {
    int32_t atom;
    int32_t start;    // first point of the chunk inside the atom's list
    int32_t count;    // <= NL_PCH
    int32_t pad;
};

struct SphereTables {
    const int64_t *pt_off;     // [natom+1] offset of atom a's points in idx
    const int64_t *beta_off;   // [natom]   offset of atom a's beta block ([nproj][npts]) in beta
    const int32_t *idx;        // grid indices, sorted ascending per atom
    const double *beta;
    const int32_t *nproj;      // [natom]
    const double *D;           // [natom][maxproj*maxproj] (row-major nproj x nproj in the top-left)
    const SphereChunk *chunks; // [nchunks], sorted by (colour, atom, start)
    const int32_t *atom_chunk0; // [natom+1] chunk ids of atom a = atom_chunk0[a] .. atom_chunk0[a+1]-1 (in atom order)
    const int32_t *atom_chunks; // chunk ids grouped per atom (ascending start)
    int32_t natom, maxproj, nchunks;
};

// scatter: CG complex values in flight per point.
#ifndef RSDFT_NL_CG9
#define RSDFT_NL_CG9 4
#endif
template <int NP> struct NlCols {
    static constexpr int CGS = NP <= 4 ? 8 : (NP <= 9 ? RSDFT_NL_CG9 : 2);
};

// Projection as a skinny FP64 tensor-core contraction with a gathered operand:
//   P[i][c] = sum_s beta[i][s] * psi_c(idx[s]),   M = projectors (MT tiles of 8), K = sphere points,
//   N = columns; real and imaginary parts of 8 columns are two N-tiles fed by ONE 16-byte gather.
// One warp owns (chunk, 8*G8 columns): beta and idx are read once per chunk and reused for all its
// columns, partial sums live in DMMA accumulators (no cross-lane reduction), and 8 k-steps of gathers
// are in flight per lane.  mma.m8n8k4 fragments: A[row = lane/4][k = lane%4], B[k = lane%4][col = lane/4],
// D[row = lane/4][col = 2*(lane%4) + {0, 1}].
template <int MT, int G8>
__global__ void __launch_bounds__(128) project_kernel(SphereTables t, const double2 *__restrict__ X, int64_t ldx,
                                                      int32_t ncol, double dV, double2 *__restrict__ pp)
{
    const int lane = threadIdx.x & 31;
    const int chunk_id = blockIdx.x * 4 + (threadIdx.x >> 5);
    if (chunk_id >= t.nchunks) return;                       // warp-uniform; the kernel has no block barrier
    const SphereChunk ch = t.chunks[chunk_id];
    const int c0 = (gridDim.y - 1 - blockIdx.y) * 8 * G8;   // last columns first: the FFT that follows starts on column 0 (L2)
    const int a = ch.atom;
    const int64_t o = t.pt_off[a];
    const int npts = (int)(t.pt_off[a + 1] - o);
    const int np = t.nproj[a];
    const int32_t *idx = t.idx + o + ch.start;
    const double *beta = t.beta + t.beta_off[a] + ch.start;
    const int kq = lane & 3, r8 = lane >> 2;
    const double2 *colp[G8];
    bool colok[G8];
#pragma unroll
    for (int g = 0; g < G8; ++g) {
        const int c = c0 + g * 8 + r8;
        colok[g] = c < ncol;
        colp[g] = X + (int64_t)(colok[g] ? c : 0) * ldx;
    }
    const double *brow[MT];
    bool rowok[MT];
#pragma unroll
    for (int m = 0; m < MT; ++m) {
        const int i = m * 8 + r8;
        rowok[m] = i < np;
        brow[m] = beta + (int64_t)(rowok[m] ? i : 0) * npts;
    }
    double are[MT][G8][2], aim[MT][G8][2];
#pragma unroll
    for (int m = 0; m < MT; ++m)
#pragma unroll
        for (int g = 0; g < G8; ++g) { are[m][g][0] = are[m][g][1] = aim[m][g][0] = aim[m][g][1] = 0.0; }
    for (int s0 = 0; s0 < ch.count; s0 += 32) {
        const int32_t my_idx = idx[min(s0 + lane, ch.count - 1)];            // one coalesced read per 8 k-steps
#pragma unroll
        for (int j = 0; j < 8; ++j) {
            const int s = s0 + 4 * j + kq;
            const bool ok = s < ch.count;                                     // past the end: beta = 0 on a valid address
            const int64_t g = __shfl_sync(0xffffffffu, my_idx, 4 * j + kq);
            double av[MT];
#pragma unroll
            for (int m = 0; m < MT; ++m) av[m] = (ok && rowok[m]) ? __ldg(brow[m] + s) : 0.0;
#pragma unroll
            for (int gg = 0; gg < G8; ++gg) {
                const double2 v = colok[gg] ? __ldg(colp[gg] + g) : make_double2(0.0, 0.0);
#pragma unroll
                for (int m = 0; m < MT; ++m) {
                    nl_dmma884(are[m][gg][0], are[m][gg][1], av[m], v.x);
                    nl_dmma884(aim[m][gg][0], aim[m][gg][1], av[m], v.y);
                }
            }
        }
    }
#pragma unroll
    for (int m = 0; m < MT; ++m) {
        const int i = m * 8 + r8;
        if (i >= np) continue;
#pragma unroll
        for (int g = 0; g < G8; ++g)
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                const int c = c0 + g * 8 + 2 * kq + e;
                if (c < ncol) pp[((int64_t)chunk_id * t.maxproj + i) * ncol + c] = make_double2(dV * are[m][g][e], dV * aim[m][g][e]);
            }
    }
}

// q[a][i][c] = sum_j D_a[i][j] * (sum over the atom's chunks, ascending start, of pp[k][j][c]).
// One CTA per (atom, tile of NL_CCOLS columns): every thread sums the chunk partials of one (j, c)
// pair (independent loads, fixed order), then one (i, c) row of D.
constexpr int NL_CCOLS = 32;
__global__ void __launch_bounds__(128) combine_kernel(SphereTables t, const double2 *__restrict__ pp, int32_t ncol,
                                                      double2 *__restrict__ q)
{
    const int a = blockIdx.x;
    const int c0 = blockIdx.y * NL_CCOLS;
    const int nc = min(NL_CCOLS, ncol - c0);
    const int np = t.nproj[a], mp = t.maxproj;
    const int k0 = t.atom_chunk0[a], k1 = t.atom_chunk0[a + 1];
    __shared__ double2 ps[16][NL_CCOLS];
    for (int e = threadIdx.x; e < np * nc; e += blockDim.x) {
        const int j = e / nc, c = e - j * nc;
        const double2 *src = pp + (int64_t)j * ncol + c0 + c;
        double sr = 0.0, si = 0.0;
        int k = k0;
        for (; k + 4 <= k1; k += 4) {
            double2 v[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) v[u] = src[(int64_t)t.atom_chunks[k + u] * mp * ncol];
#pragma unroll
            for (int u = 0; u < 4; ++u) { sr += v[u].x; si += v[u].y; }
        }
        for (; k < k1; ++k) {
            const double2 v = src[(int64_t)t.atom_chunks[k] * mp * ncol];
            sr += v.x; si += v.y;
        }
        ps[j][c] = make_double2(sr, si);
    }
    __syncthreads();
    const double *D = t.D + (int64_t)a * mp * mp;
    for (int e = threadIdx.x; e < np * nc; e += blockDim.x) {
        const int i = e / nc, c = e - i * nc;
        double sr = 0.0, si = 0.0;
        for (int j = 0; j < np; ++j) {
            const double d = D[i * mp + j];          // rows of D are stored with stride maxproj
            sr = fma(d, ps[j][c].x, sr);
            si = fma(d, ps[j][c].y, si);
        }
        q[((int64_t)a * mp + i) * ncol + c0 + c] = make_double2(sr, si);
    }
}

// One CTA = one sphere chunk (<= 128 points, one per thread) x every column of the launch: a thread keeps its point's
// grid index and beta values in registers and walks the columns in groups of CG independent read-modify-writes, so
// the beta table is read ONCE per (chunk, launch) however many columns the launch carries (with large tables --
// configs 3, 4: 43 / 98 MB -- beta re-reads per column group used to outweigh the orbital traffic itself).
// q of all columns sits in shared memory ([NP][ncol], dynamic).  blockIdx.y strides over the column groups when the
// chunk list alone does not fill the GPU.
template <int NP>
__global__ void __launch_bounds__(NL_THREADS) scatter_kernel(SphereTables t, int32_t chunk0, const double2 *__restrict__ q,
                                                             int32_t ncol, double2 *__restrict__ HX, int64_t ldhx)
{
    // chunk0: first chunk of one colour class (spheres of one class are pairwise disjoint, so the
    // read-modify-write below is race-free and the result is deterministic)
    constexpr int CG = NlCols<NP>::CGS;
    extern __shared__ __align__(16) unsigned char nl_smem_raw[];
    double2 *qs = reinterpret_cast<double2 *>(nl_smem_raw);          // [NP][ncol]
    const SphereChunk ch = t.chunks[chunk0 + blockIdx.x];
    const int a = ch.atom;
    const int64_t o = t.pt_off[a];
    const int npts = (int)(t.pt_off[a + 1] - o);
    const int np = t.nproj[a];
    for (int e = threadIdx.x; e < NP * ncol; e += NL_THREADS) {
        const int i = e / ncol, c = e - i * ncol;
        qs[e] = i < np ? q[((int64_t)a * t.maxproj + i) * ncol + c] : make_double2(0.0, 0.0);
    }
    const int s = threadIdx.x;
    const bool live = s < ch.count;
    int64_t g = 0;
    double b[NP];
#pragma unroll
    for (int i = 0; i < NP; ++i) b[i] = 0.0;
    if (live) {
        g = t.idx[o + ch.start + s];
        const double *beta = t.beta + t.beta_off[a] + ch.start + s;
#pragma unroll
        for (int i = 0; i < NP; ++i) b[i] = i < np ? __ldg(beta + (int64_t)i * npts) : 0.0;
    }
    __syncthreads();
    if (!live) return;
    const int ngroups = (ncol + CG - 1) / CG;
    for (int gy = ngroups - 1 - (int)blockIdx.y; gy >= 0; gy -= (int)gridDim.y) {   // last columns first: the FFT before ended there (L2)
        const int c0 = gy * CG;
        const int nc = min(CG, ncol - c0);
        double2 *hx = HX + (int64_t)c0 * ldhx + g;
        double2 v[CG];
#pragma unroll
        for (int c = 0; c < CG; ++c) v[c] = c < nc ? hx[(int64_t)c * ldhx] : make_double2(0.0, 0.0);
#pragma unroll
        for (int i = 0; i < NP; ++i) {
#pragma unroll
            for (int c = 0; c < CG; ++c) {
                const double2 qq = qs[i * ncol + min(c0 + c, ncol - 1)];
                v[c].x = fma(b[i], qq.x, v[c].x);
                v[c].y = fma(b[i], qq.y, v[c].y);
            }
        }
#pragma unroll
        for (int c = 0; c < CG; ++c)
            if (c < nc) hx[(int64_t)c * ldhx] = v[c];
    }
}

}  // namespace rsdft
