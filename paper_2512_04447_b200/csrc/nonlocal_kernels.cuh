// Kleinman-Bylander nonlocal projectors (PAPER.md:19 task (4), "memory-bandwidth-bound";
// PAPER.md:69 "dedicated GPU kernels"):
//   project:  pp[k][i][c] = dV * sum_{s in chunk k} beta[a][i][s] * psi_c(idx[a][s])
//   combine:  q[a][i][c]  = sum_j D_a[i][j] * sum_{k in chunks(a)} pp[k][j][c]      (fixed order)
//   scatter:  HX_c(idx[a][s]) += sum_i beta[a][i][s] * q[a][i][c]
// Every sphere is cut into chunks of <= PCH points; one CTA owns (chunk, group of CG columns):
// idx and beta are read ONCE per point and reused for the CG columns, whose gathers are
// independent loads in flight.  Partial projections are combined in a fixed order, and the
// scatter runs one launch per colour class (spheres of a class are pairwise disjoint), so the
// result is deterministic and bitwise independent of the column batching.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace rsdft {

constexpr int NL_PCH = 256;       // sphere points per chunk
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

// columns per CTA.  project: NP*CG complex accumulators (4 registers each) stay <= 72 registers;
// scatter: CG complex values in flight per point.
template <int NP> struct NlCols {
    static constexpr int CGP = NP <= 4 ? 4 : (NP <= 9 ? 2 : 1);
    static constexpr int CGS = NP <= 4 ? 8 : (NP <= 9 ? 4 : 2);
};

template <int NP>
__global__ void __launch_bounds__(NL_THREADS) project_kernel(SphereTables t, const double2 *__restrict__ X, int64_t ldx,
                                                             int32_t ncol, double dV, double2 *__restrict__ pp)
{
    constexpr int CG = NlCols<NP>::CGP;
    const SphereChunk ch = t.chunks[blockIdx.x];
    const int c0 = blockIdx.y * CG;
    const int a = ch.atom;
    const int64_t o = t.pt_off[a];
    const int npts = (int)(t.pt_off[a + 1] - o);
    const int np = t.nproj[a];
    const int32_t *idx = t.idx + o + ch.start;
    const double *beta = t.beta + t.beta_off[a] + ch.start;
    const double2 *psi = X + (int64_t)c0 * ldx;
    const int nc = min(CG, ncol - c0);
    double ar[NP][CG], ai[NP][CG];
#pragma unroll
    for (int i = 0; i < NP; ++i)
#pragma unroll
        for (int c = 0; c < CG; ++c) { ar[i][c] = 0.0; ai[i][c] = 0.0; }
    for (int s = threadIdx.x; s < ch.count; s += NL_THREADS) {
        const int64_t g = idx[s];
        double2 v[CG];
#pragma unroll
        for (int c = 0; c < CG; ++c) v[c] = c < nc ? __ldg(psi + (int64_t)c * ldx + g) : make_double2(0.0, 0.0);
#pragma unroll
        for (int i = 0; i < NP; ++i) {
            const double b = i < np ? __ldg(beta + (int64_t)i * npts + s) : 0.0;
#pragma unroll
            for (int c = 0; c < CG; ++c) {
                ar[i][c] = fma(b, v[c].x, ar[i][c]);
                ai[i][c] = fma(b, v[c].y, ai[i][c]);
            }
        }
    }
    __shared__ double red[NL_THREADS / 32][NP][CG][2];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
#pragma unroll
    for (int i = 0; i < NP; ++i)
#pragma unroll
        for (int c = 0; c < CG; ++c) {
            double r = ar[i][c], m = ai[i][c];
#pragma unroll
            for (int sft = 16; sft > 0; sft >>= 1) {
                r += __shfl_xor_sync(0xffffffffu, r, sft);
                m += __shfl_xor_sync(0xffffffffu, m, sft);
            }
            if (lane == 0) { red[w][i][c][0] = r; red[w][i][c][1] = m; }
        }
    __syncthreads();
    for (int e = threadIdx.x; e < NP * CG; e += NL_THREADS) {
        const int i = e / CG, c = e - i * CG;
        if (i < np && c < nc) {
            const double sr = (red[0][i][c][0] + red[1][i][c][0]) + (red[2][i][c][0] + red[3][i][c][0]);
            const double si = (red[0][i][c][1] + red[1][i][c][1]) + (red[2][i][c][1] + red[3][i][c][1]);
            pp[((int64_t)blockIdx.x * t.maxproj + i) * ncol + c0 + c] = make_double2(dV * sr, dV * si);
        }
    }
}

// q[a][i][c] = sum_j D_a[i][j] * (sum over the atom's chunks, ascending start, of pp[k][j][c])
__global__ void __launch_bounds__(128) combine_kernel(SphereTables t, const double2 *__restrict__ pp, int32_t ncol,
                                                      double2 *__restrict__ q)
{
    const int a = blockIdx.y;
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= ncol) return;
    const int np = t.nproj[a], mp = t.maxproj;
    const int k0 = t.atom_chunk0[a], k1 = t.atom_chunk0[a + 1];
    double pr[16], pi[16];
    for (int j = 0; j < np; ++j) {
        double sr = 0.0, si = 0.0;
        for (int k = k0; k < k1; ++k) {
            const double2 v = pp[((int64_t)t.atom_chunks[k] * mp + j) * ncol + c];
            sr += v.x; si += v.y;
        }
        pr[j] = sr; pi[j] = si;
    }
    const double *D = t.D + (int64_t)a * mp * mp;
    for (int i = 0; i < np; ++i) {
        double sr = 0.0, si = 0.0;
        for (int j = 0; j < np; ++j) {
            sr = fma(D[i * np + j], pr[j], sr);
            si = fma(D[i * np + j], pi[j], si);
        }
        q[((int64_t)a * mp + i) * ncol + c] = make_double2(sr, si);
    }
}

template <int NP>
__global__ void __launch_bounds__(NL_THREADS) scatter_kernel(SphereTables t, int32_t chunk0, const double2 *__restrict__ q,
                                                             int32_t ncol, double2 *__restrict__ HX, int64_t ldhx)
{
    // chunk0: first chunk of one colour class (spheres of one class are pairwise disjoint, so the
    // read-modify-write below is race-free and the result is deterministic)
    constexpr int CG = NlCols<NP>::CGS;
    const SphereChunk ch = t.chunks[chunk0 + blockIdx.x];
    const int c0 = blockIdx.y * CG;
    const int a = ch.atom;
    const int64_t o = t.pt_off[a];
    const int npts = (int)(t.pt_off[a + 1] - o);
    const int np = t.nproj[a];
    const int32_t *idx = t.idx + o + ch.start;
    const double *beta = t.beta + t.beta_off[a] + ch.start;
    const int nc = min(CG, ncol - c0);
    __shared__ double2 qs[NP][CG];
    for (int e = threadIdx.x; e < NP * CG; e += NL_THREADS) {
        const int i = e / CG, c = e - i * CG;
        qs[i][c] = (i < np && c < nc) ? q[((int64_t)a * t.maxproj + i) * ncol + c0 + c] : make_double2(0.0, 0.0);
    }
    __syncthreads();
    double2 *hx = HX + (int64_t)c0 * ldhx;
    for (int s = threadIdx.x; s < ch.count; s += NL_THREADS) {
        const int64_t g = idx[s];
        double2 v[CG];
#pragma unroll
        for (int c = 0; c < CG; ++c) v[c] = c < nc ? hx[(int64_t)c * ldhx + g] : make_double2(0.0, 0.0);
#pragma unroll
        for (int i = 0; i < NP; ++i) {
            const double b = i < np ? __ldg(beta + (int64_t)i * npts + s) : 0.0;
#pragma unroll
            for (int c = 0; c < CG; ++c) {
                const double2 qq = qs[i][c];
                v[c].x = fma(b, qq.x, v[c].x);
                v[c].y = fma(b, qq.y, v[c].y);
            }
        }
#pragma unroll
        for (int c = 0; c < CG; ++c)
            if (c < nc) hx[(int64_t)c * ldhx + g] = v[c];
    }
}

}  // namespace rsdft
