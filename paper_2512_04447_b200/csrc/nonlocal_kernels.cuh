// Kleinman-Bylander nonlocal projectors (PAPER.md:19 task (4), "memory-bandwidth-bound";
// PAPER.md:69 "dedicated GPU kernels"):
//   project:  p[a][i][c] = dV * sum_{s in S_a} beta[a][i][s] * psi_c(idx[a][s])
//   scatter:  HX_c(idx[a][s]) += sum_i beta[a][i][s] * q[a][i][c],   q = D_a p
// One CTA per (atom, column); sphere points are walked with coalesced idx/beta reads and a
// gather/scatter on the orbital; projections are reduced with warp shuffles then shared memory.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace rsdft {

struct SphereTables {
    const int64_t *pt_off;   // [natom+1] offset of atom a's points in idx
    const int64_t *beta_off; // [natom]   offset of atom a's beta block ([nproj][npts]) in beta
    const int32_t *idx;      // grid indices, sorted ascending per atom
    const double *beta;
    const int32_t *nproj;    // [natom]
    const double *D;         // [natom][maxproj*maxproj] (row-major nproj x nproj in the top-left)
    int32_t natom, maxproj;
};

template <int NP>
__global__ void __launch_bounds__(128) project_kernel(SphereTables t, const double2 *__restrict__ X, int64_t ldx,
                                                      int32_t ncol, double dV, double2 *__restrict__ p)
{
    const int a = blockIdx.x, c = blockIdx.y;   // all atoms
    const int64_t o = t.pt_off[a];
    const int npts = (int)(t.pt_off[a + 1] - o);
    const int np = t.nproj[a];
    const int32_t *idx = t.idx + o;
    const double *beta = t.beta + t.beta_off[a];
    const double2 *psi = X + (int64_t)c * ldx;
    double ar[NP], ai[NP];
#pragma unroll
    for (int i = 0; i < NP; ++i) { ar[i] = 0.0; ai[i] = 0.0; }
    for (int s = threadIdx.x; s < npts; s += blockDim.x) {
        const double2 v = __ldg(psi + idx[s]);
#pragma unroll
        for (int i = 0; i < NP; ++i)
            if (i < np) {
                const double b = __ldg(beta + (int64_t)i * npts + s);
                ar[i] = fma(b, v.x, ar[i]);
                ai[i] = fma(b, v.y, ai[i]);
            }
    }
    __shared__ double red[4][NP][2];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
#pragma unroll
    for (int i = 0; i < NP; ++i) {
#pragma unroll
        for (int sft = 16; sft > 0; sft >>= 1) {
            ar[i] += __shfl_xor_sync(0xffffffffu, ar[i], sft);
            ai[i] += __shfl_xor_sync(0xffffffffu, ai[i], sft);
        }
        if (lane == 0) { red[w][i][0] = ar[i]; red[w][i][1] = ai[i]; }
    }
    __syncthreads();
    if (threadIdx.x < np) {
        const int i = threadIdx.x;
        const double sr = (red[0][i][0] + red[1][i][0]) + (red[2][i][0] + red[3][i][0]);
        const double si = (red[0][i][1] + red[1][i][1]) + (red[2][i][1] + red[3][i][1]);
        p[((int64_t)a * t.maxproj + i) * ncol + c] = make_double2(dV * sr, dV * si);
    }
}

template <int NP, bool ATOMIC>
__global__ void __launch_bounds__(128) scatter_kernel(SphereTables t, const int32_t *__restrict__ alist,
                                                      const double2 *__restrict__ p, int32_t ncol,
                                                      double2 *__restrict__ HX, int64_t ldhx)
{
    // alist: the atoms of one colour class (spheres of one class are pairwise disjoint, so the
    // read-modify-write below is race-free and the result is deterministic)
    const int a = alist[blockIdx.x], c = blockIdx.y;
    const int64_t o = t.pt_off[a];
    const int npts = (int)(t.pt_off[a + 1] - o);
    const int np = t.nproj[a];
    const int32_t *idx = t.idx + o;
    const double *beta = t.beta + t.beta_off[a];
    __shared__ double qs[NP][2];
    if (threadIdx.x < np) {
        const int i = threadIdx.x;
        const double *D = t.D + (int64_t)a * t.maxproj * t.maxproj + (int64_t)i * np;
        double sr = 0.0, si = 0.0;
        for (int j = 0; j < np; ++j) {
            const double2 pj = p[((int64_t)a * t.maxproj + j) * ncol + c];
            sr = fma(D[j], pj.x, sr);
            si = fma(D[j], pj.y, si);
        }
        qs[i][0] = sr; qs[i][1] = si;
    }
    __syncthreads();
    double qr[NP], qi[NP];
#pragma unroll
    for (int i = 0; i < NP; ++i) { qr[i] = i < np ? qs[i][0] : 0.0; qi[i] = i < np ? qs[i][1] : 0.0; }
    double2 *hx = HX + (int64_t)c * ldhx;
    for (int s = threadIdx.x; s < npts; s += blockDim.x) {
        double sr = 0.0, si = 0.0;
#pragma unroll
        for (int i = 0; i < NP; ++i)
            if (i < np) {
                const double b = __ldg(beta + (int64_t)i * npts + s);
                sr = fma(b, qr[i], sr);
                si = fma(b, qi[i], si);
            }
        double2 *dst = hx + idx[s];
        if constexpr (ATOMIC) {
            atomicAdd(&dst->x, sr);
            atomicAdd(&dst->y, si);
        } else {
            const double2 v = *dst;
            *dst = make_double2(v.x + sr, v.y + si);
        }
    }
}

}  // namespace rsdft
