// librsdft: host plan + C ABI (include/rsdft.h) over the sm_100a kernels in this directory.
// PAPER.md:19 (tasks (1) FFT Laplacian, (2) H/S matrices, (4) nonlocal operator); the problem
// statement is BASELINE.json north_star/configs; readings R1..R18 are listed in DESIGN.md.
// Nothing here is shared with oracle/ (the CPU oracle is test infrastructure).
#include "../../include/rsdft.h"

#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <string>
#include <vector>

#include "eig_kernels.cuh"
#include "fft3_kernels.cuh"
#include "fft3_tma_kernels.cuh"
#include "gram_kernels.cuh"
#include "nonlocal_kernels.cuh"
#include "rotate_kernels.cuh"

namespace {

thread_local std::string g_err;

int fail(int code, const std::string &msg)
{
    g_err = msg;
    return code;
}

#define RS_CUDA(call)                                                                              \
    do {                                                                                           \
        cudaError_t e_ = (call);                                                                   \
        if (e_ != cudaSuccess)                                                                     \
            return fail(e_ == cudaErrorMemoryAllocation ? RSDFT_ALLOC : RSDFT_CUDA,                \
                        std::string(#call) + ": " + cudaGetErrorString(e_));                       \
    } while (0)

const long double PI_L = 3.14159265358979323846264338327950288L;

template <class T>
struct DevBuf {
    T *p = nullptr;
    size_t n = 0;
    ~DevBuf() { release(); }
    void release()
    {
        if (p) cudaFree(p);
        p = nullptr;
        n = 0;
    }
    cudaError_t alloc(size_t count)
    {
        release();
        if (count == 0) return cudaSuccess;
        cudaError_t e = cudaMalloc((void **)&p, count * sizeof(T));
        if (e == cudaSuccess) n = count;
        return e;
    }
    cudaError_t ensure(size_t count) { return count <= n ? cudaSuccess : alloc(count); }
    cudaError_t upload(const std::vector<T> &h)
    {
        cudaError_t e = alloc(h.size());
        if (e != cudaSuccess || h.empty()) return e;
        return cudaMemcpy(p, h.data(), h.size() * sizeof(T), cudaMemcpyHostToDevice);
    }
    // stream-ordered upload for buffers that kernels on `st` read next: the pageable source is staged
    // before cudaMemcpyAsync returns, and the copy is ordered before later work on `st`
    cudaError_t upload_async(const std::vector<T> &h, cudaStream_t st)
    {
        cudaError_t e = ensure(h.size());
        if (e != cudaSuccess || h.empty()) return e;
        return cudaMemcpyAsync(p, h.data(), h.size() * sizeof(T), cudaMemcpyHostToDevice, st);
    }
    size_t bytes() const { return n * sizeof(T); }
};

}  // namespace

struct rsdft_plan {
    int n[3];
    double len[3];
    int64_t ng;
    double dV;
    int device = 0;
    int num_sms = 148;

    // FFT tables
    DevBuf<double2> tw[3];        // per axis: w_N^m = (cos, -sin)(2 pi m / N)
    DevBuf<double> kin_x;         // t_x[kx] / Ng                       [Nx]
    DevBuf<double> kin_yz;        // (t_y[ky(r)] + t_z[kz(p)]) / Ng at r*Nz + p, permuted positions (fft3_kernels.cuh)
    DevBuf<double> vloc;          // [Ng], zero until set

    // projector tables
    int natom = 0, maxproj = 0;
    int64_t total_pts = 0, max_pts = 0;
    DevBuf<int64_t> pt_off, beta_off;
    DevBuf<int32_t> idx, nproj_a;
    DevBuf<double> beta, Dmat;
    int ncolour = 0, nchunks = 0;
    std::vector<int> colour_chunk_off;                // chunks of colour c = [off[c], off[c+1])
    DevBuf<rsdft::SphereChunk> chunks;                // sorted by (colour, atom, start)
    DevBuf<int32_t> atom_chunk0, atom_chunks;         // per-atom chunk id lists
    static constexpr int MAX_STREAMS = 4;
    DevBuf<double2> pp[MAX_STREAMS];                  // [nchunks][maxproj][batch] partial projections
    DevBuf<double2> pq[MAX_STREAMS];                  // [natom][maxproj][batch]   q = D p
    int nstreams = 3;                                 // batches round-robin over internal streams (rsdft_plan_set_streams)
    cudaStream_t s_batch[MAX_STREAMS] = {nullptr, nullptr, nullptr, nullptr};
    cudaEvent_t ev_fork = nullptr, ev_join[MAX_STREAMS] = {nullptr, nullptr, nullptr, nullptr};

    // apply_h batching
    int batch = 0;                // columns per kernel sequence
    int user_batch = 0;
    int pipeline = 2;             // FFT path (rsdft_plan_set_pipeline): 0 three kernels, 1 persistent pipeline kernel, 2 three kernels with the TMA-staged x kernel (default:
                                  // measured 4-11 % faster than path 0 on every config it has a shape for)
    DevBuf<uint32_t> pipe_pattern;
    DevBuf<int32_t> pipe_counters;
    int pipe_key = -1, pipe_npattern = 0;

    // gram workspace
    DevBuf<double2> gram_work;
    DevBuf<rsdft::GramTile> gram_tiles;
    int gram_tiles_n = -1, gram_ntiles = 0;
    DevBuf<rsdft::GramTile> gram_panel_tiles;         // panel-ordered list of the host entry point
    std::vector<int> gram_panel_off;
    int gram_panel_n = -1;
    int gram_h_upper = 0;                             // 1: H_sub from its upper tiles, mirrored (rsdft_plan_set_gram_mode)
    int gram_bulk = 0;                                // 1: TMA bulk-copy operand staging (rsdft_plan_set_gram_staging; measured slower)

    // host-buffer entry point
    DevBuf<double2> hostY, hostHY, hostHS;
    cudaStream_t s_copy = nullptr, s_comp = nullptr, s_h = nullptr;
    std::vector<cudaEvent_t> ev;
    cudaEvent_t ev_vloc = nullptr;                    // recorded by set_vloc on the caller's stream; block_step_host waits on it
    bool vloc_pending = false;

    // generalized eigen-solve (rsdft_subspace_eig): workspace, created on first use
    DevBuf<double2> eg_L, eg_B, eg_Z, eg_Dinv, eg_Kp, eg_Tp, eg_V0, eg_V1, eg_J, eg_Zs;
    DevBuf<double> eg_scal;                           // [0] ||K||_F^2, [1] rotation threshold, [2] off(K)^2, [8..] partial sums
    DevBuf<int> eg_info, eg_perm;
    DevBuf<int2> eg_pairs;
    int eg_pairs_nblk = -1;
    int eg_n = 0;                                     // size of the last successful solve (rsdft_subspace_eig_get)
    int eig_mode = 0;                                 // 0: two triangular solves (the paper's route), 1: ZHEGST-style
    int eig_inner = 1;                                // inner sweeps of the 64 x 64 sub-problems per visit
    double eig_stats[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    cudaEvent_t eg_ev[6] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
    // block Jacobi runs its critical chain (sub-problems, K update) on a high-priority stream and the V updates on a second one
    cudaStream_t eg_s_hi = nullptr, eg_s_lo = nullptr;
    cudaEvent_t eg_sync[6] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};   // J ready [2], V update done [2], fork, join

    int64_t last_launches = 0;

    ~rsdft_plan()
    {
        for (auto e : eg_ev) if (e) cudaEventDestroy(e);
        for (auto e : eg_sync) if (e) cudaEventDestroy(e);
        if (eg_s_hi) cudaStreamDestroy(eg_s_hi);
        if (eg_s_lo) cudaStreamDestroy(eg_s_lo);
        for (auto e : ev) cudaEventDestroy(e);
        for (int i = 0; i < MAX_STREAMS; ++i) {
            if (s_batch[i]) cudaStreamDestroy(s_batch[i]);
            if (ev_join[i]) cudaEventDestroy(ev_join[i]);
        }
        if (ev_fork) cudaEventDestroy(ev_fork);
        if (ev_vloc) cudaEventDestroy(ev_vloc);
        if (s_copy) cudaStreamDestroy(s_copy);
        if (s_comp) cudaStreamDestroy(s_comp);
        if (s_h) cudaStreamDestroy(s_h);
    }
    size_t device_bytes() const
    {
        size_t b = 0;
        for (int a = 0; a < 3; ++a) b += tw[a].bytes();
        b += kin_x.bytes() + kin_yz.bytes() + vloc.bytes() + pt_off.bytes() + beta_off.bytes() + idx.bytes() +
             nproj_a.bytes() + beta.bytes() + Dmat.bytes() + chunks.bytes() + atom_chunk0.bytes() + atom_chunks.bytes() +
             gram_work.bytes() + gram_tiles.bytes() + gram_panel_tiles.bytes() + hostY.bytes() + hostHY.bytes() + hostHS.bytes() +
             eg_L.bytes() + eg_B.bytes() + eg_Z.bytes() + eg_Dinv.bytes() + eg_Kp.bytes() + eg_Tp.bytes() + eg_V0.bytes() +
             eg_V1.bytes() + eg_J.bytes() + eg_Zs.bytes();
        for (int i = 0; i < MAX_STREAMS; ++i) b += pp[i].bytes() + pq[i].bytes();
        return b;
    }
};

namespace {

// ------------------------------------------------------------------------------------------
// host-side table construction (long double, rounded once)

// kappa(j) = j for j < N/2 else j - N  (BASELINE.json configs[0]; R2)
inline long kappa_of(long j, long n) { return 2 * j < n ? j : j - n; }

// real spherical harmonics, orthonormal on the unit sphere (R7, R8)
long double real_ylm(int l, int m, long double x, long double y, long double z)
{
    if (l == 0) return 0.5L / sqrtl(PI_L);
    const long double r2 = x * x + y * y + z * z;
    if (r2 == 0.0L) return 0.0L;
    if (l == 1) {
        const long double c = sqrtl(0.75L / PI_L) / sqrtl(r2);
        return c * (m < 0 ? y : (m == 0 ? z : x));
    }
    const long double a = sqrtl(15.0L / PI_L) / r2, b = sqrtl(5.0L / PI_L) / r2;
    switch (m) {
    case -2: return 0.5L * a * x * y;
    case -1: return 0.5L * a * y * z;
    case 0: return 0.25L * b * (3.0L * z * z - r2);
    case 1: return 0.5L * a * x * z;
    default: return 0.25L * a * (x * x - y * y);
    }
}

long double radial_part(const rsdft_species_t &sp, int i, long double r)
{
    if (sp.radial_kind == 0) return expl(-(long double)sp.alpha[i] * r * r);
    const long double u = r / (long double)sp.dr;
    const long j = (long)floorl(u);
    if (j >= sp.nr - 1) return 0.0L;
    const double *tab = sp.radial + (size_t)i * sp.nr;
    return (long double)tab[j] + (u - (long double)j) * ((long double)tab[j + 1] - (long double)tab[j]);
}

// minimum-image displacement, evaluated in double (R5, R6: membership is decided in
// double as dx*dx + dy*dy + dz*dz < rc*rc)
inline double min_img(double r, double R, double L)
{
    const double d = r - R;
    return d - L * std::nearbyint(d / L);
}

int validate_species(const rsdft_species_t &sp, const double len[3], int s)
{
    const std::string tag = "species " + std::to_string(s) + ": ";
    if (!(sp.rc > 0.0)) return fail(RSDFT_INVALID_ARG, tag + "rc must be > 0");
    if (sp.nproj < 1 || sp.nproj > 16) return fail(RSDFT_INVALID_ARG, tag + "nproj must be in 1..16");
    if (!sp.l || !sp.m || !sp.D) return fail(RSDFT_INVALID_ARG, tag + "null l/m/D");
    for (int i = 0; i < sp.nproj; ++i) {
        if (sp.l[i] < 0 || sp.l[i] > 2) return fail(RSDFT_INVALID_ARG, tag + "l must be 0..2");
        if (std::abs(sp.m[i]) > sp.l[i]) return fail(RSDFT_INVALID_ARG, tag + "|m| > l");
    }
    if (sp.radial_kind == 0) {
        if (!sp.alpha) return fail(RSDFT_INVALID_ARG, tag + "null alpha");
    } else if (sp.radial_kind == 1) {
        if (!sp.radial || sp.nr < 2 || !(sp.dr > 0.0)) return fail(RSDFT_INVALID_ARG, tag + "bad radial table");
    } else {
        return fail(RSDFT_INVALID_ARG, tag + "radial_kind must be 0 or 1");
    }
    for (int i = 0; i < sp.nproj; ++i)
        for (int j = 0; j < i; ++j)
            if (sp.D[i * sp.nproj + j] != sp.D[j * sp.nproj + i]) return fail(RSDFT_INVALID_ARG, tag + "D not symmetric");
    const double lmin = std::min(len[0], std::min(len[1], len[2]));
    if (!(2.0 * sp.rc < lmin)) return fail(RSDFT_UNSUPPORTED, tag + "2*rc >= min box length (one periodic image only)");
    return RSDFT_OK;
}

int build_spheres(rsdft_plan *P, const rsdft_atoms_t *atoms, const rsdft_projectors_t *proj)
{
    const int natom = atoms->natom;
    P->natom = natom;
    int maxproj = 0;
    for (int a = 0; a < natom; ++a) {
        const int s = atoms->species[a];
        if (s < 0 || s >= proj->nspecies) return fail(RSDFT_INVALID_ARG, "atom species index out of range");
        maxproj = std::max(maxproj, proj->species[s].nproj);
    }
    P->maxproj = maxproj;
    const double h[3] = {P->len[0] / P->n[0], P->len[1] / P->n[1], P->len[2] / P->n[2]};

    std::vector<int64_t> pt_off(natom + 1, 0), beta_off(natom, 0);
    std::vector<int32_t> idx, nproj_a(natom);
    std::vector<double> beta, Dm((size_t)natom * maxproj * maxproj, 0.0);
    int64_t max_pts = 0;
    for (int a = 0; a < natom; ++a) {
        const rsdft_species_t &sp = proj->species[atoms->species[a]];
        const double *R = atoms->pos + 3 * a;
        const double rc2 = sp.rc * sp.rc;
        // per-axis candidates: |d_axis|^2 < rc^2 is necessary for membership
        std::vector<int> cand[3];
        std::vector<double> dc[3];
        for (int ax = 0; ax < 3; ++ax)
            for (int i = 0; i < P->n[ax]; ++i) {
                const double d = min_img(i * h[ax], R[ax], P->len[ax]);
                if (d * d < rc2) { cand[ax].push_back(i); dc[ax].push_back(d); }
            }
        std::vector<int32_t> my;
        std::vector<double> mx, myy, mz;
        for (size_t ix = 0; ix < cand[0].size(); ++ix)
            for (size_t iy = 0; iy < cand[1].size(); ++iy)
                for (size_t iz = 0; iz < cand[2].size(); ++iz) {
                    const double dx = dc[0][ix], dy = dc[1][iy], dz = dc[2][iz];
                    const double d2 = dx * dx + dy * dy + dz * dz;
                    if (!(d2 < rc2)) continue;
                    my.push_back((int32_t)(((int64_t)cand[0][ix] * P->n[1] + cand[1][iy]) * P->n[2] + cand[2][iz]));
                    mx.push_back(dx); myy.push_back(dy); mz.push_back(dz);
                }
        const int64_t np = (int64_t)my.size();
        max_pts = std::max(max_pts, np);
        pt_off[a + 1] = pt_off[a] + np;
        beta_off[a] = (int64_t)beta.size();
        nproj_a[a] = sp.nproj;
        idx.insert(idx.end(), my.begin(), my.end());
        beta.resize(beta.size() + (size_t)np * sp.nproj);
        double *bt = beta.data() + beta_off[a];
        for (int64_t s = 0; s < np; ++s) {
            const long double x = mx[s], y = myy[s], z = mz[s];
            const long double r = sqrtl(x * x + y * y + z * z);
            for (int i = 0; i < sp.nproj; ++i)
                bt[(int64_t)i * np + s] = (double)(radial_part(sp, i, r) * real_ylm(sp.l[i], sp.m[i], x, y, z));
        }
        for (int i = 0; i < sp.nproj; ++i)
            for (int j = 0; j < sp.nproj; ++j)
                Dm[((size_t)a * maxproj + i) * maxproj + j] = sp.D[i * sp.nproj + j];
    }
    P->total_pts = pt_off[natom];
    P->max_pts = max_pts;

    // colour classes: atoms of one colour have pairwise DISJOINT point sets (exact test on the
    // index lists), so the scatter-add runs one launch per class without atomics.
    std::vector<uint64_t> ptmask((size_t)P->ng, 0);
    std::vector<int> colour(natom, 0);
    int ncolour = 0;
    for (int a = 0; a < natom; ++a) {
        uint64_t used = 0;
        for (int64_t s = pt_off[a]; s < pt_off[a + 1]; ++s) used |= ptmask[idx[s]];
        int c = 0;
        while (c < 64 && ((used >> c) & 1)) ++c;
        if (c == 64) return fail(RSDFT_UNSUPPORTED, "rsdft_plan_create: more than 64 mutually overlapping projector spheres");
        colour[a] = c;
        for (int64_t s = pt_off[a]; s < pt_off[a + 1]; ++s) ptmask[idx[s]] |= (uint64_t)1 << c;
        if (pt_off[a + 1] > pt_off[a]) ncolour = std::max(ncolour, c + 1);
    }
    P->ncolour = ncolour;
    // chunks of <= NL_PCH points, sorted by (colour, atom, start); per-atom chunk id lists
    std::vector<rsdft::SphereChunk> chunks;
    std::vector<std::vector<int32_t>> ids(natom);
    P->colour_chunk_off.assign(1, 0);
    for (int c = 0; c < ncolour; ++c) {
        for (int a = 0; a < natom; ++a) {
            if (colour[a] != c) continue;
            const int64_t np = pt_off[a + 1] - pt_off[a];
            for (int64_t st = 0; st < np; st += rsdft::NL_PCH) {
                ids[a].push_back((int32_t)chunks.size());
                chunks.push_back({a, (int32_t)st, (int32_t)std::min<int64_t>(rsdft::NL_PCH, np - st), 0});
            }
        }
        P->colour_chunk_off.push_back((int)chunks.size());
    }
    P->nchunks = (int)chunks.size();
    std::vector<int32_t> atom_chunk0(natom + 1, 0), atom_chunks;
    for (int a = 0; a < natom; ++a) {
        atom_chunks.insert(atom_chunks.end(), ids[a].begin(), ids[a].end());
        atom_chunk0[a + 1] = (int32_t)atom_chunks.size();
    }
    RS_CUDA(P->chunks.upload(chunks));
    RS_CUDA(P->atom_chunk0.upload(atom_chunk0));
    RS_CUDA(P->atom_chunks.upload(atom_chunks));

    RS_CUDA(P->pt_off.upload(pt_off));
    RS_CUDA(P->beta_off.upload(beta_off));
    RS_CUDA(P->idx.upload(idx));
    RS_CUDA(P->nproj_a.upload(nproj_a));
    RS_CUDA(P->beta.upload(beta));
    RS_CUDA(P->Dmat.upload(Dm));
    return RSDFT_OK;
}

// first-stage radix of an axis: 16 when it divides N, else 12 (fft3_kernels.cuh); 0 = length not supported
int first_radix(int N)
{
    if (rsdft::radix16_ok(N)) return 16;
    if (N % 12 == 0) {
        const int M = N / 12;
        return (M == 1 || M == 2 || M == 3 || M == 5 || M == 6 || M == 7 || M == 10 || M == 12) ? 12 : 0;
    }
    return 0;
}

int build_fft_tables(rsdft_plan *P)
{
    for (int ax = 0; ax < 3; ++ax) {
        const int N = P->n[ax];
        std::vector<double2> w(N);
        for (int m = 0; m < N; ++m) {
            // exact octant symmetries are kept by reducing the angle before cosl/sinl
            const long double ang = 2.0L * PI_L * (long double)m / (long double)N;
            w[m] = make_double2((double)cosl(ang), (double)(-sinl(ang)));
        }
        RS_CUDA(P->tw[ax].upload(w));
    }
    const long double inv_ng = 1.0L / (long double)P->ng;
    auto t_axis = [&](int ax, int k) -> long double {
        const long double g = 2.0L * PI_L * (long double)kappa_of(k, P->n[ax]) / (long double)P->len[ax];
        return 0.5L * g * g;
    };
    std::vector<double> kx(P->n[0]), kyz((size_t)P->n[1] * P->n[2]);
    for (int i = 0; i < P->n[0]; ++i) kx[i] = (double)(t_axis(0, i) * inv_ng);
    // k-space positions are permuted by the in-place transforms (N = R2*M, R2 = 16 or 12): y row r = k1*My + k2
    // holds ky = k1 + R2y*k2 ("R2-first"), z position p = k1*R2z + k2 holds kz = k1 + Mz*k2 ("M-first"); x is
    // indexed naturally.
    const int R2y = first_radix(P->n[1]), R2z = first_radix(P->n[2]);
    const int My = P->n[1] / R2y, Mz = P->n[2] / R2z;
    for (int r = 0; r < P->n[1]; ++r)
        for (int p = 0; p < P->n[2]; ++p) {
            const int ky = r / My + R2y * (r % My), kz = p / R2z + Mz * (p % R2z);
            kyz[(size_t)r * P->n[2] + p] = (double)((t_axis(1, ky) + t_axis(2, kz)) * inv_ng);
        }
    RS_CUDA(P->kin_x.upload(kx));
    RS_CUDA(P->kin_yz.upload(kyz));
    RS_CUDA(P->vloc.alloc((size_t)P->ng));
    RS_CUDA(cudaMemset(P->vloc.p, 0, P->vloc.bytes()));
    return RSDFT_OK;
}

}  // namespace

namespace {

// ------------------------------------------------------------------------------------------
// kernel launchers

using namespace rsdft;

// RSDFT_LAB_N: development builds that instantiate a single axis length (seconds instead of minutes to compile)
#ifdef RSDFT_LAB_N
#define RS_DISPATCH_N(ERR_, N_, FN_, ...)                                    \
    switch (N_) {                                                            \
    case RSDFT_LAB_N: ERR_ = FN_<RSDFT_LAB_N>(__VA_ARGS__); break;           \
    default: ERR_ = cudaErrorInvalidValue; break;                            \
    }
#else
#define RS_DISPATCH_N(ERR_, N_, FN_, ...)                                    \
    switch (N_) {                                                            \
    case 12: ERR_ = FN_<12>(__VA_ARGS__); break;                             \
    case 16: ERR_ = FN_<16>(__VA_ARGS__); break;                             \
    case 24: ERR_ = FN_<24>(__VA_ARGS__); break;                             \
    case 32: ERR_ = FN_<32>(__VA_ARGS__); break;                             \
    case 36: ERR_ = FN_<36>(__VA_ARGS__); break;                             \
    case 48: ERR_ = FN_<48>(__VA_ARGS__); break;                             \
    case 60: ERR_ = FN_<60>(__VA_ARGS__); break;                             \
    case 64: ERR_ = FN_<64>(__VA_ARGS__); break;                             \
    case 72: ERR_ = FN_<72>(__VA_ARGS__); break;                             \
    case 80: ERR_ = FN_<80>(__VA_ARGS__); break;                             \
    case 84: ERR_ = FN_<84>(__VA_ARGS__); break;                             \
    case 96: ERR_ = FN_<96>(__VA_ARGS__); break;                             \
    case 112: ERR_ = FN_<112>(__VA_ARGS__); break;                           \
    case 120: ERR_ = FN_<120>(__VA_ARGS__); break;                           \
    case 128: ERR_ = FN_<128>(__VA_ARGS__); break;                           \
    case 144: ERR_ = FN_<144>(__VA_ARGS__); break;                           \
    case 160: ERR_ = FN_<160>(__VA_ARGS__); break;                           \
    case 192: ERR_ = FN_<192>(__VA_ARGS__); break;                           \
    case 256: ERR_ = FN_<256>(__VA_ARGS__); break;                           \
    default: ERR_ = cudaErrorInvalidValue; break;                            \
    }
#endif

// CTAs per SM that fit by shared memory (1 KB reserved per CTA), capped
inline int occ_by_smem(size_t smem, int cap)
{
    return (int)std::max<size_t>(1, std::min<size_t>((size_t)cap, (size_t)(228 * 1024) / (smem + 2048)));
}

template <int NZ, int R2Y>
cudaError_t launch_fwd_zy_r(const Fft3Args &a, int sms, cudaStream_t st)
{
    auto k = fft3_fwd_zy_kernel<NZ, R2Y, 4>;
    const size_t smem = ZyCfg<NZ, R2Y>::SMEM_FWD;
    cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    // G plane-walkers for each of the my row classes, two CTA generations of the resident set
    const int64_t planes = (int64_t)a.ncol * a.nx;
    const int64_t g = std::max<int64_t>(1, std::min<int64_t>(planes, (int64_t)sms * 2 * occ_by_smem(smem, 4) / a.my));
    k<<<(int)(g * a.my), 128, smem, st>>>(a);
    return cudaSuccess;
}
template <int NZ>
cudaError_t launch_fwd_zy(const Fft3Args &a, int sms, cudaStream_t st)
{
    return a.r2y == 16 ? launch_fwd_zy_r<NZ, 16>(a, sms, st) : launch_fwd_zy_r<NZ, 12>(a, sms, st);
}
template <int NZ, int R2Y>
cudaError_t launch_inv_yz_r(const Fft3Args &a, int sms, cudaStream_t st)
{
    auto k = fft3_inv_yz_kernel<NZ, R2Y, 2>;
    const size_t smem = ZyCfg<NZ, R2Y>::SMEM_INV;
    cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    // G x-plane walkers per row class; every walker runs over all columns of the batch
    const int64_t gmax = std::max<int64_t>(1, (int64_t)sms * occ_by_smem(smem, 2) / a.my);
    const int64_t rounds = (a.nx + gmax - 1) / gmax;
    const int64_t g = (a.nx + rounds - 1) / rounds;
    k<<<(int)(g * a.my), 128, smem, st>>>(a);
    return cudaSuccess;
}
template <int NZ>
cudaError_t launch_inv_yz(const Fft3Args &a, int sms, cudaStream_t st)
{
    return a.r2y == 16 ? launch_inv_yz_r<NZ, 16>(a, sms, st) : launch_inv_yz_r<NZ, 12>(a, sms, st);
}

template <int NX, int TZ, int NT, int MINB>
cudaError_t launch_x_cfg(const Fft3Args &a, int sms, cudaStream_t st)
{
    const size_t smem = (size_t)NX * (a.my * TZ + 1) * sizeof(double2);
    if (smem + 4096 > 227 * 1024 || a.nz % TZ != 0) return cudaErrorInvalidConfiguration;
    const int64_t ntiles = (int64_t)a.ncol * a.r2y * (a.nz / TZ);
    auto k = fft3_x_kernel<NX, TZ, NT, MINB>;
    cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    const int occ = occ_by_smem(smem, MINB);
    k<<<(int)std::min<int64_t>(ntiles, (int64_t)sms * occ), NT, smem, st>>>(a);
    return cudaSuccess;
}

// cuTensorMapEncodeTiled through the runtime's driver entry point (no link against libcuda)
typedef CUresult (*TmaEncodeFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
TmaEncodeFn tma_encoder()
{
    static TmaEncodeFn fn = [] {
        void *p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) != cudaSuccess || q != cudaDriverEntryPointSuccess)
            p = nullptr;
        return (TmaEncodeFn)p;
    }();
    return fn;
}

// Tensor map of a column block seen as doubles [col][x][y][2*z]; box = one x tile (2*tz, my, nx, 1).
bool x_tile_map(CUtensorMap *tm, const Fft3Args &a, int tz)
{
    TmaEncodeFn enc = tma_encoder();
    if (!enc) return false;
    const cuuint64_t gdim[4] = {(cuuint64_t)2 * a.nz, (cuuint64_t)a.ny, (cuuint64_t)a.nx, (cuuint64_t)a.ncol};
    const cuuint64_t gstr[3] = {(cuuint64_t)a.nz * 16, (cuuint64_t)a.ny * a.nz * 16, (cuuint64_t)a.ldw * 16};
    const cuuint32_t box[4] = {(cuuint32_t)(2 * tz), (cuuint32_t)a.my, (cuuint32_t)a.nx, 1};
    const cuuint32_t estr[4] = {1, 1, 1, 1};
    // (L2 promotion 64 / 128 / 256 B: no measurable difference on the x tile)
    return enc(tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, (void *)a.W, gdim, gstr, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
               CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// TMA-staged x kernel (fft3_tma_kernels.cuh); returns cudaErrorNotSupported when the shape has none
template <int NX, int TZ, int G, int NTG, int SPG>
cudaError_t launch_x_tma_cfg(const Fft3Args &a, int sms, cudaStream_t st)
{
    if (a.ny != a.nx || a.r2y != Axis<NX>::R2 || Axis<NX>::R2 != 16 || a.nz % TZ != 0 || ((uintptr_t)a.W & 15) != 0) return cudaErrorNotSupported;
    CUtensorMap tm;
    if (!x_tile_map(&tm, a, TZ)) return cudaErrorNotSupported;
    auto k = fft3_x_tma_kernel<NX, TZ, G, NTG, SPG>;
    const size_t smem = XTmaSmem<NX, TZ, G, SPG>::bytes;
    cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    const int64_t ntiles = (int64_t)a.ncol * a.r2y * (a.nz / TZ);
    const int64_t grid = std::min<int64_t>(sms, (ntiles + G - 1) / G);
    k<<<(int)grid, G * NTG, smem, st>>>(a, tm);
    return cudaSuccess;
}
template <int NX>
cudaError_t launch_x_tma(const Fft3Args &a, int sms, cudaStream_t st)
{
    using Cc = XTmaCfg<NX>;
    if constexpr (Cc::TZ == 0) {
        return cudaErrorNotSupported;
    } else {
#ifdef RSDFT_LAB_N
        if (const char *e = getenv("RSDFT_LAB_XCFG")) {
            switch (atoi(e)) {
            case 1: return launch_x_tma_cfg<NX, 8, 2, 160, 1>(a, sms, st);
            case 2: return launch_x_tma_cfg<NX, 8, 2, 128, 1>(a, sms, st);
            case 3: return launch_x_tma_cfg<NX, 8, 2, 96, 1>(a, sms, st);
            case 4: return launch_x_tma_cfg<NX, 8, 2, 288, 1>(a, sms, st);
            case 5: return launch_x_tma_cfg<NX, 8, 3, 96, 1>(a, sms, st);
            default: break;
            }
        }
#endif
        return launch_x_tma_cfg<NX, Cc::TZ, Cc::G, Cc::NTG, Cc::SPG>(a, sms, st);
    }
}

template <int NX>
cudaError_t launch_x(const Fft3Args &a, int sms, cudaStream_t st)
{
    if (a.x_tma) {
        const cudaError_t e = launch_x_tma<NX>(a, sms, st);
        if (e != cudaErrorNotSupported) return e;
    }
    // the tile is NX x (my*TZ) elements: fall back to narrower z chunks when a large ny makes it too big or
    // when nz is not a multiple of the preferred chunk (nz = 12*M with odd M)
    auto fits = [&](int tz) { return a.nz % tz == 0 && (size_t)NX * (a.my * tz + 1) * sizeof(double2) + 4096 <= (size_t)227 * 1024; };
    if (fits(XCfg<NX>::TZ)) return launch_x_cfg<NX, XCfg<NX>::TZ, XCfg<NX>::NT, XCfg<NX>::MINB>(a, sms, st);
    if (fits(4)) return launch_x_cfg<NX, 4, 256, 1>(a, sms, st);
    return launch_x_cfg<NX, 2, 256, 1>(a, sms, st);
}

// Shapes of the persistent pipeline kernel (fft3_tma_kernels.cuh): cubic grids with a radix-16 first stage whose
// regions fit the 227 KB of shared memory.  TZ = z points per x tile, NS = fwd / inv slots per group.
template <int N> struct PipeShape { static constexpr int TZ = 0, NS = 0; };
template <> struct PipeShape<48> { static constexpr int TZ = 8, NS = 3; };
template <> struct PipeShape<64> { static constexpr int TZ = 8, NS = 3; };
template <> struct PipeShape<80> { static constexpr int TZ = 8, NS = 3; };
template <> struct PipeShape<96> { static constexpr int TZ = 8, NS = 3; };
template <> struct PipeShape<112> { static constexpr int TZ = 4, NS = 2; };
template <> struct PipeShape<128> { static constexpr int TZ = 4, NS = 2; };
template <int N> constexpr int pipe_tz() { return PipeShape<N>::TZ; }

// tensor maps of the pipeline kernel
bool rows_map(CUtensorMap *tm, const void *base, int64_t ld, const Fft3Args &a)
{
    TmaEncodeFn enc = tma_encoder();
    if (!enc || ((uintptr_t)base & 15) != 0 || 2 * a.nz > 256) return false;
    const cuuint64_t gdim[5] = {(cuuint64_t)2 * a.nz, (cuuint64_t)a.my, (cuuint64_t)a.r2y, (cuuint64_t)a.nx, (cuuint64_t)a.ncol};
    const cuuint64_t gstr[4] = {(cuuint64_t)a.nz * 16, (cuuint64_t)a.my * a.nz * 16, (cuuint64_t)a.ny * a.nz * 16, (cuuint64_t)ld * 16};
    const cuuint32_t box[5] = {(cuuint32_t)(2 * a.nz), 1, (cuuint32_t)a.r2y, 1, 1};
    const cuuint32_t estr[5] = {1, 1, 1, 1, 1};
    return enc(tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 5, const_cast<void *>(base), gdim, gstr, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
               CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}
bool vrows_map(CUtensorMap *tm, const Fft3Args &a)
{
    TmaEncodeFn enc = tma_encoder();
    if (!enc || ((uintptr_t)a.vloc & 15) != 0 || a.nz > 256 || (a.nz & 1)) return false;
    const cuuint64_t gdim[4] = {(cuuint64_t)a.nz, (cuuint64_t)a.my, (cuuint64_t)a.r2y, (cuuint64_t)a.nx};
    const cuuint64_t gstr[3] = {(cuuint64_t)a.nz * 8, (cuuint64_t)a.my * a.nz * 8, (cuuint64_t)a.ny * a.nz * 8};
    const cuuint32_t box[4] = {(cuuint32_t)a.nz, 1, (cuuint32_t)a.r2y, 1};
    const cuuint32_t estr[4] = {1, 1, 1, 1};
    return enc(tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, const_cast<double *>(a.vloc), gdim, gstr, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
               CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}
template <int N>
cudaError_t launch_pipeline(const Fft3Args &a, const PipeArgs &q, int sms, cudaStream_t st)
{
    using Sh = PipeShape<N>;
    if constexpr (Sh::TZ == 0) {
        return cudaErrorNotSupported;
    } else {
        constexpr int G = 3, NTG = 96;
        PipeMaps maps;
        if (!rows_map(&maps.x_rows, a.X, a.ldx, a) || !rows_map(&maps.w_rows, a.W, a.ldw, a) || !x_tile_map(&maps.w_xtile, a, Sh::TZ) ||
            !vrows_map(&maps.v_rows, a))
            return cudaErrorNotSupported;
        auto k = fft3_pipeline_kernel<N, 16, Sh::TZ, Sh::NS, G, NTG>;
        const size_t smem = (size_t)G * PipeCfg<N, 16, Sh::TZ, Sh::NS>::REGION + 1024;
        cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        const int64_t total = (int64_t)(a.ncol + q.lag_inv) * q.npattern;
        k<<<(int)std::min<int64_t>((total + G - 1) / G, (int64_t)sms), G * (NTG + 64), smem, st>>>(a, q, maps);
        return cudaSuccess;
    }
}

#ifdef RSDFT_LAB_N
#define RS_PIPE_LENGTHS(X_) X_(RSDFT_LAB_N)
#else
#define RS_PIPE_LENGTHS(X_) X_(48) X_(64) X_(80) X_(96) X_(112) X_(128)
#endif
inline bool pipeline_available(const int n[3])
{
    if (n[0] != n[1] || n[1] != n[2] || !tma_encoder()) return false;
#define RS_PIPE_OK(N_) case N_: return true;
    switch (n[0]) { RS_PIPE_LENGTHS(RS_PIPE_OK) default: return false; }
#undef RS_PIPE_OK
}

template <int MT>
void launch_project_mt(const SphereTables &t, const double2 *X, int64_t ldx, int ncol, double dV, double2 *pp,
                       int sms, cudaStream_t st)
{
    // widest column group (most beta/idx reuse) that still leaves >= ~8 CTAs of 4 warps per SM: the
    // kernel is latency-bound on its gathers, so warps in flight matter more than reuse
    const int gx = (t.nchunks + 3) / 4;
    const int64_t want = (int64_t)sms * 8;
#ifdef RSDFT_LAB_N
    if (const char *e = getenv("RSDFT_LAB_PG8")) {
        const int g8 = atoi(e);
        if (g8 == 4) project_kernel<MT, 4><<<dim3(gx, (ncol + 31) / 32), 128, 0, st>>>(t, X, ldx, ncol, dV, pp);
        else if (g8 == 2) project_kernel<MT, 2><<<dim3(gx, (ncol + 15) / 16), 128, 0, st>>>(t, X, ldx, ncol, dV, pp);
        else project_kernel<MT, 1><<<dim3(gx, (ncol + 7) / 8), 128, 0, st>>>(t, X, ldx, ncol, dV, pp);
        return;
    }
#endif
    // (two 8-row projector tiles with 32 columns per warp need 140 registers: 12 warps per SM; 16 columns measured 2 % faster at config 4)
    if (MT == 1 && ncol > 16 && (int64_t)gx * ((ncol + 31) / 32) >= want)
        project_kernel<MT, 4><<<dim3(gx, (ncol + 31) / 32), 128, 0, st>>>(t, X, ldx, ncol, dV, pp);
    else if (ncol > 8 && (int64_t)gx * ((ncol + 15) / 16) >= want)
        project_kernel<MT, 2><<<dim3(gx, (ncol + 15) / 16), 128, 0, st>>>(t, X, ldx, ncol, dV, pp);
    else
        project_kernel<MT, 1><<<dim3(gx, (ncol + 7) / 8), 128, 0, st>>>(t, X, ldx, ncol, dV, pp);
}
template <int NP>
void launch_scatter_np(const SphereTables &t, int chunk0, int nlist, const double2 *q, int ncol, double2 *HX,
                       int64_t ldhx, int sms, cudaStream_t st)
{
    constexpr int CG = NlCols<NP>::CGS;
    const int ngroups = (ncol + CG - 1) / CG;
    // enough CTAs for ~4 per SM when the chunk list is short; otherwise one CTA per chunk walks all column groups
    const int gy = std::max(1, std::min(ngroups, (4 * sms + nlist - 1) / nlist));
    const size_t smem = (size_t)NP * ncol * sizeof(double2);
    if (smem > 48 * 1024) cudaFuncSetAttribute(scatter_kernel<NP>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    scatter_kernel<NP><<<dim3(nlist, gy), NL_THREADS, smem, st>>>(t, chunk0, q, ncol, HX, ldhx);
}

SphereTables sphere_tables(const rsdft_plan *P)
{
    SphereTables t;
    t.pt_off = P->pt_off.p; t.beta_off = P->beta_off.p; t.idx = P->idx.p; t.beta = P->beta.p;
    t.nproj = P->nproj_a.p; t.D = P->Dmat.p; t.natom = P->natom; t.maxproj = P->maxproj;
    t.chunks = P->chunks.p; t.atom_chunk0 = P->atom_chunk0.p; t.atom_chunks = P->atom_chunks.p; t.nchunks = P->nchunks;
    return t;
}

int default_batch(const rsdft_plan *P)
{
    // columns per kernel sequence: ~540 MB of orbitals per launch (38 / 24 / 16 columns at 96^3 / 112^3 / 128^3, 68 at 80^3).  Measured on B200
    // (configs 2-4, 80^3): the kernels need >= 10-20 M points per launch to reach their asymptotic rate, the k-space scratch stops being
    // L2-resident beyond ~4 columns of 96^3 anyway (small L2-sized batches only lose), and 540 MB is 0-5 % faster than 270 MB.
    const int64_t per_col = P->ng * 16;
    int64_t b = (int64_t)(540ll << 20) / per_col;
    return (int)std::max<int64_t>(1, std::min<int64_t>(b, 72));      // (small grids: 64-72 columns measured better than 96)
}

Fft3Args fft3_args(const rsdft_plan *P, int nb, const double2 *X, int64_t ldx, double2 *HX, int64_t ldhx)
{
    Fft3Args fa;
    fa.X = X; fa.W = HX; fa.HX = HX; fa.ldx = ldx; fa.ldw = ldhx; fa.ldhx = ldhx;
    fa.ncol = nb; fa.nx = P->n[0]; fa.ny = P->n[1]; fa.nz = P->n[2];
    fa.r2y = first_radix(P->n[1]); fa.my = P->n[1] / fa.r2y;
    fa.twx = P->tw[0].p; fa.twy = P->tw[1].p; fa.twz = P->tw[2].p;
    fa.kin_x = P->kin_x.p; fa.kin_yz = P->kin_yz.p; fa.vloc = P->vloc.p;
    fa.hint_stream = 1; fa.hint_keep = 0;       // measured: X / psi / HX evict_first halves the pipeline kernel's DRAM traffic; evict_last on k-space adds nothing
    fa.x_tma = P->pipeline != 0;
#ifdef RSDFT_LAB_N
    if (const char *e = getenv("RSDFT_LAB_XTMA")) fa.x_tma = atoi(e);
    if (const char *e = getenv("RSDFT_LAB_HINTS")) { fa.hint_stream = (e[0] - '0'); fa.hint_keep = (e[1] - '0'); }
#endif
    return fa;
}

void launch_project(rsdft_plan *P, const SphereTables &tabs, int nb, const double2 *X, int64_t ldx, double2 *pp, double2 *pq, cudaStream_t st)
{
    if (P->maxproj <= 8) launch_project_mt<1>(tabs, X, ldx, nb, P->dV, pp, P->num_sms, st);
    else launch_project_mt<2>(tabs, X, ldx, nb, P->dV, pp, P->num_sms, st);
    combine_kernel<<<dim3(P->natom, (nb + NL_CCOLS - 1) / NL_CCOLS), 128, 0, st>>>(tabs, pp, nb, pq);
    P->last_launches += 2;
}

void launch_scatter(rsdft_plan *P, const SphereTables &tabs, int nb, const double2 *pq, double2 *HX, int64_t ldhx, cudaStream_t st)
{
    for (int c = 0; c < P->ncolour; ++c) {
        const int ch0 = P->colour_chunk_off[c], nlist = P->colour_chunk_off[c + 1] - ch0;
        if (nlist == 0) continue;
        if (P->maxproj <= 4) launch_scatter_np<4>(tabs, ch0, nlist, pq, nb, HX, ldhx, P->num_sms, st);
        else if (P->maxproj <= 9) launch_scatter_np<9>(tabs, ch0, nlist, pq, nb, HX, ldhx, P->num_sms, st);
        else launch_scatter_np<16>(tabs, ch0, nlist, pq, nb, HX, ldhx, P->num_sms, st);
        ++P->last_launches;
    }
}

// One unit of columns through the whole operator, on stream slot `slot`: the projections of all `nb` columns, then
// the three FFT kernels per sub-batch of `fft_batch` columns, then the scatter-adds of all `nb` columns.
int apply_h_batch(rsdft_plan *P, int slot, int nb, int fft_batch, const double2 *X, int64_t ldx, double2 *HX, int64_t ldhx, cudaStream_t st)
{
    const int Nx = P->n[0], Nz = P->n[2];
    const bool nl = P->natom > 0 && P->total_pts > 0;
    const SphereTables tabs = sphere_tables(P);
    double2 *pp = P->pp[slot].p, *pq = P->pq[slot].p;
    if (nl) launch_project(P, tabs, nb, X, ldx, pp, pq, st);    // projections read the INPUT orbitals
    for (int c0 = 0; c0 < nb; c0 += fft_batch) {
        const Fft3Args fa = fft3_args(P, std::min(fft_batch, nb - c0), X + (int64_t)c0 * ldx, ldx, HX + (int64_t)c0 * ldhx, ldhx);
        cudaError_t ke = cudaSuccess;
        RS_DISPATCH_N(ke, Nz, launch_fwd_zy, fa, P->num_sms, st)              // z fwd, y fwd stage A:  X -> HX
        RS_CUDA(ke);
        RS_DISPATCH_N(ke, Nx, launch_x, fa, P->num_sms, st)                   // y B, x fwd, t(k)/Ng, x inv, y B'
        RS_CUDA(ke);
        RS_DISPATCH_N(ke, Nz, launch_inv_yz, fa, P->num_sms, st)              // y A', z inv, + v(r) psi(r)
        RS_CUDA(ke);
        P->last_launches += 3;
    }
    if (nl) launch_scatter(P, tabs, nb, pq, HX, ldhx, st);
    RS_CUDA(cudaGetLastError());
    return RSDFT_OK;
}

// item order inside one super-step of the pipeline queue: the three phases interleaved in proportion
int pipeline_pattern(rsdft_plan *P, const Fft3Args &fa, int tz, PipeArgs &q, cudaStream_t st)
{
    q.n_fwd = fa.nx * fa.my;
    q.zchunks = fa.nz / tz;
    q.n_x = fa.r2y * q.zchunks;
    q.n_inv = q.n_fwd;
    const int key = fa.nx * 1024 + fa.my;
    if (P->pipe_key != key) {
        // Two parts per super-step: part 1 = fwd(s) interleaved with the first half of x(s-1), part 2 = inv(s-3)
        // interleaved with the second half of x(s-1).  Every dependency (all fwd items of a column before its x
        // items, all x items before its inv items) then lies at least one whole part back in the queue, so CTAs
        // rarely wait, while the compute-bound x tiles stay mixed with the memory-bound ones.
        std::vector<std::pair<double, uint32_t>> items;
        const int half_x = q.n_x / 2;
        for (int t = 0; t < q.n_fwd; ++t) items.push_back({(t + 0.5) / q.n_fwd, (0u << 28) | (uint32_t)t});
        for (int t = 0; t < half_x; ++t) items.push_back({(t + 0.5) / std::max(1, half_x) + 1e-9, (1u << 28) | (uint32_t)t});
        for (int t = 0; t < q.n_inv; ++t) items.push_back({1.0 + (t + 0.5) / q.n_inv, (2u << 28) | (uint32_t)t});
        for (int t = half_x; t < q.n_x; ++t)
            items.push_back({1.0 + (t - half_x + 0.5) / std::max(1, q.n_x - half_x) + 1e-9, (1u << 28) | (uint32_t)t});
        std::sort(items.begin(), items.end());
        std::vector<uint32_t> pat(items.size());
        for (size_t e = 0; e < items.size(); ++e) pat[e] = items[e].second;
        RS_CUDA(P->pipe_pattern.upload_async(pat, st));
        P->pipe_key = key;
        P->pipe_npattern = (int)pat.size();
    }
    q.pattern = P->pipe_pattern.p;
    q.npattern = P->pipe_npattern;
    q.lag_x = 1;
    q.lag_inv = 3;      // measured at configs[2] (FFT only, us per column): lag 2 -> 23.2, 3 -> 17.6, 4 -> 17.7; lag_x 2 / lag_inv 4 -> 18.3
#ifdef RSDFT_LAB_N
    if (const char *e = getenv("RSDFT_LAB_LAG")) q.lag_inv = atoi(e);
    if (const char *e = getenv("RSDFT_LAB_LAGX")) q.lag_x = atoi(e);
#endif
    return RSDFT_OK;
}

// All columns through ONE persistent FFT kernel (k-space handed over through L2); the projections of every batch
// run before it, the scatter-adds after it, everything on the caller's stream.
int apply_h_pipeline(rsdft_plan *P, int ncol, const double2 *X, int64_t ldx, double2 *HX, int64_t ldhx, int batch, cudaStream_t st)
{
    const bool nl = P->natom > 0 && P->total_pts > 0;
    const SphereTables tabs = sphere_tables(P);
    const size_t qstride = (size_t)P->natom * P->maxproj * batch;
    const int nbatches = (ncol + batch - 1) / batch;
    if (nl) {
        RS_CUDA(P->pp[0].ensure((size_t)P->nchunks * P->maxproj * batch));
        RS_CUDA(P->pq[0].ensure(qstride * nbatches));
        for (int k = 0; k < nbatches; ++k) {
            const int c0 = k * batch, nb = std::min(batch, ncol - c0);
            launch_project(P, tabs, nb, X + (int64_t)c0 * ldx, ldx, P->pp[0].p, P->pq[0].p + qstride * k, st);
        }
    }
    const Fft3Args fa = fft3_args(P, ncol, X, ldx, HX, ldhx);
    PipeArgs q;
    int tz = 0;
#define RS_PIPE_TZ(N_) case N_: tz = pipe_tz<N_>(); break;
    switch (P->n[0]) { RS_PIPE_LENGTHS(RS_PIPE_TZ) default: break; }
#undef RS_PIPE_TZ
    if (int rc = pipeline_pattern(P, fa, tz, q, st)) return rc;
    RS_CUDA(P->pipe_counters.ensure((size_t)3 * ncol + 4));
    RS_CUDA(cudaMemsetAsync(P->pipe_counters.p, 0, ((size_t)3 * ncol + 4) * sizeof(int32_t), st));
    q.head = P->pipe_counters.p;
    q.done = P->pipe_counters.p + 4;
    cudaError_t ke = cudaErrorInvalidValue;
#define RS_PIPE_LAUNCH(N_) case N_: ke = launch_pipeline<N_>(fa, q, P->num_sms, st); break;
    switch (P->n[0]) { RS_PIPE_LENGTHS(RS_PIPE_LAUNCH) default: break; }
#undef RS_PIPE_LAUNCH
    RS_CUDA(ke);
    ++P->last_launches;
    if (nl)
        for (int k = 0; k < nbatches; ++k) {
            const int c0 = k * batch, nb = std::min(batch, ncol - c0);
            launch_scatter(P, tabs, nb, P->pq[0].p + qstride * k, HX + (int64_t)c0 * ldhx, ldhx, st);
        }
    RS_CUDA(cudaGetLastError());
    return RSDFT_OK;
}

int apply_h_impl(rsdft_plan *P, int ncol, const double2 *X, int64_t ldx, double2 *HX, int64_t ldhx, cudaStream_t st)
{
    const int batch = P->user_batch > 0 ? P->user_batch : default_batch(P);
    P->batch = batch;
    if (P->pipeline == 1 && pipeline_available(P->n)) return apply_h_pipeline(P, ncol, X, ldx, HX, ldhx, batch, st);
    // With large projector tables (configs 3, 4: 43 / 98 MB of beta) the projector kernels work on units of 4 FFT
    // batches: project and scatter read beta once per unit, so its traffic per column drops 4x.
    const bool big_beta = P->natom > 0 && P->beta.bytes() >= ((size_t)32 << 20);
    const int unit = P->user_batch > 0 ? batch : (big_beta ? std::min(4 * batch, 64) : batch);
    const int nunits = (ncol + unit - 1) / unit;
    const int ns = std::max(1, std::min(std::min(P->nstreams, (int)rsdft_plan::MAX_STREAMS), nunits));
    if (P->natom > 0 && P->total_pts > 0)
        for (int i = 0; i < ns; ++i) {
            RS_CUDA(P->pp[i].ensure((size_t)P->nchunks * P->maxproj * unit));
            RS_CUDA(P->pq[i].ensure((size_t)P->natom * P->maxproj * unit));
        }
    if (ns > 1) {
        if (!P->ev_fork) RS_CUDA(cudaEventCreateWithFlags(&P->ev_fork, cudaEventDisableTiming));
        for (int i = 0; i < ns; ++i) {
            if (!P->s_batch[i]) RS_CUDA(cudaStreamCreateWithFlags(&P->s_batch[i], cudaStreamNonBlocking));
            if (!P->ev_join[i]) RS_CUDA(cudaEventCreateWithFlags(&P->ev_join[i], cudaEventDisableTiming));
        }
    }
    // the streams are re-aligned after every round of ns units: concurrent project/scatter kernels of the ns
    // streams then read the same beta lines through L2 (measured +6-8 %); with small tables free-running streams
    // are as fast or faster.
    const bool rounds = ns > 1 && big_beta;
    auto fork = [&]() -> cudaError_t {      // the internal streams start after everything already queued on `st`
        cudaError_t e = cudaEventRecord(P->ev_fork, st);
        for (int i = 0; i < ns && e == cudaSuccess; ++i) e = cudaStreamWaitEvent(P->s_batch[i], P->ev_fork, 0);
        return e;
    };
    auto join = [&]() -> cudaError_t {
        cudaError_t e = cudaSuccess;
        for (int i = 0; i < ns && e == cudaSuccess; ++i) {
            e = cudaEventRecord(P->ev_join[i], P->s_batch[i]);
            if (e == cudaSuccess) e = cudaStreamWaitEvent(st, P->ev_join[i], 0);
        }
        return e;
    };
    if (ns > 1) RS_CUDA(fork());
    int k = 0;
    for (int c0 = 0; c0 < ncol; c0 += unit, ++k) {
        const int nb = std::min(unit, ncol - c0);
        const int slot = ns > 1 ? k % ns : 0;
        if (rounds && k > 0 && slot == 0) {
            RS_CUDA(join());
            RS_CUDA(fork());
        }
        const int rc = apply_h_batch(P, slot, nb, batch, X + (int64_t)c0 * ldx, ldx, HX + (int64_t)c0 * ldhx, ldhx,
                                     ns > 1 ? P->s_batch[slot] : st);
        if (rc != RSDFT_OK) {
            if (ns > 1) (void)join();            // keep the caller's stream ordered after whatever was queued
            return rc;
        }
    }
    if (ns > 1) RS_CUDA(join());
    return RSDFT_OK;
}

// Gram configuration: 48 x 48 complex tile, 4 warps (2 x 2), each 24 x 24 = 3 x 3 DMMA tiles with three accumulator sets (3M
// complex product, gram_kernels.cuh), two CTAs per SM
#ifndef RSDFT_GRAM_WGM      // warps along M, warps along N, fragments per warp along M, along N, stages, 3M product, CTAs per SM
#define RSDFT_GRAM_WGM 2    // (the 4-product form of round 1: 2, 4, 6, 3, 3, false, 1 -- a 96 x 96 tile)
#define RSDFT_GRAM_WGN 2
#define RSDFT_GRAM_FA 3
#define RSDFT_GRAM_FB 3
#define RSDFT_GRAM_STAGES 3
#define RSDFT_GRAM_M3 true
#define RSDFT_GRAM_MINB 2
#endif
#ifndef RSDFT_GRAM_KC       // grid points per pipeline stage
#define RSDFT_GRAM_KC 16
#endif
#define RSDFT_GRAM_SHAPE RSDFT_GRAM_WGM, RSDFT_GRAM_WGN, RSDFT_GRAM_FA, RSDFT_GRAM_FB, RSDFT_GRAM_KC, RSDFT_GRAM_STAGES
using GCfg = GramCfg<RSDFT_GRAM_SHAPE>;
constexpr int GRAM_KC = RSDFT_GRAM_KC;

int choose_kslabs(int64_t ntiles, int64_t nchunks, int sms)
{
    // time model: units run in waves of `sms` CTAs; a unit costs its slab length plus a fixed
    // fill/epilogue overhead (~48 chunks' worth).  Pick the split with the least modelled time.
    const int64_t ksmax = std::max<int64_t>(1, std::min<int64_t>(64, nchunks / 64));
    int best = 1;
    double best_cost = 1e300;
    for (int64_t ks = 1; ks <= ksmax; ++ks) {
        const int64_t waves = (ntiles * ks + sms - 1) / sms;
        const double cost = (double)waves * ((double)((nchunks + ks - 1) / ks) + 48.0);
        if (cost < best_cost) { best_cost = cost; best = (int)ks; }
    }
    return best;
}

// One launch of the Gram kernels over `ntiles` tiles of a device tile list (any subset of the
// [S|H] tiles): split-K contraction into the tile-indexed workspace, then the fixed-order reduce.
int gram_launch(rsdft_plan *P, int n, const double2 *Y, int64_t ldy, const double2 *HY, int64_t ldhy, double2 *H, double2 *S,
                int lds, const GramTile *dtiles, int ntiles, cudaStream_t st, int ks_fixed = 0)
{
    if (ntiles == 0) return RSDFT_OK;
    const int64_t nchunks = P->ng / GRAM_KC;
    const int ks = ks_fixed > 0 ? ks_fixed : choose_kslabs(ntiles, nchunks, P->num_sms * RSDFT_GRAM_MINB);
    if ((size_t)ks * ntiles * GCfg::TM * GCfg::TN > P->gram_work.n)
        return fail(RSDFT_ALLOC, "gram_launch: workspace smaller than the launch needs (internal)");
    GramArgs a;
    a.Y = Y; a.HY = HY; a.ldy = ldy; a.ldhy = ldhy; a.n = n; a.ntiles = ntiles; a.kslabs = ks;
    a.nchunks = nchunks; a.tiles = dtiles; a.work = P->gram_work.p;
    // operand staging: TMA bulk copies (gram_bulk, rsdft_plan_set_gram_mode) or per-thread cp.async
    auto kern = P->gram_bulk ? gram_dmma_kernel<RSDFT_GRAM_SHAPE, true, RSDFT_GRAM_M3, RSDFT_GRAM_MINB> : gram_dmma_kernel<RSDFT_GRAM_SHAPE, false, RSDFT_GRAM_M3, RSDFT_GRAM_MINB>;
    // the attribute is per device/context: set it on every launch (cheap), never cache it per thread
    RS_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)GCfg::SMEM));
    kern<<<ntiles * ks, GCfg::THREADS, GCfg::SMEM, st>>>(a);
    GramReduceArgs r;
    r.work = P->gram_work.p; r.tiles = dtiles; r.H = H; r.S = S; r.n = n; r.lds = lds; r.kslabs = ks; r.ntiles = ntiles;
    r.tm = GCfg::TM; r.tn = GCfg::TN;
    gram_reduce_kernel<<<ntiles, 256, 0, st>>>(r);
    P->last_launches += 2;
    RS_CUDA(cudaGetLastError());
    return RSDFT_OK;
}

// workspace elements a launch of `ntiles` tiles needs
size_t gram_work_need(const rsdft_plan *P, int ntiles)
{
    if (ntiles == 0) return 0;
    return (size_t)choose_kslabs(ntiles, P->ng / GRAM_KC, P->num_sms * RSDFT_GRAM_MINB) * ntiles * GCfg::TM * GCfg::TN;
}

// the whole [S|H]: H tiles row-major, then the upper S tiles
int gram_impl(rsdft_plan *P, int n, const double2 *Y, int64_t ldy, const double2 *HY, int64_t ldhy, double2 *H, double2 *S,
              int lds, cudaStream_t st)
{
    const int tm = (n + GCfg::TM - 1) / GCfg::TM;
    const int key = n * 8 + (P->gram_h_upper ? 4 : 0) + (H ? 2 : 0) + (S ? 1 : 0);
    if (P->gram_tiles_n != key) {
        std::vector<GramTile> tiles;
        if (H)
            for (int i = 0; i < tm; ++i)
                for (int j = P->gram_h_upper ? i : 0; j < tm; ++j)
                    tiles.push_back({(int16_t)i, (int16_t)j, (int16_t)(P->gram_h_upper ? 2 : 0), 0});
        if (S)
            for (int i = 0; i < tm; ++i)
                for (int j = i; j < tm; ++j) tiles.push_back({(int16_t)i, (int16_t)j, 1, 0});
        RS_CUDA(P->gram_tiles.upload_async(tiles, st));
        P->gram_ntiles = (int)tiles.size();
        P->gram_tiles_n = key;
    }
    // the K split is the one of the full [S|H] launch whichever outputs are asked for, so that S_sub (or H_sub) alone
    // comes out bit for bit as it does together with the other matrix
    const int full = tm * tm + tm * (tm + 1) / 2;              // (also the same in both Gram modes)
    const int ks = choose_kslabs(full, P->ng / GRAM_KC, P->num_sms * RSDFT_GRAM_MINB);
    RS_CUDA(P->gram_work.ensure((size_t)ks * P->gram_ntiles * GCfg::TM * GCfg::TN));
    return gram_launch(P, n, Y, ldy, HY, ldhy, H, S, lds, P->gram_tiles.p, P->gram_ntiles, st, ks);
}

// tile list ordered by column panel (panel t = tile column t): panel t holds every [S|H] tile that
// becomes computable when columns [0, TM(t+1)) are on the device (TM = the Gram tile width): H(i<=t, t), H(t, j<t), S(i<=t, t).
int gram_panel_lists(rsdft_plan *P, int n, cudaStream_t st)
{
    const int key = 2 * n + P->gram_h_upper;
    if (P->gram_panel_n == key) return RSDFT_OK;
    const int tm = (n + GCfg::TM - 1) / GCfg::TM;
    std::vector<GramTile> tiles;
    P->gram_panel_off.assign(1, 0);
    for (int t = 0; t < tm; ++t) {
        for (int i = 0; i <= t; ++i) tiles.push_back({(int16_t)i, (int16_t)t, (int16_t)(P->gram_h_upper ? 2 : 0), 0});
        if (!P->gram_h_upper)
            for (int j = 0; j < t; ++j) tiles.push_back({(int16_t)t, (int16_t)j, 0, 0});
        for (int i = 0; i <= t; ++i) tiles.push_back({(int16_t)i, (int16_t)t, 1, 0});
        P->gram_panel_off.push_back((int)tiles.size());
    }
    RS_CUDA(P->gram_panel_tiles.upload_async(tiles, st));
    P->gram_panel_n = key;
    return RSDFT_OK;
}

// the compute calls launch on the current device: it must be the one the plan was created on
int check_device(const rsdft_plan *P, const char *who)
{
    int dev = -1;
    RS_CUDA(cudaGetDevice(&dev));
    if (dev != P->device)
        return fail(RSDFT_INVALID_ARG, std::string(who) + ": current CUDA device " + std::to_string(dev) +
                                           " is not the plan's device " + std::to_string(P->device));
    return RSDFT_OK;
}

bool overlaps(const void *a, size_t na, const void *b, size_t nb)
{
    const char *pa = (const char *)a, *pb = (const char *)b;
    return pa < pb + nb && pb < pa + na;
}

#include "eig_driver.cuh"

}  // namespace

// ------------------------------------------------------------------------------------------
// rsdft_subspace_gram_static: the Gram contraction for callers that cannot allocate (CUDA graph capture, serving loops).
// Its split-K partial tiles and its tile list live in the two file-scope arrays below instead of plan-owned cudaMalloc
// buffers: RSDFT_GRAM_STATIC_WORK_BYTES (64 MiB) + 12.1 KiB of device memory on every GPU that loads the library, held
// until exit.  Every call on a device shares them.  In host code the array names are host-side stand-ins, not device
// addresses: gram_static_scratch() resolves them with cudaGetSymbolAddress once per device.
constexpr int GRAM_STATIC_MAX_N = RSDFT_GRAM_STATIC_MAX_N;
constexpr int GRAM_STATIC_MAX_TCOLS = (GRAM_STATIC_MAX_N + GCfg::TM - 1) / GCfg::TM;
constexpr int GRAM_STATIC_MAX_TILES = GRAM_STATIC_MAX_TCOLS * GRAM_STATIC_MAX_TCOLS + GRAM_STATIC_MAX_TCOLS * (GRAM_STATIC_MAX_TCOLS + 1) / 2;
constexpr size_t GRAM_STATIC_WORK_ELEMS = (size_t)RSDFT_GRAM_STATIC_WORK_BYTES / sizeof(double2);
static_assert((size_t)GRAM_STATIC_MAX_TILES * GCfg::TM * GCfg::TN <= GRAM_STATIC_WORK_ELEMS,
              "RSDFT_GRAM_STATIC_WORK_BYTES too small for RSDFT_GRAM_STATIC_MAX_N columns at one K slab");

static __device__ __align__(256) double2 g_gram_static_work[GRAM_STATIC_WORK_ELEMS];        // [kslabs][ntiles][TN][TM]
static __device__ __align__(256) rsdft::GramTile g_gram_static_tiles[GRAM_STATIC_MAX_TILES];

// The tile list gram_impl builds on the host (H tiles row-major -- from the diagonal on in the Hermitian mode -- then the
// upper S tiles), written on the device so that no upload buffer is needed.  tc = tile columns.
__global__ void gram_static_tiles_kernel(int tc, int want_h, int want_s, int h_upper)
{
    const int upper = tc * (tc + 1) / 2;
    const int nh = want_h ? (h_upper ? upper : tc * tc) : 0;
    const int nt = nh + (want_s ? upper : 0);
    for (int e = blockIdx.x * blockDim.x + threadIdx.x; e < nt; e += gridDim.x * blockDim.x) {
        const bool is_h = e < nh;
        int i, j;
        if (is_h && !h_upper) { i = e / tc; j = e - i * tc; }
        else {                                   // e-th pair (i <= j) in row-major order
            int r = is_h ? e : e - nh;
            i = 0;
            while (r >= tc - i) { r -= tc - i; ++i; }
            j = i + r;
        }
        rsdft::GramTile t;
        t.ti = (int16_t)i; t.tj = (int16_t)j; t.mat = (int16_t)(is_h ? (h_upper ? 2 : 0) : 1); t.pad = 0;
        g_gram_static_tiles[e] = t;              // device code names the array directly
    }
}

namespace {

struct GramStaticScratch { double2 *work; rsdft::GramTile *tiles; };

// Device addresses of the two arrays for the CURRENT device (`dev`), resolved once per device.
int gram_static_scratch(int dev, GramStaticScratch &out)
{
    constexpr int MAXDEV = 64;
    static std::mutex mu;
    static GramStaticScratch cache[MAXDEV];
    static bool have[MAXDEV];
    if (dev < 0 || dev >= MAXDEV) return fail(RSDFT_UNSUPPORTED, "rsdft_subspace_gram_static: device ordinal beyond 63");
    std::lock_guard<std::mutex> lock(mu);
    if (!have[dev]) {
        GramStaticScratch s{nullptr, nullptr};
        RS_CUDA(cudaGetSymbolAddress((void **)&s.work, g_gram_static_work));
        RS_CUDA(cudaGetSymbolAddress((void **)&s.tiles, g_gram_static_tiles));
        if (!s.work || !s.tiles || ((uintptr_t)s.work & 255))
            return fail(RSDFT_CUDA, "rsdft_subspace_gram_static: cudaGetSymbolAddress returned an unusable address");
        cache[dev] = s;
        have[dev] = true;
    }
    out = cache[dev];
    return RSDFT_OK;
}

}  // namespace

// ------------------------------------------------------------------------------------------
// C ABI

extern "C" {

const char *rsdft_last_error(void) { return g_err.c_str(); }

int rsdft_plan_create(const rsdft_grid_t *grid, const rsdft_box_t *box, const rsdft_atoms_t *atoms,
                      const rsdft_projectors_t *projectors, rsdft_plan_t **out)
{
    if (!grid || !box || !out) return fail(RSDFT_INVALID_ARG, "rsdft_plan_create: null grid/box/out");
    *out = nullptr;
    for (int a = 0; a < 3; ++a) {
        const int N = grid->n[a];
        if (N <= 0) return fail(RSDFT_INVALID_ARG, "rsdft_plan_create: grid length <= 0");
        if (first_radix(N) == 0)
            return fail(RSDFT_UNSUPPORTED, "rsdft_plan_create: grid length " + std::to_string(N) +
                                               " not in {12,16,24,32,36,48,60,64,72,80,84,96,112,120,128,144,160,192,256}");
        if (!(box->len[a] > 0.0) || !std::isfinite(box->len[a]))
            return fail(RSDFT_UNSUPPORTED, "rsdft_plan_create: box length must be positive and finite");
    }
    const bool have_atoms = atoms && atoms->natom > 0 && projectors && projectors->nspecies > 0;
    if (atoms && atoms->natom < 0) return fail(RSDFT_INVALID_ARG, "rsdft_plan_create: natom < 0");
    if (atoms && atoms->natom > 0 && (!projectors || projectors->nspecies <= 0 || !projectors->species))
        return fail(RSDFT_INVALID_ARG, "rsdft_plan_create: atoms given without projectors");
    if (have_atoms) {
        if (!atoms->pos || !atoms->species) return fail(RSDFT_INVALID_ARG, "rsdft_plan_create: null atom arrays");
        for (int s = 0; s < projectors->nspecies; ++s) {
            const int rc = validate_species(projectors->species[s], box->len, s);
            if (rc != RSDFT_OK) return rc;
        }
        for (int a = 0; a < 3 * atoms->natom; ++a)
            if (!std::isfinite(atoms->pos[a])) return fail(RSDFT_INVALID_ARG, "rsdft_plan_create: non-finite atom position");
    }
    rsdft_plan *P = new (std::nothrow) rsdft_plan();
    if (!P) return fail(RSDFT_ALLOC, "rsdft_plan_create: host allocation failed");
    for (int a = 0; a < 3; ++a) { P->n[a] = grid->n[a]; P->len[a] = box->len[a]; }
    P->ng = (int64_t)P->n[0] * P->n[1] * P->n[2];
    P->dV = (double)(((long double)P->len[0] / P->n[0]) * ((long double)P->len[1] / P->n[1]) *
                     ((long double)P->len[2] / P->n[2]));
    int rc = RSDFT_OK;
    cudaError_t e = cudaGetDevice(&P->device);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&P->num_sms, cudaDevAttrMultiProcessorCount, P->device);
    if (e != cudaSuccess) rc = fail(RSDFT_CUDA, std::string("rsdft_plan_create: ") + cudaGetErrorString(e));
    try {
        if (rc == RSDFT_OK) rc = build_fft_tables(P);
        if (rc == RSDFT_OK && have_atoms) rc = build_spheres(P, atoms, projectors);
    } catch (const std::bad_alloc &) {
        rc = fail(RSDFT_ALLOC, "rsdft_plan_create: host allocation failed");
    }
    if (rc == RSDFT_OK) {
        // the table uploads above ran on the legacy stream: finish them before the plan can be used
        // from a non-blocking stream
        const cudaError_t se = cudaDeviceSynchronize();
        if (se != cudaSuccess) rc = fail(RSDFT_CUDA, std::string("rsdft_plan_create: ") + cudaGetErrorString(se));
    }
    if (rc != RSDFT_OK) { delete P; return rc; }
    *out = P;
    return RSDFT_OK;
}

int rsdft_plan_destroy(rsdft_plan_t *plan)
{
    if (!plan) return RSDFT_OK;
    cudaDeviceSynchronize();
    delete plan;
    return RSDFT_OK;
}

int rsdft_plan_set_vloc(rsdft_plan_t *plan, const double *vloc_dev, void *stream)
{
    if (!plan) return fail(RSDFT_INVALID_ARG, "rsdft_plan_set_vloc: null plan");
    if (int rc = check_device(plan, "rsdft_plan_set_vloc")) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    if (vloc_dev) RS_CUDA(cudaMemcpyAsync(plan->vloc.p, vloc_dev, plan->vloc.bytes(), cudaMemcpyDeviceToDevice, st));
    else RS_CUDA(cudaMemsetAsync(plan->vloc.p, 0, plan->vloc.bytes(), st));
    // rsdft_block_step_host runs on plan-owned streams: it orders itself after this copy through the event
    if (!plan->ev_vloc) RS_CUDA(cudaEventCreateWithFlags(&plan->ev_vloc, cudaEventDisableTiming));
    RS_CUDA(cudaEventRecord(plan->ev_vloc, st));
    plan->vloc_pending = true;
    return RSDFT_OK;
}

int rsdft_plan_set_batch(rsdft_plan_t *plan, int32_t batch_cols)
{
    if (!plan || batch_cols < 0 || batch_cols > 65535) return fail(RSDFT_INVALID_ARG, "rsdft_plan_set_batch: bad argument");
    plan->user_batch = batch_cols;
    return RSDFT_OK;
}

int rsdft_plan_set_pipeline(rsdft_plan_t *plan, int32_t mode)
{
    if (!plan || mode < 0 || mode > 2) return fail(RSDFT_INVALID_ARG, "rsdft_plan_set_pipeline: mode must be 0, 1 or 2");
    plan->pipeline = mode;
    return RSDFT_OK;
}

int rsdft_plan_set_streams(rsdft_plan_t *plan, int32_t nstreams)
{
    if (!plan || nstreams < 0 || nstreams > rsdft_plan::MAX_STREAMS)
        return fail(RSDFT_INVALID_ARG, "rsdft_plan_set_streams: nstreams must be in 0..4");
    plan->nstreams = nstreams == 0 ? 3 : nstreams;
    return RSDFT_OK;
}

int rsdft_plan_set_gram_mode(rsdft_plan_t *plan, int32_t h_upper_only)
{
    if (!plan || (h_upper_only != 0 && h_upper_only != 1))
        return fail(RSDFT_INVALID_ARG, "rsdft_plan_set_gram_mode: mode must be 0 or 1");
    plan->gram_h_upper = h_upper_only;
    return RSDFT_OK;
}

int rsdft_plan_set_gram_staging(rsdft_plan_t *plan, int32_t bulk)
{
    if (!plan || (bulk != 0 && bulk != 1)) return fail(RSDFT_INVALID_ARG, "rsdft_plan_set_gram_staging: bulk must be 0 or 1");
    plan->gram_bulk = bulk;
    return RSDFT_OK;
}

int rsdft_plan_info(const rsdft_plan_t *plan, int64_t *out8)
{
    if (!plan || !out8) return fail(RSDFT_INVALID_ARG, "rsdft_plan_info: null argument");
    out8[0] = plan->natom; out8[1] = plan->total_pts; out8[2] = plan->max_pts; out8[3] = (int64_t)plan->device_bytes();
    out8[4] = plan->user_batch > 0 ? plan->user_batch : default_batch(plan); out8[5] = plan->last_launches;
    out8[6] = plan->ng; out8[7] = plan->ncolour;
    return RSDFT_OK;
}

int rsdft_apply_h(rsdft_plan_t *plan, int32_t ncol, const void *X, int64_t ldx, void *HX, int64_t ldhx, void *stream)
{
    if (!plan || !X || !HX) return fail(RSDFT_INVALID_ARG, "rsdft_apply_h: null argument");
    if (ncol <= 0) return fail(RSDFT_INVALID_ARG, "rsdft_apply_h: ncol <= 0");
    if (ldx < plan->ng || ldhx < plan->ng) return fail(RSDFT_INVALID_ARG, "rsdft_apply_h: ld < Ng");
    if (((uintptr_t)X | (uintptr_t)HX) & 15) return fail(RSDFT_INVALID_ARG, "rsdft_apply_h: pointers must be 16-byte aligned");
    const size_t bx = ((size_t)(ncol - 1) * ldx + plan->ng) * 16, bh = ((size_t)(ncol - 1) * ldhx + plan->ng) * 16;
    if (overlaps(X, bx, HX, bh)) return fail(RSDFT_INVALID_ARG, "rsdft_apply_h: X and HX overlap");
    if (int rc = check_device(plan, "rsdft_apply_h")) return rc;
    plan->last_launches = 0;
    return apply_h_impl(plan, ncol, (const double2 *)X, ldx, (double2 *)HX, ldhx, (cudaStream_t)stream);
}

int rsdft_subspace_gram(rsdft_plan_t *plan, int32_t n, const void *Y, int64_t ldy, const void *HY, int64_t ldhy,
                        void *H_sub, void *S_sub, int32_t lds, void *stream)
{
    if (!plan || !Y) return fail(RSDFT_INVALID_ARG, "rsdft_subspace_gram: null argument");
    if (n <= 0 || n > 32767 * GCfg::TM) return fail(RSDFT_INVALID_ARG, "rsdft_subspace_gram: n out of range");
    if (!H_sub && !S_sub) return fail(RSDFT_INVALID_ARG, "rsdft_subspace_gram: both outputs null");
    if (H_sub && !HY) return fail(RSDFT_INVALID_ARG, "rsdft_subspace_gram: H_sub requested without HY");
    if (ldy < plan->ng || (H_sub && ldhy < plan->ng)) return fail(RSDFT_INVALID_ARG, "rsdft_subspace_gram: ld < Ng");
    if (lds < n) return fail(RSDFT_INVALID_ARG, "rsdft_subspace_gram: lds < n");
    if (((uintptr_t)Y | (uintptr_t)HY | (uintptr_t)H_sub | (uintptr_t)S_sub) & 15)
        return fail(RSDFT_INVALID_ARG, "rsdft_subspace_gram: pointers must be 16-byte aligned");
    if (int rc = check_device(plan, "rsdft_subspace_gram")) return rc;
    plan->last_launches = 0;
    return gram_impl(plan, n, (const double2 *)Y, ldy, H_sub ? (const double2 *)HY : nullptr, ldhy, (double2 *)H_sub,
                     (double2 *)S_sub, lds, (cudaStream_t)stream);
}

int rsdft_subspace_gram_static(rsdft_plan_t *plan, int32_t n, const void *Y, int64_t ldy, const void *HY, int64_t ldhy,
                               void *H_sub, void *S_sub, int32_t lds, void *stream)
{
    if (!plan || !Y) return fail(RSDFT_INVALID_ARG, "rsdft_subspace_gram_static: null argument");
    if (n <= 0) return fail(RSDFT_INVALID_ARG, "rsdft_subspace_gram_static: n out of range");
    if (n > GRAM_STATIC_MAX_N)
        return fail(RSDFT_UNSUPPORTED, "rsdft_subspace_gram_static: n = " + std::to_string(n) + " exceeds RSDFT_GRAM_STATIC_MAX_N = " +
                                           std::to_string(GRAM_STATIC_MAX_N) + " (the static scratch of " +
                                           std::to_string(RSDFT_GRAM_STATIC_WORK_BYTES >> 20) + " MiB holds no more); use rsdft_subspace_gram");
    if (!H_sub && !S_sub) return fail(RSDFT_INVALID_ARG, "rsdft_subspace_gram_static: both outputs null");
    if (H_sub && !HY) return fail(RSDFT_INVALID_ARG, "rsdft_subspace_gram_static: H_sub requested without HY");
    if (ldy < plan->ng || (H_sub && ldhy < plan->ng)) return fail(RSDFT_INVALID_ARG, "rsdft_subspace_gram_static: ld < Ng");
    if (lds < n) return fail(RSDFT_INVALID_ARG, "rsdft_subspace_gram_static: lds < n");
    if (((uintptr_t)Y | (uintptr_t)HY | (uintptr_t)H_sub | (uintptr_t)S_sub) & 15)
        return fail(RSDFT_INVALID_ARG, "rsdft_subspace_gram_static: pointers must be 16-byte aligned");
    if (int rc = check_device(plan, "rsdft_subspace_gram_static")) return rc;
    GramStaticScratch sc;
    if (int rc = gram_static_scratch(plan->device, sc)) return rc;

    const cudaStream_t st = (cudaStream_t)stream;
    const int tc = (n + GCfg::TM - 1) / GCfg::TM;
    const int upper = tc * (tc + 1) / 2;
    const int ntiles = (H_sub ? (plan->gram_h_upper ? upper : tc * tc) : 0) + (S_sub ? upper : 0);
    // the K split rsdft_subspace_gram takes (so that the two agree bit for bit), cut down to what the scratch holds
    const int64_t nchunks = plan->ng / GRAM_KC;
    int ks = choose_kslabs(tc * tc + upper, nchunks, plan->num_sms * RSDFT_GRAM_MINB);
    ks = (int)std::max<size_t>(1, std::min<size_t>((size_t)ks, GRAM_STATIC_WORK_ELEMS / ((size_t)ntiles * GCfg::TM * GCfg::TN)));

    gram_static_tiles_kernel<<<(ntiles + 255) / 256, 256, 0, st>>>(tc, H_sub != nullptr, S_sub != nullptr, plan->gram_h_upper);
    GramArgs a;
    a.Y = (const double2 *)Y; a.HY = H_sub ? (const double2 *)HY : nullptr; a.ldy = ldy; a.ldhy = ldhy; a.n = n; a.ntiles = ntiles;
    a.kslabs = ks; a.nchunks = nchunks; a.tiles = sc.tiles; a.work = sc.work;
    auto kern = gram_dmma_kernel<RSDFT_GRAM_SHAPE, false, RSDFT_GRAM_M3, RSDFT_GRAM_MINB>;
    RS_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)GCfg::SMEM));
    kern<<<ntiles * ks, GCfg::THREADS, GCfg::SMEM, st>>>(a);      // every (slab, tile) of the scratch it reads later is written here in full:
    GramReduceArgs r;                                             // nothing has to start at zero
    r.work = sc.work; r.tiles = sc.tiles; r.H = (double2 *)H_sub; r.S = (double2 *)S_sub; r.n = n; r.lds = lds; r.kslabs = ks; r.ntiles = ntiles;
    r.tm = GCfg::TM; r.tn = GCfg::TN;
    gram_reduce_kernel<<<ntiles, 256, 0, st>>>(r);
    plan->last_launches = 3;
    RS_CUDA(cudaGetLastError());
    return RSDFT_OK;
}

int rsdft_subspace_rotate(rsdft_plan_t *plan, int32_t n, int32_t m, const void *Y, int64_t ldy, const void *Cmat, int32_t ldc,
                          void *Out, int64_t ldo, void *stream)
{
    if (!plan || !Y || !Cmat || !Out) return fail(RSDFT_INVALID_ARG, "rsdft_subspace_rotate: null argument");
    if (n <= 0 || m <= 0) return fail(RSDFT_INVALID_ARG, "rsdft_subspace_rotate: n, m must be > 0");
    if (ldy < plan->ng || ldo < plan->ng) return fail(RSDFT_INVALID_ARG, "rsdft_subspace_rotate: ld < Ng");
    if (ldc < n) return fail(RSDFT_INVALID_ARG, "rsdft_subspace_rotate: ldc < n");
    if (((uintptr_t)Y | (uintptr_t)Cmat | (uintptr_t)Out) & 15)
        return fail(RSDFT_INVALID_ARG, "rsdft_subspace_rotate: pointers must be 16-byte aligned");
    const size_t by = ((size_t)(n - 1) * ldy + plan->ng) * 16, bo = ((size_t)(m - 1) * ldo + plan->ng) * 16;
    if (overlaps(Y, by, Out, bo)) return fail(RSDFT_INVALID_ARG, "rsdft_subspace_rotate: Y and Out overlap");
    if (int rc = check_device(plan, "rsdft_subspace_rotate")) return rc;
    RotateArgs a;
    a.Y = (const double2 *)Y; a.C = (const double2 *)Cmat; a.Out = (double2 *)Out;
    a.ldy = ldy; a.ldo = ldo; a.ng = plan->ng; a.n = n; a.m = m; a.ldc = ldc;
    // 3M complex product (rotate_kernels.cuh): output tile 48 x 48 or 48 x 64 (rows x columns), whichever pads m less
    // (m = 480 -> 48, m = 512 -> 64), four warps with three accumulator sets, two CTAs per SM
    const bool wide = ((m + 63) / 64) * 64 < ((m + 47) / 48) * 48;
    using R48 = RotateCfg<2, 2, 3, 3, 16, 3>;
    using R64 = RotateCfg<2, 2, 3, 4, 16, 3>;
    const int tm = wide ? R64::TM : R48::TM, tn = wide ? R64::TN : R48::TN;
    a.jtiles = (m + tn - 1) / tn;
    const int64_t units = ((plan->ng + tm - 1) / tm) * a.jtiles;
    if (units > 0x7fffffffll) return fail(RSDFT_UNSUPPORTED, "rsdft_subspace_rotate: too many tiles for one launch");
    if (wide) {
        auto kern = rotate_dmma_kernel<2, 2, 3, 4, 16, 3, true, 2>;
        RS_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)R64::SMEM));
        kern<<<(unsigned)units, R64::THREADS, R64::SMEM, (cudaStream_t)stream>>>(a);
    } else {
        auto kern = rotate_dmma_kernel<2, 2, 3, 3, 16, 3, true, 2>;
        RS_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)R48::SMEM));
        kern<<<(unsigned)units, R48::THREADS, R48::SMEM, (cudaStream_t)stream>>>(a);
    }
    plan->last_launches = 1;
    RS_CUDA(cudaGetLastError());
    return RSDFT_OK;
}

int rsdft_block_step_host(rsdft_plan_t *plan, int32_t n, const void *Y_host, int64_t ldy, void *HY_host, int64_t ldhy,
                          void *H_sub_host, void *S_sub_host, int32_t lds)
{
    if (!plan || !Y_host || !H_sub_host || !S_sub_host) return fail(RSDFT_INVALID_ARG, "rsdft_block_step_host: null argument");
    if (n <= 0) return fail(RSDFT_INVALID_ARG, "rsdft_block_step_host: n <= 0");
    if (ldy < plan->ng || (HY_host && ldhy < plan->ng)) return fail(RSDFT_INVALID_ARG, "rsdft_block_step_host: ld < Ng");
    if (lds < n) return fail(RSDFT_INVALID_ARG, "rsdft_block_step_host: lds < n");
    if (int rc = check_device(plan, "rsdft_block_step_host")) return rc;
    rsdft_plan *P = plan;
    const int64_t ng = P->ng;
    RS_CUDA(P->hostY.ensure((size_t)n * ng));
    RS_CUDA(P->hostHY.ensure((size_t)n * ng));
    RS_CUDA(P->hostHS.ensure((size_t)2 * n * n));
    if (!P->s_copy) RS_CUDA(cudaStreamCreateWithFlags(&P->s_copy, cudaStreamNonBlocking));
    if (!P->s_comp) RS_CUDA(cudaStreamCreateWithFlags(&P->s_comp, cudaStreamNonBlocking));
    if (!P->s_h) {
        int plo = 0, phi = 0;
        RS_CUDA(cudaDeviceGetStreamPriorityRange(&plo, &phi));
        RS_CUDA(cudaStreamCreateWithPriority(&P->s_h, cudaStreamNonBlocking, phi));
    }
    const cudaStream_t sh = P->s_h;     // apply_h on its own high-priority stream: panel k+1 goes through H in the tail of panel k's Gram launch
    // a V_loc set on some caller stream must have landed before the plan-owned streams read it
    if (P->vloc_pending) {
        RS_CUDA(cudaStreamWaitEvent(P->s_comp, P->ev_vloc, 0));
        RS_CUDA(cudaStreamWaitEvent(P->s_h, P->ev_vloc, 0));
        P->vloc_pending = false;
    }
    // Column panels of two Gram tile widths (96 columns; apply_h keeps efficient batches) on three plan-owned streams (copy, H, Gram): the
    // H2D copy of panel k+1 overlaps apply_h and the Gram tiles of panel k, and apply_h of panel k+1 fills the tail of panel k's Gram launch.  After panel t has been through H, every [S|H] tile that involves only
    // columns < TM(t+1) and touches panel t is contracted, so the Gram (the long part of the step) runs
    // while the rest of Y is still crossing PCIe instead of after the last byte has arrived.
    constexpr int TPP = 2;                                     // Gram tile columns per upload panel
    const int chunk = TPP * GCfg::TM;
    const int nchunk = (n + chunk - 1) / chunk;
    const int ntcol = (n + GCfg::TM - 1) / GCfg::TM;          // tile columns = entries of gram_panel_off - 1
    while ((int)P->ev.size() < 2 * nchunk) {
        cudaEvent_t e;
        RS_CUDA(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
        P->ev.push_back(e);
    }
    int rc = gram_panel_lists(P, n, P->s_comp);
    if (rc != RSDFT_OK) return rc;
    size_t need = 0;
    auto tiles_of = [&](int k, int &first) {                   // tile-list range that becomes computable with upload panel k
        const int t0 = std::min(k * TPP, ntcol), t1 = std::min((k + 1) * TPP, ntcol);
        first = P->gram_panel_off[t0];
        return P->gram_panel_off[t1] - first;
    };
    for (int k = 0; k < nchunk; ++k) { int f; need = std::max(need, gram_work_need(P, tiles_of(k, f))); }
    RS_CUDA(P->gram_work.ensure(need));
    double2 *Hd = P->hostHS.p, *Sd = P->hostHS.p + (size_t)n * n;
    P->last_launches = 0;
    int64_t launches = 0;
    // everything below is queued on the two plan-owned streams; on ANY error both are drained before the
    // call returns, so no copy or kernel of a failed call is still touching the caller's host buffers
#ifdef RSDFT_LAB_TIMELINE      // lab builds only: per-panel event times on stderr
    std::vector<cudaEvent_t> tl(3 * nchunk + 1);
    for (auto &e : tl) cudaEventCreate(&e);
    cudaEventRecord(tl[3 * nchunk], P->s_copy);
#endif
    auto body = [&]() -> int {
        for (int k = 0; k < nchunk; ++k) {
            const int c0 = k * chunk, nc = std::min(chunk, n - c0);
            RS_CUDA(cudaMemcpy2DAsync(P->hostY.p + (int64_t)c0 * ng, (size_t)ng * 16,
                                      (const char *)Y_host + (size_t)c0 * ldy * 16, (size_t)ldy * 16, (size_t)ng * 16, nc,
                                      cudaMemcpyHostToDevice, P->s_copy));
            RS_CUDA(cudaEventRecord(P->ev[2 * k], P->s_copy));
#ifdef RSDFT_LAB_TIMELINE
            cudaEventRecord(tl[3 * k], P->s_copy);
#endif
            RS_CUDA(cudaStreamWaitEvent(sh, P->ev[2 * k], 0));
            int r = apply_h_impl(P, nc, P->hostY.p + (int64_t)c0 * ng, ng, P->hostHY.p + (int64_t)c0 * ng, ng, sh);
            if (r != RSDFT_OK) return r;
            RS_CUDA(cudaEventRecord(P->ev[2 * k + 1], sh));
            RS_CUDA(cudaStreamWaitEvent(P->s_comp, P->ev[2 * k + 1], 0));
#ifdef RSDFT_LAB_TIMELINE
            cudaEventRecord(tl[3 * k + 1], sh);
#endif
            launches += P->last_launches;
            P->last_launches = 0;
            int first = 0;
            const int nt = tiles_of(k, first);
            r = gram_launch(P, n, P->hostY.p, ng, P->hostHY.p, ng, Hd, Sd, n, P->gram_panel_tiles.p + first, nt, P->s_comp);
            if (r != RSDFT_OK) return r;
#ifdef RSDFT_LAB_TIMELINE
            cudaEventRecord(tl[3 * k + 2], P->s_comp);
#endif
            launches += P->last_launches;
            P->last_launches = 0;
        }
        P->last_launches = launches;
        RS_CUDA(cudaMemcpy2DAsync(H_sub_host, (size_t)lds * 16, Hd, (size_t)n * 16, (size_t)n * 16, n, cudaMemcpyDeviceToHost, P->s_comp));
        RS_CUDA(cudaMemcpy2DAsync(S_sub_host, (size_t)lds * 16, Sd, (size_t)n * 16, (size_t)n * 16, n, cudaMemcpyDeviceToHost, P->s_comp));
        if (HY_host) {   // HY goes back on the copy stream, behind the uploads, while the Gram runs
            for (int k = 0; k < nchunk; ++k) {
                const int c0 = k * chunk, nc = std::min(chunk, n - c0);
                RS_CUDA(cudaStreamWaitEvent(P->s_copy, P->ev[2 * k + 1], 0));
                RS_CUDA(cudaMemcpy2DAsync((char *)HY_host + (size_t)c0 * ldhy * 16, (size_t)ldhy * 16,
                                          P->hostHY.p + (int64_t)c0 * ng, (size_t)ng * 16, (size_t)ng * 16, nc,
                                          cudaMemcpyDeviceToHost, P->s_copy));
            }
        }
        return RSDFT_OK;
    };
    rc = body();
    const cudaError_t e0 = cudaStreamSynchronize(P->s_h), e1 = cudaStreamSynchronize(P->s_comp), e2 = cudaStreamSynchronize(P->s_copy);
#ifdef RSDFT_LAB_TIMELINE
    for (int k = 0; k < nchunk; ++k) {
        float t[3];
        for (int j = 0; j < 3; ++j) cudaEventElapsedTime(&t[j], tl[3 * nchunk], tl[3 * k + j]);
        int f;
        fprintf(stderr, "panel %2d: upload done %8.2f  apply_h done %8.2f  gram done %8.2f ms  (%d tiles)\n", k, t[0], t[1], t[2], tiles_of(k, f));
    }
    for (auto &e : tl) cudaEventDestroy(e);
#endif
    if (rc != RSDFT_OK) return rc;
    RS_CUDA(e0);
    RS_CUDA(e1);
    RS_CUDA(e2);
    return RSDFT_OK;
}

int rsdft_subspace_rotate2(rsdft_plan_t *plan, int32_t n, int32_t m, const void *Y, int64_t ldy, const void *HY, int64_t ldhy,
                           const void *Cmat, int32_t ldc, const double *lambda, void *Xout, int64_t ldx, void *HXout, int64_t ldhx,
                           void *R, int64_t ldr, void *stream)
{
    if (!plan || !Y || !HY || !Cmat) return fail(RSDFT_INVALID_ARG, "rsdft_subspace_rotate2: null argument");
    if (!Xout && !HXout && !R) return fail(RSDFT_INVALID_ARG, "rsdft_subspace_rotate2: all outputs null");
    if (R && !lambda) return fail(RSDFT_INVALID_ARG, "rsdft_subspace_rotate2: R requested without lambda");
    if (n <= 0 || m <= 0) return fail(RSDFT_INVALID_ARG, "rsdft_subspace_rotate2: n, m must be > 0");
    const int64_t ng = plan->ng;
    if (ldy < ng || ldhy < ng || (Xout && ldx < ng) || (HXout && ldhx < ng) || (R && ldr < ng))
        return fail(RSDFT_INVALID_ARG, "rsdft_subspace_rotate2: ld < Ng");
    if (ldc < n) return fail(RSDFT_INVALID_ARG, "rsdft_subspace_rotate2: ldc < n");
    if (((uintptr_t)Y | (uintptr_t)HY | (uintptr_t)Cmat | (uintptr_t)Xout | (uintptr_t)HXout | (uintptr_t)R) & 15)
        return fail(RSDFT_INVALID_ARG, "rsdft_subspace_rotate2: pointers must be 16-byte aligned");
    const size_t by = ((size_t)(n - 1) * ldy + ng) * 16, bh = ((size_t)(n - 1) * ldhy + ng) * 16;
    const void *outs[3] = {Xout, HXout, R};
    const int64_t lds3[3] = {ldx, ldhx, ldr};
    for (int i = 0; i < 3; ++i) {
        if (!outs[i]) continue;
        const size_t bo = ((size_t)(m - 1) * lds3[i] + ng) * 16;
        if (overlaps(Y, by, outs[i], bo) || overlaps(HY, bh, outs[i], bo))
            return fail(RSDFT_INVALID_ARG, "rsdft_subspace_rotate2: an output overlaps Y or HY");
        for (int j = i + 1; j < 3; ++j)
            if (outs[j] && overlaps(outs[i], bo, outs[j], ((size_t)(m - 1) * lds3[j] + ng) * 16))
                return fail(RSDFT_INVALID_ARG, "rsdft_subspace_rotate2: outputs overlap each other");
    }
    if (int rc = check_device(plan, "rsdft_subspace_rotate2")) return rc;
    Rotate2Args a;
    a.Y = (const double2 *)Y; a.HY = (const double2 *)HY; a.C = (const double2 *)Cmat; a.lambda = lambda;
    a.X = (double2 *)Xout; a.HX = (double2 *)HXout; a.R = (double2 *)R;
    a.ldy = ldy; a.ldhy = ldhy; a.ldx = ldx; a.ldhx = ldhx; a.ldr = ldr; a.ng = ng; a.n = n; a.m = m; a.ldc = ldc;
    // 3M complex product with six accumulator sets (X': K1..K3, HX': K1..K3): 48 x 32 output tile (rows x columns), four
    // warps of 3 x 2 fragments, two CTAs per SM
    using R32 = Rotate2Cfg<2, 2, 3, 2, 16, 3>;
    const int tm = R32::TM, tn = R32::TN;
    a.jtiles = (m + tn - 1) / tn;
    const int64_t units = ((ng + tm - 1) / tm) * a.jtiles;
    if (units > 0x7fffffffll) return fail(RSDFT_UNSUPPORTED, "rsdft_subspace_rotate2: too many tiles for one launch");
    {
        auto kern = rotate2_dmma_kernel<2, 2, 3, 2, 16, 3, true, 2>;
        RS_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)R32::SMEM));
        kern<<<(unsigned)units, R32::THREADS, R32::SMEM, (cudaStream_t)stream>>>(a);
    }
    plan->last_launches = 1;
    RS_CUDA(cudaGetLastError());
    return RSDFT_OK;
}

int rsdft_subspace_eig(rsdft_plan_t *plan, int32_t n, const void *H_sub, const void *S_sub, int32_t lds, int32_t m,
                       double *lambda, void *Cmat, int32_t ldc, void *stream)
{
    if (!plan || !H_sub || !S_sub || !lambda || !Cmat) return fail(RSDFT_INVALID_ARG, "rsdft_subspace_eig: null argument");
    if (n <= 0 || n > 16384) return fail(RSDFT_INVALID_ARG, "rsdft_subspace_eig: n out of range (1..16384)");
    if (m <= 0 || m > n) return fail(RSDFT_INVALID_ARG, "rsdft_subspace_eig: m must be in 1..n");
    if (lds < n || ldc < n) return fail(RSDFT_INVALID_ARG, "rsdft_subspace_eig: leading dimension < n");
    if (((uintptr_t)H_sub | (uintptr_t)S_sub | (uintptr_t)Cmat) & 15 || ((uintptr_t)lambda & 7))
        return fail(RSDFT_INVALID_ARG, "rsdft_subspace_eig: misaligned pointer");
    if (int rc = check_device(plan, "rsdft_subspace_eig")) return rc;
    plan->last_launches = 0;
    const int rc = eig_impl(plan, n, (const double2 *)H_sub, (const double2 *)S_sub, lds, m, lambda, (double2 *)Cmat, ldc,
                            (cudaStream_t)stream);
    if (rc != RSDFT_OK) cudaStreamSynchronize((cudaStream_t)stream);      // nothing of a failed call stays in flight
    return rc;
}

int rsdft_subspace_eig_get(rsdft_plan_t *plan, int32_t what, void *out, int32_t ld, void *stream)
{
    if (!plan || !out) return fail(RSDFT_INVALID_ARG, "rsdft_subspace_eig_get: null argument");
    if (plan->eg_n <= 0) return fail(RSDFT_INVALID_ARG, "rsdft_subspace_eig_get: no successful rsdft_subspace_eig on this plan yet");
    if (what != 0 && what != 1) return fail(RSDFT_INVALID_ARG, "rsdft_subspace_eig_get: what must be 0 (L) or 1 (K)");
    if (ld < plan->eg_n) return fail(RSDFT_INVALID_ARG, "rsdft_subspace_eig_get: ld < n");
    if (int rc = check_device(plan, "rsdft_subspace_eig_get")) return rc;
    const int n = plan->eg_n;
    mat_copy_kernel<<<296, 256, 0, (cudaStream_t)stream>>>(what == 0 ? plan->eg_L.p : plan->eg_Z.p, n, (double2 *)out, ld, n, n, what == 0 ? 1 : 0);
    RS_CUDA(cudaGetLastError());
    return RSDFT_OK;
}

int rsdft_plan_set_eig_mode(rsdft_plan_t *plan, int32_t reduction, int32_t inner_sweeps)
{
    if (!plan || (reduction != 0 && reduction != 1) || inner_sweeps < 0 || inner_sweeps > 16)
        return fail(RSDFT_INVALID_ARG, "rsdft_plan_set_eig_mode: reduction must be 0 or 1, inner_sweeps in 0..16");
    plan->eig_mode = reduction;
    plan->eig_inner = inner_sweeps == 0 ? 1 : inner_sweeps;
    return RSDFT_OK;
}

int rsdft_subspace_eig_stats(const rsdft_plan_t *plan, double *out8)
{
    if (!plan || !out8) return fail(RSDFT_INVALID_ARG, "rsdft_subspace_eig_stats: null argument");
    for (int i = 0; i < 8; ++i) out8[i] = plan->eig_stats[i];
    return RSDFT_OK;
}

int rsdft_plan_release_workspace(rsdft_plan_t *plan)
{
    if (!plan) return fail(RSDFT_INVALID_ARG, "rsdft_plan_release_workspace: null plan");
    if (int rc = check_device(plan, "rsdft_plan_release_workspace")) return rc;
    RS_CUDA(cudaDeviceSynchronize());
    plan->hostY.release(); plan->hostHY.release(); plan->hostHS.release();
    plan->gram_work.release();
    for (int i = 0; i < rsdft_plan::MAX_STREAMS; ++i) { plan->pp[i].release(); plan->pq[i].release(); }
    plan->eg_L.release(); plan->eg_B.release(); plan->eg_Z.release(); plan->eg_Dinv.release(); plan->eg_Kp.release();
    plan->eg_Tp.release(); plan->eg_V0.release(); plan->eg_V1.release(); plan->eg_J.release(); plan->eg_Zs.release();
    plan->eg_n = 0;
    return RSDFT_OK;
}

}  // extern "C"
