// Host orchestration of rsdft_subspace_eig (eq. 1) over the kernels of
// eig_kernels.cuh.  Included by rsdft.cu inside its anonymous namespace (uses fail(), RS_CUDA, DevBuf, rsdft_plan).
//
//   eig_potrf        S = L L^H: right-looking blocked Cholesky, 64-column panels; diagonal block factored and
//                    inverted by one CTA, panel = S21 inv(L11)^H and trailing update S22 -= L21 L21^H on DMMA.
//   eig_trsm_lower   X = L^-1 B: forward substitution by blocks, diagonal blocks applied as inverses (GEMM only).
//   reduce (mode 0)  the paper's route: K = L^-1 H L^-H as TWO triangular solves, Z = L^-1 H, K = L^-1 Z^H.
//   reduce (mode 1)  the ZHEGST-style blocked two-sided reduction the paper replaces (same algorithm as LAPACK's
//                    zhegst, itype 1, lower), built from the same GEMM kernel, for the comparison of PAPER.md:101.
//   eig_jacobi       K Z = Z Lambda by block Jacobi, ascending order.
//   eig_backsolve    C = L^-H Z for the m lowest.
#pragma once

struct EigBufs;   // (members live in rsdft_plan; see rsdft.cu)

static cudaError_t eig_zgemm(bool ta, bool tb, int M, int N, int K, double alpha, const double2 *A, int64_t lda,
                             const double2 *B, int64_t ldb, double beta, double2 *C, int64_t ldc, int lower, cudaStream_t st,
                             int64_t *launches)
{
    if (M <= 0 || N <= 0) return cudaSuccess;
    rsdft::ZgemmArgs a;
    a.A = A; a.B = B; a.C = C; a.lda = lda; a.ldb = ldb; a.ldc = ldc; a.M = M; a.N = N; a.K = K;
    a.alpha = alpha; a.beta = beta; a.lower = lower;
    const dim3 grid((M + 63) / 64, (N + 63) / 64);
    if (!ta && !tb) rsdft::zgemm_kernel<false, false><<<grid, 256, 0, st>>>(a);
    else if (!ta && tb) rsdft::zgemm_kernel<false, true><<<grid, 256, 0, st>>>(a);
    else if (ta && !tb) rsdft::zgemm_kernel<true, false><<<grid, 256, 0, st>>>(a);
    else rsdft::zgemm_kernel<true, true><<<grid, 256, 0, st>>>(a);
    if (launches) ++*launches;
    return cudaGetLastError();
}

// W (n x n, ld n): working copy of S, destroyed.  L (n x n, ld n): receives the factor, strict upper part zero.
static int eig_potrf(rsdft_plan *P, int n, double2 *W, double2 *L, cudaStream_t st)
{
    constexpr int NB = rsdft::EIG_NB;
    const size_t smem = (size_t)2 * NB * (NB + 1) * sizeof(double2);
    RS_CUDA(cudaFuncSetAttribute(rsdft::potf2_trtri_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    RS_CUDA(cudaMemsetAsync(L, 0, (size_t)n * n * sizeof(double2), st));
    for (int k0 = 0, kb = 0; k0 < n; k0 += NB, ++kb) {
        const int nb = std::min(NB, n - k0), rem = n - k0 - nb;
        // the diagonal block is factored in place in W, then copied into L with its inverse kept aside
        rsdft::potf2_trtri_kernel<<<1, 256, smem, st>>>(W, n, k0, nb, P->eg_Dinv.p + (size_t)kb * NB * NB, P->eg_info.p);
        rsdft::mat_copy_kernel<<<4, 256, 0, st>>>(W + (int64_t)k0 * n + k0, n, L + (int64_t)k0 * n + k0, n, nb, nb, 1);
        P->last_launches += 2;
        if (rem > 0) {
            // L21 = S21 inv(L11)^H
            RS_CUDA(eig_zgemm(false, true, rem, nb, nb, 1.0, W + (int64_t)k0 * n + k0 + nb, n, P->eg_Dinv.p + (size_t)kb * NB * NB, NB,
                              0.0, L + (int64_t)k0 * n + k0 + nb, n, 0, st, &P->last_launches));
            // S22 -= L21 L21^H (lower tiles)
            RS_CUDA(eig_zgemm(false, true, rem, rem, nb, -1.0, L + (int64_t)k0 * n + k0 + nb, n, L + (int64_t)k0 * n + k0 + nb, n,
                              1.0, W + (int64_t)(k0 + nb) * n + k0 + nb, n, 1, st, &P->last_launches));
        }
    }
    RS_CUDA(cudaGetLastError());
    return RSDFT_OK;
}

// X (n x nc, ldx) = L^-1 B; B (n x nc, ldb) is destroyed.  Dinv: inverted 64 x 64 diagonal blocks of L.
static int eig_trsm_lower(rsdft_plan *P, int n, int nc, const double2 *L, double2 *B, int64_t ldb, double2 *X, int64_t ldx, cudaStream_t st)
{
    constexpr int NB = rsdft::EIG_NB;
    for (int k0 = 0, kb = 0; k0 < n; k0 += NB, ++kb) {
        const int nb = std::min(NB, n - k0), rem = n - k0 - nb;
        RS_CUDA(eig_zgemm(false, false, nb, nc, nb, 1.0, P->eg_Dinv.p + (size_t)kb * NB * NB, NB, B + k0, ldb, 0.0, X + k0, ldx, 0, st,
                          &P->last_launches));
        RS_CUDA(eig_zgemm(false, false, rem, nc, nb, -1.0, L + (int64_t)k0 * n + k0 + nb, n, X + k0, ldx, 1.0, B + k0 + nb, ldb, 0, st,
                          &P->last_launches));
    }
    return RSDFT_OK;
}

// C (n x m, ldc) = L^-H T; T (n x m, ld n) is destroyed.
static int eig_backsolve(rsdft_plan *P, int n, int m, const double2 *L, double2 *T, double2 *C, int64_t ldc, cudaStream_t st)
{
    constexpr int NB = rsdft::EIG_NB;
    const int nblk = (n + NB - 1) / NB;
    for (int kb = nblk - 1; kb >= 0; --kb) {
        const int k0 = kb * NB, nb = std::min(NB, n - k0);
        RS_CUDA(eig_zgemm(true, false, nb, m, nb, 1.0, P->eg_Dinv.p + (size_t)kb * NB * NB, NB, T + k0, n, 0.0, C + k0, ldc, 0, st,
                          &P->last_launches));
        RS_CUDA(eig_zgemm(true, false, k0, m, nb, -1.0, L + k0, n, C + k0, ldc, 1.0, T, n, 0, st, &P->last_launches));
    }
    return RSDFT_OK;
}

// mode 0 (the paper's proposal): K = L^-1 H L^-H by two triangular solves.
//   Z = L^-1 H;  K = L^-1 Z^H  (= L^-1 H^H L^-H = K for Hermitian H).   Result in P->eg_Z (ld n), both triangles.
static int eig_reduce_trsm(rsdft_plan *P, int n, const double2 *H, int64_t ldh, cudaStream_t st)
{
    double2 *B = P->eg_B.p, *Z = P->eg_Z.p, *L = P->eg_L.p;
    rsdft::mat_copy_kernel<<<296, 256, 0, st>>>(H, ldh, B, n, n, n, 0);
    ++P->last_launches;
    int rc = eig_trsm_lower(P, n, n, L, B, n, Z, n, st);
    if (rc != RSDFT_OK) return rc;
    const dim3 tg((n + 31) / 32, (n + 31) / 32);
    rsdft::conj_transpose_kernel<<<tg, 256, 0, st>>>(Z, n, B, n, n, n);
    ++P->last_launches;
    rc = eig_trsm_lower(P, n, n, L, B, n, Z, n, st);
    RS_CUDA(cudaGetLastError());
    return rc;
}

// mode 1: the blocked two-sided reduction of LAPACK's zhegst (itype 1, lower) with the same kernels, i.e. what
// "(P)ZHEGST" does.  Per 64-column block k (A = working copy of H, L21 = L[below, k], A21 likewise):
//   A11 <- inv(L11) A11 inv(L11)^H;  A21 <- A21 inv(L11)^H;  A21 -= 1/2 L21 A11;  A22 -= A21 L21^H + L21 A21^H (lower);
//   A21 -= 1/2 L21 A11;  A21 <- inv(L22) A21   (a triangular solve with the whole trailing factor).
// Result: K in the LOWER triangle (diagonal blocks full) of P->eg_Z.
static int eig_reduce_hegst(rsdft_plan *P, int n, const double2 *H, int64_t ldh, cudaStream_t st)
{
    constexpr int NB = rsdft::EIG_NB;
    double2 *A = P->eg_Z.p, *L = P->eg_L.p, *T = P->eg_B.p;       // T: scratch panel (n x 64) + 64 x 64 block
    rsdft::mat_copy_kernel<<<296, 256, 0, st>>>(H, ldh, A, n, n, n, 0);
    ++P->last_launches;
    double2 *T11 = T + (size_t)n * NB;
    for (int k0 = 0, kb = 0; k0 < n; k0 += NB, ++kb) {
        const int nb = std::min(NB, n - k0), rem = n - k0 - nb;
        const double2 *Di = P->eg_Dinv.p + (size_t)kb * NB * NB;
        double2 *A11 = A + (int64_t)k0 * n + k0, *A21 = A + (int64_t)k0 * n + k0 + nb, *A22 = A + (int64_t)(k0 + nb) * n + k0 + nb;
        const double2 *L21 = L + (int64_t)k0 * n + k0 + nb;
        RS_CUDA(eig_zgemm(false, false, nb, nb, nb, 1.0, Di, NB, A11, n, 0.0, T11, NB, 0, st, &P->last_launches));
        RS_CUDA(eig_zgemm(false, true, nb, nb, nb, 1.0, T11, NB, Di, NB, 0.0, A11, n, 0, st, &P->last_launches));
        if (rem <= 0) continue;
        RS_CUDA(eig_zgemm(false, true, rem, nb, nb, 1.0, A21, n, Di, NB, 0.0, T, n, 0, st, &P->last_launches));          // T = A21 inv(L11)^H
        RS_CUDA(eig_zgemm(false, false, rem, nb, nb, -0.5, L21, n, A11, n, 1.0, T, n, 0, st, &P->last_launches));        // T -= 1/2 L21 A11
        RS_CUDA(eig_zgemm(false, true, rem, rem, nb, -1.0, T, n, L21, n, 1.0, A22, n, 1, st, &P->last_launches));         // A22 -= T L21^H
        RS_CUDA(eig_zgemm(false, true, rem, rem, nb, -1.0, L21, n, T, n, 1.0, A22, n, 1, st, &P->last_launches));         // A22 -= L21 T^H
        RS_CUDA(eig_zgemm(false, false, rem, nb, nb, -0.5, L21, n, A11, n, 1.0, T, n, 0, st, &P->last_launches));        // T -= 1/2 L21 A11
        // A21 = inv(L22) T: forward substitution over the trailing blocks
        for (int j0 = k0 + nb, jb = kb + 1; j0 < n; j0 += NB, ++jb) {
            const int mb = std::min(NB, n - j0), below = n - j0 - mb;
            RS_CUDA(eig_zgemm(false, false, mb, nb, mb, 1.0, P->eg_Dinv.p + (size_t)jb * NB * NB, NB, T + (j0 - k0 - nb), n, 0.0,
                              A + (int64_t)k0 * n + j0, n, 0, st, &P->last_launches));
            RS_CUDA(eig_zgemm(false, false, below, nb, mb, -1.0, L + (int64_t)j0 * n + j0 + mb, n, A + (int64_t)k0 * n + j0, n, 1.0,
                              T + (j0 + mb - k0 - nb), n, 0, st, &P->last_launches));
        }
    }
    return RSDFT_OK;
}

// Round-robin tournament over nblk (even) blocks: nblk - 1 rounds of nblk / 2 disjoint pairs visit every pair once.
static void eig_pair_table(int nblk, std::vector<int2> &pairs)
{
    std::vector<int> arr(nblk);
    for (int i = 0; i < nblk; ++i) arr[i] = i;
    pairs.clear();
    for (int r = 0; r < nblk - 1; ++r) {
        for (int i = 0; i < nblk / 2; ++i) {
            const int a = arr[i], b = arr[nblk - 1 - i];
            pairs.push_back(make_int2(std::min(a, b), std::max(a, b)));
        }
        const int last = arr[nblk - 1];                       // keep arr[0], rotate the rest by one
        for (int i = nblk - 1; i > 1; --i) arr[i] = arr[i - 1];
        arr[1] = last;
    }
}

// K (n x n in P->eg_Z, ld n; lower_only: read the lower triangle only) -> eigenvalues ascending in lambda[m]
// (device), the m lowest eigenvectors in P->eg_Zs (n x m, ld n).  Synchronises `st` with the host once per sweep.
static int eig_jacobi(rsdft_plan *P, int n, int m, int lower_only, double *lambda, cudaStream_t st)
{
    constexpr int JB = rsdft::EIG_JB, D = 2 * JB;
    const int npad = (n + D - 1) / D * D, nblk = npad / JB, npairs = nblk / 2, rounds = nblk - 1;
    double2 *Kp = P->eg_Kp.p, *Tp = P->eg_Tp.p, *Va = P->eg_V0.p, *Vb = P->eg_V1.p;
    double *scal = P->eg_scal.p;
    const int nred = 148;
    if (lower_only) {       // mirror the lower triangle first so that the symmetrising loads below see a full matrix
        const dim3 tg((n + 31) / 32, (n + 31) / 32);
        rsdft::conj_transpose_kernel<<<tg, 256, 0, st>>>(P->eg_Z.p, n, P->eg_B.p, n, n, n);
        rsdft::mat_copy_kernel<<<296, 256, 0, st>>>(P->eg_B.p, n, P->eg_Z.p, n, n, n, 2);
        P->last_launches += 2;
    }
    rsdft::jacobi_prepare_kernel<<<nred, 256, 0, st>>>(P->eg_Z.p, n, n, npad, Kp, Va, scal + 8);
    rsdft::sum_partials_kernel<<<1, 32, 0, st>>>(scal + 8, nred, scal);
    rsdft::jacobi_pad_diag_kernel<<<(npad - n + 63) / 64 + 1, 64, 0, st>>>(Kp, n, npad, scal);
    P->last_launches += 3;
    if (P->eg_pairs_nblk != nblk) {
        std::vector<int2> pairs;
        eig_pair_table(nblk, pairs);
        RS_CUDA(P->eg_pairs.upload_async(pairs, st));
        P->eg_pairs_nblk = nblk;
    }
    const size_t smem_sub = (size_t)2 * D * (D + 1) * sizeof(double2);
    const size_t smem_upd = (size_t)3 * D * (D + 4) * sizeof(double2);
    RS_CUDA(cudaFuncSetAttribute(rsdft::jacobi_subeig_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_sub));
    const size_t smem_cross = (size_t)D * (D + 1) * sizeof(double2);
    RS_CUDA(cudaFuncSetAttribute(rsdft::jacobi_subeig_cross_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_cross));
    RS_CUDA(cudaFuncSetAttribute(rsdft::jacobi_block_update_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_upd));
    double host[3] = {0.0, 0.0, 0.0};
    RS_CUDA(cudaMemcpyAsync(host, scal, sizeof(double), cudaMemcpyDeviceToHost, st));
    RS_CUDA(cudaStreamSynchronize(st));
    const double norm2 = host[0];
    // entries below 1e-18 ||K||_F are not rotated (they are far under the round-off of the updates)
    const double tiny = 1e-18 * std::sqrt(norm2);
    RS_CUDA(cudaMemcpyAsync(scal + 1, &tiny, sizeof(double), cudaMemcpyHostToDevice, st));
    const int tiles = npad / 64;
    // Two streams per round: `hi` carries the chain sub-problems -> K update -> next sub-problems (the 23 sub-problem
    // CTAs are a latency chain on 23 SMs), `lo` carries V <- V Jt, which nothing needs before the end and which fills
    // the other SMs meanwhile.  J is double-buffered by round parity; ev J[p] = J of that parity written, V[p] = read.
    if (!P->eg_s_hi) {
        int plo = 0, phi = 0;
        RS_CUDA(cudaDeviceGetStreamPriorityRange(&plo, &phi));
        RS_CUDA(cudaStreamCreateWithPriority(&P->eg_s_hi, cudaStreamNonBlocking, phi));
        RS_CUDA(cudaStreamCreateWithPriority(&P->eg_s_lo, cudaStreamNonBlocking, plo));
        for (auto &e : P->eg_sync) RS_CUDA(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
    }
    const cudaStream_t hi = P->eg_s_hi, lo = P->eg_s_lo;
    RS_CUDA(cudaEventRecord(P->eg_sync[4], st));                // fork: both streams start behind the caller's stream
    RS_CUDA(cudaStreamWaitEvent(hi, P->eg_sync[4], 0));
    RS_CUDA(cudaStreamWaitEvent(lo, P->eg_sync[4], 0));
    const size_t jsz = (size_t)npairs * D * D;
    double prev = -1.0;
    int sweep = 0;
    int64_t gr = 0;                                             // rounds so far (parity picks the J buffer)
    bool converged = norm2 == 0.0;
    const int max_sweeps = 30;
    for (; sweep < max_sweeps && !converged; ++sweep) {
        for (int r = 0; r < rounds; ++r, ++gr) {
            const int par = (int)(gr & 1);
            double2 *Jb = P->eg_J.p + (size_t)par * jsz;
            const int2 *pr = P->eg_pairs.p + (size_t)r * npairs;
            if (gr >= 2) RS_CUDA(cudaStreamWaitEvent(hi, P->eg_sync[2 + par], 0));    // the V update two rounds back has read this J buffer
            if (r > 0) rsdft::jacobi_subeig_cross_kernel<<<npairs, 1024, smem_cross, hi>>>(Kp, npad, pr, Jb, P->eig_inner, scal);   // cross pairs
            else rsdft::jacobi_subeig_kernel<<<npairs, rsdft::EIG_SUB_NT, smem_sub, hi>>>(Kp, npad, pr, Jb, P->eig_inner, scal);     // all pairs
            rsdft::BlockUpdArgs u;
            u.Kin = Kp; u.Kout = Tp; u.Vin = Va; u.Vout = Vb;
            u.npad = npad; u.npairs = npairs; u.nk = npairs * (npairs + 1) / 2; u.tiles = tiles;
            u.pairs = pr; u.Jbuf = Jb; u.item0 = 0;
            RS_CUDA(cudaEventRecord(P->eg_sync[par], hi));
            rsdft::jacobi_block_update_kernel<<<u.nk, 256, smem_upd, hi>>>(u);                           // K = Jt^H K Jt
            RS_CUDA(cudaStreamWaitEvent(lo, P->eg_sync[par], 0));
            u.item0 = u.nk;
            rsdft::jacobi_block_update_kernel<<<npairs * tiles, 256, smem_upd, lo>>>(u);                 // V = V Jt
            RS_CUDA(cudaEventRecord(P->eg_sync[2 + par], lo));
            P->last_launches += 3;
            std::swap(Kp, Tp);
            std::swap(Va, Vb);
        }
        rsdft::jacobi_offnorm_kernel<<<nred, 256, 0, hi>>>(Kp, n, npad, scal + 8);
        rsdft::sum_partials_kernel<<<1, 32, 0, hi>>>(scal + 8, nred, scal + 2);
        P->last_launches += 2;
        RS_CUDA(cudaGetLastError());
        RS_CUDA(cudaMemcpyAsync(host + 2, scal + 2, sizeof(double), cudaMemcpyDeviceToHost, hi));
        RS_CUDA(cudaStreamSynchronize(hi));
        const double off = host[2];
#ifdef RSDFT_LAB_N
        if (getenv("RSDFT_LAB_EIGTRACE")) fprintf(stderr, "sweep %d: off/norm = %.3e\n", sweep, std::sqrt(off / norm2));
#endif
        // converged: off(K) <= 1e-13 ||K||_F, or the round-off floor is reached (no further decrease below 1e-10)
        if (off <= 1e-26 * norm2) converged = true;
        else if (prev >= 0.0 && off > 0.25 * prev && off <= 1e-20 * norm2) converged = true;
        prev = off;
    }
    RS_CUDA(cudaEventRecord(P->eg_sync[5], lo));                // join: the caller's stream continues behind both
    RS_CUDA(cudaStreamWaitEvent(st, P->eg_sync[5], 0));
    RS_CUDA(cudaEventRecord(P->eg_sync[5], hi));
    RS_CUDA(cudaStreamWaitEvent(st, P->eg_sync[5], 0));
    P->eig_stats[0] = sweep;
    P->eig_stats[5] = norm2 > 0.0 ? std::sqrt(prev < 0.0 ? 0.0 : prev / norm2) : 0.0;
    if (!converged) return fail(RSDFT_NO_CONVERGENCE, "rsdft_subspace_eig: block Jacobi did not converge in 30 sweeps");
    rsdft::eig_rank_kernel<<<(n + 255) / 256, 256, 0, st>>>(Kp, n, npad, m, lambda, P->eg_perm.p);
    rsdft::eig_gather_kernel<<<m, 256, 0, st>>>(Va, npad, n, m, P->eg_perm.p, P->eg_Zs.p, n);
    P->last_launches += 2;
    RS_CUDA(cudaGetLastError());
    return RSDFT_OK;
}

static int eig_impl(rsdft_plan *P, int n, const double2 *H, const double2 *S, int64_t lds, int m, double *lambda, double2 *C,
                    int64_t ldc, cudaStream_t st)
{
    constexpr int NB = rsdft::EIG_NB, D = 2 * rsdft::EIG_JB;
    const int nblk = (n + NB - 1) / NB, npad = (n + D - 1) / D * D;
    const size_t nn = (size_t)n * n, np2 = (size_t)npad * npad;
    RS_CUDA(P->eg_L.ensure(nn));
    RS_CUDA(P->eg_B.ensure(std::max(nn, (size_t)n * NB + (size_t)NB * NB)));
    RS_CUDA(P->eg_Z.ensure(nn));
    RS_CUDA(P->eg_Dinv.ensure((size_t)nblk * NB * NB));
    RS_CUDA(P->eg_Kp.ensure(np2)); RS_CUDA(P->eg_Tp.ensure(np2)); RS_CUDA(P->eg_V0.ensure(np2)); RS_CUDA(P->eg_V1.ensure(np2));
    RS_CUDA(P->eg_J.ensure((size_t)2 * (npad / D) * D * D));      // two buffers (round parity)
    RS_CUDA(P->eg_Zs.ensure((size_t)n * m));
    RS_CUDA(P->eg_scal.ensure(8 + 148));
    RS_CUDA(P->eg_info.ensure(1));
    RS_CUDA(P->eg_perm.ensure((size_t)n));
    for (int i = 0; i < 6; ++i)
        if (!P->eg_ev[i]) RS_CUDA(cudaEventCreate(&P->eg_ev[i]));
    P->eg_n = 0;
    RS_CUDA(cudaMemsetAsync(P->eg_info.p, 0, sizeof(int), st));
    RS_CUDA(cudaEventRecord(P->eg_ev[0], st));
    // 1. Cholesky of S (working copy in eg_B)
    rsdft::mat_copy_kernel<<<296, 256, 0, st>>>(S, lds, P->eg_B.p, n, n, n, 0);
    ++P->last_launches;
    int rc = eig_potrf(P, n, P->eg_B.p, P->eg_L.p, st);
    if (rc != RSDFT_OK) return rc;
    int info = 0;
    RS_CUDA(cudaMemcpyAsync(&info, P->eg_info.p, sizeof(int), cudaMemcpyDeviceToHost, st));
    RS_CUDA(cudaEventRecord(P->eg_ev[1], st));
    RS_CUDA(cudaStreamSynchronize(st));
    if (info != 0)
        return fail(RSDFT_NOT_POSITIVE_DEFINITE, "rsdft_subspace_eig: S_sub is not positive definite (pivot " + std::to_string(info) + ")");
    // 2. K = L^-1 H L^-H
    rc = P->eig_mode == 1 ? eig_reduce_hegst(P, n, H, lds, st) : eig_reduce_trsm(P, n, H, lds, st);
    if (rc != RSDFT_OK) return rc;
    RS_CUDA(cudaEventRecord(P->eg_ev[2], st));
    // keep K for rsdft_subspace_eig_get (the Jacobi stage works on its own padded copy)
    // 3. K Z = Z Lambda
    rc = eig_jacobi(P, n, m, P->eig_mode == 1, lambda, st);
    if (rc != RSDFT_OK) return rc;
    RS_CUDA(cudaEventRecord(P->eg_ev[3], st));
    // 4. C = L^-H Z
    rc = eig_backsolve(P, n, m, P->eg_L.p, P->eg_Zs.p, C, ldc, st);
    if (rc != RSDFT_OK) return rc;
    RS_CUDA(cudaEventRecord(P->eg_ev[4], st));
    RS_CUDA(cudaStreamSynchronize(st));
    float ms = 0.f;
    for (int i = 0; i < 4; ++i) {
        RS_CUDA(cudaEventElapsedTime(&ms, P->eg_ev[i], P->eg_ev[i + 1]));
        P->eig_stats[1 + i] = ms;
    }
    P->eig_stats[6] = P->eig_mode;
    P->eg_n = n;
    return RSDFT_OK;
}
