"""GPU parity of NEXT-1 (rsdft_subspace_eig: eq. 1) and NEXT-2 (rsdft_subspace_rotate2 with the LOBPCG
residual) against the oracle, through the C ABI.

What is unique is compared element by element: the Cholesky factor L (lower, positive diagonal), the standard-form
matrix K = L^-1 H L^-H, the eigenvalues.  Eigenvectors are NOT unique (a phase per vector, any basis inside a
degenerate eigenspace), so for them the test is a complete validity check: residual ||H C - S C Lambda||, S-orthonormality
C^H S C = I, and, per cluster of close eigenvalues, equality of the spanned subspace with the oracle's (projector
difference).  Inputs are seeded synthetic pencils from workloads.subspace_pencil (both sides read the same H, S) or the
two sides' own apply_h -> gram chains.  Every test needs a B200 (pytest -m gpu)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL = 1e-12


@pytest.fixture(scope="module")
def env():
    import torch
    from oracle import oracle
    from paper_2512_04447_b200 import rsdft, workloads
    assert torch.cuda.is_available()
    rsdft.load()
    plan = rsdft.rsdft_plan_create((16, 16, 16), (10.0, 10.0, 10.0))      # the eigen-solve does not depend on the grid
    return dict(torch=torch, oracle=oracle, rsdft=rsdft, wl=workloads, plan=plan)


def dev(env, M):
    """numpy M[i, j] -> CUDA tensor holding the column-major matrix (t[j, i] = M[i, j])"""
    return env["torch"].as_tensor(np.ascontiguousarray(M.T)).cuda()


def host(t):
    return t.cpu().numpy().T.copy()


def clusters(w, tol):
    """index ranges [a, b) of eigenvalues chained closer than tol"""
    out, a = [], 0
    for i in range(1, len(w) + 1):
        if i == len(w) or w[i] - w[i - 1] > tol:
            out.append((a, i))
            a = i
    return out


def check_eig(env, H, S, m, solver, lam, Cg, Lg=None, Kg=None):
    """the complete check of one GPU result (lam, Cg) for the pencil (H, S) against the oracle"""
    oracle = env["oracle"]
    n = H.shape[0]
    lam_o, C_o, L_o, K_o = oracle.subspace_eig(H, S, n, solver=solver, return_factors=True)
    kn = np.max(np.abs(lam_o))                                   # ||K||_2
    if Lg is not None:
        assert np.all(np.triu(Lg, 1) == 0.0)
        assert np.max(np.abs(Lg - L_o)) <= TOL * np.max(np.abs(L_o))                 # unique: element-wise
    if Kg is not None:
        assert np.max(np.abs(Kg - K_o)) <= TOL * np.max(np.abs(K_o))
    assert lam.shape == (m,) and Cg.shape == (n, m)
    assert np.all(np.diff(lam) >= 0.0)
    assert np.max(np.abs(lam - lam_o[:m])) <= TOL * kn
    SC = S @ Cg
    hn, sn = np.linalg.norm(H, 2), np.linalg.norm(S, 2)
    cn = np.sqrt(np.max(np.sum(np.abs(Cg) ** 2, axis=0)))
    assert np.max(np.linalg.norm(H @ Cg - SC * lam, axis=0)) <= 1e-11 * (hn + kn * sn) * cn   # residual per column
    assert np.max(np.abs(Cg.conj().T @ SC - np.eye(m))) <= TOL * max(1.0, np.linalg.cond(S) / 10)
    # subspaces: every cluster of eigenvalues closer than 1e-8 ||K|| that lies wholly inside the first m
    for a, b in clusters(lam_o, 1e-8 * kn):
        if b > m:
            break
        gap = min(lam_o[a] - lam_o[a - 1] if a > 0 else np.inf, lam_o[b] - lam_o[b - 1] if b < n else np.inf)
        Pg = Cg[:, a:b] @ Cg[:, a:b].conj().T
        Po = C_o[:, a:b] @ C_o[:, a:b].conj().T
        assert np.max(np.abs(Pg - Po)) <= 1e-11 * np.max(np.abs(Po)) * max(1.0, kn / gap), (a, b, gap)


def gpu_eig(env, H, S, m, factors=True):
    torch, rsdft, plan = env["torch"], env["rsdft"], env["plan"]
    n = H.shape[0]
    lam, Cm = rsdft.rsdft_subspace_eig(plan, dev(env, H), dev(env, S), m)
    torch.cuda.synchronize()
    out = [lam.cpu().numpy(), host(Cm)]
    if factors:
        out += [host(rsdft.rsdft_subspace_eig_get(plan, "L", n)), host(rsdft.rsdft_subspace_eig_get(plan, "K", n))]
        torch.cuda.synchronize()
    return out


# ------------------------------------------------------------------ seeded pencils, both sides read the same H, S
@pytest.mark.parametrize("n,m", [(1, 1), (2, 2), (7, 3), (24, 8), (63, 63), (64, 20), (65, 65), (100, 34), (130, 130), (192, 64)])
def test_eig_parity_small_and_ragged(env, n, m):
    H, S = env["wl"].subspace_pencil(n, 5)
    lam, Cg, Lg, Kg = gpu_eig(env, H, S, m)
    check_eig(env, H, S, m, "jacobi", lam, Cg, Lg, Kg)


@pytest.mark.parametrize("n", [60, 150])
def test_eig_degenerate_levels(env, n):
    """shells of 6, 12, 8 ... equal eigenvalues: the eigenvalues and each shell's SUBSPACE must match the oracle"""
    H, S, w = env["wl"].subspace_pencil(n, 9, degenerate=True)
    lam, Cg, Lg, Kg = gpu_eig(env, H, S, n)
    assert np.max(np.abs(lam - w)) <= 1e-12 * np.max(np.abs(w)) * np.linalg.cond(S)
    check_eig(env, H, S, n, "jacobi", lam, Cg, Lg, Kg)


@pytest.mark.parametrize("n,m", [(1440, 480), (1536, 512)])
def test_eig_parity_config_sizes(env, n, m):
    """configs[2] (n = 1440) and configs[3, 4] (n = 1536): L and K element by element against the long-double
    oracle; the standard problem against the library routine the paper names there (oracle solver "heevd")."""
    H, S = env["wl"].subspace_pencil(n, 2)
    lam, Cg, Lg, Kg = gpu_eig(env, H, S, m)
    check_eig(env, H, S, m, "heevd", lam, Cg, Lg, Kg)
    st = env["rsdft"].rsdft_subspace_eig_stats(env["plan"])
    assert 1 <= st["sweeps"] <= 20 and st["off_rel"] <= 1e-12


def test_eig_hegst_mode_agrees_with_trsm_mode(env):
    """The ZHEGST-style reduction (kept for the paper's comparison) reaches the same K (its lower
    triangle is what it defines), the same eigenvalues and valid eigenvectors."""
    rsdft, plan = env["rsdft"], env["plan"]
    n, m = 200, 70
    H, S = env["wl"].subspace_pencil(n, 3)
    lam0, C0, L0, K0 = gpu_eig(env, H, S, m)
    rsdft.rsdft_plan_set_eig_mode(plan, 1, 0)
    try:
        lam1, C1, L1, K1 = gpu_eig(env, H, S, m)
    finally:
        rsdft.rsdft_plan_set_eig_mode(plan, 0, 0)
    assert np.array_equal(L0, L1)
    assert np.max(np.abs(np.tril(K1) - np.tril(K0))) <= TOL * np.max(np.abs(K0))
    check_eig(env, H, S, m, "jacobi", lam1, C1, L1, None)
    assert np.max(np.abs(lam1 - lam0)) <= TOL * np.max(np.abs(lam0))


def test_eig_inner_sweeps_knob_and_reuse(env):
    """results do not depend (beyond round-off) on the sub-problem sweep count; a plan can be reused across sizes"""
    rsdft, plan = env["rsdft"], env["plan"]
    H, S = env["wl"].subspace_pencil(97, 4)
    ref = gpu_eig(env, H, S, 97, factors=False)
    for inner in (1, 4):
        rsdft.rsdft_plan_set_eig_mode(plan, 0, inner)
        lam, Cg = gpu_eig(env, H, S, 97, factors=False)
        assert np.max(np.abs(lam - ref[0])) <= TOL * np.max(np.abs(ref[0]))
        check_eig(env, H, S, 97, "jacobi", lam, Cg)
    rsdft.rsdft_plan_set_eig_mode(plan, 0, 0)


def test_eig_error_paths(env):
    torch, rsdft, plan = env["torch"], env["rsdft"], env["plan"]
    H, S = env["wl"].subspace_pencil(40, 6)
    bad = S.copy()
    bad[17, 17] = -1.0
    with pytest.raises(rsdft.RsdftError) as e:
        rsdft.rsdft_subspace_eig(plan, dev(env, H), dev(env, bad))
    assert e.value.code == rsdft.RSDFT_NOT_POSITIVE_DEFINITE and "18" in str(e.value)
    with pytest.raises(rsdft.RsdftError):
        rsdft.rsdft_subspace_eig(plan, dev(env, H), dev(env, S), 41)              # m > n
    with pytest.raises(ValueError):
        rsdft.rsdft_subspace_eig(plan, dev(env, H), dev(env, S)[:, :30])           # wrong shape
    with pytest.raises(ValueError):
        rsdft.rsdft_subspace_eig(plan, dev(env, H).cpu(), dev(env, S))             # host tensor
    lam, Cm = rsdft.rsdft_subspace_eig(plan, dev(env, H), dev(env, S), 5)          # the plan still works afterwards
    torch.cuda.synchronize()
    check_eig(env, H, S, 5, "jacobi", lam.cpu().numpy(), host(Cm))


def test_eig_padded_leading_dimensions(env):
    torch, rsdft, plan = env["torch"], env["rsdft"], env["plan"]
    n, m = 50, 12
    H, S = env["wl"].subspace_pencil(n, 8)
    Hd = torch.full((n, n + 6), float("nan"), dtype=torch.complex128, device="cuda")
    Sd = torch.full((n, n + 6), float("nan"), dtype=torch.complex128, device="cuda")
    Hd[:, :n] = dev(env, H); Sd[:, :n] = dev(env, S)
    Cm = torch.full((m, n + 3), float("nan"), dtype=torch.complex128, device="cuda")
    lam, _ = rsdft.rsdft_subspace_eig(plan, Hd, Sd, m, Cmat=Cm)
    torch.cuda.synchronize()
    assert bool(torch.isnan(Cm[:, n:].real).all())
    check_eig(env, H, S, m, "jacobi", lam.cpu().numpy(), Cm[:, :n].cpu().numpy().T.copy())


# ------------------------------------------------------------------ the two sides' own chains
@pytest.mark.parametrize("cfg", [0, 1])
def test_block_step_then_eig_chain(env, cfg):
    """configs[0] (n = 24) and configs[1] (n = 192): apply_h -> gram -> eig on the CUDA path against the same chain in
    the oracle, each side on its own intermediate results (Ritz values of the seeded random block)."""
    torch, oracle, rsdft, wl = env["torch"], env["oracle"], env["rsdft"], env["wl"]
    system = wl.make_system(cfg)
    ng = int(np.prod(system["n"]))
    m = system["m"]
    plan = rsdft.plan_from_system(system)
    Y = torch.cat([wl.orbital_block(ng, range(m), system["seed"], s, device="cuda") for s in range(3)], dim=0)
    HY = torch.empty_like(Y)
    rsdft.rsdft_apply_h(plan, Y, HY)
    Hs, Ss = rsdft.rsdft_subspace_gram(plan, Y, HY)
    lam, Cm = rsdft.rsdft_subspace_eig(plan, Hs, Ss, m)
    torch.cuda.synchronize()
    Yh = Y.cpu().numpy()
    HY_ref = oracle.apply_h(system, Yh)
    H_ref, S_ref = oracle.gram(Yh, HY_ref)
    H_ref = 0.5 * (H_ref + H_ref.conj().T)
    check_eig(env, H_ref, S_ref, m, "jacobi", lam.cpu().numpy(), host(Cm))
    # rotate2 on the CUDA path against the oracle's own chain: X' and R agree up to the eigenvector phases, so compare
    # phase-invariant quantities: |R| column norms and the Gram matrix of X'
    Xn, HXn, R = rsdft.rsdft_subspace_rotate2(plan, Y, HY, Cm, lam)
    torch.cuda.synchronize()
    lam_o, C_o = oracle.subspace_eig(H_ref, S_ref, m)
    Xo, HXo, Ro = oracle.rotate2(Yh, HY_ref, C_o, lam_o)
    rn_g = np.linalg.norm(R.cpu().numpy(), axis=1)
    rn_o = np.linalg.norm(Ro, axis=1)
    assert np.max(np.abs(rn_g - rn_o)) <= 1e-9 * np.max(rn_o)          # simple spectrum: residual norms are unique
    plan.close()


def test_rayleigh_ritz_chain_recovers_free_electron_levels_on_device(env):
    """apply_h -> gram -> rsdft_subspace_eig -> rsdft_subspace_rotate2 entirely on the CUDA path: for V = 0 and no
    projectors a subspace spanned by plane waves is invariant, so one Rayleigh-Ritz step returns the free-electron levels
    1/2 |G|^2 (closed form; north_star's Ritz-value pin) with a vanishing residual R = HX' - X' Lambda."""
    torch, rsdft = env["torch"], env["rsdft"]
    n3, L = (16, 16, 32), (10.0, 10.0, 12.0)
    ng = int(np.prod(n3))
    rng = np.random.default_rng(11)
    ks = set()
    while len(ks) < 24:
        ks.add(tuple(int(v) for v in rng.integers(0, [16, 16, 32])))
    ks = sorted(ks)
    ii = np.indices(n3).reshape(3, -1)
    PW = np.stack([np.exp(2j * np.pi * sum(k[a] * ii[a] / n3[a] for a in range(3))) for k in ks]) / np.sqrt(ng)
    M = rng.standard_normal((24, 24)) + 1j * rng.standard_normal((24, 24)) + 4.0 * np.eye(24)
    plan = rsdft.rsdft_plan_create(n3, L)
    Y = torch.as_tensor(M @ PW).cuda()
    HY = torch.empty_like(Y)
    rsdft.rsdft_apply_h(plan, Y, HY)
    H, S = rsdft.rsdft_subspace_gram(plan, Y, HY)
    lam, Cm = rsdft.rsdft_subspace_eig(plan, H, S, 8)
    Xn, HXn, R = rsdft.rsdft_subspace_rotate2(plan, Y, HY, Cm, lam)
    torch.cuda.synchronize()
    kap = lambda j, N: j if 2 * j < N else j - N
    t = np.sort([0.5 * sum((2 * np.pi * kap(k[a], n3[a]) / L[a]) ** 2 for a in range(3)) for k in ks])
    assert np.max(np.abs(lam.cpu().numpy() - t[:8])) <= 1e-11 * t.max()
    assert float(R.abs().max()) <= 1e-10 * t.max() * float(Xn.abs().max())
    HXn2 = torch.empty_like(Xn)
    rsdft.rsdft_apply_h(plan, Xn, HXn2)                                     # H (Y C) == (H Y) C
    torch.cuda.synchronize()
    assert float((HXn2 - HXn).abs().max() / HXn.abs().max()) <= 1e-12
    plan.close()


# ------------------------------------------------------------------ NEXT-2: rotate2 element by element
@pytest.mark.parametrize("n,m", [(1, 1), (24, 8), (97, 50), (200, 96), (192, 200), (40, 128), (33, 250)])
def test_rotate2_parity_small_and_ragged(env, n, m):
    torch, oracle, rsdft, wl = env["torch"], env["oracle"], env["rsdft"], env["wl"]
    plan = rsdft.rsdft_plan_create((16, 32, 16), (5.0, 9.0, 5.0))
    ng = 16 * 32 * 16                                       # 8192 = 85 row tiles of 96 + 32
    Y = wl.orbital_block(ng, range(n), 51, 0, device="cuda", ld=ng + 8)
    HY = wl.orbital_block(ng, range(n), 51, 2, device="cuda", ld=ng + 24)
    Cs = wl.orbital_block(n, range(m), 52, 1, device="cuda", ld=n + 3)       # stored [m, ldc]: column-major n x m
    lam = torch.as_tensor(np.random.default_rng(n * 1000 + m).uniform(-1.0, 3.0, m)).cuda()
    mk = lambda pad: torch.full((m, ng + pad), float("nan"), dtype=torch.complex128, device="cuda")
    Xn, HXn, R = mk(16), mk(0), mk(40)
    rsdft.rsdft_subspace_rotate2(plan, Y, HY, Cs, lam, Xn, HXn, R)
    torch.cuda.synchronize()
    Xo, HXo, Ro = oracle.rotate2(Y[:, :ng].cpu().numpy(), HY[:, :ng].cpu().numpy(), Cs[:, :n].cpu().numpy().T, lam.cpu().numpy())
    for got, ref in ((Xn, Xo), (HXn, HXo), (R, Ro)):
        g = got[:, :ng].cpu().numpy()
        assert np.max(np.max(np.abs(g - ref), axis=1) / np.max(np.abs(ref), axis=1)) <= TOL
        assert bool(torch.isnan(got[:, ng:].real).all())    # padding untouched
    # P' = [W, P] C_P is the same call through pointer offsets into the block (sub-block of rows of Y, rows of C)
    if n >= 3:
        a = n // 3
        Pn, _, _ = rsdft.rsdft_subspace_rotate2(plan, Y[a:], HY[a:], Cs[:, a:], None, want_r=False)
        torch.cuda.synchronize()
        ref = oracle.rotate(Y[a:, :ng].cpu().numpy(), Cs[:, a:n].cpu().numpy().T)
        assert np.max(np.abs(Pn[:, :ng].cpu().numpy() - ref)) <= TOL * np.max(np.abs(ref))
    # the single-output kernel agrees
    X1 = rsdft.rsdft_subspace_rotate(plan, Y, Cs)
    torch.cuda.synchronize()
    assert float((X1[:, :ng] - Xn[:, :ng]).abs().max()) <= 1e-13 * float(Xn[:, :ng].abs().max())
    plan.close()


def test_rotate2_full_size_config2_sampled(env):
    """configs[2] shapes: n = 1440, m = 480 on the 96^3 grid, Y and HY random seeded blocks; the oracle recomputes a
    sample of grid points (all 480 outputs of X', HX', R at each)."""
    torch, oracle, rsdft, wl = env["torch"], env["oracle"], env["rsdft"], env["wl"]
    system = wl.make_system(2)
    m = system["m"]; n = 3 * m
    ng = int(np.prod(system["n"]))
    plan = rsdft.rsdft_plan_create(system["n"], system["len"])
    Y = wl.block_y(system, device="cuda")
    HY = torch.empty_like(Y)
    for s in range(3):
        wl.orbital_block(ng, range(m), 97, s, out=HY[s * m:(s + 1) * m])
    Cs = wl.orbital_block(n, range(m), 77, 0, device="cuda")
    lam = torch.as_tensor(np.random.default_rng(5).uniform(-1.0, 3.0, m)).cuda()
    Xn, HXn, R = rsdft.rsdft_subspace_rotate2(plan, Y, HY, Cs, lam)
    torch.cuda.synchronize()
    pts = np.unique(np.concatenate([[0, 95, 96, ng - 1], np.random.default_rng(3).integers(0, ng, 60)]))
    Xo, HXo, Ro = oracle.rotate2(Y[:, pts].cpu().numpy(), HY[:, pts].cpu().numpy(), Cs.cpu().numpy().T, lam.cpu().numpy())
    for got, ref in ((Xn, Xo), (HXn, HXo), (R, Ro)):
        assert np.max(np.abs(got[:, pts].cpu().numpy() - ref)) <= TOL * np.max(np.abs(ref))
    plan.close()
