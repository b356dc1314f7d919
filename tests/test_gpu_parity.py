"""GPU parity: the CUDA path through the C ABI vs the CPU oracle on the same seeded inputs.

Bar (BASELINE.json north_star; R16): max_g |gpu - oracle| / max_g |oracle| <= 1e-12 per
column for HX, per matrix for H_sub and S_sub, complex128.  Integer work (sphere point counts)
is compared exactly.  Every test here needs a B200 (pytest -m gpu)."""
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
    rsdft.load()          # fails loudly if the extension is missing
    return dict(torch=torch, oracle=oracle, rsdft=rsdft, wl=workloads)


def col_err(gpu, ref):
    """per-row normwise error of [ncol, Ng] arrays"""
    num = np.max(np.abs(gpu - ref), axis=1)
    den = np.max(np.abs(ref), axis=1)
    return float(np.max(num / den))


def mat_err(gpu, ref):
    return float(np.max(np.abs(gpu - ref)) / np.max(np.abs(ref)))


def blocks(env, system, cols_per_block=None, ld=None):
    """X, W, P seeded blocks (streams 0, 1, 2) stacked into Y [3m, ld] on the device."""
    wl, torch = env["wl"], env["torch"]
    m = system["m"] if cols_per_block is None else cols_per_block
    ng = int(np.prod(system["n"]))
    return torch.cat([wl.orbital_block(ng, range(m), system["seed"], s, device="cuda", ld=ld) for s in range(3)], dim=0)


def gpu_apply(env, plan, X):
    torch, rsdft = env["torch"], env["rsdft"]
    HX = torch.full_like(X, float("nan"))
    rsdft.rsdft_apply_h(plan, X, HX)
    torch.cuda.synchronize()
    return HX


# ------------------------------------------------------------------ configs 0 and 1, everything
@pytest.mark.parametrize("cfg", [0, 1])
def test_block_step_parity_full(env, cfg):
    torch, oracle, rsdft, wl = env["torch"], env["oracle"], env["rsdft"], env["wl"]
    system = wl.make_system(cfg)
    ng = int(np.prod(system["n"]))
    plan = rsdft.plan_from_system(system)
    info = rsdft.rsdft_plan_info(plan)
    Y = blocks(env, system)
    HY = gpu_apply(env, plan, Y)
    Yh = Y.cpu().numpy()
    HY_ref, p_ref = oracle.apply_h(system, Yh, return_p=True)
    assert col_err(HY.cpu().numpy(), HY_ref) <= TOL
    # integer work: sphere sizes agree exactly with the oracle's all-grid scan
    npts = sum(len(oracle.sphere(system["n"], system["len"], R, system["species"][0])[0]) for R in system["pos"])
    assert info["sphere_points"] == npts and info["ng"] == ng
    H, S = rsdft.rsdft_subspace_gram(plan, Y, HY)
    torch.cuda.synchronize()
    H_ref, S_ref = oracle.gram(Yh, HY_ref)
    Hg, Sg = H.cpu().numpy().T, S.cpu().numpy().T          # column-major storage -> M[i, j]
    assert mat_err(Hg, H_ref) <= TOL
    assert mat_err(Sg, S_ref) <= TOL
    assert np.array_equal(Sg, Sg.conj().T)                  # exactly Hermitian
    assert np.all(np.diagonal(Sg).imag == 0.0)
    assert mat_err(Hg, Hg.conj().T) <= 1e-13                # Hermitian to round-off
    np.linalg.cholesky(Sg)                                  # positive definite
    plan.close()


def test_apply_h_only_x_block_config0(env):
    """configs[0]: 'one rsdft_apply_h on X' (8 columns)."""
    oracle, rsdft, wl = env["oracle"], env["rsdft"], env["wl"]
    system = wl.make_system(0)
    plan = rsdft.plan_from_system(system)
    X = wl.orbital_block(4096, range(8), 0, 0, device="cuda")
    HX = gpu_apply(env, plan, X)
    assert col_err(HX.cpu().numpy(), oracle.apply_h(system, X.cpu().numpy())) <= TOL


# ------------------------------------------------------------------ every supported length on every axis
@pytest.mark.parametrize("N", [12, 16, 24, 32, 36, 48, 60, 64, 72, 80, 84, 96, 112, 120, 128, 144, 160, 192, 256])
@pytest.mark.parametrize("axis", [0, 1, 2])
def test_kinetic_every_length_every_axis(env, N, axis):
    torch, oracle, rsdft, wl = env["torch"], env["oracle"], env["rsdft"], env["wl"]
    n = [16, 16, 16]
    n[axis] = N
    L = [6.0, 7.0, 8.0]
    L[axis] = 0.31 * N
    ng = int(np.prod(n))
    rng = np.random.default_rng(100 + N + axis)
    system = dict(n=tuple(n), len=tuple(L), vloc=rng.standard_normal(ng))
    plan = rsdft.plan_from_system(system)
    X = wl.orbital_block(ng, range(3), 77, axis, device="cuda")
    HX = gpu_apply(env, plan, X)
    assert col_err(HX.cpu().numpy(), oracle.apply_h(system, X.cpu().numpy())) <= TOL
    # plane wave with negative frequency along `axis` is an eigenvector of T (V_loc = 0)
    rsdft.rsdft_plan_set_vloc(plan, None)
    k = N - 3
    idx = np.indices(n)[axis].reshape(-1)
    pw = torch.as_tensor(np.exp(2j * np.pi * k * idx / N)[None, :]).cuda()
    Tpw = gpu_apply(env, plan, pw).cpu().numpy()
    lam = 0.5 * (2 * np.pi * (k - N) / L[axis]) ** 2
    # round-off in the empty Fourier modes is amplified by their own t(k): scale by max_k t(k)
    tmax = 0.5 * sum((np.pi * n[a] / L[a]) ** 2 for a in range(3))
    assert np.max(np.abs(Tpw - lam * pw.cpu().numpy())) <= 1e-13 * tmax


@pytest.mark.parametrize("n3", [(60, 36, 24), (12, 60, 84), (24, 16, 60), (60, 60, 60)])
def test_lengths_with_first_radix_12(env, n3):
    """Grids whose lengths are 12*M (the paper's 60^3 among them), mixed with 16*M ones, with projectors."""
    oracle, rsdft, wl = env["oracle"], env["rsdft"], env["wl"]
    L = tuple(0.23 * v for v in n3)
    system = wl.small_system(n=n3, L=L, natom=3, seed=4, nproj=9, rc=1.3)
    ng = int(np.prod(n3))
    plan = rsdft.plan_from_system(system)
    X = wl.orbital_block(ng, range(3), 15, 0, device="cuda")
    HX = gpu_apply(env, plan, X)
    assert col_err(HX.cpu().numpy(), oracle.apply_h(system, X.cpu().numpy())) <= TOL
    plan.close()


@pytest.mark.parametrize("N,ncol", [(48, 13), (60, 9), (64, 7), (80, 5), (96, 7), (112, 4), (128, 3)])
def test_pipeline_kernel_matches_three_kernel_path(env, N, ncol):
    """rsdft_plan_set_pipeline(1): the persistent FFT kernel (work queue, per-column completion counters, TMA boxes issued
    by control warps) and rsdft_plan_set_pipeline(2): the TMA-staged x kernel give the same bits as the three-kernel
    path, on a caller's side stream, with overlapping projector spheres; and they match the oracle on sampled columns.
    (60 = 12*5 has no pipeline kernel: the call silently runs path 0.)"""
    torch, oracle, rsdft, wl = env["torch"], env["oracle"], env["rsdft"], env["wl"]
    L = (0.22 * N,) * 3
    system = wl.small_system(n=(N, N, N), L=L, natom=6, seed=N, nproj=4, rc=1.8)
    ng = N ** 3
    plan = rsdft.plan_from_system(system)
    X = wl.orbital_block(ng, range(ncol), 31, 0, device="cuda", ld=ng + 16)
    rsdft.rsdft_plan_set_pipeline(plan, 0)
    ref = gpu_apply(env, plan, X)
    side = torch.cuda.Stream()
    outs = []
    for mode, batch in ((1, 0), (1, 2), (2, 0), (2, 2)):
        rsdft.rsdft_plan_set_pipeline(plan, mode)
        rsdft.rsdft_plan_set_batch(plan, batch)
        with torch.cuda.stream(side):
            HX = torch.full_like(X, float("nan"))
            rsdft.rsdft_apply_h(plan, X, HX)
            outs.append(HX.clone())
        side.synchronize()
    for o in outs:
        assert torch.equal(torch.view_as_real(o[:, :ng]), torch.view_as_real(ref[:, :ng]))
        assert bool(torch.isnan(o[:, ng:].real).all())
    cols = [0, ncol - 1]
    assert col_err(outs[0][cols, :ng].cpu().numpy(), oracle.apply_h(system, X[cols, :ng].cpu().numpy())) <= TOL
    assert rsdft.rsdft_plan_info(plan)["last_launches"] >= 1
    plan.close()


# ------------------------------------------------------------------ degenerate / ragged inputs
def test_no_atoms_no_vloc_is_kinetic_only(env):
    oracle, rsdft, wl = env["oracle"], env["rsdft"], env["wl"]
    system = dict(n=(32, 16, 48), len=(9.0, 5.0, 13.0), vloc=None)
    plan = rsdft.rsdft_plan_create(system["n"], system["len"])
    ng = 32 * 16 * 48
    X = wl.orbital_block(ng, range(5), 5, 0, device="cuda")
    HX = gpu_apply(env, plan, X)
    assert col_err(HX.cpu().numpy(), oracle.apply_h(system, X.cpu().numpy())) <= TOL
    assert rsdft.rsdft_plan_info(plan)["natom"] == 0


@pytest.mark.parametrize("radial_kind", [0, 1])
def test_noncubic_spd_projectors_full_D_padded_ld(env, radial_kind):
    """9 s+p+d projectors, full symmetric D, tabulated radial part, overlapping spheres, ld > Ng,
    ncol not a multiple of the batch width; result independent of the batch width and of the
    number of internal streams (bitwise)."""
    torch, oracle, rsdft, wl = env["torch"], env["oracle"], env["rsdft"], env["wl"]
    system = wl.small_system(n=(32, 16, 48), L=(7.0, 4.1, 9.5), natom=5, seed=11, nproj=9, rc=1.9,
                             radial_kind=radial_kind)
    ng = 32 * 16 * 48
    plan = rsdft.plan_from_system(system)
    assert rsdft.rsdft_plan_info(plan)["colour_classes"] >= 2          # spheres do overlap here
    X = wl.orbital_block(ng, range(7), 3, 0, device="cuda", ld=ng + 24)
    ref = oracle.apply_h(system, X[:, :ng].cpu().numpy())
    outs = []
    for batch, streams in ((0, 0), (1, 1), (3, 4), (7, 2), (16, 3), (2, 3)):
        rsdft.rsdft_plan_set_batch(plan, batch)
        rsdft.rsdft_plan_set_streams(plan, streams)
        HX = gpu_apply(env, plan, X)
        assert col_err(HX[:, :ng].cpu().numpy(), ref) <= TOL
        assert bool(torch.isnan(HX[:, ng:].real).all())                 # padding untouched
        outs.append(HX[:, :ng].clone())
    for o in outs[1:]:
        assert torch.equal(torch.view_as_real(o), torch.view_as_real(outs[0]))


def test_single_column_and_sphere_wrapping(env):
    """One column; atoms placed at the box corner and outside [0, L) so spheres wrap periodically."""
    oracle, rsdft, wl = env["oracle"], env["rsdft"], env["wl"]
    system = wl.small_system(n=(16, 16, 16), L=(5.0, 5.0, 5.0), natom=3, seed=5, nproj=4, rc=1.7)
    system["pos"] = np.array([[0.01, 0.02, 4.99], [-1.3, 6.2, 2.5], [2.5, 2.5, 2.5]])
    plan = rsdft.plan_from_system(system)
    X = wl.orbital_block(4096, [0], 9, 0, device="cuda")
    HX = gpu_apply(env, plan, X)
    assert col_err(HX.cpu().numpy(), oracle.apply_h(system, X.cpu().numpy())) <= TOL


@pytest.mark.parametrize("n", [1, 7, 96, 97, 200])
def test_gram_ragged_sizes_and_options(env, n):
    torch, oracle, rsdft, wl = env["torch"], env["oracle"], env["rsdft"], env["wl"]
    plan = rsdft.rsdft_plan_create((16, 32, 16), (5.0, 9.0, 5.0))
    ng = 16 * 32 * 16
    Y = wl.orbital_block(ng, range(n), 21, 0, device="cuda", ld=ng + 8)
    HY = wl.orbital_block(ng, range(n), 21, 1, device="cuda")
    H_ref, S_ref = oracle.gram(Y[:, :ng].cpu().numpy(), HY.cpu().numpy())
    H, S = rsdft.rsdft_subspace_gram(plan, Y, HY)
    torch.cuda.synchronize()
    assert mat_err(H.cpu().numpy().T, H_ref) <= TOL
    assert mat_err(S.cpu().numpy().T, S_ref) <= TOL
    _, S2 = rsdft.rsdft_subspace_gram(plan, Y, None, want_h=False)
    H2, _ = rsdft.rsdft_subspace_gram(plan, Y, HY, want_s=False)
    torch.cuda.synchronize()
    assert torch.equal(torch.view_as_real(S2), torch.view_as_real(S))    # deterministic, bitwise
    assert torch.equal(torch.view_as_real(H2), torch.view_as_real(H))


def test_gram_bulk_copy_staging_is_bitwise_identical(env):
    """rsdft_plan_set_gram_staging(1): the TMA bulk-copy (cp.async.bulk + mbarrier) operand pipeline computes exactly what
    the cp.async pipeline computes, ragged last tile and H-upper mode included."""
    torch, rsdft, wl = env["torch"], env["rsdft"], env["wl"]
    plan = rsdft.rsdft_plan_create((16, 32, 48), (5.0, 9.0, 14.0))
    ng = 16 * 32 * 48
    for n in (7, 200):
        Y = wl.orbital_block(ng, range(n), 23, 0, device="cuda", ld=ng + 8)
        HY = wl.orbital_block(ng, range(n), 23, 1, device="cuda")
        for mode in (0, 1):
            rsdft.rsdft_plan_set_gram_mode(plan, mode)
            rsdft.rsdft_plan_set_gram_staging(plan, 0)
            H0, S0 = rsdft.rsdft_subspace_gram(plan, Y, HY)
            rsdft.rsdft_plan_set_gram_staging(plan, 1)
            H1, S1 = rsdft.rsdft_subspace_gram(plan, Y, HY)
            torch.cuda.synchronize()
            assert torch.equal(torch.view_as_real(H0), torch.view_as_real(H1))
            assert torch.equal(torch.view_as_real(S0), torch.view_as_real(S1))
    plan.close()


def test_repeated_calls_are_bitwise_reproducible(env):
    """Race evidence without a sanitizer (compute-sanitizer is closed on this GPU pool): five repetitions of apply_h with
    overlapping spheres (colour-class scatter), of the Gram, of the eigen-solve and of rotate2 give identical bits, on
    both apply_h FFT paths."""
    torch, rsdft, wl = env["torch"], env["rsdft"], env["wl"]
    system = wl.small_system(n=(48, 48, 48), L=(9.0, 9.0, 9.0), natom=10, seed=77, nproj=9, rc=2.2)
    ng = 48 ** 3
    plan = rsdft.plan_from_system(system)
    assert rsdft.rsdft_plan_info(plan)["colour_classes"] >= 2
    Y = wl.orbital_block(ng, range(60), 19, 0, device="cuda")
    ref = None
    for rep in range(5):
        rsdft.rsdft_plan_set_pipeline(plan, rep % 3)
        HY = torch.full_like(Y, float("nan"))
        rsdft.rsdft_apply_h(plan, Y, HY)
        H, S = rsdft.rsdft_subspace_gram(plan, Y, HY)
        lam, Cm = rsdft.rsdft_subspace_eig(plan, H, S, 20)
        Xn, HXn, R = rsdft.rsdft_subspace_rotate2(plan, Y, HY, Cm, lam)
        torch.cuda.synchronize()
        cur = [torch.view_as_real(t).clone() for t in (HY, H, S, Cm, Xn, HXn, R)] + [lam.clone()]
        if ref is None:
            ref = cur
        else:
            for a, b in zip(ref, cur):
                assert torch.equal(a, b)
    plan.close()


def test_gram_plane_waves_closed_form(env):
    """Plane-wave columns: S_sub = Ng I, H_sub = Ng diag(t) (V = 0, no projectors) -- closed form."""
    torch, rsdft = env["torch"], env["rsdft"]
    n, L = (16, 16, 32), (10.0, 10.0, 12.0)
    ng = int(np.prod(n))
    plan = rsdft.rsdft_plan_create(n, L)
    ks = [(0, 0, 0), (1, 0, 0), (0, 15, 0), (0, 0, 16), (3, 2, 31), (8, 8, 1)]
    ii = np.indices(n).reshape(3, -1)
    Y = np.stack([np.exp(2j * np.pi * sum(k[a] * ii[a] / n[a] for a in range(3))) for k in ks])
    Yd = torch.as_tensor(Y).cuda()
    HY = gpu_apply(env, plan, Yd)
    H, S = rsdft.rsdft_subspace_gram(plan, Yd, HY)
    torch.cuda.synchronize()
    kap = lambda j, N: j if 2 * j < N else j - N
    t = np.array([0.5 * sum((2 * np.pi * kap(k[a], n[a]) / L[a]) ** 2 for a in range(3)) for k in ks])
    assert np.max(np.abs(S.cpu().numpy().T - ng * np.eye(len(ks)))) <= 1e-12 * ng
    assert np.max(np.abs(H.cpu().numpy().T - ng * np.diag(t))) <= 1e-12 * ng * t.max()


def test_error_paths_on_device(env):
    torch, rsdft = env["torch"], env["rsdft"]
    plan = rsdft.rsdft_plan_create((16, 16, 16), (10.0,) * 3)
    X = torch.zeros((2, 4096), dtype=torch.complex128, device="cuda")
    with pytest.raises(rsdft.RsdftError) as e:
        rsdft.rsdft_apply_h(plan, X, X)                                   # aliasing
    assert e.value.code == rsdft.RSDFT_INVALID_ARG and "overlap" in str(e.value)
    short = torch.zeros((2, 4000), dtype=torch.complex128, device="cuda")
    with pytest.raises(ValueError):
        rsdft.rsdft_apply_h(plan, short, torch.zeros_like(short))         # ld < Ng: caught by the binding
    with pytest.raises(ValueError):
        rsdft.rsdft_subspace_gram(plan, short, short)
    lib0 = rsdft.load()                                                   # ... and by the C ABI itself
    assert lib0.rsdft_apply_h(plan.handle, 2, X.data_ptr(), 4000, X.data_ptr() + 2 * 4096 * 16, 4096, None) == rsdft.RSDFT_INVALID_ARG
    assert lib0.rsdft_subspace_gram(plan.handle, 2, X.data_ptr(), 4000, X.data_ptr(), 4000, X.data_ptr(), X.data_ptr(), 2, None) == rsdft.RSDFT_INVALID_ARG
    with pytest.raises(ValueError):
        rsdft.rsdft_apply_h(plan, X.cpu(), X)                             # host tensor
    lib = rsdft.load()
    assert lib.rsdft_apply_h(plan.handle, 0, X.data_ptr(), 4096, X.data_ptr(), 4096, None) == rsdft.RSDFT_INVALID_ARG


def test_block_step_host_matches_device_path(env):
    torch, oracle, rsdft, wl = env["torch"], env["oracle"], env["rsdft"], env["wl"]
    system = wl.make_system(1)
    ng = 48 ** 3
    plan = rsdft.plan_from_system(system)
    Y = blocks(env, system, cols_per_block=8)
    Yh = Y.cpu().pin_memory()
    HYh = torch.empty_like(Yh).pin_memory()
    H, S = rsdft.rsdft_block_step_host(plan, Yh, HYh)
    HY_ref = oracle.apply_h(system, Yh.numpy())
    H_ref, S_ref = oracle.gram(Yh.numpy(), HY_ref)
    assert col_err(HYh.numpy(), HY_ref) <= TOL
    assert mat_err(H.numpy().T, H_ref) <= TOL and mat_err(S.numpy().T, S_ref) <= TOL
    HY = gpu_apply(env, plan, Y)
    assert torch.equal(torch.view_as_real(HY.cpu()), torch.view_as_real(HYh))
    assert rsdft.rsdft_plan_info(plan)["last_launches"] > 0


def test_block_step_host_padded_ld_and_ragged_last_panel(env):
    """rsdft_block_step_host with ld > Ng on both host blocks, n = 200 = two full 96-column panels + a ragged one,
    lds > n on the host matrices; then rsdft_plan_release_workspace and a second call."""
    torch, oracle, rsdft, wl = env["torch"], env["oracle"], env["rsdft"], env["wl"]
    system = wl.small_system(n=(32, 16, 48), L=(7.0, 4.1, 9.5), natom=5, seed=11, nproj=9, rc=1.9)
    ng = 32 * 16 * 48
    n = 200
    plan = rsdft.plan_from_system(system)
    Yh = wl.orbital_block(ng, range(n), 13, 0, ld=ng + 40).pin_memory()
    HYh = torch.full((n, ng + 8), float("nan"), dtype=torch.complex128).pin_memory()
    Hh = torch.full((n, n + 5), float("nan"), dtype=torch.complex128).pin_memory()
    Sh = torch.full((n, n + 5), float("nan"), dtype=torch.complex128).pin_memory()
    rsdft.rsdft_block_step_host(plan, Yh, HYh, Hh, Sh)
    Yn = Yh[:, :ng].numpy()
    HY_ref = oracle.apply_h(system, Yn)
    H_ref, S_ref = oracle.gram(Yn, HY_ref)
    assert col_err(HYh[:, :ng].numpy(), HY_ref) <= TOL
    assert bool(torch.isnan(HYh[:, ng:].real).all()) and bool(torch.isnan(Hh[:, n:].real).all())
    assert mat_err(Hh[:, :n].numpy().T, H_ref) <= TOL and mat_err(Sh[:, :n].numpy().T, S_ref) <= TOL
    before = rsdft.rsdft_plan_info(plan)["device_bytes"]
    rsdft.rsdft_plan_release_workspace(plan)
    assert rsdft.rsdft_plan_info(plan)["device_bytes"] < before - 2 * n * ng * 16 + 1
    H2, S2 = rsdft.rsdft_block_step_host(plan, Yh, None)
    assert np.array_equal(H2.numpy(), Hh[:, :n].numpy()) and np.array_equal(S2.numpy(), Sh[:, :n].numpy())
    plan.close()


def test_set_vloc_on_another_stream_is_ordered_before_block_step_host(env):
    """rsdft_plan_set_vloc queued on a busy side stream, then rsdft_block_step_host right away (plan-owned streams):
    the step must see the NEW potential (the plan orders itself after the copy through an event)."""
    torch, rsdft, wl = env["torch"], env["rsdft"], env["wl"]
    system = wl.make_system(1)
    ng = 48 ** 3
    plan = rsdft.plan_from_system(system)
    Yh = wl.orbital_block(ng, range(12), 3, 0).pin_memory()
    v2 = torch.as_tensor(np.random.default_rng(2).standard_normal(ng)).cuda()
    ref_plan = rsdft.plan_from_system(dict(system, vloc=v2.cpu().numpy()))
    HY_ref = torch.empty_like(Yh).pin_memory()
    rsdft.rsdft_block_step_host(ref_plan, Yh, HY_ref)
    side = torch.cuda.Stream()
    big = torch.zeros(1 << 28, dtype=torch.float64, device="cuda")
    HY = torch.empty_like(Yh).pin_memory()
    with torch.cuda.stream(side):
        for _ in range(20):
            big.add_(1.0)                                   # ~40 ms of queued work ahead of the copy
        rsdft.rsdft_plan_set_vloc(plan, v2)
    rsdft.rsdft_block_step_host(plan, Yh, HY)
    assert torch.equal(torch.view_as_real(HY), torch.view_as_real(HY_ref))
    side.synchronize()
    plan.close(); ref_plan.close()


def test_two_devices_in_one_thread(env):
    """a plan per device used from one thread (the Gram kernel's shared-memory attribute is per device)"""
    torch, rsdft, wl = env["torch"], env["rsdft"], env["wl"]
    if torch.cuda.device_count() < 2:
        pytest.skip("needs 2 GPUs")
    outs = []
    for d in (0, 1):
        with torch.cuda.device(d):
            plan = rsdft.rsdft_plan_create((16, 32, 16), (5.0, 9.0, 5.0))
            Y = wl.orbital_block(8192, range(20), 21, 0, device="cuda:%d" % d)
            HY = torch.empty_like(Y)
            rsdft.rsdft_apply_h(plan, Y, HY)
            H, S = rsdft.rsdft_subspace_gram(plan, Y, HY)
            torch.cuda.synchronize()
            outs.append((H.cpu(), S.cpu()))
            plan.close()
    assert torch.equal(torch.view_as_real(outs[0][0]), torch.view_as_real(outs[1][0]))
    assert torch.equal(torch.view_as_real(outs[0][1]), torch.view_as_real(outs[1][1]))


def test_binding_rejects_wrong_output_tensors(env):
    torch, rsdft = env["torch"], env["rsdft"]
    plan = rsdft.rsdft_plan_create((16, 16, 16), (10.0,) * 3)
    Y = torch.zeros((4, 4096), dtype=torch.complex128, device="cuda")
    HY = torch.zeros_like(Y)
    with pytest.raises(ValueError):
        rsdft.rsdft_subspace_gram(plan, Y, HY, H_sub=torch.zeros((4, 3), dtype=torch.complex128, device="cuda"))
    with pytest.raises(ValueError):
        rsdft.rsdft_subspace_gram(plan, Y, HY, S_sub=torch.zeros((4, 4), dtype=torch.complex64, device="cuda"))
    with pytest.raises(ValueError):
        rsdft.rsdft_subspace_gram(plan, Y, HY, H_sub=torch.zeros((4, 4), dtype=torch.complex128))       # host
    with pytest.raises(ValueError):
        rsdft.rsdft_apply_h(plan, Y[:, :4000], HY)                                                       # view shorter than Ng
    with pytest.raises(ValueError):
        rsdft.rsdft_block_step_host(plan, Y.cpu(), None, torch.zeros((4, 4), dtype=torch.complex128, device="cuda"))
    Hs = torch.full((4, 9), float("nan"), dtype=torch.complex128, device="cuda")
    Ss = torch.full((4, 9), float("nan"), dtype=torch.complex128, device="cuda")
    rsdft.rsdft_subspace_gram(plan, Y, HY, Hs, Ss)                                                       # lds = 9 > n is passed through
    torch.cuda.synchronize()
    assert bool(torch.isnan(Hs[:, 4:].real).all()) and bool((Hs[:, :4] == 0).all())
    plan.close()


# ------------------------------------------------------------------ BASELINE.json full sizes, bench.py's launch configuration
@pytest.mark.parametrize("cfg", [2, 3, 4, 5, 6])
def test_full_size_block_step_sampled_parity(env, cfg):
    """configs[2..4] (and the paper's own shapes, workloads.CONFIGS[5, 6]: diamond-216 on 60^3 with 436 orbitals, W-128 on
    80^3 with 901) at full size (n = 3m columns, whole block resident in HBM), the library's default
    batching/streams, i.e. exactly what bench.py times.  The oracle recomputes a seeded sample of columns
    spread over X, W, P (HX element by element) and the matching |C| x |C| sub-blocks of H_sub and S_sub
    over the full grid; the rest of the matrices is checked through invariants that hold at any size."""
    torch, oracle, rsdft, wl = env["torch"], env["oracle"], env["rsdft"], env["wl"]
    system = wl.make_system(cfg)
    m = system["m"]
    n = 3 * m
    ng = int(np.prod(system["n"]))
    need = 2 * n * ng * 16 + (8 << 30)
    import gc
    gc.collect()
    torch.cuda.empty_cache()                     # blocks of the previous case are still cached by torch
    free, _ = torch.cuda.mem_get_info()
    assert free >= need, "configs[%d] needs %.0f GB of free HBM, %.0f GB are free: the full-size case cannot be skipped" % (
        cfg, need / 1e9, free / 1e9)
    plan = rsdft.plan_from_system(system)
    info = rsdft.rsdft_plan_info(plan)
    # integer work at full size: the plan's sphere lists hold exactly the points the oracle's all-grid scan finds
    npts = sum(len(oracle.sphere(system["n"], system["len"], R, system["species"][0])[0]) for R in system["pos"])
    assert info["sphere_points"] == npts and info["ng"] == ng
    Y = wl.block_y(system, device="cuda")
    HY = torch.empty_like(Y)
    rsdft.rsdft_apply_h(plan, Y, HY)
    H, S = rsdft.rsdft_subspace_gram(plan, Y, HY)
    torch.cuda.synchronize()
    # 16+ sampled columns: the ends of X, W, P, both sides of an internal column-batch boundary and of a stream-round
    # boundary (3 batches), the ragged last batch, plus seeded random ones
    b = info["batch_cols"]
    C = {0, b - 1, b, 3 * b - 1, 3 * b, m - 1, m, 2 * m - 3, 2 * m + 7, n - 1, (n // b) * b - 1, min((n // b) * b, n - 1)}
    C |= {int(v) for v in np.random.default_rng(cfg).integers(0, n, 6)}
    C = sorted(c for c in C if 0 <= c < n)
    assert len(C) >= 16
    Yc = Y[C].cpu().numpy()
    HY_ref = oracle.apply_h(system, Yc)
    assert col_err(HY[C].cpu().numpy(), HY_ref) <= TOL
    H_ref, S_ref = oracle.gram(Yc, HY_ref)
    Hg, Sg = H.cpu().numpy().T, S.cpu().numpy().T
    scale_h, scale_s = np.max(np.abs(Hg)), np.max(np.abs(Sg))
    assert np.max(np.abs(Hg[np.ix_(C, C)] - H_ref)) <= TOL * scale_h
    assert np.max(np.abs(Sg[np.ix_(C, C)] - S_ref)) <= TOL * scale_s
    # whole-matrix properties
    assert np.array_equal(Sg, Sg.conj().T)
    assert np.max(np.abs(Hg - Hg.conj().T)) <= 1e-12 * scale_h
    rows = lambda f: torch.cat([f(c0, min(c0 + 32, n)) for c0 in range(0, n, 32)]).cpu().numpy()   # chunked: no 50 GB temporaries
    norms = rows(lambda a, b: (Y[a:b].real ** 2 + Y[a:b].imag ** 2).sum(dim=1))
    assert np.max(np.abs(np.diagonal(Sg).real - norms)) <= 1e-12 * scale_s
    hd = rows(lambda a, b: (Y[a:b].conj() * HY[a:b]).sum(dim=1))       # diag(H_sub) = <y_i | H y_i>
    assert np.max(np.abs(np.diagonal(Hg) - hd)) <= 1e-12 * scale_h
    np.linalg.cholesky(Sg)
    # the other FFT paths at full size: three plain kernels and the persistent pipeline kernel (where the grid has one)
    # rewrite the same HY bit for bit -- compared through per-column integer checksums of the bit patterns, so that no
    # third block has to be resident
    bits = lambda T: torch.view_as_real(T).view(torch.int64).sum(dim=(1, 2))
    ref_bits = bits(HY)
    for mode in (0, 1):
        rsdft.rsdft_plan_set_pipeline(plan, mode)
        HY.fill_(float("nan"))
        rsdft.rsdft_apply_h(plan, Y, HY)
        torch.cuda.synchronize()
        assert torch.equal(bits(HY), ref_bits), "FFT path %d differs from the default path at full size" % mode
    plan.close()


def test_gram_hermitian_mode_matches_full(env):
    """rsdft_plan_set_gram_mode(1): H_sub from its upper tiles + conjugate mirror equals the fully contracted H_sub
    to round-off when HY really is H Y (H Hermitian), is exactly Hermitian, and matches the oracle; the host
    entry point honours the mode too."""
    torch, oracle, rsdft, wl = env["torch"], env["oracle"], env["rsdft"], env["wl"]
    system = wl.small_system(n=(16, 32, 16), L=(5.0, 9.0, 5.0), natom=4, seed=3, nproj=9, rc=1.6)
    ng = 16 * 32 * 16
    n = 200                                                   # 3 tile columns, ragged last tile
    plan = rsdft.plan_from_system(system)
    Y = wl.orbital_block(ng, range(n), 31, 0, device="cuda")
    HY = gpu_apply(env, plan, Y)
    H0, S0 = rsdft.rsdft_subspace_gram(plan, Y, HY)
    rsdft.rsdft_plan_set_gram_mode(plan, 1)
    H1, S1 = rsdft.rsdft_subspace_gram(plan, Y, HY)
    torch.cuda.synchronize()
    H0n, H1n = H0.cpu().numpy().T, H1.cpu().numpy().T
    assert np.array_equal(H1n, H1n.conj().T) and np.all(np.diagonal(H1n).imag == 0.0)
    assert mat_err(H1n, H0n) <= 1e-13
    assert torch.equal(torch.view_as_real(S1), torch.view_as_real(S0))
    Yh = Y.cpu().numpy()
    H_ref, _ = oracle.gram(Yh, oracle.apply_h(system, Yh))
    assert mat_err(H1n, H_ref) <= TOL
    Hh, Sh = rsdft.rsdft_block_step_host(plan, Y.cpu().pin_memory(), None)
    assert mat_err(Hh.numpy().T, H_ref) <= TOL
    assert np.array_equal(Hh.numpy(), Hh.numpy().conj().T)
    plan.close()


# ------------------------------------------------------------------ properties of the CUDA operator itself (any size)
def test_gpu_operator_is_hermitian_and_linear(env):
    """<x|H y> = conj(<y|H x>) and H(ax + by) = a Hx + b Hy on the CUDA path (north_star's invariants, applied to
    the product rather than the oracle): overlapping spheres, non-cubic grid with three different radix mixes."""
    torch, rsdft, wl = env["torch"], env["rsdft"], env["wl"]
    system = wl.small_system(n=(48, 80, 32), L=(9.0, 15.5, 6.1), natom=9, seed=21, nproj=9, rc=2.1)
    ng = 48 * 80 * 32
    plan = rsdft.plan_from_system(system)
    X = wl.orbital_block(ng, range(5), 41, 0, device="cuda")
    Y = wl.orbital_block(ng, range(5), 41, 1, device="cuda")
    HX, HY = gpu_apply(env, plan, X), gpu_apply(env, plan, Y)
    A = X.conj() @ HY.T                      # A[i, j] = <x_i | H y_j>
    B = Y.conj() @ HX.T                      # B[j, i] = <y_j | H x_i>
    scale = float(A.abs().max())
    assert float((A - B.conj().T).abs().max()) <= 1e-12 * scale
    a, b = 0.7 - 1.3j, -2.1 + 0.4j
    HZ = gpu_apply(env, plan, a * X + b * Y)
    ref = a * HX + b * HY
    assert float((HZ - ref).abs().max() / ref.abs().max()) <= 1e-13
    plan.close()


def test_gpu_translation_covariance(env):
    """Shifting psi, v and the atoms by an integer grid vector shifts H psi identically (exercises the periodic
    wrap of the sphere lists and of every FFT axis on the CUDA path)."""
    torch, rsdft, wl = env["torch"], env["rsdft"], env["wl"]
    n, L = (32, 48, 16), (8.0, 12.0, 4.0)
    system = wl.small_system(n=n, L=L, natom=4, seed=8, nproj=4, rc=1.5)
    ng = int(np.prod(n))
    sh = (5, 31, 9)
    h = [L[a] / n[a] for a in range(3)]
    shifted = dict(system)
    shifted["pos"] = system["pos"] + np.array([sh[a] * h[a] for a in range(3)])
    shifted["vloc"] = np.roll(system["vloc"].reshape(n), sh, axis=(0, 1, 2)).reshape(-1).copy()
    X = wl.orbital_block(ng, range(3), 12, 0, device="cuda")
    Xs = torch.roll(X.reshape(3, *n), sh, dims=(1, 2, 3)).reshape(3, ng).contiguous()
    p1, p2 = rsdft.plan_from_system(system), rsdft.plan_from_system(shifted)
    HX = gpu_apply(env, p1, X)
    HXs = gpu_apply(env, p2, Xs)
    ref = torch.roll(HX.reshape(3, *n), sh, dims=(1, 2, 3)).reshape(3, ng)
    assert float((HXs - ref).abs().max() / ref.abs().max()) <= 1e-13
    p1.close(); p2.close()


def test_calls_are_ordered_on_the_callers_stream(env):
    """apply_h forks to internal streams and joins back: work queued on the caller's (non-default) stream right after
    the call must see the finished result, and the call must wait for work queued before it."""
    torch, rsdft, wl = env["torch"], env["rsdft"], env["wl"]
    system = wl.make_system(1)
    ng = 48 ** 3
    plan = rsdft.plan_from_system(system)
    rsdft.rsdft_plan_set_batch(plan, 4)
    rsdft.rsdft_plan_set_streams(plan, 4)
    X0 = wl.orbital_block(ng, range(24), 1, 0, device="cuda")
    ref = gpu_apply(env, plan, X0)
    torch.cuda.synchronize()
    side = torch.cuda.Stream()
    X = torch.zeros_like(X0)
    HX = torch.empty_like(X0)
    with torch.cuda.stream(side):
        for _ in range(3):                              # keep the stream busy so ordering mistakes show
            X.copy_(X0 * 0.0)
            X.copy_(X0)                                 # queued BEFORE the call on the same stream
            rsdft.rsdft_apply_h(plan, X, HX)
            out = HX.clone()                            # queued AFTER the call on the same stream
            H, S = rsdft.rsdft_subspace_gram(plan, X, HX)
            Hc = H.clone()
    side.synchronize()
    assert torch.equal(torch.view_as_real(out), torch.view_as_real(ref))
    H2, _ = rsdft.rsdft_subspace_gram(plan, X0, ref)
    torch.cuda.synchronize()
    assert torch.equal(torch.view_as_real(Hc), torch.view_as_real(H2))
    plan.close()


# ------------------------------------------------------------------ NEXT-2: Rayleigh-Ritz update Out = Y C
@pytest.mark.parametrize("n,m", [(1, 1), (24, 8), (97, 50), (200, 96), (192, 200), (40, 128), (33, 250)])
def test_rotate_parity_small_and_ragged(env, n, m):
    """rsdft_subspace_rotate vs the oracle, element by element: ragged n (K), m (N) and a grid whose size is not a
    multiple of the 96-point tile; padded ld on every operand."""
    torch, oracle, rsdft, wl = env["torch"], env["oracle"], env["rsdft"], env["wl"]
    plan = rsdft.rsdft_plan_create((16, 32, 16), (5.0, 9.0, 5.0))
    ng = 16 * 32 * 16                                       # 8192 = 85 tiles of 96 + 32
    Y = wl.orbital_block(ng, range(n), 51, 0, device="cuda", ld=ng + 8)
    Cs = wl.orbital_block(n, range(m), 52, 1, device="cuda", ld=n + 3)       # stored [m, ldc]: column-major n x m
    Out = torch.full((m, ng + 16), float("nan"), dtype=torch.complex128, device="cuda")
    rsdft.rsdft_subspace_rotate(plan, Y, Cs, Out)
    torch.cuda.synchronize()
    ref = oracle.rotate(Y[:, :ng].cpu().numpy(), Cs[:, :n].cpu().numpy().T)
    assert col_err(Out[:, :ng].cpu().numpy(), ref) <= TOL
    assert bool(torch.isnan(Out[:, ng:].real).all())        # padding untouched
    plan.close()


def test_rotate_full_size_config2_sampled(env):
    """configs[2] shapes: X' = Y C_X with n = 1440, m = 480 on the 96^3 grid; the oracle recomputes a sample of
    grid points (all 480 outputs at each) and the identity (YC)^H (YC) = C^H S_sub C ties it to the Gram kernel."""
    torch, oracle, rsdft, wl = env["torch"], env["oracle"], env["rsdft"], env["wl"]
    system = wl.make_system(2)
    m = system["m"]; n = 3 * m
    ng = int(np.prod(system["n"]))
    plan = rsdft.rsdft_plan_create(system["n"], system["len"])
    Y = wl.block_y(system, device="cuda")
    Cs = wl.orbital_block(n, range(m), 77, 0, device="cuda")
    Out = rsdft.rsdft_subspace_rotate(plan, Y, Cs)
    torch.cuda.synchronize()
    pts = np.unique(np.concatenate([[0, 95, 96, ng - 1], np.random.default_rng(3).integers(0, ng, 60)]))
    ref = oracle.rotate(Y[:, pts].cpu().numpy(), Cs.cpu().numpy().T)
    got = Out[:, pts].cpu().numpy()
    assert np.max(np.abs(got - ref)) <= TOL * np.max(np.abs(ref))
    _, S = rsdft.rsdft_subspace_gram(plan, Y, None, want_h=False)
    _, S2 = rsdft.rsdft_subspace_gram(plan, Out, None, want_h=False)
    torch.cuda.synchronize()
    Cm = Cs.cpu().numpy().T
    want = Cm.conj().T @ S.cpu().numpy().T @ Cm
    assert np.max(np.abs(S2.cpu().numpy().T - want)) <= 1e-11 * np.max(np.abs(want))
    plan.close()


def test_two_species_with_different_projector_counts(env):
    """Atoms of two species (4 s+p projectors with a diagonal D, 9 s+p+d projectors with a full symmetric D,
    different cut-off radii) in one plan: the per-atom projector count is smaller than the plan's maximum."""
    oracle, rsdft, wl = env["oracle"], env["rsdft"], env["wl"]
    a = wl.small_system(n=(32, 32, 16), L=(7.0, 7.5, 4.0), natom=6, seed=17, nproj=9, rc=1.7)
    b = wl.small_system(n=(32, 32, 16), L=(7.0, 7.5, 4.0), natom=6, seed=18, nproj=4, rc=1.3)
    system = dict(a)
    system["species"] = [a["species"][0], b["species"][0]]
    system["species_of"] = np.array([0, 1, 1, 0, 1, 0], np.int32)
    ng = 32 * 32 * 16
    plan = rsdft.plan_from_system(system)
    X = wl.orbital_block(ng, range(9), 4, 0, device="cuda")
    HX = gpu_apply(env, plan, X)
    assert col_err(HX.cpu().numpy(), oracle.apply_h(system, X.cpu().numpy())) <= TOL
    plan.close()


@pytest.mark.parametrize("n3", [(112, 256, 16), (256, 16, 192), (16, 160, 256)])
def test_mixed_large_lengths_with_projectors(env, n3):
    """Lengths 160, 192, 256 (M = 10, 12, 16) mixed with small ones, projectors included: exercises the x kernel's
    narrower-tile fallback for a large ny and the one-CTA-per-SM shapes of the 256-point kernels."""
    oracle, rsdft, wl = env["oracle"], env["rsdft"], env["wl"]
    L = tuple(0.21 * v for v in n3)
    system = wl.small_system(n=n3, L=L, natom=3, seed=9, nproj=4, rc=1.2)
    ng = int(np.prod(n3))
    plan = rsdft.plan_from_system(system)
    X = wl.orbital_block(ng, range(2), 14, 0, device="cuda")
    HX = gpu_apply(env, plan, X)
    assert col_err(HX.cpu().numpy(), oracle.apply_h(system, X.cpu().numpy())) <= TOL
    plan.close()
