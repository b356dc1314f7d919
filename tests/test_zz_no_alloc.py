"""rsdft_subspace_gram_static: the Gram entry point that allocates nothing (its scratch is a file-scope static __device__
array inside librsdft.so) against the existing rsdft_subspace_gram on the same seeded inputs, on calls in a row that
share the scratch.  Bar as in test_gpu_parity.py (R16): normwise 1e-12 per matrix; bit for bit where the
static scratch holds the K split the existing path takes.

This file is collected last on purpose (pytest -x: a failure here hides no other test) and does not depend
on anything the other test files leave behind: it passes alone in a fresh process and after them."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL = 1e-12


@pytest.fixture(scope="module")
def env():
    import torch
    from paper_2512_04447_b200 import rsdft, workloads
    assert torch.cuda.is_available()
    rsdft.load()          # fails loudly if the extension is missing
    return dict(torch=torch, rsdft=rsdft, wl=workloads)


def mat_err(a, b):
    a, b = a.cpu().numpy(), b.cpu().numpy()
    return float(np.max(np.abs(a - b)) / np.max(np.abs(b)))


def nan_matrix(torch, n, ld=None):
    return torch.full((n, n if ld is None else ld), float("nan"), dtype=torch.complex128, device="cuda")[:, :n]


def bits_equal(torch, a, b):
    return torch.equal(torch.view_as_real(a.resolve_conj().contiguous()), torch.view_as_real(b.resolve_conj().contiguous()))


def test_static_gram_matches_existing_path_on_calls_in_a_row(env):
    """Calls back to back on one stream, each with another n, other data and another output selection, so that every call
    finds the previous call's partial tiles and tile list in the scratch: ragged n (200 = 4 tiles + 8 columns), a smaller
    n after a larger one, S_sub alone, the Hermitian H mode, and the first case again."""
    torch, rsdft, wl = env["torch"], env["rsdft"], env["wl"]
    plan = rsdft.rsdft_plan_create((16, 32, 48), (5.0, 9.0, 14.0))
    ng = 16 * 32 * 48
    cases = [(200, 31, 0, True), (97, 32, 0, True), (200, 33, 0, False), (7, 34, 1, True), (96, 35, 1, True), (200, 31, 0, True)]
    first = None
    for n, seed, mode, want_h in cases:
        Y = wl.orbital_block(ng, range(n), seed, 0, device="cuda", ld=ng + 8)
        HY = wl.orbital_block(ng, range(n), seed, 1, device="cuda")
        rsdft.rsdft_plan_set_gram_mode(plan, mode)
        H_ref, S_ref = rsdft.rsdft_subspace_gram(plan, Y, HY, want_h=want_h)            # the existing path
        H = nan_matrix(torch, n, n + 3) if want_h else None                           # caller-owned outputs, lds > n
        S = nan_matrix(torch, n, n + 3)
        rsdft.rsdft_subspace_gram_static(plan, Y, HY if want_h else None, H, S)
        torch.cuda.synchronize()
        assert rsdft.rsdft_plan_info(plan)["last_launches"] == 3
        assert mat_err(S, S_ref) <= TOL
        assert bits_equal(torch, S, S_ref)              # same K split (it fits the scratch) => same bits
        assert bits_equal(torch, S, S.conj().T)         # exactly Hermitian, as the existing path's
        if want_h:
            assert mat_err(H, H_ref) <= TOL
            assert bits_equal(torch, H, H_ref)
        if first is None:
            first = (H.clone(), S.clone())
    assert bits_equal(torch, H, first[0]) and bits_equal(torch, S, first[1])           # the first case again, four calls later
    plan.close()


def test_static_gram_with_the_k_split_cut_to_the_scratch(env):
    """64^3 grid, n = 480 (155 tiles): the existing path splits K further than 64 MiB of partial tiles allow, the static
    entry point cuts the split down -- another summation order, so the comparison is the 1e-12 bar, twice in a row, and the
    second call must not take device memory."""
    torch, rsdft, wl = env["torch"], env["rsdft"], env["wl"]
    plan = rsdft.rsdft_plan_create((64, 64, 64), (12.0, 12.0, 12.0))
    ng, n = 64 ** 3, 480
    Y = wl.orbital_block(ng, range(n), 41, 0, device="cuda")
    HY = wl.orbital_block(ng, range(n), 41, 1, device="cuda")
    H_ref, S_ref = rsdft.rsdft_subspace_gram(plan, Y, HY)
    H, S = nan_matrix(torch, n), nan_matrix(torch, n)
    rsdft.rsdft_subspace_gram_static(plan, Y, HY, H, S)
    torch.cuda.synchronize()
    assert mat_err(H, H_ref) <= TOL and mat_err(S, S_ref) <= TOL
    H2, S2 = nan_matrix(torch, n), nan_matrix(torch, n)
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    rsdft.rsdft_subspace_gram_static(plan, Y, HY, H2, S2)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= free_before, "the call took device memory"
    assert mat_err(H2, H_ref) <= TOL and mat_err(S2, S_ref) <= TOL
    assert bits_equal(torch, H2, H) and bits_equal(torch, S2, S)                       # deterministic
    plan.close()


def test_static_gram_rejects_sizes_beyond_its_scratch(env):
    torch, rsdft = env["torch"], env["rsdft"]
    plan = rsdft.rsdft_plan_create((16, 16, 16), (5.0, 5.0, 5.0))
    n = rsdft.RSDFT_GRAM_STATIC_MAX_N + 1
    Y = torch.zeros((n, 4096), dtype=torch.complex128, device="cuda")
    S = nan_matrix(torch, n)
    with pytest.raises(rsdft.RsdftError) as e:
        rsdft.rsdft_subspace_gram_static(plan, Y, None, None, S)
    assert e.value.code == rsdft.RSDFT_UNSUPPORTED
    assert "RSDFT_GRAM_STATIC_MAX_N" in str(e.value) and "rsdft_subspace_gram" in str(e.value)
    torch.cuda.synchronize()
    assert bool(torch.isnan(S.real).all())                                             # nothing was launched
    # the largest size it takes: n = MAX_N, every tile of [S|H] at one K slab
    n = rsdft.RSDFT_GRAM_STATIC_MAX_N
    Y = torch.randn((n, 4096), dtype=torch.complex128, device="cuda", generator=torch.Generator(device="cuda").manual_seed(5))
    HY = torch.randn((n, 4096), dtype=torch.complex128, device="cuda", generator=torch.Generator(device="cuda").manual_seed(6))
    H_ref, S_ref = rsdft.rsdft_subspace_gram(plan, Y, HY)
    H, S = nan_matrix(torch, n), nan_matrix(torch, n)
    rsdft.rsdft_subspace_gram_static(plan, Y, HY, H, S)
    torch.cuda.synchronize()
    assert mat_err(H, H_ref) <= TOL and mat_err(S, S_ref) <= TOL
    plan.close()
