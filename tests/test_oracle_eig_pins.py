"""Pins for the NEXT-1 / NEXT-2 oracle (oracle/rsdft_eig_oracle.c, oracle.rotate2): the generalized Hermitian
eigen-solve by the paper's route (eq. 1: S = L L^H, K = L^-1 H L^-H by two triangular solves,
K Z = Z Lambda, X = L^-H Z) and the Rayleigh-Ritz update with residual, checked against what the mathematics
fixes: uniqueness of the Cholesky factor, closed forms for 2 x 2, pencils built from a prescribed spectrum,
eq. 1's identity against the library's generalized solver, the free-electron levels of the golden file.
Each pin is chosen so that a plausible slip (L^H instead of L, a missing conjugate, a transposed solve, an
unsorted spectrum) fails it.  CPU only."""
import os

import numpy as np
import pytest
import scipy.linalg

from oracle import oracle

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def crandn(rng, *shape):
    return (rng.standard_normal(shape) + 1j * rng.standard_normal(shape)) * np.sqrt(0.5)


def hpd(rng, n, cond=50.0):
    """Hermitian positive definite with a prescribed condition number"""
    Q, _ = np.linalg.qr(crandn(rng, n, n))
    d = np.geomspace(1.0, cond, n)
    S = (Q * d) @ Q.conj().T
    return 0.5 * (S + S.conj().T)


def herm(rng, n):
    A = crandn(rng, n, n)
    return 0.5 * (A + A.conj().T)


# ----------------------------------------------------------------------------- Cholesky
def test_potrf_2x2_closed_form():
    a, d, b = 4.0, 3.0, 1.0 - 2.0j
    S = np.array([[a, b], [np.conj(b), d]])
    L = oracle.potrf(S)
    want = np.array([[2.0, 0.0], [np.conj(b) / 2.0, np.sqrt(d - abs(b) ** 2 / a)]])
    assert np.max(np.abs(L - want)) < 1e-15


@pytest.mark.parametrize("n", [1, 5, 33, 150])
def test_potrf_is_the_unique_lower_factor(n):
    rng = np.random.default_rng(n)
    S = hpd(rng, n)
    L = oracle.potrf(S)
    assert np.all(np.triu(L, 1) == 0.0)                          # lower
    assert np.all(np.diagonal(L).imag == 0.0) and np.all(np.diagonal(L).real > 0.0)
    assert np.max(np.abs(L @ L.conj().T - S)) < 1e-15 * np.max(np.abs(S)) * n
    assert np.max(np.abs(L - np.linalg.cholesky(S))) < 1e-14 * np.max(np.abs(L)) * max(1, n // 8)   # library cross-check


def test_potrf_reads_only_the_lower_triangle_and_rejects_indefinite():
    rng = np.random.default_rng(3)
    S = hpd(rng, 12)
    junk = S.copy()
    junk[np.triu_indices(12, 1)] = 99.0
    assert np.array_equal(oracle.potrf(junk), oracle.potrf(S))
    bad = S.copy()
    bad[5, 5] = -1.0
    with pytest.raises(np.linalg.LinAlgError):
        oracle.potrf(bad)


# ----------------------------------------------------------------------------- K = L^-1 H L^-H
@pytest.mark.parametrize("n", [2, 17, 96])
def test_reduce_inverts_back_and_keeps_the_spectrum(n):
    """L K L^H = H (pins both substitutions: L^H K L = H, or K = L^-H H L^-1, fail), K Hermitian, and eq. 1's
    identity: eigenvalues of K = generalized eigenvalues of (H, S) (library generalized solver)."""
    rng = np.random.default_rng(10 + n)
    H, S = herm(rng, n), hpd(rng, n)
    L = oracle.potrf(S)
    K = oracle.reduce_to_standard(H, S)
    assert np.max(np.abs(L @ K @ L.conj().T - H)) < 1e-13 * np.max(np.abs(H))
    assert np.max(np.abs(K - K.conj().T)) < 1e-14 * np.max(np.abs(K))
    w_lib = scipy.linalg.eigh(H, S, eigvals_only=True)
    w_k = np.linalg.eigvalsh(0.5 * (K + K.conj().T))
    assert np.max(np.abs(w_k - w_lib)) < 1e-12 * np.max(np.abs(w_lib))


def test_reduce_with_identity_overlap_and_diagonal_overlap():
    rng = np.random.default_rng(4)
    H = herm(rng, 9)
    assert np.max(np.abs(oracle.reduce_to_standard(H, np.eye(9)) - H)) == 0.0
    d = rng.uniform(0.5, 2.0, 9)
    K = oracle.reduce_to_standard(H, np.diag(d * d))
    assert np.max(np.abs(K - H / np.outer(d, d))) < 1e-15 * np.max(np.abs(K))


# ----------------------------------------------------------------------------- standard problem: Jacobi
def test_jacobi_2x2_closed_form():
    a, d, b = 1.5, -0.5, 0.75 + 0.25j
    w, Z = oracle.jacobi_eigh(np.array([[a, b], [np.conj(b), d]]))
    mid, rad = 0.5 * (a + d), np.sqrt((0.5 * (a - d)) ** 2 + abs(b) ** 2)
    assert np.max(np.abs(w - [mid - rad, mid + rad])) < 1e-15
    assert np.max(np.abs(Z.conj().T @ Z - np.eye(2))) < 1e-15


@pytest.mark.parametrize("n", [1, 3, 24, 120])
def test_jacobi_prescribed_spectrum_with_degenerate_levels(n):
    rng = np.random.default_rng(20 + n)
    w0 = np.sort(rng.standard_normal(n))
    if n >= 24:
        w0[3:9] = w0[3]                        # a six-fold level, like the free-electron shells
        w0[10:12] = w0[10]
        w0 = np.sort(w0)
    Q, _ = np.linalg.qr(crandn(rng, n, n))
    K = (Q * w0) @ Q.conj().T
    K = 0.5 * (K + K.conj().T)
    w, Z = oracle.jacobi_eigh(K)
    scale = max(1.0, np.max(np.abs(w0)))
    assert np.all(np.diff(w) >= 0.0)                                         # ascending
    assert np.max(np.abs(w - w0)) < 1e-14 * scale
    assert np.max(np.abs(Z.conj().T @ Z - np.eye(n))) < 1e-14                # unitary
    assert np.max(np.abs(K @ Z - Z * w)) < 1e-14 * scale * max(1, n // 8)    # eigenpairs
    assert np.max(np.abs(w - np.linalg.eigvalsh(K))) < 1e-13 * scale         # library cross-check


def test_jacobi_on_a_diagonal_matrix_is_a_sort():
    d = np.array([3.0, -1.0, 2.0, -1.0, 0.0])
    w, Z = oracle.jacobi_eigh(np.diag(d))
    assert np.array_equal(w, np.sort(d))
    assert np.array_equal(np.abs(Z), np.eye(5)[:, np.argsort(d, kind="stable")])


# ----------------------------------------------------------------------------- back substitution
def test_backsolve_inverts_l_dagger():
    rng = np.random.default_rng(6)
    L = oracle.potrf(hpd(rng, 30))
    Z = crandn(rng, 30, 7)
    Cm = oracle.backsolve(L, Z)
    assert np.max(np.abs(L.conj().T @ Cm - Z)) < 1e-14 * np.max(np.abs(Z))
    assert np.max(np.abs(Cm - scipy.linalg.solve_triangular(L.conj().T, Z, lower=False))) < 1e-13 * np.max(np.abs(Cm))


# ----------------------------------------------------------------------------- the whole of eq. 1
@pytest.mark.parametrize("solver", ["jacobi", "heevd"])
@pytest.mark.parametrize("n,m", [(2, 2), (24, 8), (75, 25), (96, 96)])
def test_subspace_eig_recovers_a_prescribed_pencil(solver, n, m):
    """H = B^H diag(w) B, S = B^H B: the generalized eigenvalues are exactly w and the eigenvector of w_i is
    B^-1 e_i (up to a phase).  Independent of any eigen-solver."""
    rng = np.random.default_rng(100 + n)
    B = crandn(rng, n, n) + 2.0 * np.eye(n)
    w0 = np.sort(rng.uniform(-1.0, 3.0, n))
    H = B.conj().T @ np.diag(w0) @ B
    S = B.conj().T @ B
    H, S = 0.5 * (H + H.conj().T), 0.5 * (S + S.conj().T)
    lam, Cm, L, K = oracle.subspace_eig(H, S, m, solver=solver, return_factors=True)
    cond = np.linalg.cond(S)
    assert lam.shape == (m,) and Cm.shape == (n, m)
    assert np.max(np.abs(lam - w0[:m])) < 1e-15 * cond * 10
    assert np.max(np.abs(Cm.conj().T @ S @ Cm - np.eye(m))) < 1e-15 * cond * 10       # S-orthonormal
    assert np.max(np.abs(H @ Cm - S @ Cm * lam)) < 1e-14 * np.max(np.abs(H)) * np.sqrt(cond)
    X0 = np.linalg.inv(B)[:, :m]                                                     # exact eigenvectors (unnormalised)
    X0 = X0 / np.sqrt(np.real(np.einsum("ij,ij->j", X0.conj(), S @ X0)))
    overlap = np.abs(np.einsum("ij,ij->j", X0.conj(), S @ Cm))                       # |<x0_i|S|c_i>| = 1 (gaps are O(1/n))
    gaps = np.min(np.diff(w0))
    assert np.max(np.abs(overlap - 1.0)) < 1e-13 * cond / max(gaps, 1e-3)
    assert np.max(np.abs(L @ L.conj().T - S)) < 1e-14 * np.max(np.abs(S)) and np.all(np.triu(L, 1) == 0.0)
    assert np.max(np.abs(L @ K @ L.conj().T - H)) < 1e-13 * np.max(np.abs(H)) * np.sqrt(cond)


def test_subspace_eig_jacobi_and_heevd_routes_agree_and_match_the_library():
    rng = np.random.default_rng(77)
    n = 60
    H, S = herm(rng, n), hpd(rng, n, cond=200.0)
    l1, C1 = oracle.subspace_eig(H, S)
    l2, C2 = oracle.subspace_eig(H, S, solver="heevd")
    w = scipy.linalg.eigh(H, S, eigvals_only=True)
    assert np.max(np.abs(l1 - w)) < 1e-12 * np.max(np.abs(w))
    assert np.max(np.abs(l2 - l1)) < 1e-12 * np.max(np.abs(w))
    # eigenvectors agree up to a phase per column (this spectrum is simple)
    ph = np.einsum("ij,ij->j", C1.conj(), S @ C2)
    assert np.max(np.abs(np.abs(ph) - 1.0)) < 1e-10


def test_subspace_eig_rejects_an_indefinite_overlap():
    rng = np.random.default_rng(8)
    S = hpd(rng, 6)
    S[2, 2] = -0.1
    with pytest.raises(np.linalg.LinAlgError):
        oracle.subspace_eig(herm(rng, 6), S)


def test_free_electron_levels_through_the_whole_oracle_chain():
    """apply_h -> gram -> subspace_eig with V = 0 and no projectors on random mixes of the 27 lowest plane waves:
    the Ritz values are the free-electron levels of tests/golden/free_electron_levels.txt (north_star), the
    Ritz vectors are S-orthonormal, and the rotated block has zero residual (oracle.rotate2)."""
    n, L = (16, 16, 16), (10.0, 10.0, 10.0)
    levels = []
    for line in open(os.path.join(GOLD, "free_electron_levels.txt")):
        if line.startswith("#") or not line.strip():
            continue
        _, deg, e = line.split()
        levels += [float(e)] * int(deg)
    levels = np.array(levels[:27])
    grids = np.meshgrid(*[np.arange(k) for k in n], indexing="ij")
    pw = np.array([np.exp(2j * np.pi * (kx * grids[0] + ky * grids[1] + kz * grids[2]) / 16).ravel()
                   for kx in (-1, 0, 1) for ky in (-1, 0, 1) for kz in (-1, 0, 1)])
    rng = np.random.default_rng(9)
    Y = (crandn(rng, 27, 27) + 2.0 * np.eye(27)) @ pw
    HY = oracle.apply_h(dict(n=n, len=L), Y)
    H, S = oracle.gram(Y, HY)
    lam, Cm = oracle.subspace_eig(H, S)
    assert np.max(np.abs(lam - levels)) < 1e-11
    assert np.max(np.abs(Cm.conj().T @ S @ Cm - np.eye(27))) < 1e-11
    Xn, HXn, R = oracle.rotate2(Y, HY, Cm[:, :7], lam[:7])
    assert np.max(np.abs(R)) < 1e-11 * np.max(np.abs(Xn))                 # exact eigenpairs: zero residual
    assert np.max(np.abs(oracle.apply_h(dict(n=n, len=L), Xn) - HXn)) < 1e-12 * np.max(np.abs(HXn))


# ----------------------------------------------------------------------------- NEXT-2: rotate2
def test_rotate2_pins():
    """X' and HX' equal oracle.rotate of each operand (whose own pins are in test_oracle_pins.py), R is the plain
    column-wise combination written out as loops, and everything is linear in C."""
    rng = np.random.default_rng(12)
    n, m, ng = 6, 4, 50
    Y, HY = crandn(rng, n, ng), crandn(rng, n, ng)
    Cm, lam = crandn(rng, n, m), rng.standard_normal(m)
    X, HX, R = oracle.rotate2(Y, HY, Cm, lam)
    assert np.array_equal(X, oracle.rotate(Y, Cm)) and np.array_equal(HX, oracle.rotate(HY, Cm))
    ref = np.zeros((m, ng), dtype=complex)
    for j in range(m):
        for r in range(ng):
            acc = 0.0
            for c in range(n):
                acc += (HY[c, r] - lam[j] * Y[c, r]) * Cm[c, j]
            ref[j, r] = acc
    assert np.max(np.abs(R - ref)) < 1e-14 * np.max(np.abs(ref))
    X2, HX2, R2 = oracle.rotate2(Y, HY, 2.0 * Cm, lam)
    assert np.allclose(R2, 2.0 * R, rtol=1e-15, atol=0) and np.allclose(X2, 2.0 * X, rtol=1e-15, atol=0)
    # lam = 0 gives R = HX'; a permutation matrix C picks columns exactly
    _, HX0, R0 = oracle.rotate2(Y, HY, Cm, np.zeros(m))
    assert np.array_equal(R0, HX0)
    P = np.zeros((n, 2)); P[[4, 1], [0, 1]] = 1.0
    Xp, HXp, Rp = oracle.rotate2(Y, HY, P, np.array([2.0, -3.0]))
    assert np.array_equal(Xp, Y[[4, 1]])
    assert np.allclose(Rp, HY[[4, 1]] - np.array([[2.0], [-3.0]]) * Y[[4, 1]], rtol=4e-16, atol=1e-15)
