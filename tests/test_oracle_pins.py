"""Pins for the CPU oracle (oracle/rsdft_oracle.c) against things OTHER than itself:
the DFT definition by brute force, numpy.fft, closed forms, the paper's printed cut-offs
(tests/golden/paper_cutoffs.txt), textbook free-electron levels
(tests/golden/free_electron_levels.txt), scipy's spherical harmonics, symmetry and
invariants (north_star list; SURVEY 8(c) "Pins").  CPU only."""
import os

import numpy as np
import pytest
import scipy.linalg
import scipy.special

from oracle import oracle
from paper_2512_04447_b200 import workloads as wl

GOLD = os.path.join(os.path.dirname(__file__), "golden")
RNG = np.random.default_rng(1234)


def crandn(*shape):
    return (RNG.standard_normal(shape) + 1j * RNG.standard_normal(shape)) * np.sqrt(0.5)


def relerr(a, b):
    return np.max(np.abs(a - b)) / np.max(np.abs(b))


# ----------------------------------------------------------------------------- FFT
def test_fft_bruteforce_full_matrix_small_odd_grid():
    """Full O(Ng^2) DFT definition, non-cubic grid with odd and even lengths."""
    n = (6, 5, 4)
    ng = int(np.prod(n))
    ix, iy, iz = np.meshgrid(*[np.arange(k) for k in n], indexing="ij")
    ix, iy, iz = ix.ravel(), iy.ravel(), iz.ravel()
    phase = (np.outer(ix, ix) / n[0] + np.outer(iy, iy) / n[1] + np.outer(iz, iz) / n[2])
    F = np.exp(-2j * np.pi * phase)                       # F[k, r]
    x = crandn(3, ng)
    assert relerr(oracle.fft3d(n, x, -1), x @ F.T) < 1e-13
    assert relerr(oracle.fft3d(n, x, +1), (x @ F.conj().T) / ng) < 1e-13


def test_fft_definition_16cubed():
    """16^3 (config 0's grid): the definition applied axis by axis with explicit DFT matrices."""
    n = (16, 16, 16)
    x = crandn(int(np.prod(n)))
    Fm = np.exp(-2j * np.pi * np.outer(np.arange(16), np.arange(16)) / 16)
    ref = np.einsum("ax,by,cz,xyz->abc", Fm, Fm, Fm, x.reshape(n), optimize=True).ravel()
    assert relerr(oracle.fft3d(n, x, -1), ref) < 1e-13


@pytest.mark.parametrize("n", [(48, 4, 3), (3, 96, 2), (2, 3, 112), (128, 2, 2), (14, 24, 18), (32, 32, 32)])
def test_fft_vs_numpy_library(n):
    """Mixed-radix path (lengths whose recursion ends in direct DFTs of 3, 7, 9, 12, 14) vs numpy.fft."""
    x = crandn(2, int(np.prod(n)))
    ref = np.fft.fftn(x.reshape((2,) + n), axes=(1, 2, 3)).reshape(2, -1)
    assert relerr(oracle.fft3d(n, x, -1), ref) < 1e-13
    refi = np.fft.ifftn(x.reshape((2,) + n), axes=(1, 2, 3)).reshape(2, -1)
    assert relerr(oracle.fft3d(n, x, +1), refi) < 1e-13


def test_fft_invariants():
    n = (12, 16, 10)
    ng = int(np.prod(n))
    x = crandn(ng)
    X = oracle.fft3d(n, x, -1)
    assert relerr(oracle.fft3d(n, X, +1), x) < 1e-14                       # inverse(forward) = id
    assert abs(np.vdot(X, X).real / ng - np.vdot(x, x).real) < 1e-12 * ng   # Parseval
    d = np.zeros(ng, complex); d[0] = 1.0
    assert relerr(oracle.fft3d(n, d, -1), np.ones(ng)) < 1e-15              # delta -> constant
    # shift theorem: delta at (1,0,0) -> e^{-2 pi i kx/nx}
    d = np.zeros(n, complex); d[1, 0, 0] = 1.0
    ref = np.exp(-2j * np.pi * np.arange(n[0]) / n[0])[:, None, None] * np.ones(n)
    assert relerr(oracle.fft3d(n, d.ravel(), -1), ref.ravel()) < 1e-14   # numpy exp error on the ref side


# ------------------------------------------------------------------------- kinetic
def test_paper_cutoffs_fix_hartree_units():
    """max_k t(k) along one axis = 1/2 (pi/h)^2 Ha = (pi/h)^2 / 2 ... in Ry: (pi/h)^2.
    The paper prints 86.7 Ry for 60^3 and 110.7 Ry for 80^3."""
    for line in open(os.path.join(GOLD, "paper_cutoffs.txt")):
        if line.startswith("#") or not line.strip():
            continue
        npts, L, ecut_ry = line.split()
        npts, L, ecut_ry = int(npts), float(L), float(ecut_ry)
        n = (npts, 2, 2)
        t = oracle.kinetic_table(n, (L, 1.0, 1.0)).reshape(n)
        e_ha = t[:, 0, 0].max()          # Nyquist along x only
        assert abs(2.0 * e_ha - ecut_ry) / ecut_ry < 5e-3


@pytest.mark.parametrize("n,L", [((16, 16, 16), (10.0, 10.0, 10.0)), ((12, 10, 6), (7.0, 6.0, 5.0))])
def test_plane_waves_are_kinetic_eigenvectors(n, L):
    """e^{iG.r} is an eigenvector with eigenvalue |G|^2/2 (north_star), including the
    Nyquist index and negative frequencies."""
    system = dict(n=n, len=L)
    grids = np.meshgrid(*[np.arange(k) for k in n], indexing="ij")
    ks = [(0, 0, 0), (1, 0, 0), (0, 2, 0), (n[0] - 1, 0, 1), (n[0] // 2, n[1] // 2, n[2] // 2),
          (3, n[1] - 2, n[2] // 2), (n[0] // 2 + 1, 1, n[2] - 1)]
    X, ev = [], []
    for k in ks:
        X.append(np.exp(2j * np.pi * sum(k[a] * grids[a] / n[a] for a in range(3))).ravel())
        kap = [k[a] if 2 * k[a] < n[a] else k[a] - n[a] for a in range(3)]
        ev.append(0.5 * sum((2 * np.pi * kap[a] / L[a]) ** 2 for a in range(3)))
    X = np.array(X)
    HX = oracle.apply_h(system, X)
    for x, hx, e in zip(X, HX, ev):
        assert np.max(np.abs(hx - e * x)) < 1e-13 * max(1.0, e)


def test_cosine_potential_closed_form():
    """v = 2 V0 cos(g x), psi = e^{iGx}: H psi = G^2/2 psi + V0 (e^{i(G+g)x} + e^{i(G-g)x}) exactly."""
    n, L = (24, 6, 4), (9.0, 5.0, 4.0)
    x = np.arange(n[0]) * L[0] / n[0]
    g, G, V0 = 2 * np.pi / L[0] * 2, 2 * np.pi / L[0] * 5, 0.7
    ones = np.ones(n)
    v = (2 * V0 * np.cos(g * x))[:, None, None] * ones
    psi = np.exp(1j * G * x)[:, None, None] * ones
    ref = (G * G / 2 * np.exp(1j * G * x) + V0 * (np.exp(1j * (G + g) * x) + np.exp(1j * (G - g) * x)))[:, None, None] * ones
    HX = oracle.apply_h(dict(n=n, len=L, vloc=v.ravel()), psi.reshape(1, -1))
    assert relerr(HX[0], ref.ravel()) < 1e-13


# ---------------------------------------------------------------------- projectors
def _real_ylm_scipy(l, m, d):
    """Real spherical harmonics from scipy's complex ones (library pin of normalisation,
    ordering and sign: Y_{l,-|m|} ~ sin(|m| phi), Y_{l,|m|} ~ cos(|m| phi), no Condon-Shortley
    phase in the real form)."""
    r = np.linalg.norm(d, axis=-1)
    theta = np.arccos(np.clip(d[..., 2] / r, -1, 1))       # polar
    phi = np.arctan2(d[..., 1], d[..., 0])                 # azimuth
    if hasattr(scipy.special, "sph_harm_y"):
        Y = scipy.special.sph_harm_y(l, abs(m), theta, phi)
    else:  # pragma: no cover
        Y = scipy.special.sph_harm(abs(m), l, phi, theta)
    if m == 0:
        return Y.real
    if m > 0:
        return np.sqrt(2) * (-1) ** m * Y.real
    return np.sqrt(2) * (-1) ** m * Y.imag


def _dense_beta(system, a):
    """beta_i(r) on ALL grid points by an independent numpy construction (zeros outside the sphere)."""
    n, L = system["n"], system["len"]
    sp = system["species"][system["species_of"][a]]
    R = system["pos"][a]
    grids = np.meshgrid(*[np.arange(k) * (L[i] / k) for i, k in enumerate(n)], indexing="ij")
    d = np.stack([g - R[i] for i, g in enumerate(grids)], axis=-1)
    d = d - np.array(L) * np.round(d / np.array(L))
    r = np.linalg.norm(d, axis=-1)
    inside = (d ** 2).sum(-1) < sp["rc"] ** 2
    out = []
    for i, (l, m) in enumerate(zip(sp["l"], sp["m"])):
        if sp.get("radial_kind", 0) == 0:
            f = np.exp(-sp["alpha"][i] * r * r)
        else:
            f = np.interp(r, np.arange(sp["radial"].shape[1]) * sp["dr"], sp["radial"][i], right=0.0)
        with np.errstate(invalid="ignore", divide="ignore"):
            y = _real_ylm_scipy(int(l), int(m), d)
        y = np.where(r == 0, (0.5 / np.sqrt(np.pi)) if l == 0 else 0.0, y)
        out.append(np.where(inside, f * y, 0.0).ravel())
    return np.array(out)


@pytest.mark.parametrize("kind", [0, 1])
def test_sphere_tables_vs_dense_numpy_scipy(kind):
    system = wl.small_system(radial_kind=kind)
    for a in range(len(system["pos"])):
        idx, beta = oracle.sphere(system["n"], system["len"], system["pos"][a], system["species"][0])
        dense = _dense_beta(system, a)
        mine = np.zeros_like(dense)
        mine[:, idx] = beta
        assert len(idx) == np.count_nonzero(np.abs(dense[0]))      # s projector never vanishes inside
        assert np.max(np.abs(mine - dense)) < 1e-14
        assert len(idx) > 50


def test_apply_h_vs_dense_operator():
    """Whole H on a small non-cubic system against dense linear algebra: T from numpy.fft,
    V_loc pointwise, V_NL = dV * B^T D B with B built densely on all grid points."""
    system = wl.small_system()
    n, L = system["n"], system["len"]
    ng = int(np.prod(n))
    X = crandn(5, ng)
    dV = np.prod([L[i] / n[i] for i in range(3)])
    kap = [np.fft.fftfreq(n[i], d=1.0 / n[i]) for i in range(3)]
    KX, KY, KZ = np.meshgrid(*kap, indexing="ij")
    t = 0.5 * ((2 * np.pi * KX / L[0]) ** 2 + (2 * np.pi * KY / L[1]) ** 2 + (2 * np.pi * KZ / L[2]) ** 2)
    ref = np.fft.ifftn(t * np.fft.fftn(X.reshape((5,) + n), axes=(1, 2, 3)), axes=(1, 2, 3)).reshape(5, -1)
    ref = ref + system["vloc"] * X
    sp = system["species"][0]
    for a in range(len(system["pos"])):
        B = _dense_beta(system, a)                      # [nproj, Ng]
        p = dV * (X @ B.T)                              # [ncol, nproj]
        ref = ref + (p @ sp["D"].T) @ B
    HX, p_orc = oracle.apply_h(system, X, return_p=True)
    assert relerr(HX, ref) < 1e-13
    B0 = _dense_beta(system, 0)
    assert relerr(p_orc[0].T, dV * (X @ B0.T)) < 1e-13


def test_h_is_hermitian_under_plain_inner_product():
    """<x|Hy> = conj(<y|Hx>) (north_star)."""
    system = wl.small_system()
    ng = int(np.prod(system["n"]))
    X = crandn(4, ng)
    HX = oracle.apply_h(system, X)
    M = X.conj() @ HX.T            # M[i,j] = <x_i | H x_j>
    assert np.max(np.abs(M - M.conj().T)) < 1e-12 * np.max(np.abs(M))


def test_translation_covariance():
    """Shifting psi, v and the atoms by an integer grid vector shifts H psi identically
    (exercises the periodic wrap of the sphere lists)."""
    system = wl.small_system()
    n, L = system["n"], system["len"]
    ng = int(np.prod(n))
    X = crandn(2, ng)
    HX = oracle.apply_h(system, X)
    s = (5, 7, 3)
    shifted = dict(system)
    shifted["pos"] = np.mod(system["pos"] + np.array([s[i] * L[i] / n[i] for i in range(3)]), np.array(L))
    roll = lambda a: np.roll(a.reshape((-1,) + n), s, axis=(1, 2, 3)).reshape(a.shape[0] if a.ndim == 2 else 1, -1)
    shifted["vloc"] = roll(system["vloc"][None, :])[0]
    HXs = oracle.apply_h(shifted, roll(X))
    assert relerr(HXs, roll(HX)) < 1e-12


def test_nonlocal_energy_identity_and_null_space():
    """<psi|V_NL psi> = (1/dV) sum_a p_a^H D p_a;  psi supported outside every sphere -> V_NL psi = 0."""
    system = wl.small_system(n=(16, 16, 16), L=(10.0, 10.0, 10.0), natom=2, rc=2.0)
    n, L = system["n"], system["len"]
    ng = int(np.prod(n))
    dV = np.prod([L[i] / n[i] for i in range(3)])
    bare = dict(n=n, len=L, vloc=system["vloc"])
    X = crandn(3, ng)
    HX, p = oracle.apply_h(system, X, return_p=True)
    VX = HX - oracle.apply_h(bare, X)
    D = system["species"][0]["D"]
    for c in range(3):
        lhs = np.vdot(X[c], VX[c])
        rhs = sum(np.vdot(p[a, :, c], D @ p[a, :, c]) for a in range(p.shape[0])) / dV
        assert abs(lhs - rhs) < 1e-12 * abs(rhs)
    mask = np.ones(ng, bool)
    for a in range(len(system["pos"])):
        idx, _ = oracle.sphere(n, L, system["pos"][a], system["species"][0])
        mask[idx] = False
    Xo = X * mask
    VXo = oracle.apply_h(system, Xo) - oracle.apply_h(bare, Xo)
    assert np.max(np.abs(VXo)) == 0.0


def test_cubic_symmetry_orthogonality_atom_on_grid_point():
    """Atom on a grid point of a cubic grid: B B^T is diagonal, the three p norms are equal,
    {xy,yz,xz} equal, {z^2, x^2-y^2} equal (cubic harmonics); Y_lm(0)=0 for l>0."""
    n, L = (20, 20, 20), (8.0, 8.0, 8.0)
    sp = dict(rc=2.2, l=wl._L_SPD, m=wl._M_SPD, radial_kind=0, alpha=np.full(9, 0.8), D=np.eye(9))
    R = np.array([3, 7, 19]) * (L[0] / n[0])
    idx, beta = oracle.sphere(n, L, R, sp)
    G = beta @ beta.T
    off = G - np.diag(np.diag(G))
    assert np.max(np.abs(off)) < 1e-13 * np.max(np.diag(G))
    d = np.diag(G)
    assert np.ptp(d[1:4]) < 1e-13 * d[1]
    assert np.ptp(d[[4, 5, 7]]) < 1e-13 * d[4]
    assert np.ptp(d[[6, 8]]) < 1e-13 * d[6]
    centre = int((3 * n[1] + 7) * n[2] + 19)
    j = int(np.nonzero(idx == centre)[0][0])
    assert beta[0, j] == pytest.approx(0.5 / np.sqrt(np.pi), rel=1e-15)
    assert np.all(beta[1:, j] == 0.0)


def test_projector_norms_approach_continuum_integral():
    """dV sum beta_i^2 -> int_0^rc f(r)^2 r^2 dr as h -> 0 (orthonormal Y_lm); loose, 1e-2."""
    n, L = (64, 64, 64), (6.0, 6.0, 6.0)
    alpha, rc = 1.3, 2.2
    sp = dict(rc=rc, l=wl._L_SPD, m=wl._M_SPD, radial_kind=0, alpha=np.full(9, alpha), D=np.eye(9))
    idx, beta = oracle.sphere(n, L, np.array([3.01, 2.97, 3.05]), sp)
    dV = (L[0] / n[0]) ** 3
    r = np.linspace(0, rc, 200001)
    exact = np.trapezoid(np.exp(-2 * alpha * r * r) * r * r, r)
    got = dV * (beta ** 2).sum(1)
    assert np.max(np.abs(got - exact)) < 1e-2 * exact


def test_radial_table_reproduces_linear_function_exactly():
    """kind 1 (linear interpolation): a table sampled from a + b r gives beta = (a + b|d|) Y_lm."""
    n, L = (12, 12, 12), (6.0, 6.0, 6.0)
    nr, dr = 40, 0.06
    r = np.arange(nr) * dr
    sp = dict(rc=2.0, l=[0, 1], m=[0, 0], radial_kind=1, dr=dr, radial=np.stack([1.0 - 0.25 * r, 0.5 + 0.1 * r]),
              D=np.eye(2))
    R = np.array([2.9, 3.2, 3.1])
    idx, beta = oracle.sphere(n, L, R, sp)
    system = dict(n=n, len=L, pos=R[None, :], species_of=np.zeros(1, np.int32), species=[sp])
    dense = _dense_beta(system, 0)
    assert np.max(np.abs(dense[:, idx] - beta)) < 1e-14
    g = np.stack(np.unravel_index(idx, n), -1) * (L[0] / n[0]) - R
    g = g - L[0] * np.round(g / L[0])
    rr = np.linalg.norm(g, axis=1)
    assert np.max(np.abs(beta[0] - (1.0 - 0.25 * rr) * 0.5 / np.sqrt(np.pi))) < 1e-14


# ---------------------------------------------------------------------------- Gram
def test_gram_vs_matmul_and_invariants():
    ng, n = 3000, 7
    Y, HY = crandn(n, ng), crandn(n, ng)
    H, S = oracle.gram(Y, HY)
    assert relerr(S, Y.conj() @ Y.T) < 1e-14         # S[i,j] = sum_r conj(Y[r,i]) Y[r,j]
    assert relerr(H, Y.conj() @ HY.T) < 1e-14
    assert np.max(np.abs(S - S.conj().T)) < 1e-15 * np.max(np.abs(S))
    scipy.linalg.cholesky(S)                           # Hermitian positive definite
    assert np.all(np.abs(np.diag(S).imag) < 1e-15 * ng)


def test_gram_plane_waves_give_ng_identity_and_kinetic_diagonal():
    n, L = (8, 6, 10), (5.0, 4.0, 6.0)
    ng = int(np.prod(n))
    grids = np.meshgrid(*[np.arange(k) for k in n], indexing="ij")
    ks = [(0, 0, 0), (1, 0, 0), (7, 5, 9), (4, 3, 5), (2, 1, 3)]
    Y = np.array([np.exp(2j * np.pi * sum(k[a] * grids[a] / n[a] for a in range(3))).ravel() for k in ks])
    HY = oracle.apply_h(dict(n=n, len=L), Y)
    H, S = oracle.gram(Y, HY)
    t = oracle.kinetic_table(n, L).reshape(n)
    assert np.max(np.abs(S - ng * np.eye(len(ks)))) < 1e-12 * ng
    assert np.max(np.abs(H - ng * np.diag([t[k] for k in ks]))) < 1e-12 * ng * t.max()


def test_free_electron_ritz_values():
    """V = 0, no projectors, Y = random mixes of the 27 lowest plane waves: the generalized
    eigenvalues of (H_sub, S_sub) are the free-electron levels (north_star)."""
    n, L = (16, 16, 16), (10.0, 10.0, 10.0)
    levels = []
    for line in open(os.path.join(GOLD, "free_electron_levels.txt")):
        if line.startswith("#") or not line.strip():
            continue
        k2, deg, e = line.split()
        levels += [float(e)] * int(deg)
    levels = np.array(levels[:27])        # |kappa|^2 <= 3: 1 + 6 + 12 + 8
    grids = np.meshgrid(*[np.arange(k) for k in n], indexing="ij")
    pw = []
    for kx in (-1, 0, 1):
        for ky in (-1, 0, 1):
            for kz in (-1, 0, 1):
                pw.append(np.exp(2j * np.pi * (kx * grids[0] + ky * grids[1] + kz * grids[2]) / 16).ravel())
    pw = np.array(pw)
    Y = crandn(27, 27) @ pw
    HY = oracle.apply_h(dict(n=n, len=L), Y)
    H, S = oracle.gram(Y, HY)
    assert np.max(np.abs(H - H.conj().T)) < 1e-12 * np.max(np.abs(H))   # Hermitian to round-off
    w = scipy.linalg.eigh(H, S, eigvals_only=True)
    assert np.max(np.abs(np.sort(w) - np.sort(levels))) < 1e-10


def test_config0_system_shapes():
    s = wl.make_system(0)
    assert s["n"] == (16, 16, 16) and len(s["pos"]) == 2 and s["vloc"].shape == (4096,)
    idx, beta = oracle.sphere(s["n"], s["len"], s["pos"][0], s["species"][0])
    assert 120 <= len(idx) <= 160 and beta.shape[0] == 4     # ~137 points per sphere


# ------------------------------------------------------------------ NEXT-2: Rayleigh-Ritz update Out = Y C
def test_rotate_pins():
    """oracle.rotate against what the mathematics fixes: a permutation matrix reorders columns exactly, a diagonal
    matrix scales them, an explicit triple loop on a tiny case, linearity, and the Gram identity
    (YC)^H (YC) = C^H (Y^H Y) C that ties it to oracle.gram (a transposed or conjugated C fails at least one)."""
    rng = np.random.default_rng(5)
    n, m, ng = 7, 4, 60
    Y = rng.standard_normal((n, ng)) + 1j * rng.standard_normal((n, ng))
    perm = [3, 0, 6, 2]
    P = np.zeros((n, m)); P[perm, range(m)] = 1.0
    assert np.array_equal(oracle.rotate(Y, P), Y[perm])
    d = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    assert np.allclose(oracle.rotate(Y, np.diag(d)), d[:, None] * Y, rtol=1e-15, atol=0)
    C = rng.standard_normal((n, m)) + 1j * rng.standard_normal((n, m))
    out = oracle.rotate(Y, C)
    brute = np.zeros((m, ng), dtype=complex)
    for j in range(m):
        for r in range(ng):
            for c in range(n):
                brute[j, r] += Y[c, r] * C[c, j]
    assert np.max(np.abs(out - brute)) <= 1e-14 * np.max(np.abs(brute))
    C2 = rng.standard_normal((n, m)) + 1j * rng.standard_normal((n, m))
    lin = oracle.rotate(Y, 0.3 * C - 2j * C2)
    assert np.max(np.abs(lin - (0.3 * out - 2j * oracle.rotate(Y, C2)))) <= 1e-14 * np.max(np.abs(lin))
    _, S = oracle.gram(Y, None)
    _, S_rot = oracle.gram(out, None)
    ref = C.conj().T @ S @ C
    assert np.max(np.abs(S_rot - ref)) <= 1e-13 * np.max(np.abs(ref))
