"""ctypes wrapper around oracle/rsdft_oracle.c -- TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this module.  It does not import paper_2512_04447_b200 and shares
nothing with the CUDA path; the arithmetic lives in rsdft_oracle.c (each function
there cites the passage it follows).

A "system" here is a plain dict (see paper_2512_04447_b200.workloads for the seeded
generators that produce it; that module holds no method arithmetic):
    n: (nx, ny, nz)   len: (Lx, Ly, Lz) bohr
    pos: [natom, 3] float64   species_of: [natom] int32
    species: list of dicts {rc, l, m, radial_kind, alpha | (dr, radial), D}
    vloc: [Ng] float64 or None
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "rsdft_oracle.c")
_SRCS = [_SRC, os.path.join(_HERE, "rsdft_eig_oracle.c")]
_LIB = os.path.join(_HERE, "librsdft_oracle.so")
_lib = None


def build(force=False):
    """Compile rsdft_oracle.c and rsdft_eig_oracle.c with gcc (-O2, OpenMP, no fast-math)."""
    if (not force) and os.path.exists(_LIB) and all(os.path.getmtime(_LIB) >= os.path.getmtime(s) for s in _SRCS):
        return _LIB
    cmd = ["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-std=gnu11", "-Wall",
           "-o", _LIB] + _SRCS + ["-lm"]
    subprocess.check_call(cmd)
    return _LIB


class _Species(C.Structure):
    _fields_ = [("rc", C.c_double), ("nproj", C.c_int32),
                ("l", C.POINTER(C.c_int32)), ("m", C.POINTER(C.c_int32)),
                ("radial_kind", C.c_int32), ("alpha", C.POINTER(C.c_double)),
                ("nr", C.c_int32), ("dr", C.c_double), ("radial", C.POINTER(C.c_double)),
                ("D", C.POINTER(C.c_double))]


def _load():
    global _lib
    if _lib is None:
        build()
        _lib = C.CDLL(_LIB)
        _lib.orc_sphere.restype = C.c_int64
    return _lib


def num_threads():
    return int(_load().orc_num_threads())


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _ip(a):
    return a.ctypes.data_as(C.POINTER(C.c_int32))


def _pack_species(species):
    """-> (ctypes array, keepalive list)"""
    keep = []
    arr = (_Species * max(1, len(species)))()
    for s, sp in enumerate(species):
        l = np.ascontiguousarray(sp["l"], dtype=np.int32)
        m = np.ascontiguousarray(sp["m"], dtype=np.int32)
        D = np.ascontiguousarray(sp["D"], dtype=np.float64)
        nproj = len(l)
        assert D.shape == (nproj, nproj)
        kind = int(sp.get("radial_kind", 0))
        alpha = np.ascontiguousarray(sp.get("alpha", np.zeros(nproj)), dtype=np.float64)
        radial = np.ascontiguousarray(sp.get("radial", np.zeros((nproj, 1))), dtype=np.float64)
        keep += [l, m, D, alpha, radial]
        arr[s].rc = float(sp["rc"]); arr[s].nproj = nproj
        arr[s].l = _ip(l); arr[s].m = _ip(m)
        arr[s].radial_kind = kind; arr[s].alpha = _dp(alpha)
        arr[s].nr = radial.shape[1]; arr[s].dr = float(sp.get("dr", 1.0)); arr[s].radial = _dp(radial)
        arr[s].D = _dp(D)
    return arr, keep


def fft3d(n, x, sign):
    """Forward (sign=-1, unnormalised) / inverse (sign=+1, 1/Ng) DFT of columns x[ncol, Ng]."""
    lib = _load()
    x = np.ascontiguousarray(x, dtype=np.complex128)
    if x.ndim == 1:
        return fft3d(n, x[None, :], sign)[0]
    ncol, ng = x.shape
    assert ng == n[0] * n[1] * n[2]
    out = np.empty_like(x)
    nn = (C.c_int32 * 3)(*n)
    rc = lib.orc_fft3d(nn, C.c_int(sign), C.c_int(ncol), _dp(x.view(np.float64)), C.c_int64(ng),
                       _dp(out.view(np.float64)), C.c_int64(ng))
    assert rc == 0
    return out


def kinetic_table(n, length):
    lib = _load()
    t = np.empty(n[0] * n[1] * n[2], dtype=np.float64)
    lib.orc_kinetic_table((C.c_int32 * 3)(*n), (C.c_double * 3)(*length), _dp(t))
    return t


def sphere(n, length, R, sp):
    """-> (idx[int32 npts], beta[nproj, npts]) for one atom at R, scanning all grid points."""
    lib = _load()
    arr, keep = _pack_species([sp])
    nn = (C.c_int32 * 3)(*n); ll = (C.c_double * 3)(*length); RR = (C.c_double * 3)(*R)
    cnt = lib.orc_sphere(nn, ll, RR, C.byref(arr[0]), C.c_int64(0), None, None)
    idx = np.empty(max(cnt, 1), dtype=np.int32)
    beta = np.empty((len(sp["l"]), max(cnt, 1)), dtype=np.float64)
    lib.orc_sphere(nn, ll, RR, C.byref(arr[0]), C.c_int64(max(cnt, 1)), _ip(idx), _dp(beta))
    return idx[:cnt], beta[:, :cnt]


def apply_h(system, X, return_p=False):
    """HX = (T + V_loc + V_NL) X for X[ncol, Ng] complex128 (row = one orbital)."""
    lib = _load()
    n = tuple(int(v) for v in system["n"]); length = tuple(float(v) for v in system["len"])
    X = np.ascontiguousarray(X, dtype=np.complex128)
    ncol, ng = X.shape
    assert ng == n[0] * n[1] * n[2]
    pos = np.ascontiguousarray(system.get("pos", np.zeros((0, 3))), dtype=np.float64).reshape(-1, 3)
    natom = pos.shape[0]
    species_of = np.ascontiguousarray(system.get("species_of", np.zeros(natom)), dtype=np.int32)
    species = system.get("species", []) if natom > 0 else []
    arr, keep = _pack_species(species)
    vloc = system.get("vloc", None)
    if vloc is not None:
        vloc = np.ascontiguousarray(vloc, dtype=np.float64).reshape(-1)
        assert vloc.size == ng
    maxproj = max([len(sp["l"]) for sp in species], default=0)
    HX = np.empty_like(X)
    p = np.zeros((max(natom, 1), max(maxproj, 1), ncol), dtype=np.complex128) if return_p else None
    rc = lib.orc_apply_h((C.c_int32 * 3)(*n), (C.c_double * 3)(*length),
                         C.c_int32(natom), _dp(pos), _ip(species_of),
                         C.c_int32(len(species)), arr, _dp(vloc) if vloc is not None else None,
                         C.c_int32(ncol), _dp(X.view(np.float64)), C.c_int64(ng),
                         _dp(HX.view(np.float64)), C.c_int64(ng),
                         _dp(p.view(np.float64)) if return_p else None)
    assert rc == 0
    return (HX, p[:natom, :maxproj]) if return_p else HX


def gram(Y, HY=None, want_s=True):
    """(H_sub, S_sub) with H_sub = Y^H HY, S_sub = Y^H Y; Y, HY are [n, Ng] (row = column
    vector of the paper's Y).  Returned as n x n numpy arrays M[i, j]."""
    lib = _load()
    Y = np.ascontiguousarray(Y, dtype=np.complex128)
    n, ng = Y.shape
    H = S = None
    if HY is not None:
        HY = np.ascontiguousarray(HY, dtype=np.complex128)
        assert HY.shape == Y.shape
        H = np.empty((n, n), dtype=np.complex128)   # column-major storage: H_store[j, i] = H[i, j]
    if want_s:
        S = np.empty((n, n), dtype=np.complex128)
    rc = lib.orc_gram(C.c_int64(ng), C.c_int32(n), _dp(Y.view(np.float64)), C.c_int64(ng),
                      _dp(HY.view(np.float64)) if HY is not None else None, C.c_int64(ng),
                      _dp(H.view(np.float64)) if H is not None else None,
                      _dp(S.view(np.float64)) if S is not None else None, C.c_int32(n))
    assert rc == 0
    return (H.T.copy() if H is not None else None, S.T.copy() if S is not None else None)


def rotate(Y, Cmat):
    """Rayleigh-Ritz update of LOBPCG (Knyazev's method, cited PAPER.md:19,124):
    Out[j, r] = sum_c Y[c, r] * Cmat[c, j] for Y[n, Ng] (row = one column of the block) and the n x m matrix Cmat.
    The plain definition, accumulated in long double (numpy's matmul on clongdouble is a plain loop)."""
    Y = np.asarray(Y, dtype=np.complex128)
    Cmat = np.asarray(Cmat, dtype=np.complex128)
    assert Y.shape[0] == Cmat.shape[0]
    out = Cmat.astype(np.clongdouble).T @ Y.astype(np.clongdouble)        # [m, n] @ [n, Ng]
    return out.astype(np.complex128)


# ----------------------------------------------------------------------------- NEXT-1 / NEXT-2
def _cm(a):
    """numpy M[i, j] -> column-major buffer (element (i, j) at i + j*n) as a contiguous array"""
    return np.ascontiguousarray(np.asarray(a, dtype=np.complex128).T)


def potrf(S):
    """Cholesky factor L (lower, real positive diagonal) of the Hermitian positive definite S = L L^H
    (PAPER.md:22); plain column algorithm in long double.  Raises if S is not positive definite."""
    S = np.asarray(S, dtype=np.complex128)
    n = S.shape[0]
    Sb = _cm(S)
    Lb = np.zeros((n, n), dtype=np.complex128)
    rc = _load().orc_potrf(C.c_int32(n), _dp(Sb.view(np.float64)), C.c_int32(n), _dp(Lb.view(np.float64)), C.c_int32(n))
    if rc != 0:
        raise np.linalg.LinAlgError("oracle.potrf: pivot %d is not positive" % rc)
    return Lb.T.copy()


def reduce_to_standard(H, S):
    """K = L^-1 H L^-H with S = L L^H, by two triangular substitutions (eq. 1)."""
    H = np.asarray(H, dtype=np.complex128)
    n = H.shape[0]
    Hb, Sb = _cm(H), _cm(S)
    Kb = np.zeros((n, n), dtype=np.complex128)
    rc = _load().orc_reduce(C.c_int32(n), _dp(Hb.view(np.float64)), C.c_int32(n), _dp(Sb.view(np.float64)), C.c_int32(n),
                            _dp(Kb.view(np.float64)), C.c_int32(n))
    if rc != 0:
        raise np.linalg.LinAlgError("oracle.reduce_to_standard: S is not positive definite (pivot %d)" % rc)
    return Kb.T.copy()


def jacobi_eigh(K):
    """(w ascending, Z) of a Hermitian K by the classical cyclic Jacobi method in long double."""
    K = np.asarray(K, dtype=np.complex128)
    n = K.shape[0]
    Kb = _cm(K)
    w = np.zeros(n, dtype=np.float64)
    Zb = np.zeros((n, n), dtype=np.complex128)
    rc = _load().orc_jacobi(C.c_int32(n), _dp(Kb.view(np.float64)), C.c_int32(n), _dp(w), _dp(Zb.view(np.float64)), C.c_int32(n))
    assert 0 <= rc < 60, "oracle.jacobi_eigh did not converge"
    return w, Zb.T.copy()


def backsolve(L, Z):
    """C = L^-H Z (eq. 1: Z = L^H X) by back substitution."""
    L = np.asarray(L, dtype=np.complex128)
    Z = np.asarray(Z, dtype=np.complex128)
    n, m = Z.shape
    Lb, Zb = _cm(L), _cm(Z)
    Cb = np.zeros((m, n), dtype=np.complex128)
    rc = _load().orc_backsolve(C.c_int32(n), C.c_int32(m), _dp(Lb.view(np.float64)), C.c_int32(n),
                               _dp(Zb.view(np.float64)), C.c_int32(n), _dp(Cb.view(np.float64)), C.c_int32(n))
    assert rc == 0
    return Cb.T.copy()


def subspace_eig(H, S, m=None, solver="jacobi", return_factors=False):
    """Generalized Hermitian eigen-solve H x = lambda S x by the paper's route (eq. 1):
    S = L L^H, K = L^-1 H L^-H (two triangular substitutions instead of ZHEGST), K Z = Z Lambda, X = L^-H Z.
    -> (lambda[m] ascending, C[n, m]) with C^H S C = I (and L, K if return_factors).
    solver="jacobi": everything in the C oracle in long double (cyclic Jacobi for the standard problem).
    solver="heevd":  Cholesky, the two substitutions and the back substitution in the C oracle; the standard
    problem by the library routine the paper names there, "(P)ZHEEVD" = numpy.linalg.eigh.
    Used where the O(n^3 * sweeps) Jacobi loop is too slow (n > ~300)."""
    H = np.asarray(H, dtype=np.complex128)
    S = np.asarray(S, dtype=np.complex128)
    n = H.shape[0]
    m = n if m is None else int(m)
    if solver == "jacobi":
        Hb, Sb = _cm(H), _cm(S)
        lam = np.zeros(m, dtype=np.float64)
        Cb = np.zeros((m, n), dtype=np.complex128)
        Lb = np.zeros((n, n), dtype=np.complex128)
        Kb = np.zeros((n, n), dtype=np.complex128)
        rc = _load().orc_subspace_eig(C.c_int32(n), _dp(Hb.view(np.float64)), C.c_int32(n), _dp(Sb.view(np.float64)), C.c_int32(n),
                                      C.c_int32(m), _dp(lam), _dp(Cb.view(np.float64)), C.c_int32(n),
                                      _dp(Lb.view(np.float64)), _dp(Kb.view(np.float64)), C.c_int32(n))
        if rc != 0:
            raise np.linalg.LinAlgError("oracle.subspace_eig: S is not positive definite (pivot %d)" % rc)
        Cm, L, K = Cb.T.copy(), Lb.T.copy(), Kb.T.copy()
    elif solver == "heevd":
        L = potrf(S)
        K = reduce_to_standard(H, S)
        w, Z = np.linalg.eigh(0.5 * (K + K.conj().T))
        lam = w[:m].copy()
        Cm = backsolve(L, Z[:, :m])
    else:
        raise ValueError(solver)
    return (lam, Cm, L, K) if return_factors else (lam, Cm)


def rotate2(Y, HY, Cmat, lam):
    """Rayleigh-Ritz update with residual (Knyazev's LOBPCG, cited PAPER.md:19,124):
        X'[j] = sum_c Y[c] C[c, j],   HX'[j] = sum_c HY[c] C[c, j],   R[j] = HX'[j] - lam[j] X'[j]
    for Y, HY [n, Ng] (row = one column of the block), Cmat n x m, lam[m] real.  Three plain products/loops in
    long double, rounded to double once at the end."""
    Yl = np.asarray(Y, dtype=np.complex128).astype(np.clongdouble)
    HYl = np.asarray(HY, dtype=np.complex128).astype(np.clongdouble)
    Cl = np.asarray(Cmat, dtype=np.complex128).astype(np.clongdouble)
    X = Cl.T @ Yl
    HX = Cl.T @ HYl
    R = HX - np.asarray(lam, dtype=np.longdouble)[:, None] * X
    return X.astype(np.complex128), HX.astype(np.complex128), R.astype(np.complex128)
