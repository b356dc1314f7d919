"""Thin ctypes binding over librsdft.so (include/rsdft.h) -- argument marshalling only.

Every step of the path runs in the CUDA kernels behind the C ABI; there is no CPU fallback:
if the library is missing, or it reports an error, the call raises.  torch is used for device
memory and streams only (torch tensors' data_ptr() / torch.cuda.current_stream()).

Function names follow the C ABI: rsdft_plan_create, rsdft_plan_set_vloc, rsdft_apply_h,
rsdft_subspace_gram, rsdft_subspace_gram_static, rsdft_subspace_rotate, rsdft_subspace_rotate2, rsdft_subspace_eig, rsdft_subspace_eig_get,
rsdft_plan_set_eig_mode, rsdft_subspace_eig_stats, rsdft_block_step_host, rsdft_plan_release_workspace, rsdft_plan_info,
rsdft_plan_set_batch, rsdft_plan_set_streams, rsdft_plan_set_gram_mode, rsdft_plan_destroy, rsdft_last_error.  Orbital blocks are torch complex128 tensors of shape
[ncol, ld] (row c = column c of the paper's block, contiguous in the grid index)."""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "librsdft.so")

SYMBOLS = ["rsdft_plan_create", "rsdft_plan_set_vloc", "rsdft_apply_h", "rsdft_subspace_gram", "rsdft_subspace_gram_static",
           "rsdft_subspace_rotate",
           "rsdft_subspace_rotate2", "rsdft_subspace_eig", "rsdft_subspace_eig_get", "rsdft_plan_set_eig_mode",
           "rsdft_subspace_eig_stats", "rsdft_plan_release_workspace", "rsdft_plan_set_pipeline", "rsdft_plan_set_gram_staging",
           "rsdft_block_step_host", "rsdft_plan_info", "rsdft_plan_set_batch", "rsdft_plan_set_streams", "rsdft_plan_set_gram_mode", "rsdft_plan_destroy",
           "rsdft_last_error"]

RSDFT_OK, RSDFT_INVALID_ARG, RSDFT_UNSUPPORTED, RSDFT_ALLOC, RSDFT_CUDA = 0, -1, -2, -3, -4
RSDFT_NOT_POSITIVE_DEFINITE, RSDFT_NO_CONVERGENCE = -5, -6


class RsdftError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("librsdft error %d: %s" % (code, msg))
        self.code = code


class _Grid(C.Structure):
    _fields_ = [("n", C.c_int32 * 3)]


class _Box(C.Structure):
    _fields_ = [("len", C.c_double * 3)]


class _Atoms(C.Structure):
    _fields_ = [("natom", C.c_int32), ("pos", C.POINTER(C.c_double)), ("species", C.POINTER(C.c_int32))]


class _Species(C.Structure):
    _fields_ = [("rc", C.c_double), ("nproj", C.c_int32),
                ("l", C.POINTER(C.c_int32)), ("m", C.POINTER(C.c_int32)),
                ("radial_kind", C.c_int32), ("alpha", C.POINTER(C.c_double)),
                ("nr", C.c_int32), ("dr", C.c_double), ("radial", C.POINTER(C.c_double)),
                ("D", C.POINTER(C.c_double))]


class _Projectors(C.Structure):
    _fields_ = [("nspecies", C.c_int32), ("species", C.POINTER(_Species))]


_lib = None


def load():
    """dlopen librsdft.so; raises (never falls back) when it has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError("librsdft.so is not built: run `python -m paper_2512_04447_b200.build` "
                           "(there is no CPU fallback for the CUDA path)")
    lib = C.CDLL(LIB_PATH)
    vp, i32, i64 = C.c_void_p, C.c_int32, C.c_int64
    lib.rsdft_plan_create.argtypes = [C.POINTER(_Grid), C.POINTER(_Box), C.POINTER(_Atoms),
                                      C.POINTER(_Projectors), C.POINTER(vp)]
    lib.rsdft_plan_set_vloc.argtypes = [vp, vp, vp]
    lib.rsdft_apply_h.argtypes = [vp, i32, vp, i64, vp, i64, vp]
    lib.rsdft_subspace_gram.argtypes = [vp, i32, vp, i64, vp, i64, vp, vp, i32, vp]
    lib.rsdft_subspace_gram_static.argtypes = [vp, i32, vp, i64, vp, i64, vp, vp, i32, vp]
    lib.rsdft_subspace_rotate.argtypes = [vp, i32, i32, vp, i64, vp, i32, vp, i64, vp]
    lib.rsdft_subspace_rotate2.argtypes = [vp, i32, i32, vp, i64, vp, i64, vp, i32, vp, vp, i64, vp, i64, vp, i64, vp]
    lib.rsdft_subspace_eig.argtypes = [vp, i32, vp, vp, i32, i32, vp, vp, i32, vp]
    lib.rsdft_subspace_eig_get.argtypes = [vp, i32, vp, i32, vp]
    lib.rsdft_plan_set_eig_mode.argtypes = [vp, i32, i32]
    lib.rsdft_subspace_eig_stats.argtypes = [vp, C.POINTER(C.c_double)]
    lib.rsdft_plan_release_workspace.argtypes = [vp]
    lib.rsdft_plan_set_pipeline.argtypes = [vp, i32]
    lib.rsdft_plan_set_gram_staging.argtypes = [vp, i32]
    lib.rsdft_block_step_host.argtypes = [vp, i32, vp, i64, vp, i64, vp, vp, i32]
    lib.rsdft_plan_info.argtypes = [vp, C.POINTER(i64)]
    lib.rsdft_plan_set_batch.argtypes = [vp, i32]
    lib.rsdft_plan_set_streams.argtypes = [vp, i32]
    lib.rsdft_plan_set_gram_mode.argtypes = [vp, i32]
    lib.rsdft_plan_destroy.argtypes = [vp]
    lib.rsdft_last_error.restype = C.c_char_p
    for name in SYMBOLS:
        if name != "rsdft_last_error":
            getattr(lib, name).restype = C.c_int
    _lib = lib
    return lib


def rsdft_last_error():
    return load().rsdft_last_error().decode()


def _check(rc):
    if rc != RSDFT_OK:
        raise RsdftError(rc, rsdft_last_error())


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _ip(a):
    return a.ctypes.data_as(C.POINTER(C.c_int32))


def _stream(stream):
    if stream is None:
        import torch
        stream = torch.cuda.current_stream().cuda_stream
    return C.c_void_p(int(stream))


class Plan:
    """Owner of an rsdft_plan_t* (destroyed on close() / garbage collection)."""

    def __init__(self, handle, n, length):
        self.handle = handle
        self.n = tuple(n)
        self.len = tuple(length)
        self.ng = int(n[0]) * int(n[1]) * int(n[2])

    def close(self):
        if self.handle:
            load().rsdft_plan_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def rsdft_plan_create(grid, box, atoms=None, projectors=None):
    """grid: (Nx, Ny, Nz); box: (Lx, Ly, Lz) bohr; atoms: (pos[natom,3], species_of[natom]) or
    None; projectors: list of species dicts {rc, l, m, D, radial_kind, alpha | (dr, radial)}."""
    lib = load()
    g = _Grid((C.c_int32 * 3)(*[int(v) for v in grid]))
    b = _Box((C.c_double * 3)(*[float(v) for v in box]))
    keep = []
    a_ptr = p_ptr = None
    if atoms is not None:
        pos = np.ascontiguousarray(atoms[0], dtype=np.float64).reshape(-1, 3)
        spo = np.ascontiguousarray(atoms[1], dtype=np.int32).reshape(-1)
        if spo.shape[0] != pos.shape[0]:
            raise ValueError("species_of and pos disagree on natom")
        keep += [pos, spo]
        a_ptr = C.pointer(_Atoms(pos.shape[0], _dp(pos), _ip(spo)))
    if projectors is not None:
        arr = (_Species * max(1, len(projectors)))()
        for s, sp in enumerate(projectors):
            l = np.ascontiguousarray(sp["l"], dtype=np.int32)
            m = np.ascontiguousarray(sp["m"], dtype=np.int32)
            D = np.ascontiguousarray(sp["D"], dtype=np.float64)
            nproj = int(l.shape[0])
            alpha = np.ascontiguousarray(sp.get("alpha", np.zeros(nproj)), dtype=np.float64)
            radial = np.ascontiguousarray(sp.get("radial", np.zeros((nproj, 2))), dtype=np.float64)
            keep += [l, m, D, alpha, radial]
            arr[s] = _Species(float(sp["rc"]), nproj, _ip(l), _ip(m), int(sp.get("radial_kind", 0)), _dp(alpha),
                              int(radial.shape[1]), float(sp.get("dr", 1.0)), _dp(radial), _dp(D))
        keep.append(arr)
        p_ptr = C.pointer(_Projectors(len(projectors), arr))
    out = C.c_void_p()
    _check(lib.rsdft_plan_create(C.byref(g), C.byref(b), a_ptr, p_ptr, C.byref(out)))
    return Plan(out, grid, box)


def plan_from_system(system):
    """Convenience: plan for a workloads.make_system() dict, V_loc uploaded if present."""
    import torch
    natom = len(system.get("pos", []))
    plan = rsdft_plan_create(system["n"], system["len"],
                             (system["pos"], system["species_of"]) if natom else None,
                             system["species"] if natom else None)
    if system.get("vloc") is not None:
        v = torch.as_tensor(np.ascontiguousarray(system["vloc"], dtype=np.float64)).cuda()
        rsdft_plan_set_vloc(plan, v)
        torch.cuda.current_stream().synchronize()
    return plan


def rsdft_plan_set_vloc(plan, vloc, stream=None):
    """vloc: torch float64 CUDA tensor [Ng], or None to reset V_loc to 0."""
    ptr = None
    if vloc is not None:
        if not (vloc.is_cuda and vloc.is_contiguous() and vloc.numel() == plan.ng and vloc.element_size() == 8):
            raise ValueError("vloc must be a contiguous float64 CUDA tensor of Ng elements")
        ptr = C.c_void_p(vloc.data_ptr())
    _check(load().rsdft_plan_set_vloc(plan.handle, ptr, _stream(stream)))


def _block(t, name, plan=None, host=False):
    """An orbital block [ncol, ld]: complex128, unit inner stride, on the device (or the host), ld >= Ng.
    -> (ncol, ld).  Everything the C ABI cannot check from a raw pointer is checked here."""
    import torch
    if not isinstance(t, torch.Tensor) or t.dtype != torch.complex128 or t.dim() != 2 or t.stride(1) != 1:
        raise ValueError("%s must be a complex128 tensor [ncol, ld] with unit inner stride" % name)
    if host and t.is_cuda:
        raise ValueError("%s must be a HOST tensor" % name)
    if not host and not t.is_cuda:
        raise ValueError("%s must be a CUDA tensor" % name)
    if t.shape[0] < 1:
        raise ValueError("%s has no columns" % name)
    if plan is not None and t.shape[1] < plan.ng:
        raise ValueError("%s has %d elements per column, the plan's grid has %d" % (name, t.shape[1], plan.ng))
    ld = t.stride(0) if t.shape[0] > 1 else max(t.shape[1], t.stride(0))
    if t.shape[0] > 1 and ld < t.shape[1]:
        raise ValueError("%s: rows overlap (stride %d < %d)" % (name, ld, t.shape[1]))
    return t.shape[0], ld


def _matrix(t, name, rows, cols, host=False):
    """A column-major rows x cols complex128 matrix held as a torch tensor [cols, ld >= rows] (t[j, i] = M[i, j]).
    -> ld."""
    import torch
    if not isinstance(t, torch.Tensor) or t.dtype != torch.complex128 or t.dim() != 2 or t.stride(1) != 1:
        raise ValueError("%s must be a complex128 tensor [%d, ld >= %d] with unit inner stride" % (name, cols, rows))
    if bool(t.is_cuda) == bool(host):
        raise ValueError("%s must be a %s tensor" % (name, "HOST" if host else "CUDA"))
    if t.shape[0] != cols or t.shape[1] < rows:
        raise ValueError("%s must have shape [%d, >= %d], got %s" % (name, cols, rows, tuple(t.shape)))
    ld = t.stride(0) if cols > 1 else max(t.shape[1], t.stride(0))
    if cols > 1 and ld < rows:
        raise ValueError("%s: columns overlap" % name)
    if ld >= 2 ** 31:
        raise ValueError("%s: leading dimension does not fit int32" % name)
    return ld


def rsdft_apply_h(plan, X, HX, stream=None):
    """HX[c, :Ng] = (T + V_loc + V_NL) X[c, :Ng] for every row c.  X, HX: [ncol, ld] CUDA complex128."""
    ncol, ldx = _block(X, "X", plan)
    ncol2, ldhx = _block(HX, "HX", plan)
    if ncol != ncol2:
        raise ValueError("X and HX disagree on ncol")
    _check(load().rsdft_apply_h(plan.handle, ncol, C.c_void_p(X.data_ptr()), ldx, C.c_void_p(HX.data_ptr()), ldhx,
                                _stream(stream)))
    return HX


RSDFT_GRAM_STATIC_MAX_N = 1536


def rsdft_subspace_gram_static(plan, Y, HY, H_sub, S_sub, stream=None):
    """rsdft_subspace_gram through the entry point that allocates nothing: the caller passes the outputs ([n, lds >= n]
    complex128 CUDA tensors, column-major as rsdft_subspace_gram's; None skips one, HY may be None without H_sub); the
    scratch is the library's static device array; n <= RSDFT_GRAM_STATIC_MAX_N.  -> (H_sub, S_sub)."""
    if H_sub is None and S_sub is None:
        raise ValueError("rsdft_subspace_gram_static: the caller passes at least one output")
    n, ldy = _block(Y, "Y", plan)
    ldhy = ldy
    if H_sub is not None:
        n2, ldhy = _block(HY, "HY", plan)
        if n2 != n:
            raise ValueError("Y and HY disagree on n")
    lds = None
    for t, name in ((H_sub, "H_sub"), (S_sub, "S_sub")):
        if t is not None:
            ld = _matrix(t, name, n, n)
            if lds is not None and ld != lds:
                raise ValueError("H_sub and S_sub must share one leading dimension")
            lds = ld
    _check(load().rsdft_subspace_gram_static(plan.handle, n, C.c_void_p(Y.data_ptr()), ldy,
                                             C.c_void_p(HY.data_ptr()) if H_sub is not None else None, ldhy,
                                             C.c_void_p(H_sub.data_ptr()) if H_sub is not None else None,
                                             C.c_void_p(S_sub.data_ptr()) if S_sub is not None else None, lds, _stream(stream)))
    return H_sub, S_sub


def rsdft_subspace_gram(plan, Y, HY, H_sub=None, S_sub=None, stream=None, want_h=True, want_s=True):
    """-> (H_sub, S_sub) as torch [n, lds >= n] complex128 CUDA tensors holding the COLUMN-MAJOR
    matrices: M_store[j, i] = M[i, j] (so M = M_store.T).  Y, HY: [n, ld].  Given outputs must share one lds."""
    import torch
    n, ldy = _block(Y, "Y", plan)
    ldhy = ldy
    if want_h:
        n2, ldhy = _block(HY, "HY", plan)
        if n2 != n:
            raise ValueError("Y and HY disagree on n")
    if want_h and H_sub is None:
        H_sub = torch.empty((n, n), dtype=torch.complex128, device=Y.device)
    if want_s and S_sub is None:
        S_sub = torch.empty((n, n), dtype=torch.complex128, device=Y.device)
    lds = None
    for t, name, want in ((H_sub, "H_sub", want_h), (S_sub, "S_sub", want_s)):
        if want:
            ld = _matrix(t, name, n, n)
            if lds is not None and ld != lds:
                raise ValueError("H_sub and S_sub must share one leading dimension")
            lds = ld
    _check(load().rsdft_subspace_gram(plan.handle, n, C.c_void_p(Y.data_ptr()), ldy,
                                      C.c_void_p(HY.data_ptr()) if want_h else None, ldhy,
                                      C.c_void_p(H_sub.data_ptr()) if want_h else None,
                                      C.c_void_p(S_sub.data_ptr()) if want_s else None, lds, _stream(stream)))
    return H_sub, S_sub


def rsdft_subspace_rotate(plan, Y, Cmat, Out=None, stream=None):
    """Out[j, :Ng] = sum_c Cmat[c, j] * Y[c, :Ng].  Y: [n, ld] CUDA complex128 block; Cmat: torch [m, n] CUDA
    complex128 tensor [m, ldc >= n] holding the COLUMN-MAJOR n x m matrix (Cmat_store[j, c] = C[c, j], like the
    Gram outputs); Out: [m, ldo] block (allocated if None)."""
    import torch
    n, ldy = _block(Y, "Y", plan)
    if not isinstance(Cmat, torch.Tensor) or Cmat.dim() != 2:
        raise ValueError("Cmat must be a CUDA complex128 tensor [m, ldc >= n] (column-major n x m)")
    m = Cmat.shape[0]
    ldc = _matrix(Cmat, "Cmat", n, m)
    if Out is None:
        Out = torch.empty((m, ldy), dtype=torch.complex128, device=Y.device)
    m2, ldo = _block(Out, "Out", plan)
    if m2 != m:
        raise ValueError("Out and Cmat disagree on m")
    _check(load().rsdft_subspace_rotate(plan.handle, n, m, C.c_void_p(Y.data_ptr()), ldy, C.c_void_p(Cmat.data_ptr()), ldc,
                                        C.c_void_p(Out.data_ptr()), ldo, _stream(stream)))
    return Out


def rsdft_subspace_rotate2(plan, Y, HY, Cmat, lam=None, Xout=None, HXout=None, R=None, stream=None, want_r=True):
    """One pass: Xout = Y C, HXout = HY C, R = HXout - lam * Xout (column-wise).  Y, HY: [n, ld] blocks; Cmat: [m, ldc >= n]
    (column-major n x m); lam: CUDA float64 [m].  Outputs [m, ld] blocks, allocated if None (R only if want_r).
    -> (Xout, HXout, R)."""
    import torch
    n, ldy = _block(Y, "Y", plan)
    n2, ldhy = _block(HY, "HY", plan)
    if n2 != n:
        raise ValueError("Y and HY disagree on n")
    if not isinstance(Cmat, torch.Tensor) or Cmat.dim() != 2:
        raise ValueError("Cmat must be a CUDA complex128 tensor [m, ldc >= n]")
    m = Cmat.shape[0]
    ldc = _matrix(Cmat, "Cmat", n, m)
    if want_r:
        if lam is None or not (lam.is_cuda and lam.dtype == torch.float64 and lam.dim() == 1 and lam.is_contiguous() and lam.numel() >= m):
            raise ValueError("lam must be a contiguous CUDA float64 tensor of m elements")
    outs = []
    for t, name, want in ((Xout, "Xout", True), (HXout, "HXout", True), (R, "R", want_r)):
        if want and t is None:
            t = torch.empty((m, plan.ng), dtype=torch.complex128, device=Y.device)
        if want:
            m2, ld = _block(t, name, plan)
            if m2 != m:
                raise ValueError("%s and Cmat disagree on m" % name)
            outs.append((t, ld))
        else:
            outs.append((None, 0))
    p = lambda t: C.c_void_p(t.data_ptr()) if t is not None else None
    _check(load().rsdft_subspace_rotate2(plan.handle, n, m, p(Y), ldy, p(HY), ldhy, p(Cmat), ldc,
                                         C.c_void_p(lam.data_ptr()) if want_r else None,
                                         p(outs[0][0]), outs[0][1], p(outs[1][0]), outs[1][1], p(outs[2][0]), outs[2][1],
                                         _stream(stream)))
    return outs[0][0], outs[1][0], outs[2][0]


def rsdft_subspace_eig(plan, H_sub, S_sub, m=None, lam=None, Cmat=None, stream=None):
    """Generalized eigen-solve H_sub x = lam S_sub x (eq. 1) on the device.  H_sub, S_sub: [n, lds >= n]
    CUDA complex128 (column-major, as rsdft_subspace_gram returns them).  -> (lam[m] float64 CUDA ascending,
    Cmat [m, n] CUDA complex128 holding the column-major n x m eigenvector matrix: Cmat[j] = eigenvector j)."""
    import torch
    if not isinstance(H_sub, torch.Tensor) or H_sub.dim() != 2:
        raise ValueError("H_sub must be a 2-D CUDA complex128 tensor")
    n = H_sub.shape[0]
    lds = _matrix(H_sub, "H_sub", n, n)
    if _matrix(S_sub, "S_sub", n, n) != lds:
        raise ValueError("H_sub and S_sub must share one leading dimension")
    m = n if m is None else int(m)
    if lam is None:
        lam = torch.empty(m, dtype=torch.float64, device=H_sub.device)
    if not (lam.is_cuda and lam.dtype == torch.float64 and lam.dim() == 1 and lam.is_contiguous() and lam.numel() >= m):
        raise ValueError("lam must be a contiguous CUDA float64 tensor of m elements")
    if Cmat is None:
        Cmat = torch.empty((m, n), dtype=torch.complex128, device=H_sub.device)
    ldc = _matrix(Cmat, "Cmat", n, m)
    _check(load().rsdft_subspace_eig(plan.handle, n, C.c_void_p(H_sub.data_ptr()), C.c_void_p(S_sub.data_ptr()), lds, m,
                                     C.c_void_p(lam.data_ptr()), C.c_void_p(Cmat.data_ptr()), ldc, _stream(stream)))
    return lam, Cmat


def rsdft_subspace_eig_get(plan, what, n, stream=None):
    """what = "L": Cholesky factor, "K": standard-form matrix of the last rsdft_subspace_eig; -> [n, n] CUDA tensor
    (column-major storage: t[j, i] = M[i, j])."""
    import torch
    out = torch.empty((n, n), dtype=torch.complex128, device="cuda")
    _check(load().rsdft_subspace_eig_get(plan.handle, {"L": 0, "K": 1}[what], C.c_void_p(out.data_ptr()), n, _stream(stream)))
    return out


def rsdft_plan_set_eig_mode(plan, reduction=0, inner_sweeps=0):
    _check(load().rsdft_plan_set_eig_mode(plan.handle, int(reduction), int(inner_sweeps)))


def rsdft_subspace_eig_stats(plan):
    out = (C.c_double * 8)()
    _check(load().rsdft_subspace_eig_stats(plan.handle, out))
    keys = ["sweeps", "ms_potrf", "ms_reduce", "ms_eig", "ms_back", "off_rel", "reduction_mode"]
    return dict(zip(keys, [float(v) for v in out]))


def rsdft_plan_release_workspace(plan):
    _check(load().rsdft_plan_release_workspace(plan.handle))


def rsdft_block_step_host(plan, Y_host, HY_host=None, H_sub_host=None, S_sub_host=None):
    """One whole block step from HOST tensors (pinned recommended): uploads Y in chunks overlapped
    with apply_h, forms the Gram matrices, downloads them (and HY if HY_host is given)."""
    import torch
    n, ldy = _block(Y_host, "Y_host", plan, host=True)
    ldhy = 0
    if HY_host is not None:
        n2, ldhy = _block(HY_host, "HY_host", plan, host=True)
        if n2 != n:
            raise ValueError("Y_host and HY_host disagree on n")
    if H_sub_host is None:
        H_sub_host = torch.empty((n, n), dtype=torch.complex128).pin_memory()
    if S_sub_host is None:
        S_sub_host = torch.empty((n, n), dtype=torch.complex128).pin_memory()
    lds = _matrix(H_sub_host, "H_sub_host", n, n, host=True)
    if _matrix(S_sub_host, "S_sub_host", n, n, host=True) != lds:
        raise ValueError("H_sub_host and S_sub_host must share one leading dimension")
    _check(load().rsdft_block_step_host(plan.handle, n, C.c_void_p(Y_host.data_ptr()), ldy,
                                        C.c_void_p(HY_host.data_ptr()) if HY_host is not None else None, ldhy,
                                        C.c_void_p(H_sub_host.data_ptr()), C.c_void_p(S_sub_host.data_ptr()), lds))
    return H_sub_host, S_sub_host


def rsdft_plan_info(plan):
    out = (C.c_int64 * 8)()
    _check(load().rsdft_plan_info(plan.handle, out))
    keys = ["natom", "sphere_points", "max_sphere_points", "device_bytes", "batch_cols", "last_launches", "ng",
            "colour_classes"]
    return dict(zip(keys, [int(v) for v in out]))


def rsdft_plan_set_batch(plan, batch_cols):
    _check(load().rsdft_plan_set_batch(plan.handle, int(batch_cols)))


def rsdft_plan_set_streams(plan, nstreams):
    _check(load().rsdft_plan_set_streams(plan.handle, int(nstreams)))


def rsdft_plan_set_pipeline(plan, mode):
    _check(load().rsdft_plan_set_pipeline(plan.handle, int(mode)))


def rsdft_plan_set_gram_staging(plan, bulk):
    _check(load().rsdft_plan_set_gram_staging(plan.handle, int(bulk)))


def rsdft_plan_set_gram_mode(plan, h_upper_only):
    _check(load().rsdft_plan_set_gram_mode(plan.handle, int(h_upper_only)))


def rsdft_plan_destroy(plan):
    plan.close()
