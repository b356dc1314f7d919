"""Seeded synthetic inputs for the five workloads of BASELINE.json `configs`.

This module serves BOTH the CUDA path's tests/bench and the oracle's tests.  It holds
none of the method's arithmetic (no FFT, no projector sums, no Gram): it only draws
atoms, builds the *input arrays* (V_loc is an input array, SURVEY 8(c) reading 12) and
draws random orbital blocks.  It imports neither `oracle` nor the CUDA binding.

The inputs stand in for the paper's diamond-216 / W-128 benchmark inputs,
which need QUMASUN input files and ONCV pseudopotentials that are not available here;
shapes follow BASELINE.json (recipe in DESIGN.md "Input recipe").
"""
import numpy as np

# real spherical harmonics labels: s + 3 real p (+ 5 real d); SURVEY 8(c) reading 7
_L_SP = [0, 1, 1, 1]
_M_SP = [0, -1, 0, 1]
_L_SPD = _L_SP + [2, 2, 2, 2, 2]
_M_SPD = _M_SP + [-2, -1, 0, 1, 2]

CONFIGS = {
    0: dict(name="cfg0-tiny16", n=16, L=10.0, m=8, seed=0, atoms="uniform", natom=2,
            depth=2.0, width=1.0, nproj=4, rc=2.0),
    1: dict(name="cfg1-small48", n=48, L=15.0, m=64, seed=1, atoms="uniform", natom=16,
            depth=2.0, width=1.0, nproj=4, rc=2.0),
    2: dict(name="cfg2-diamond96", n=96, L=20.22, m=480, seed=2, atoms="diamond", natom=216,
            depth=3.0, width=0.8, nproj=4, rc=1.4),
    3: dict(name="cfg3-tungsten112", n=112, L=23.92, m=512, seed=3, atoms="bcc", natom=128,
            depth=4.0, width=1.0, nproj=9, rc=2.2),
    4: dict(name="cfg4-large128", n=128, L=26.0, m=512, seed=4, atoms="minsep", natom=256,
            depth=4.0, width=1.0, nproj=9, rc=2.2, minsep=3.0),
    # the paper's own benchmark shapes: diamond-216 on 60^3 with N = 436 orbitals and W-128 on 80^3
    # with N = 901, with the synthetic potentials/projectors of configs 2 and 3 (the ONCV files are not available)
    5: dict(name="paper-diamond60", n=60, L=20.22, m=436, seed=5, atoms="diamond", natom=216,
            depth=3.0, width=0.8, nproj=4, rc=1.4),
    6: dict(name="paper-tungsten80", n=80, L=23.92, m=901, seed=6, atoms="bcc", natom=128,
            depth=4.0, width=1.0, nproj=9, rc=2.2),
}


def _min_image(d, L):
    return d - L * np.rint(d / L)


def _atoms(cfg, rng):
    L = cfg["L"]
    kind = cfg["atoms"]
    if kind == "uniform":
        return rng.uniform(0.0, L, size=(cfg["natom"], 3))
    if kind == "diamond":       # 8-atom conventional cell x 3^3, a = L/3 (BASELINE.json configs[2])
        a = L / 3.0
        basis = np.array([[0, 0, 0], [0, .5, .5], [.5, 0, .5], [.5, .5, 0],
                          [.25, .25, .25], [.25, .75, .75], [.75, .25, .75], [.75, .75, .25]])
        cells = np.array([[i, j, k] for i in range(3) for j in range(3) for k in range(3)], dtype=float)
        return ((cells[:, None, :] + basis[None, :, :]) * a).reshape(-1, 3)
    if kind == "bcc":           # 2-atom cell x 4^3, a = L/4 (configs[3])
        a = L / 4.0
        basis = np.array([[0, 0, 0], [.5, .5, .5]])
        cells = np.array([[i, j, k] for i in range(4) for j in range(4) for k in range(4)], dtype=float)
        return ((cells[:, None, :] + basis[None, :, :]) * a).reshape(-1, 3)
    if kind == "minsep":        # sequential rejection, minimum-image separation >= minsep (configs[4])
        pts = []
        while len(pts) < cfg["natom"]:
            p = rng.uniform(0.0, L, size=3)
            if all(np.linalg.norm(_min_image(p - q, L)) >= cfg["minsep"] for q in pts):
                pts.append(p)
        return np.array(pts)
    raise ValueError(kind)


def _species(cfg, rng):
    nproj = cfg["nproj"]
    if nproj == 4:
        l, m = _L_SP, _M_SP
        D = np.diag([1.0, -0.5, -0.5, -0.5])
    else:
        l, m = _L_SPD, _M_SPD
        D = np.diag(rng.uniform(-1.0, 1.0, size=nproj))    # configs[3]: "D drawn uniform in [-1, 1] Ha"
    # radial part exp(-r^2/0.5) = exp(-2 r^2) for every projector (configs[0])
    return dict(rc=cfg["rc"], l=np.array(l, np.int32), m=np.array(m, np.int32), radial_kind=0,
                alpha=np.full(nproj, 2.0), D=D)


def gaussian_vloc(n, L, pos, depth, width):
    """v(r) = -depth * sum_a exp(-|d|^2 / (2 w^2)), minimum image; an INPUT array."""
    out = None
    ax = []
    for a in range(3):
        r = np.arange(n[a]) * (L[a] / n[a])
        d = _min_image(r[None, :] - pos[:, a:a + 1], L[a])
        ax.append(np.exp(-d * d / (2.0 * width * width)))
    out = -depth * np.einsum("ax,ay,az->xyz", ax[0], ax[1], ax[2], optimize=True)
    return np.ascontiguousarray(out.reshape(-1))


def sphere_margin(system):
    """min over atoms and grid points of | |d|^2 - rc^2 |: an input-validity check (the oracle and the plan must
    agree on sphere membership point for point).  Only the grid points within rc + 2h of an atom along each axis
    can come near its sphere boundary, so each atom scans its own bounding box."""
    n, L = system["n"], system["len"]
    best = np.inf
    for a, R in enumerate(system["pos"]):
        rc = system["species"][system["species_of"][a]]["rc"]
        d2 = 0.0
        for ax in range(3):
            h = L[ax] / n[ax]
            r = np.arange(n[ax]) * h
            d = _min_image(r - R[ax], L[ax])
            d = d[np.abs(d) <= rc + 2.0 * h]
            shape = [1, 1, 1]; shape[ax] = -1
            d2 = d2 + (d * d).reshape(shape)
        best = min(best, float(np.min(np.abs(d2 - rc * rc))))
    return best


def make_system(cfg_id, with_vloc=True, check_margin=None):
    """-> dict(n, len, pos, species_of, species, vloc, m, seed, name)."""
    cfg = CONFIGS[cfg_id]
    rng = np.random.default_rng(cfg["seed"])
    n = (cfg["n"],) * 3
    L = (cfg["L"],) * 3
    pos = np.mod(_atoms(cfg, rng), cfg["L"])
    sp = _species(cfg, rng)
    system = dict(name=cfg["name"], cfg=cfg_id, n=n, len=L, pos=pos,
                  species_of=np.zeros(len(pos), np.int32), species=[sp],
                  m=cfg["m"], seed=cfg["seed"], vloc=None)
    if with_vloc:
        system["vloc"] = gaussian_vloc(n, L, pos, cfg["depth"], cfg["width"])
    if check_margin is None:
        check_margin = True
    if check_margin:
        assert sphere_margin(system) > 1e-9, "grid point on a sphere boundary; change the seed"
    return system


def small_system(n=(12, 10, 8), L=(7.0, 6.0, 5.0), natom=3, seed=7, nproj=9, rc=1.9, radial_kind=0):
    """Non-cubic, non-power-of-two little system for oracle pins and ABI edge cases."""
    rng = np.random.default_rng(seed)
    pos = rng.uniform(0, 1, size=(natom, 3)) * np.array(L)
    l, m = (_L_SPD, _M_SPD) if nproj == 9 else (_L_SP, _M_SP)
    A = rng.uniform(-1, 1, size=(nproj, nproj))
    sp = dict(rc=rc, l=np.array(l, np.int32), m=np.array(m, np.int32), radial_kind=radial_kind,
              alpha=rng.uniform(1.0, 3.0, size=nproj), D=0.5 * (A + A.T))
    if radial_kind == 1:
        nr = 64
        dr = rc / (nr - 4)
        r = np.arange(nr) * dr
        sp["dr"] = dr
        sp["radial"] = np.stack([np.exp(-a * r * r) * (1 + 0.3 * i * r) for i, a in enumerate(sp["alpha"])])
    system = dict(name="small", cfg=-1, n=tuple(n), len=tuple(L), pos=pos,
                  species_of=np.zeros(natom, np.int32), species=[sp], m=4, seed=seed,
                  vloc=rng.standard_normal(int(np.prod(n))))
    return system


def subspace_pencil(n, seed, degenerate=False):
    """Seeded synthetic (H_sub, S_sub) pencil of size n for the eigen-solve (NEXT-1), shaped like the Gram matrices
    of a random orbital block: S = G^H G (Hermitian positive definite, well conditioned), H = G^H diag(d) G with
    d in (-1, 3) (the Ritz values then lie in (-1, 3)).  degenerate=True builds H = B^H diag(w) B, S = B^H B with
    repeated levels in w (shells of 6, 12, 8 like the free-electron spectrum), returning w as a third value.
    An INPUT generator: it draws random matrices and multiplies them; it holds no step of the eigen-solve."""
    rng = np.random.default_rng(1000003 * int(seed) + int(n))
    cn = lambda *shape: (rng.standard_normal(shape) + 1j * rng.standard_normal(shape)) * np.sqrt(0.5)
    if degenerate:
        B = cn(n, n) + 2.0 * np.sqrt(n) * np.eye(n)
        base = np.sort(rng.uniform(-1.0, 3.0, n))
        w = base.copy()
        i = 1
        for deg in (6, 12, 8, 6, 24):
            if i + deg <= n:
                w[i:i + deg] = base[i]
            i += deg + 3
        w = np.sort(w)
        H = B.conj().T @ (w[:, None] * B)
        S = B.conj().T @ B
        return 0.5 * (H + H.conj().T), 0.5 * (S + S.conj().T), w
    k = 4 * n
    G = cn(k, n)
    d = rng.uniform(-1.0, 3.0, k)
    S = G.conj().T @ G
    H = G.conj().T @ (d[:, None] * G)
    return 0.5 * (H + H.conj().T), 0.5 * (S + S.conj().T)


def orbital_block(ng, cols, seed, stream, device="cpu", ld=None, out=None):
    """CN(0,1) orbitals (re, im ~ N(0, 1/2) i.i.d.; SURVEY 8(c) reading 13) as a torch
    complex128 tensor [len(cols), ld] (row c = orbital cols[c]).  Each column has its own
    generator seed (seed, stream, column), so any subset of columns can be regenerated.
    `stream` separates X (0), W (1), P (2).  Values drawn on `device`; the oracle is fed a
    host copy of the very same tensor, never an independently drawn one.  `out` (rows of a
    preallocated block) is filled in place instead of allocating."""
    import torch
    ld = ng if ld is None else ld
    cols = list(cols)
    if out is None:
        out = torch.zeros((len(cols), ld), dtype=torch.complex128, device=device)
    else:
        device = out.device
        assert out.shape == (len(cols), ld) and out.dtype == torch.complex128
    view = torch.view_as_real(out)
    gen = torch.Generator(device=device)
    for r, c in enumerate(cols):
        gen.manual_seed((int(seed) * 1000003 + int(stream)) * 1000003 + int(c))
        view[r, :ng, :].normal_(0.0, 0.5 ** 0.5, generator=gen)
    return out


def block_y(system, device="cuda"):
    """Y = [X, W, P] of a config as ONE [3m, Ng] tensor, filled block by block in place (no
    concatenation copy: configs[4] holds 51.5 GB per block)."""
    import torch
    m = system["m"]
    ng = int(np.prod(system["n"]))
    Y = torch.empty((3 * m, ng), dtype=torch.complex128, device=device)
    for s in range(3):
        orbital_block(ng, range(m), system["seed"], s, out=Y[s * m:(s + 1) * m])
    return Y
