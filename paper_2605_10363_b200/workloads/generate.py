"""Seeded generators for the five BASELINE.json workloads (inputs only).

Everything here is *input construction*: molecular geometry, the synthetic uncontracted
Cartesian Gaussian shell table, atom-centred quadrature points with Becke weights, and
the idempotent-like density matrix D = 2 Q Q^T.  Nothing here evaluates a basis function,
a density, a functional or a contraction.

Recipe readings (repeated in DESIGN.md §4):
  * radial rule: Gauss-Chebyshev of the 2nd kind, x_i = cos(i*pi/51), i = 1..50,
    r = R (1+x)/(1-x), w_rad = (pi/51) sin(i*pi/51) * 2R/(1-x)^2 * r^2
  * angular rule: 110-point Fibonacci sphere, z_k = 1-(2k+1)/110, phi_k = k*pi*(3-sqrt 5),
    equal weights 4*pi/110
  * Becke fuzzy cells, plain (no atomic-size adjustment), 3 smoothing iterations
  * points are emitted atom by atom, radial-major, angular-minor ("caller order")
"""
from __future__ import annotations

import dataclasses
import math
import os
from typing import Optional

import numpy as np

ANG2BOHR = 1.0 / 0.529177210903

# synthetic basis (BASELINE.json configs[0]); C uses the O table
_BASIS = {
    "O": [(0, 5.0), (0, 1.0), (0, 0.25), (1, 1.2), (1, 0.3), (2, 0.8)],
    "C": [(0, 5.0), (0, 1.0), (0, 0.25), (1, 1.2), (1, 0.3), (2, 0.8)],
    "H": [(0, 1.5), (0, 0.3), (1, 0.7)],
}
_RADIAL_SCALE = {"H": 1.0, "O": 1.2, "C": 1.3}  # bohr
_NCART = {0: 1, 1: 3, 2: 6}
N_RAD = 50
N_ANG = 110


@dataclasses.dataclass
class Workload:
    """Flat arrays exactly as they are handed to `kldi_plan_create` (include/kldi.h)."""

    name: str
    symbols: list            # per atom
    atom_xyz: np.ndarray     # [n_atoms,3] bohr
    shell_atom: np.ndarray   # [n_shells] int32
    shell_l: np.ndarray      # [n_shells] int32
    shell_prim_off: np.ndarray  # [n_shells+1] int32
    prim_alpha: np.ndarray   # [n_prim]
    prim_coef: np.ndarray    # [n_prim] (multiplies normalised primitives)
    grid_xyz: np.ndarray     # [n_pts,3] bohr, caller order
    grid_w: np.ndarray       # [n_pts]
    D: np.ndarray            # [n_ao,n_ao] symmetric
    functional: str          # "lda" | "gga"
    eps: float
    seed: int

    @property
    def n_atoms(self) -> int:
        return self.atom_xyz.shape[0]

    @property
    def n_ao(self) -> int:
        return int(sum(_NCART[int(l)] for l in self.shell_l))

    @property
    def n_pts(self) -> int:
        return self.grid_xyz.shape[0]


# ----------------------------------------------------------------------------- geometry
def water_monomer() -> tuple[list, np.ndarray]:
    """O at the origin, O-H 0.9572 A, H-O-H 104.52 deg (BASELINE.json configs[0]); bohr."""
    r = 0.9572 * ANG2BOHR
    half = math.radians(104.52) / 2.0
    xyz = np.array(
        [[0.0, 0.0, 0.0],
         [r * math.sin(half), 0.0, r * math.cos(half)],
         [-r * math.sin(half), 0.0, r * math.cos(half)]]
    )
    return ["O", "H", "H"], xyz


def _random_rotation(rng: np.random.Generator) -> np.ndarray:
    q, r = np.linalg.qr(rng.standard_normal((3, 3)))
    q = q * np.sign(np.diag(r))
    if np.linalg.det(q) < 0:
        q[:, 0] = -q[:, 0]
    return q


def water_cluster_geometry(n_mol: int, seed: int) -> tuple[list, np.ndarray]:
    """n_mol rigid waters, O uniformly random in a cube of side (n_mol*29.9 A^3)^(1/3),
    sequential insertion with redraw until every O-O distance >= 2.7 A; random orientation."""
    rng = np.random.default_rng(seed)
    side = (n_mol * 29.9) ** (1.0 / 3.0) * ANG2BOHR
    dmin2 = (2.7 * ANG2BOHR) ** 2
    _, mono = water_monomer()
    oxy = np.zeros((n_mol, 3))
    n = 0
    while n < n_mol:
        c = rng.uniform(0.0, side, size=3)
        if n == 0 or np.min(np.sum((oxy[:n] - c) ** 2, axis=1)) >= dmin2:
            oxy[n] = c
            n += 1
    xyz = np.zeros((3 * n_mol, 3))
    symbols = []
    for m in range(n_mol):
        rot = _random_rotation(rng)
        xyz[3 * m:3 * m + 3] = mono @ rot.T + oxy[m]
        symbols += ["O", "H", "H"]
    return symbols, xyz


def alkane_geometry(n_c: int) -> tuple[list, np.ndarray]:
    """All-trans zigzag C_n H_{2n+2}: C-C 1.54 A, C-C-C 111.7 deg, C-H 1.09 A, tetrahedral H."""
    cc = 1.54 * ANG2BOHR
    ch = 1.09 * ANG2BOHR
    half = math.radians(111.7) / 2.0
    dx, dz = cc * math.sin(half), cc * math.cos(half)
    carbons = np.array([[i * dx, 0.0, dz * (i % 2)] for i in range(n_c)])
    tet = math.radians(109.4712206)
    normal = np.array([0.0, 1.0, 0.0])  # normal of the carbon plane (xz)
    symbols = ["C"] * n_c
    hs = []
    for i in range(n_c):
        nb = []
        if i > 0:
            nb.append(carbons[i - 1] - carbons[i])
        if i < n_c - 1:
            nb.append(carbons[i + 1] - carbons[i])
        if len(nb) == 2:
            b = nb[0] / np.linalg.norm(nb[0]) + nb[1] / np.linalg.norm(nb[1])
            b /= np.linalg.norm(b)
        else:
            # terminal carbon: the missing neighbour sits where the zigzag would continue
            u = nb[0] / np.linalg.norm(nb[0])
            miss = np.array([-u[0], 0.0, u[2]])
            hs.append(carbons[i] + ch * miss)
            b = u + miss
            b /= np.linalg.norm(b)
        for sgn in (+1.0, -1.0):
            hs.append(carbons[i] + ch * (-b * math.cos(tet / 2.0) + sgn * normal * math.sin(tet / 2.0)))
    symbols += ["H"] * len(hs)
    return symbols, np.vstack([carbons, np.array(hs)])


# ----------------------------------------------------------------------------- basis table
def shells_for(symbols: list):
    atom, ls, off, alpha, coef = [], [], [0], [], []
    for ia, s in enumerate(symbols):
        for (l, a) in _BASIS[s]:
            atom.append(ia)
            ls.append(l)
            alpha.append(a)
            coef.append(1.0)
            off.append(len(alpha))
    return (np.array(atom, np.int32), np.array(ls, np.int32), np.array(off, np.int32),
            np.array(alpha, np.float64), np.array(coef, np.float64))


# ----------------------------------------------------------------------------- quadrature
def atomic_grid(radial_scale: float, n_rad: int = N_RAD, n_ang: int = N_ANG):
    """Points (relative to the nucleus) and weights of one atomic grid, radial-major."""
    i = np.arange(1, n_rad + 1)
    th = i * math.pi / (n_rad + 1)
    x = np.cos(th)
    r = radial_scale * (1.0 + x) / (1.0 - x)
    w_rad = (math.pi / (n_rad + 1)) * np.sin(th) * 2.0 * radial_scale / (1.0 - x) ** 2 * r * r
    k = np.arange(n_ang)
    z = 1.0 - (2.0 * k + 1.0) / n_ang
    phi = k * math.pi * (3.0 - math.sqrt(5.0))
    s = np.sqrt(np.maximum(0.0, 1.0 - z * z))
    unit = np.stack([s * np.cos(phi), s * np.sin(phi), z], axis=1)
    pts = (r[:, None, None] * unit[None, :, :]).reshape(-1, 3)
    w = np.repeat(w_rad * (4.0 * math.pi / n_ang), n_ang)
    return pts, w


def _becke_numpy(atom_xyz: np.ndarray, pts: np.ndarray, owner: np.ndarray, chunk: int = 0):
    """P_owner / sum_B P_B with P_A = prod_{B!=A} s(mu_AB), mu_AB = (r_A-r_B)/R_AB,
    f <- 1.5 f - 0.5 f^3 three times, s = (1-f)/2."""
    n_at = atom_xyz.shape[0]
    out = np.ones(pts.shape[0])
    if n_at == 1:
        return out
    rab = np.linalg.norm(atom_xyz[:, None, :] - atom_xyz[None, :, :], axis=2)
    np.fill_diagonal(rab, 1.0)
    inv = 1.0 / rab
    if chunk <= 0:
        chunk = max(64, int(2.0e7 / (n_at * n_at)))
    for c0 in range(0, pts.shape[0], chunk):
        p = pts[c0:c0 + chunk]
        d = np.linalg.norm(p[:, None, :] - atom_xyz[None, :, :], axis=2)      # [n, A]
        mu = (d[:, :, None] - d[:, None, :]) * inv[None, :, :]                 # [n, A, B]
        for _ in range(3):
            mu = 1.5 * mu - 0.5 * mu ** 3
        s = 0.5 * (1.0 - mu)
        idx = np.arange(n_at)
        s[:, idx, idx] = 1.0
        cell = np.prod(s, axis=2)                                              # [n, A]
        tot = cell.sum(axis=1)
        own = cell[np.arange(p.shape[0]), owner[c0:c0 + chunk]]
        out[c0:c0 + chunk] = own / tot
    return out


def becke_weights(atom_xyz: np.ndarray, pts: np.ndarray, owner: np.ndarray,
                  backend: str = "auto") -> np.ndarray:
    """Becke partition factor of each point for its owning atom.

    backend "numpy" is the definition; "cuda" runs the same formula in a small CUDA helper
    (workloads/becke.cu, built by __graft_entry__.build) because the 256-water case needs
    2.5e12 cell-function evaluations.  "auto" = cuda when a GPU and the helper exist.
    """
    if backend == "auto":
        backend = "numpy"
        try:
            import torch
            if torch.cuda.is_available() and atom_xyz.shape[0] > 8:
                from . import becke_cuda
                if becke_cuda.available():
                    backend = "cuda"
        except Exception:
            backend = "numpy"
    if backend == "cuda":
        from . import becke_cuda
        return becke_cuda.becke_partition(atom_xyz, pts, owner)
    if backend == "none":   # the caller supplies the final weights (named_config(grid_w=...))
        return np.ones(pts.shape[0])
    return _becke_numpy(atom_xyz, pts, owner)


def molecular_grid(symbols: list, atom_xyz: np.ndarray, becke_backend: str = "auto"):
    pts, w, owner = [], [], []
    for ia, s in enumerate(symbols):
        p, ww = atomic_grid(_RADIAL_SCALE[s])
        pts.append(p + atom_xyz[ia])
        w.append(ww)
        owner.append(np.full(p.shape[0], ia, np.int32))
    pts = np.vstack(pts)
    w = np.concatenate(w)
    owner = np.concatenate(owner)
    w = w * becke_weights(atom_xyz, pts, owner, becke_backend)
    return np.ascontiguousarray(pts), np.ascontiguousarray(w)


# ----------------------------------------------------------------------------- density matrix
def density_matrix(n_ao: int, n_occ: int, seed: int) -> np.ndarray:
    """D = 2 Q Q^T, Q the thin-QR orthonormal factor of a seeded N(0,1) n_ao x n_occ matrix."""
    rng = np.random.default_rng(seed)
    q, _ = np.linalg.qr(rng.standard_normal((n_ao, n_occ)))
    d = 2.0 * (q @ q.T)
    return np.ascontiguousarray(0.5 * (d + d.T))


# ----------------------------------------------------------------------------- assembly
def make_workload(name: str, symbols: list, atom_xyz: np.ndarray, n_occ: int, functional: str,
                  eps: float, seed: int, becke_backend: str = "auto") -> Workload:
    sh_atom, sh_l, sh_off, alpha, coef = shells_for(symbols)
    n_ao = int(sum(_NCART[int(l)] for l in sh_l))
    pts, w = molecular_grid(symbols, atom_xyz, becke_backend)
    D = density_matrix(n_ao, n_occ, seed + 1)
    return Workload(name, list(symbols), np.ascontiguousarray(atom_xyz, dtype=np.float64), sh_atom, sh_l,
                    sh_off, alpha, coef, pts, w, D, functional, eps, seed)


_CONFIGS = {
    # name: (kind, size, functional, eps, seed)
    "cfg0": ("water", 1, "lda", 1e-12, 1000),
    "cfg1": ("water", 32, "lda", 1e-12, 1001),
    "cfg2": ("alkane", 60, "lda", 1e-12, 1002),
    "cfg3": ("water", 256, "lda", 1e-12, 1003),
    "cfg4": ("water", 64, "gga", 1e-12, 1004),
}


def named_config(name: str, *, n_override: Optional[int] = None, functional: Optional[str] = None,
                 eps: Optional[float] = None, cache: Optional[bool] = None, becke_backend: str = "auto",
                 grid_w: Optional[np.ndarray] = None) -> Workload:
    """BASELINE.json configs[0..4] as "cfg0".."cfg4".  `n_override` shrinks the molecule count
    (waters or carbons) for reduced-size parity cases; same recipe, same seed.  `grid_w`: final quadrature
    weights of this very config written earlier by this generator (e.g. with the CUDA Becke helper on a GPU box);
    the Becke step is then skipped — for CPU-only runs of the large configs."""
    kind, size, fn, e, seed = _CONFIGS[name]
    if cache is None:
        cache = os.environ.get("KLDI_WL_CACHE", "0") == "1"
    if n_override is not None:
        size = n_override
    if functional is not None:
        fn = functional
    if eps is not None:
        e = eps
    tag = f"{name}_{kind}{size}_{fn}"
    cache_dir = os.path.join(os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__)))),
                             "baseline", "_ref")
    path = os.path.join(cache_dir, f"wl_{tag}.npz")
    if cache and os.path.exists(path):
        z = np.load(path, allow_pickle=False)
        return Workload(tag, [str(s) for s in z["symbols"]], z["atom_xyz"], z["shell_atom"], z["shell_l"],
                        z["shell_prim_off"], z["prim_alpha"], z["prim_coef"], z["grid_xyz"], z["grid_w"],
                        z["D"], fn, e, seed)
    if kind == "water":
        symbols, xyz = water_monomer() if size == 1 else water_cluster_geometry(size, seed)
        n_occ = 5 * size
    else:
        symbols, xyz = alkane_geometry(size)
        n_occ = (6 * size + (2 * size + 2)) // 2
    wl = make_workload(tag, symbols, xyz, n_occ, fn, e, seed, "none" if grid_w is not None else becke_backend)
    if grid_w is not None:
        grid_w = np.ascontiguousarray(grid_w, dtype=np.float64)
        if grid_w.shape != wl.grid_w.shape:
            raise ValueError(f"grid_w has shape {grid_w.shape}, config needs {wl.grid_w.shape}")
        wl.grid_w = grid_w
        return wl
    if cache and wl.n_pts >= 200_000:
        try:
            os.makedirs(cache_dir, exist_ok=True)
            np.savez(path, symbols=np.array(wl.symbols), atom_xyz=wl.atom_xyz, shell_atom=wl.shell_atom,
                     shell_l=wl.shell_l, shell_prim_off=wl.shell_prim_off, prim_alpha=wl.prim_alpha,
                     prim_coef=wl.prim_coef, grid_xyz=wl.grid_xyz, grid_w=wl.grid_w, D=wl.D)
        except OSError:
            pass
    return wl
