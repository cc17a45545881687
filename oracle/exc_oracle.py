"""CPU ORACLE for the KerneLDI EXC hot path — TEST INFRASTRUCTURE, NOT THE PRODUCT.

Plain, slow, dense, *unscreened* FP64 numpy implementation of what the hot path computes,
written from /root/reference/PAPER.md (cited as PAPER.md:<line>) and the readings in
DESIGN.md §3.  It shares no code, tables or helpers with the CUDA path
(paper_2605_10363_b200/csrc) and imports nothing from the package.  Only tests/,
__graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import it.

What the method reaches: with thresholds -> 0 the block-filtered products (Eq. 16;
PAPER.md:209, Eq. 18) are exactly the dense products (Eq. 7), so the oracle is
the plain definition written out:

  Phi_{g,mu} = chi_mu(r_g)                                  PAPER.md:67  (Eq. 2)
  rho_g      = sum_{mu,nu} D_{mu,nu} chi_mu(r_g) chi_nu(r_g)  PAPER.md:426 (via R = D Phi, Eq. 4)
  E_xc       = sum_g w_g e(rho_g[, sigma_g])                PAPER.md:57-61 (quadrature of Eq. 1)
  V_{mu,nu}  = sum_g w_g v_g chi_mu(r_g) chi_nu(r_g)         PAPER.md:61 (Eq. 1), PAPER.md:80 (Eq. 5), b = 1

There is no blocking, screening, fusion or reordering here beyond processing the grid in
chunks (a sum over g is a sum over chunks of g).  numpy's matmul (BLAS dgemm) serves as the
dense-product step; `brute_force_lda` below is the same thing as explicit Python loops.

Pins (tests/test_oracle_pins.py, all `-m "not gpu"`): analytic Gaussian overlap => diag(S)=1 and
int rho = Tr(D S); closed-form Slater energy of one s-Gaussian; V symmetric; central finite
differences dE/dD = V (LDA and PBE-x); brute-force loops on single water; PBE-x limits; central finite
differences of E in the atom coordinates (fixed grid) = exc_nuclear_gradient_lda / _gga (AO second derivatives from
central differences of the analytic first ones); kinetic-energy density: closed
form int tau = 3 alpha n / 2 of one s-Gaussian, AO gradients from finite differences, Tr(D V^tau) = sum wv tau.
Absolute PBE-x (and Slater) energies: the four decimals the PBE paper prints for the exchange energy of
the hydrogen atom (tests/golden/pbe_x_hydrogen.txt), by a 1-D radial integral of slater() / pbe_x().
"""
from __future__ import annotations

import math

import numpy as np

# ---- constants of the spin-restricted exchange functionals
C_X = 0.75 * (3.0 / math.pi) ** (1.0 / 3.0)
K_S = (3.0 * math.pi ** 2) ** (2.0 / 3.0)
KAPPA = 0.804
MU = 0.21951
RHO_CUT = 1e-20          # reading A9: below this density e = v_rho = v_sigma = 0


# ----------------------------------------------------------------------------- basis functions
def cart_components(l: int):
    """Cartesian powers (i,j,k), i+j+k = l, in the boundary order x,y,z / xx,xy,xz,yy,yz,zz
    (reading A1)."""
    return [(i, j, l - i - j) for i in range(l, -1, -1) for j in range(l - i, -1, -1)]


def _dfact(n: int) -> float:
    """(n)!! with (-1)!! = 1."""
    out = 1.0
    while n > 1:
        out *= n
        n -= 2
    return out


def norm_const(alpha: float, i: int, j: int, k: int) -> float:
    """Normalisation of x^i y^j z^k exp(-alpha r^2) so that <chi|chi> = 1 (reading A1):
    (2a/pi)^{3/4} (4a)^{l/2} / sqrt((2i-1)!!(2j-1)!!(2k-1)!!)."""
    l = i + j + k
    return ((2.0 * alpha / math.pi) ** 0.75 * (4.0 * alpha) ** (0.5 * l)
            / math.sqrt(_dfact(2 * i - 1) * _dfact(2 * j - 1) * _dfact(2 * k - 1)))


def n_ao_of(shell_l) -> int:
    return int(sum((int(l) + 1) * (int(l) + 2) // 2 for l in shell_l))


def ao_values(atom_xyz, shell_atom, shell_l, shell_prim_off, prim_alpha, prim_coef, pts, deriv: bool = False):
    """Phi[g,mu] = chi_mu(r_g) (Eq. 2) for contracted Cartesian Gaussians
    chi = sum_prim coef * N * (x-Ax)^i (y-Ay)^j (z-Az)^k exp(-alpha |r-A|^2).
    With deriv=True also the analytic gradient dPhi[c,g,mu] = d chi_mu / d r_c:
    d/dx [x^i e^{-a r^2}] = (i x^{i-1} - 2 a x^{i+1}) e^{-a r^2}."""
    pts = np.asarray(pts, dtype=np.float64)
    n_pts = pts.shape[0]
    n_ao = n_ao_of(shell_l)
    phi = np.zeros((n_pts, n_ao))
    dphi = np.zeros((3, n_pts, n_ao)) if deriv else None
    col = 0
    for s in range(len(shell_l)):
        l = int(shell_l[s])
        dx = pts - np.asarray(atom_xyz[int(shell_atom[s])])[None, :]
        r2 = np.sum(dx * dx, axis=1)
        for (i, j, k) in cart_components(l):
            pw = (i, j, k)
            for p in range(int(shell_prim_off[s]), int(shell_prim_off[s + 1])):
                a = float(prim_alpha[p])
                c = float(prim_coef[p]) * norm_const(a, i, j, k)
                ex = np.exp(-a * r2)
                mono = [dx[:, d] ** pw[d] for d in range(3)]
                phi[:, col] += c * mono[0] * mono[1] * mono[2] * ex
                if deriv:
                    for d in range(3):
                        n = pw[d]
                        dm = -2.0 * a * dx[:, d] ** (n + 1)
                        if n > 0:
                            dm = dm + n * dx[:, d] ** (n - 1)
                        other = mono[(d + 1) % 3] * mono[(d + 2) % 3]
                        dphi[d, :, col] += c * dm * other * ex
            col += 1
    return (phi, dphi) if deriv else phi


# ----------------------------------------------------------------------------- density
def density(phi, D):
    """rho_g = sum_{mu,nu} D_{mu,nu} Phi_{g,mu} Phi_{g,nu}; X = Phi D is the
    paper's R = D Phi (Eq. 4) in grid-major storage."""
    X = phi @ D
    return np.sum(X * phi, axis=1)


def density_gradient(phi, dphi, D):
    """d_c rho_g = sum_{mu,nu} D_{mu,nu} (d_c chi_mu chi_nu + chi_mu d_c chi_nu); general
    (not assuming D symmetric) so that single-element finite differences are exact."""
    XT = phi @ D.T      # XT[g,mu] = sum_nu D[mu,nu] Phi[g,nu]
    X = phi @ D         # X[g,nu]  = sum_mu Phi[g,mu] D[mu,nu]
    return np.stack([np.sum(dphi[c] * XT, axis=1) + np.sum(X * dphi[c], axis=1) for c in range(3)])


# ----------------------------------------------------------------------------- functionals
def slater(rho):
    """Spin-restricted Slater exchange: e = -C_x rho^{4/3}, v_rho = -(4/3) C_x rho^{1/3};
    zero below RHO_CUT (reading A9)."""
    rho = np.asarray(rho, dtype=np.float64)
    ok = rho >= RHO_CUT
    r = np.where(ok, rho, 1.0)
    c = np.cbrt(r)
    e = np.where(ok, -C_X * r * c, 0.0)
    v = np.where(ok, -(4.0 / 3.0) * C_X * c, 0.0)
    return e, v


def pbe_x(rho, sigma, mu: float = MU, kappa: float = KAPPA):
    """Slater x PBE exchange enhancement F(s) = 1 + kappa - kappa/(1 + mu s^2/kappa)
    (BASELINE.json configs[4]); s^2 = sigma / (4 K_S rho^{8/3}), sigma = |grad rho|^2.
    Returns e, v_rho = de/drho, v_sigma = de/dsigma."""
    rho = np.asarray(rho, dtype=np.float64)
    sigma = np.asarray(sigma, dtype=np.float64)
    ok = rho >= RHO_CUT
    r = np.where(ok, rho, 1.0)
    c = np.cbrt(r)              # rho^{1/3}
    r43 = r * c
    s2 = np.where(ok, sigma, 0.0) / (4.0 * K_S * r43 * r43)
    den = 1.0 + mu * s2 / kappa
    F = 1.0 + kappa - kappa / den
    Fp = mu / (den * den)       # dF/d(s^2)
    e = np.where(ok, -C_X * r43 * F, 0.0)
    v_rho = np.where(ok, -C_X * c * ((4.0 / 3.0) * F - (8.0 / 3.0) * s2 * Fp), 0.0)
    v_sigma = np.where(ok, -C_X * Fp / (4.0 * K_S * r43), 0.0)
    return e, v_rho, v_sigma


# ----------------------------------------------------------------------------- potential matrix
def vxc_lda_from_wv(phi, wv):
    """V = Phi^T diag(wv) Phi (Eq. 5 with b = 1; wv = w*v_xc, Eq. 3)."""
    return phi.T @ (wv[:, None] * phi)


def vxc_lda_block_from_wv(phi, wv, rows, cols):
    """The sub-block V[rows][:, cols] of vxc_lda_from_wv, from the same definition V_{mu,nu} = sum_g wv_g chi_mu chi_nu
    (Eq. 5) restricted to the wanted AO rows and columns — for stored reference values at sizes where
    forming all of V on the CPU takes hours (tests/golden/make_cfg3_golden.py)."""
    return phi[:, rows].T @ (wv[:, None] * phi[:, cols])


def vxc_gga_from_wv(phi, dphi, wv4):
    """V = B + B^T, B = Phi^T Z, Z = 1/2 wv0 Phi + sum_c wv_c d_c Phi, with wv0 = w v_rho and
    wv_c = 2 w v_sigma d_c rho (the boundary convention of kldi_build_vxc, include/kldi.h)."""
    Z = 0.5 * wv4[0][:, None] * phi
    for c in range(3):
        Z = Z + wv4[1 + c][:, None] * dphi[c]
    B = phi.T @ Z
    return B + B.T


def _basis_args(wl):
    return (wl.atom_xyz, wl.shell_atom, wl.shell_l, wl.shell_prim_off, wl.prim_alpha, wl.prim_coef)


def exc(basis, pts, w, D, functional: str = "lda", chunk: int = 8192, want_v: bool = True):
    """The whole path, dense: AO values -> rho (-> grad rho) -> functional -> E_xc and V.

    `basis` = (atom_xyz, shell_atom, shell_l, shell_prim_off, prim_alpha, prim_coef).
    Returns dict(E, V, rho, drho (GGA), wv).  E is accumulated with math.fsum over the
    per-point terms (exactly rounded sum).  The grid is processed in chunks of `chunk` points.
    """
    pts = np.asarray(pts, dtype=np.float64)
    w = np.asarray(w, dtype=np.float64)
    D = np.asarray(D, dtype=np.float64)
    n_pts = pts.shape[0]
    n_ao = D.shape[0]
    gga = functional == "gga"
    rho = np.zeros(n_pts)
    drho = np.zeros((3, n_pts)) if gga else None
    wv = np.zeros((4, n_pts)) if gga else np.zeros(n_pts)
    V = np.zeros((n_ao, n_ao)) if want_v else None
    e_terms = []
    for c0 in range(0, n_pts, chunk):
        sl = slice(c0, min(n_pts, c0 + chunk))
        if gga:
            phi, dphi = ao_values(*basis, pts[sl], deriv=True)
            rho[sl] = density(phi, D)
            drho[:, sl] = density_gradient(phi, dphi, D)
            sigma = np.sum(drho[:, sl] ** 2, axis=0)
            e, v_rho, v_sigma = pbe_x(rho[sl], sigma)
            wv[0, sl] = w[sl] * v_rho
            for c in range(3):
                wv[1 + c, sl] = 2.0 * w[sl] * v_sigma * drho[c, sl]
            if want_v:
                V += vxc_gga_from_wv(phi, dphi, wv[:, sl])
        else:
            phi = ao_values(*basis, pts[sl])
            rho[sl] = density(phi, D)
            e, v_rho = slater(rho[sl])
            wv[sl] = w[sl] * v_rho
            if want_v:
                V += vxc_lda_from_wv(phi, wv[sl])
        e_terms.append(w[sl] * e)
    E = math.fsum(np.concatenate(e_terms).tolist())
    return {"E": E, "V": V, "rho": rho, "drho": drho, "wv": wv}


def exc_energy_from_rho(w, rho, drho=None, functional: str = "lda") -> float:
    """E_xc = sum_g w_g e_g for a given density (used to check energies at sizes where the dense
    density itself is too expensive to recompute on the CPU)."""
    if functional == "gga":
        e, _, _ = pbe_x(rho, np.sum(np.asarray(drho) ** 2, axis=0))
    else:
        e, _ = slater(rho)
    return math.fsum((np.asarray(w) * e).tolist())


# ----------------------------------------------------------------------------- meta-GGA contractions
def kinetic_energy_density(dphi, D):
    """tau_g = 1/2 sum_{mu,nu} D_{mu,nu} grad chi_mu(r_g) . grad chi_nu(r_g): the third density-like variable of the
    meta-GGA class the paper runs (M06-2X; the functional itself is out of scope).  The same product
    as the density build (Eq. 4) with d_c Phi in place of Phi, summed over c."""
    return 0.5 * sum(np.sum((dphi[c] @ D) * dphi[c], axis=1) for c in range(3))


def vtau_from_wv(dphi, wv):
    """V^tau = 1/2 sum_c (d_c Phi)^T diag(wv) (d_c Phi), wv = w * v_tau: dE/dD_{mu,nu} of E = sum_g w_g e(tau_g)
    (Eq. 5, with d_c Phi in place of Phi)."""
    return 0.5 * sum(dphi[c].T @ (wv[:, None] * dphi[c]) for c in range(3))


# ----------------------------------------------------------------------------- nuclear gradient
def exc_nuclear_gradient_lda(basis, pts, w, D, chunk: int = 8192):
    """EXC nuclear-gradient contraction, LDA, at fixed density matrix and FIXED quadrature (points and weights do not
    move with the atoms: no grid response) — the paper's second workload, for which it prints no
    formula; this is the chain rule on E_xc = sum_g w_g e(rho_g) written out (G1):

        chi_mu depends on the nucleus A it sits on through r - A  =>  d chi_mu(r_g) / d A_c = - d_c chi_mu(r_g),
        d rho_g / d A_c = -2 sum_{mu on A} d_c chi_mu(r_g) X_{g,mu},   X = Phi D  (D symmetric, Eq. 4),
        dE_xc / d A_c   = sum_g w_g v_rho(rho_g) d rho_g / d A_c
                        = -2 sum_g w_g v_g sum_{mu on A} d_c Phi_{g,mu} X_{g,mu}.

    Returns grad [n_atoms][3].  Pinned by central finite differences of the oracle's own energy in the atom
    coordinates with the same points and weights (tests/test_oracle_pins.py)."""
    atom_xyz, shell_atom, shell_l = basis[0], basis[1], basis[2]
    ao_atom = np.concatenate([[int(shell_atom[s])] * ((int(l) + 1) * (int(l) + 2) // 2) for s, l in enumerate(shell_l)])
    n_atoms = len(atom_xyz)
    grad = np.zeros((n_atoms, 3))
    for c0 in range(0, len(pts), chunk):
        phi, dphi = ao_values(*basis, pts[c0:c0 + chunk], deriv=True)
        rho = density(phi, D)
        _, v = slater(rho)
        wv = w[c0:c0 + chunk] * v
        X = phi @ D
        for c in range(3):
            per_ao = -2.0 * np.einsum("g,gm,gm->m", wv, dphi[c], X)
            np.add.at(grad[:, c], ao_atom, per_ao)
    return grad


def ao_hessians(atom_xyz, shell_atom, shell_l, shell_prim_off, prim_alpha, prim_coef, pts):
    """Second derivatives d2Phi[c, d, g, mu] = d^2 chi_mu / d r_c d r_d of the contracted Cartesian Gaussians of
    ao_values.  A primitive is a product of 1-D factors u(x) = x^n e^{-a x^2}, so
        u'  = (n x^{n-1} - 2 a x^{n+1}) e^{-a x^2},
        u'' = (n (n-1) x^{n-2} - 2 a (2 n + 1) x^n + 4 a^2 x^{n+2}) e^{-a x^2},
    the mixed second derivative is u_c' u_d' u_e and the pure one u_c'' u_d u_e.  Pinned by central differences of the
    analytic gradients of ao_values (tests/test_oracle_pins.py)."""
    pts = np.asarray(pts, dtype=np.float64)
    n_pts = pts.shape[0]
    n_ao = n_ao_of(shell_l)
    out = np.zeros((3, 3, n_pts, n_ao))
    col = 0
    for s in range(len(shell_l)):
        l = int(shell_l[s])
        dx = pts - np.asarray(atom_xyz[int(shell_atom[s])])[None, :]
        for pw in cart_components(l):
            for p in range(int(shell_prim_off[s]), int(shell_prim_off[s + 1])):
                a = float(prim_alpha[p])
                c = float(prim_coef[p]) * norm_const(a, *pw)
                u0, u1, u2 = [], [], []
                for d in range(3):
                    x, n = dx[:, d], pw[d]
                    e = np.exp(-a * x * x)
                    u0.append(x ** n * e)
                    t1 = -2.0 * a * x ** (n + 1)
                    if n > 0:
                        t1 = t1 + n * x ** (n - 1)
                    u1.append(t1 * e)
                    t2 = -2.0 * a * (2 * n + 1) * x ** n + 4.0 * a * a * x ** (n + 2)
                    if n > 1:
                        t2 = t2 + n * (n - 1) * x ** (n - 2)
                    u2.append(t2 * e)
                for d1 in range(3):
                    for d2 in range(3):
                        f = [u0[0], u0[1], u0[2]]
                        if d1 == d2:
                            f[d1] = u2[d1]
                        else:
                            f[d1], f[d2] = u1[d1], u1[d2]
                        out[d1, d2, :, col] += c * f[0] * f[1] * f[2]
            col += 1
    return out


def exc_nuclear_gradient_gga(basis, pts, w, D, chunk: int = 4096):
    """EXC nuclear-gradient contraction for the GGA functional (Slater x PBE enhancement), fixed density matrix and FIXED
    quadrature, same reading G1 as exc_nuclear_gradient_lda: the chain rule on E_xc = sum_g w_g e(rho_g, sigma_g),
    sigma = |grad rho|^2, with d chi_mu / d A_c = - d_c chi_mu for mu on A (D symmetric, X = Phi D, X^d = d_d Phi D):

        d rho / d A_c        = -2 sum_{mu on A} d_c Phi_mu X_mu
        d (d_d rho) / d A_c  = -2 sum_{mu on A} [ d_c d_d Phi_mu X_mu + d_c Phi_mu X^d_mu ]
        dE / d A_c = sum_g [ wv0 d rho / d A_c + sum_d wv_d d (d_d rho) / d A_c ],
        wv0 = w v_rho,  wv_d = 2 w v_sigma d_d rho          (the wv convention of kldi_build_vxc).

    Returns grad [n_atoms][3].  Pinned by central differences of the oracle's GGA energy in the atom coordinates."""
    atom_xyz, shell_atom, shell_l = basis[0], basis[1], basis[2]
    ao_atom = np.concatenate([[int(shell_atom[s])] * ((int(l) + 1) * (int(l) + 2) // 2) for s, l in enumerate(shell_l)])
    grad = np.zeros((len(atom_xyz), 3))
    for c0 in range(0, len(pts), chunk):
        p = pts[c0:c0 + chunk]
        phi, dphi = ao_values(*basis, p, deriv=True)
        hess = ao_hessians(*basis, p)
        rho = density(phi, D)
        drho = density_gradient(phi, dphi, D)
        _, v_rho, v_sigma = pbe_x(rho, np.sum(drho ** 2, axis=0))
        ww = w[c0:c0 + chunk]
        wv0 = ww * v_rho
        wvd = [2.0 * ww * v_sigma * drho[d] for d in range(3)]
        X = phi @ D
        Xd = [dphi[d] @ D for d in range(3)]
        for c in range(3):
            per_ao = -2.0 * np.einsum("g,gm,gm->m", wv0, dphi[c], X)
            for d in range(3):
                per_ao = per_ao - 2.0 * np.einsum("g,gm,gm->m", wvd[d], hess[c, d], X)
                per_ao = per_ao - 2.0 * np.einsum("g,gm,gm->m", wvd[d], dphi[c], Xd[d])
            np.add.at(grad[:, c], ao_atom, per_ao)
    return grad


# ----------------------------------------------------------------------------- sampled entries
def rho_at_points(basis, pts_sample, D, want_grad: bool = False):
    """rho (and grad rho) at a handful of points, each from the plain definition."""
    if want_grad:
        phi, dphi = ao_values(*basis, pts_sample, deriv=True)
        return density(phi, D), density_gradient(phi, dphi, D)
    phi = ao_values(*basis, pts_sample)
    return density(phi, D)


def single_ao_values(basis, ao_index: int, pts, deriv: bool = False, chunk: int = 262144):
    """Column `ao_index` of Phi (and of its gradient) on all points, without forming Phi."""
    atom_xyz, shell_atom, shell_l, shell_prim_off, prim_alpha, prim_coef = basis
    col = 0
    for s in range(len(shell_l)):
        n = (int(shell_l[s]) + 1) * (int(shell_l[s]) + 2) // 2
        if ao_index < col + n:
            sub = (atom_xyz, np.array([shell_atom[s]]), np.array([shell_l[s]]),
                   np.array([0, shell_prim_off[s + 1] - shell_prim_off[s]]),
                   prim_alpha[shell_prim_off[s]:shell_prim_off[s + 1]],
                   prim_coef[shell_prim_off[s]:shell_prim_off[s + 1]])
            k = ao_index - col
            vals, grads = [], []
            for c0 in range(0, len(pts), chunk):
                out = ao_values(*sub, pts[c0:c0 + chunk], deriv=deriv)
                if deriv:
                    vals.append(out[0][:, k])
                    grads.append(out[1][:, :, k])
                else:
                    vals.append(out[:, k])
            if deriv:
                return np.concatenate(vals), np.concatenate(grads, axis=1)
            return np.concatenate(vals)
        col += n
    raise IndexError(ao_index)


def vxc_entries_from_wv(basis, pts, wv, pairs, gga: bool = False):
    """Selected V_{mu,nu} = sum_g wv_g chi_mu chi_nu (LDA) or the GGA expression of
    vxc_gga_from_wv, one entry at a time over ALL grid points (for full-size sampled parity)."""
    out = []
    cache = {}

    def col(m):
        if m not in cache:
            cache[m] = single_ao_values(basis, m, pts, deriv=gga)
        return cache[m]

    for (m, n) in pairs:
        if gga:
            pm, gm = col(m)
            pn, gn = col(n)
            t = wv[0] * pm * pn
            for c in range(3):
                t = t + wv[1 + c] * (gm[c] * pn + pm * gn[c])
            out.append(math.fsum(t.tolist()))
        else:
            out.append(math.fsum((wv * col(m) * col(n)).tolist()))
    return np.array(out)


# ----------------------------------------------------------------------------- brute force
def brute_force_lda(basis, pts, w, D):
    """Invariant (v): the same LDA path as explicit Python loops over g, mu, nu — no matmul,
    no vectorisation across AOs.  Only for tiny inputs (single water)."""
    atom_xyz, shell_atom, shell_l, shell_prim_off, prim_alpha, prim_coef = basis
    aos = []   # (atom, i, j, k, [(alpha, coef*N)])
    for s in range(len(shell_l)):
        for (i, j, k) in cart_components(int(shell_l[s])):
            prims = [(float(prim_alpha[p]), float(prim_coef[p]) * norm_const(float(prim_alpha[p]), i, j, k))
                     for p in range(int(shell_prim_off[s]), int(shell_prim_off[s + 1]))]
            aos.append((int(shell_atom[s]), i, j, k, prims))
    n_ao = len(aos)
    rho = [0.0] * len(pts)
    V = [[0.0] * n_ao for _ in range(n_ao)]
    e_terms = []
    for g in range(len(pts)):
        chi = []
        for (ia, i, j, k, prims) in aos:
            x = pts[g][0] - atom_xyz[ia][0]
            y = pts[g][1] - atom_xyz[ia][1]
            z = pts[g][2] - atom_xyz[ia][2]
            r2 = x * x + y * y + z * z
            val = 0.0
            for (a, c) in prims:
                val += c * (x ** i) * (y ** j) * (z ** k) * math.exp(-a * r2)
            chi.append(val)
        r = 0.0
        for m in range(n_ao):
            for n in range(n_ao):
                r += D[m][n] * chi[m] * chi[n]
        rho[g] = r
        if r >= RHO_CUT:
            c13 = r ** (1.0 / 3.0)
            e_terms.append(w[g] * (-C_X * r * c13))
            wv = w[g] * (-(4.0 / 3.0) * C_X * c13)
            for m in range(n_ao):
                t = wv * chi[m]
                for n in range(n_ao):
                    V[m][n] += t * chi[n]
    return {"E": math.fsum(e_terms), "V": np.array(V), "rho": np.array(rho)}
