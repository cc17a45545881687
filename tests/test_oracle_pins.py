"""Pins of the CPU oracle against things the mathematics fixes (BASELINE.json invariants (i)-(v)).
None of these re-types the oracle's own formula: each uses a closed form, an identity, a finite
difference or explicit loops."""
import math
import os

import numpy as np
import pytest

from oracle import exc_oracle as O
from oracle import overlap as OV
from paper_2605_10363_b200 import workloads as W

HERE = os.path.dirname(os.path.abspath(__file__))


def basis_of(wl):
    return (wl.atom_xyz, wl.shell_atom, wl.shell_l, wl.shell_prim_off, wl.prim_alpha, wl.prim_coef)


@pytest.fixture(scope="module")
def water():
    return W.named_config("cfg0")


def test_component_order_and_count():
    assert O.cart_components(1) == [(1, 0, 0), (0, 1, 0), (0, 0, 1)]
    assert O.cart_components(2) == [(2, 0, 0), (1, 1, 0), (1, 0, 1), (0, 2, 0), (0, 1, 1), (0, 0, 2)]


def test_overlap_diagonal_is_one(water):
    S = OV.overlap_matrix(*basis_of(water))
    assert np.max(np.abs(np.diag(S) - 1.0)) < 1e-14
    assert np.max(np.abs(S - S.T)) == 0.0
    # a textbook special case: two normalised s-Gaussians a,b at distance R:
    # S = (2 sqrt(ab)/(a+b))^{3/2} exp(-ab/(a+b) R^2)
    a, b, R = 1.5, 0.3, 1.7
    xyz = np.array([[0.0, 0, 0], [0, 0, R]])
    S2 = OV.overlap_matrix(xyz, [0, 1], [0, 0], [0, 1, 2], [a, b], [1.0, 1.0])
    ref = (2 * math.sqrt(a * b) / (a + b)) ** 1.5 * math.exp(-a * b / (a + b) * R * R)
    assert abs(S2[0, 1] - ref) < 1e-15


def test_slater_closed_form_single_s_gaussian():
    """Invariant (iv) + quadrature weights: one normalised s-Gaussian, alpha=1, n=2."""
    alpha, n, ref = np.loadtxt(os.path.join(HERE, "golden", "slater_s_gaussian.txt"))
    formula = -0.75 * (3 / math.pi) ** (1 / 3) * n ** (4 / 3) * (2 * alpha / math.pi) ** 2 * (3 * math.pi / (8 * alpha)) ** 1.5
    assert abs(formula - ref) < 1e-10          # the fixture is the closed form
    pts, w = W.atomic_grid(1.0)
    basis = (np.zeros((1, 3)), np.array([0]), np.array([0]), np.array([0, 1]), np.array([alpha]), np.array([1.0]))
    out = O.exc(basis, pts, w, np.array([[n]]), "lda")
    assert abs(out["E"] - ref) < 2e-10 * abs(ref) + 1e-10
    # number of electrons: exact angular rule for an s density
    assert abs(float(np.sum(w * out["rho"])) - n) < 1e-9
    # V is a 1x1 matrix: <chi| v |chi> = -(4/3) C_x n^{1/3} int rho1^{4/3}  (rho1 = density for n=1)
    v_ref = (4.0 / 3.0) * ref / n
    assert abs(out["V"][0, 0] - v_ref) < 1e-9


def test_electron_count_equals_trace_DS(water):
    """Invariant (i): int rho = Tr(D S).  1e-6 needs a verification grid (the 110-point equal-weight
    angular rule limits the config grid to ~4e-4); the config grid must reach 1e-3."""
    S = OV.overlap_matrix(*basis_of(water))
    ne = float(np.sum(water.D * S))
    out = O.exc(basis_of(water), water.grid_xyz, water.grid_w, water.D, "lda", want_v=False)
    err_cfg = abs(float(np.sum(water.grid_w * out["rho"])) - ne) / abs(ne)
    assert err_cfg < 1e-3
    # verification grid: 80 radial x 16000 angular per atom
    pts, w, owner = [], [], []
    for ia, s in enumerate(water.symbols):
        p, ww = W.atomic_grid({"H": 1.0, "O": 1.2}[s], n_rad=80, n_ang=16000)
        pts.append(p + water.atom_xyz[ia]); w.append(ww); owner.append(np.full(len(ww), ia, np.int32))
    pts = np.vstack(pts); w = np.concatenate(w); owner = np.concatenate(owner)
    w = w * W.becke_weights(water.atom_xyz, pts, owner, backend="numpy")
    rho = np.concatenate([O.rho_at_points(basis_of(water), pts[c:c + 65536], water.D)
                          for c in range(0, len(pts), 65536)])
    err_fine = abs(float(np.sum(w * rho)) - ne) / abs(ne)
    assert err_fine < 1e-6
    assert err_fine < err_cfg


def test_v_symmetric_and_bruteforce(water):
    """Invariants (ii) and (v) on single water (every 8th grid point for the Python loops)."""
    sl = slice(0, None, 8)
    pts, w = water.grid_xyz[sl], water.grid_w[sl]
    out = O.exc(basis_of(water), pts, w, water.D, "lda", chunk=500)
    V = out["V"]
    assert np.max(np.abs(V - V.T)) <= 1e-13 * np.max(np.abs(V))
    bf = O.brute_force_lda(basis_of(water), pts.tolist(), w.tolist(), water.D.tolist())
    assert np.max(np.abs(bf["rho"] - out["rho"])) < 1e-12 * max(1.0, np.max(np.abs(out["rho"])))
    assert abs(bf["E"] - out["E"]) < 1e-11 * abs(out["E"])
    assert np.max(np.abs(bf["V"] - V)) < 1e-11 * np.max(np.abs(V))
    # chunking must not matter
    out2 = O.exc(basis_of(water), pts, w, water.D, "lda", chunk=100000)
    assert np.max(np.abs(out2["V"] - V)) < 1e-12 * np.max(np.abs(V))


@pytest.mark.parametrize("functional", ["lda", "gga"])
def test_finite_difference_dE_dD_equals_V(water, functional):
    """Invariant (iii): central differences of E_xc w.r.t. single elements D_{mu,nu} give V_{mu,nu}."""
    basis = basis_of(water)
    out = O.exc(basis, water.grid_xyz, water.grid_w, water.D, functional)
    V = out["V"]
    assert np.max(np.abs(V - V.T)) <= 1e-12 * np.max(np.abs(V))
    h = 3e-5
    scale = np.max(np.abs(V))
    for (m, n) in [(0, 0), (2, 7), (7, 2), (3, 16), (12, 24), (20, 21)]:
        Dp = water.D.copy(); Dp[m, n] += h
        Dm = water.D.copy(); Dm[m, n] -= h
        ep = O.exc(basis, water.grid_xyz, water.grid_w, Dp, functional, want_v=False)["E"]
        em = O.exc(basis, water.grid_xyz, water.grid_w, Dm, functional, want_v=False)["E"]
        fd = (ep - em) / (2 * h)
        assert abs(fd - V[m, n]) < 1e-6 * scale, (functional, m, n, fd, V[m, n])


def test_ao_gradient_matches_finite_difference(water):
    basis = basis_of(water)
    rng = np.random.default_rng(5)
    pts = rng.uniform(-2.5, 2.5, size=(40, 3))
    phi, dphi = O.ao_values(*basis, pts, deriv=True)
    h = 1e-5
    for c in range(3):
        e = np.zeros(3); e[c] = h
        fd = (O.ao_values(*basis, pts + e) - O.ao_values(*basis, pts - e)) / (2 * h)
        assert np.max(np.abs(fd - dphi[c])) < 1e-8
    # density gradient against the density at displaced points
    rho, drho = O.rho_at_points(basis, pts, water.D, want_grad=True)
    for c in range(3):
        e = np.zeros(3); e[c] = h
        fd = (O.rho_at_points(basis, pts + e, water.D) - O.rho_at_points(basis, pts - e, water.D)) / (2 * h)
        assert np.max(np.abs(fd - drho[c])) < 1e-7


def test_v_block_is_the_block_of_v(water):
    """vxc_lda_block_from_wv (used for the stored cfg3 reference) is the sub-block of the pinned full V, and one of its
    entries equals the explicit sum over grid points."""
    basis = basis_of(water)
    phi = O.ao_values(*basis, water.grid_xyz)
    wv = water.grid_w * np.cos(np.arange(water.n_pts))
    V = O.vxc_lda_from_wv(phi, wv)
    rows, cols = np.array([0, 7, 24]), np.arange(0, 25, 3)
    B = O.vxc_lda_block_from_wv(phi, wv, rows, cols)
    assert B.shape == (3, len(cols)) and np.max(np.abs(B - V[np.ix_(rows, cols)])) < 1e-13
    assert abs(B[1, 2] - sum(wv[g] * phi[g, 7] * phi[g, 6] for g in range(water.n_pts))) < 1e-12


def test_nuclear_gradient_lda_matches_finite_difference_of_energy(water):
    """the paper prints no gradient formula, so the oracle's EXC nuclear-gradient contraction is
    pinned by central differences of the (closed-form-pinned) energy in the atom coordinates, grid held fixed, and
    by the translation identity sum_A dE/dA_c = -sum_g w_g v_g d_c rho_g (moving every atom = moving the grid back)."""
    basis = basis_of(water)
    g = O.exc_nuclear_gradient_lda(basis, water.grid_xyz, water.grid_w, water.D)
    assert g.shape == (3, 3) and np.max(np.abs(g)) > 1e-3
    h = 1e-4
    for (a, c) in [(0, 0), (0, 2), (1, 1), (2, 0), (2, 2)]:
        e = []
        for sgn in (+1, -1):
            xyz = np.array(basis[0], dtype=np.float64, copy=True)
            xyz[a, c] += sgn * h
            e.append(O.exc((xyz,) + tuple(basis[1:]), water.grid_xyz, water.grid_w, water.D, "lda", want_v=False)["E"])
        fd = (e[0] - e[1]) / (2 * h)
        assert abs(fd - g[a, c]) < 1e-6 * np.max(np.abs(g)), (a, c, fd, g[a, c])
    phi, dphi = O.ao_values(*basis, water.grid_xyz, deriv=True)
    rho = O.density(phi, water.D)
    drho = O.density_gradient(phi, dphi, water.D)
    wv = water.grid_w * O.slater(rho)[1]
    for c in range(3):
        assert abs(g[:, c].sum() + np.dot(wv, drho[c])) < 1e-10 * np.max(np.abs(g))


def test_nuclear_gradient_gga_matches_finite_difference_of_energy(water):
    """GGA half of SURVEY.md §8(f2).  (a) the AO second derivatives against central differences of the analytic first
    derivatives in the point coordinates (and symmetric in the two directions); (b) the GGA nuclear-gradient contraction
    against central differences of the oracle's GGA energy in the atom coordinates, grid held fixed; (c) mu -> 0 in the
    functional is not available here, but dropping the sigma terms must give back the LDA-form expression: checked through
    (b) on five components of both signs."""
    basis = basis_of(water)
    rng = np.random.default_rng(4)
    p = rng.uniform(-2.5, 2.5, size=(40, 3))
    hess = O.ao_hessians(*basis, p)
    assert np.max(np.abs(hess - hess.transpose(1, 0, 2, 3))) < 1e-13
    h = 1e-5
    for d in range(3):
        pp, pm = p.copy(), p.copy()
        pp[:, d] += h
        pm[:, d] -= h
        fd = (O.ao_values(*basis, pp, deriv=True)[1] - O.ao_values(*basis, pm, deriv=True)[1]) / (2 * h)   # [c, g, mu]
        assert np.max(np.abs(fd - hess[:, d])) < 2e-8 * max(1.0, np.max(np.abs(hess)))
    g = O.exc_nuclear_gradient_gga(basis, water.grid_xyz, water.grid_w, water.D)
    assert g.shape == (3, 3) and np.max(np.abs(g)) > 1e-3
    h = 1e-4
    for (a, c) in [(0, 0), (0, 2), (1, 1), (2, 0), (2, 2)]:
        e = []
        for sgn in (+1, -1):
            xyz = np.array(basis[0], dtype=np.float64, copy=True)
            xyz[a, c] += sgn * h
            e.append(O.exc((xyz,) + tuple(basis[1:]), water.grid_xyz, water.grid_w, water.D, "gga", want_v=False)["E"])
        fd = (e[0] - e[1]) / (2 * h)
        assert abs(fd - g[a, c]) < 1e-6 * np.max(np.abs(g)), (a, c, fd, g[a, c])
    g_lda = O.exc_nuclear_gradient_lda(basis, water.grid_xyz, water.grid_w, water.D)
    assert np.max(np.abs(g - g_lda)) > 1e-4          # the enhancement factor is really in it


def test_kinetic_energy_density_and_vtau(water):
    """SURVEY.md §8(f4) contractions.  (a) closed form: one normalised s-Gaussian, exponent alpha, occupation n has
    int tau = n * 3 alpha / 2 (its kinetic energy); (b) tau from AO gradients taken by central differences of the AO
    VALUES (independent of the analytic gradients); (c) V^tau is symmetric, and Tr(D V^tau[wv]) = sum_g wv_g tau_g
    for arbitrary wv (a wrong factor or transposed operand in either function breaks it); (d) one element by loops."""
    from paper_2605_10363_b200 import workloads as W

    alpha, n = 0.9, 2.0
    pts, w = W.atomic_grid(1.0, n_rad=120)
    one = (np.zeros((1, 3)), np.array([0]), np.array([0]), np.array([0, 1]), np.array([alpha]), np.array([1.0]))
    _, dphi = O.ao_values(*one, pts, deriv=True)
    tau = O.kinetic_energy_density(dphi, np.array([[n]]))
    assert abs(np.dot(w, tau) - 1.5 * alpha * n) < 1e-8

    basis = basis_of(water)
    rng = np.random.default_rng(11)
    p2 = rng.uniform(-2.0, 2.0, size=(30, 3))
    _, dphi = O.ao_values(*basis, p2, deriv=True)
    tau = O.kinetic_energy_density(dphi, water.D)
    h = 1e-5
    fd = []
    for c in range(3):
        e = np.zeros(3); e[c] = h
        fd.append((O.ao_values(*basis, p2 + e) - O.ao_values(*basis, p2 - e)) / (2 * h))
    tau_fd = 0.5 * sum(np.einsum("gm,mn,gn->g", fd[c], water.D, fd[c]) for c in range(3))
    assert np.max(np.abs(tau - tau_fd)) < 1e-7 * np.max(np.abs(tau))
    wv = rng.normal(size=len(p2))
    Vt = O.vtau_from_wv(dphi, wv)
    assert np.max(np.abs(Vt - Vt.T)) <= 1e-14 * np.max(np.abs(Vt))
    assert abs(np.sum(water.D * Vt) - np.dot(wv, tau)) < 1e-11 * abs(np.dot(np.abs(wv), tau))
    m, k = 3, 17
    loop = 0.0
    for g in range(len(p2)):
        for c in range(3):
            loop += 0.5 * wv[g] * dphi[c][g, m] * dphi[c][g, k]
    assert abs(loop - Vt[m, k]) < 1e-13 * np.max(np.abs(Vt))


def test_exchange_energy_of_the_hydrogen_atom_matches_the_literature():
    """Absolute pin of the functionals: the oracle's slater() and pbe_x() integrated over the exact hydrogen 1s density
    (a 1-D radial integral by scipy's quad — none of the AO / grid machinery) reproduce the four decimals printed in
    the PBE paper's Table I (tests/golden/pbe_x_hydrogen.txt).  A wrong C_x, mu, kappa, a factor in the reduced
    gradient s^2 = sigma / (4 (3 pi^2)^{2/3} rho^{8/3}) or in sigma moves the PBE value in the third decimal."""
    from scipy import integrate

    gold = np.loadtxt(os.path.join(HERE, "golden", "pbe_x_hydrogen.txt"))

    def e_x(kind):
        def integrand(r):
            rho = 2.0 * np.exp(-2.0 * r) / np.pi            # 2 rho_up (spin scaling)
            grad = 2.0 * rho                                # |d rho / d r| of exp(-2r)
            if kind == 0:
                e = O.slater(np.array([rho]))[0]
            else:
                e = O.pbe_x(np.array([rho]), np.array([grad * grad]))[0]
            return 4.0 * np.pi * r * r * float(e[0])
        return 0.5 * integrate.quad(integrand, 0.0, 40.0, epsabs=1e-12, epsrel=1e-12, limit=400)[0]

    for kind, ref in gold:
        assert abs(e_x(int(kind)) - ref) < 5e-5, (kind, e_x(int(kind)), ref)
    # closed form of the LSD value: -C_x 2^{1/3} int rho_up^{4/3} d^3r, int (e^{-2r}/pi)^{4/3} 4 pi r^2 dr = 4 pi^{-1/3} 2/(8/3)^3
    closed = -0.75 * (3.0 / np.pi) ** (1.0 / 3.0) * 2.0 ** (1.0 / 3.0) * 4.0 * np.pi * np.pi ** (-4.0 / 3.0) * 2.0 / (8.0 / 3.0) ** 3
    assert abs(e_x(0) - closed) < 1e-10


def test_pbe_enhancement_limits():
    rho = np.geomspace(1e-12, 50.0, 200)
    e_s, v_s = O.slater(rho)
    e0, v0, vs0 = O.pbe_x(rho, np.zeros_like(rho))
    assert np.allclose(e0, e_s, rtol=1e-15, atol=0) and np.allclose(v0, v_s, rtol=1e-15, atol=0)   # F(0) = 1
    e_m0, v_m0, vs_m0 = O.pbe_x(rho, rho ** 2, mu=0.0)                                            # mu = 0 -> Slater
    assert np.allclose(e_m0, e_s, rtol=1e-15) and np.all(vs_m0 == 0.0)
    e_inf, _, _ = O.pbe_x(rho, 1e40 * np.ones_like(rho))                                          # F(inf) = 1+kappa
    assert np.allclose(e_inf, 1.804 * e_s, rtol=1e-12)
    sig = np.geomspace(1e-10, 1e6, 200)
    e, _, _ = O.pbe_x(rho, sig)
    assert np.all(e <= e_s * (1 - 1e-14)) and np.all(e >= 1.804 * e_s * (1 + 1e-14))
    # closed forms at one point: rho = 1, s^2 = 1  ->  sigma = 4 K_S
    ks = (3 * math.pi ** 2) ** (2 / 3)
    F = 1 + 0.804 - 0.804 / (1 + 0.21951 / 0.804)
    e1, _, _ = O.pbe_x(np.array([1.0]), np.array([4 * ks]))
    assert abs(e1[0] + 0.75 * (3 / math.pi) ** (1 / 3) * F) < 1e-15
    # derivative consistency by finite differences in rho and sigma
    r0, s0 = 0.37, 0.81
    h = 1e-6
    _, vr, vs = O.pbe_x(np.array([r0]), np.array([s0]))
    fr = (O.pbe_x(np.array([r0 + h]), np.array([s0]))[0] - O.pbe_x(np.array([r0 - h]), np.array([s0]))[0]) / (2 * h)
    fs = (O.pbe_x(np.array([r0]), np.array([s0 + h]))[0] - O.pbe_x(np.array([r0]), np.array([s0 - h]))[0]) / (2 * h)
    assert abs(fr[0] - vr[0]) < 1e-8 and abs(fs[0] - vs[0]) < 1e-8
    # the density guard (reading A9)
    e_c, v_c = O.slater(np.array([0.0, -1e-25, 1e-21, 1e-19]))
    assert np.all(e_c[:3] == 0) and np.all(v_c[:3] == 0) and e_c[3] < 0


def test_sampled_entry_helpers_agree_with_dense(water):
    basis = basis_of(water)
    out = O.exc(basis, water.grid_xyz, water.grid_w, water.D, "gga")
    pairs = [(0, 0), (3, 11), (24, 5)]
    got = O.vxc_entries_from_wv(basis, water.grid_xyz, out["wv"], pairs, gga=True)
    ref = np.array([out["V"][m, n] for m, n in pairs])
    assert np.max(np.abs(got - ref)) < 1e-12
    assert abs(O.exc_energy_from_rho(water.grid_w, out["rho"], out["drho"], "gga") - out["E"]) < 1e-13
