"""CPU ORACLE helper — TEST INFRASTRUCTURE, NOT THE PRODUCT.

Closed-form overlap matrix S_{mu,nu} = int chi_mu chi_nu d^3r (Eq. 8) of the
contracted Cartesian Gaussians defined in exc_oracle.ao_values.  It is evaluated analytically
(Gaussian product theorem + binomial expansion), i.e. WITHOUT the quadrature grid, so it pins
the AO normalisation, the quadrature weights and the density build through
int rho = Tr(D S) (BASELINE.json invariant (i)).

For primitives a on A, b on B: p = a+b, P = (aA+bB)/p,
  int (x-A)^i (x-B)^j e^{-a(x-A)^2 - b(x-B)^2} dx
     = e^{-ab/p (A-B)^2} sum_{s even} c_s (s-1)!! / (2p)^{s/2} sqrt(pi/p),
  c_s = sum_{t+u=s} C(i,t) C(j,u) (P-A)^{i-t} (P-B)^{j-u}.
"""
from __future__ import annotations

import math

import numpy as np

from .exc_oracle import cart_components, norm_const


def _dfact(n: int) -> float:
    out = 1.0
    while n > 1:
        out *= n
        n -= 2
    return out


def _overlap_1d(i: int, j: int, a: float, b: float, A: float, B: float) -> float:
    p = a + b
    P = (a * A + b * B) / p
    tot = 0.0
    for t in range(i + 1):
        for u in range(j + 1):
            s = t + u
            if s % 2:
                continue
            tot += (math.comb(i, t) * math.comb(j, u) * (P - A) ** (i - t) * (P - B) ** (j - u)
                    * _dfact(s - 1) / (2.0 * p) ** (s // 2))
    return tot * math.sqrt(math.pi / p) * math.exp(-a * b / p * (A - B) ** 2)


def overlap_matrix(atom_xyz, shell_atom, shell_l, shell_prim_off, prim_alpha, prim_coef) -> np.ndarray:
    aos = []
    for s in range(len(shell_l)):
        for (i, j, k) in cart_components(int(shell_l[s])):
            prims = [(float(prim_alpha[p]), float(prim_coef[p]) * norm_const(float(prim_alpha[p]), i, j, k))
                     for p in range(int(shell_prim_off[s]), int(shell_prim_off[s + 1]))]
            aos.append((np.asarray(atom_xyz[int(shell_atom[s])], dtype=np.float64), (i, j, k), prims))
    n = len(aos)
    S = np.zeros((n, n))
    for m in range(n):
        A, pa, prm = aos[m]
        for q in range(m, n):
            B, pb, prq = aos[q]
            v = 0.0
            for (a, ca) in prm:
                for (b, cb) in prq:
                    t = ca * cb
                    for d in range(3):
                        t *= _overlap_1d(pa[d], pb[d], a, b, float(A[d]), float(B[d]))
                    v += t
            S[m, q] = S[q, m] = v
    return S
