"""the overlap-signature ordering of the AO blocks (Eq. 8-10, 444-457 Eq. 21) —
host logic of libkldi (kldi_ao_order), checked on the CPU: its closed-form overlaps against the oracle's analytic
overlap matrix (a different derivation: binomial expansion vs Obara-Saika recursion), the cosine distances, the
clustering on cases whose answer is known, and a brute-force average-linkage reference on a small molecule."""
import numpy as np

from oracle import overlap as OV
from paper_2605_10363_b200 import binding as K
from paper_2605_10363_b200.workloads import generate as G


def _basis(symbols, xyz):
    sa, sl, so, al, co = G.shells_for(symbols)
    return (xyz, sa, sl, so, al, co)


def _atom_of_ao(basis):
    ncart = {0: 1, 1: 3, 2: 6}
    return np.concatenate([np.full(ncart[int(l)], int(a)) for a, l in zip(basis[1], basis[2])])


def test_cosine_distances_follow_eq21_on_the_oracle_overlap():
    symbols, xyz = G.water_cluster_geometry(3, 5)
    basis = _basis(symbols, xyz)
    order, dist = K.ao_order(*basis, want_dist=True)
    S = OV.overlap_matrix(*basis)
    at = _atom_of_ao(basis)
    n = len(symbols)
    T = np.array([[np.linalg.norm(S[np.ix_(at == a, at == b)]) for b in range(n)] for a in range(n)])
    ref = 1.0 - (T @ T.T) / np.outer(np.linalg.norm(T, axis=1), np.linalg.norm(T, axis=1))
    np.fill_diagonal(ref, 0.0)
    assert np.max(np.abs(dist - ref)) <= 1e-12
    assert np.array_equal(np.sort(order), np.arange(n))


def _reference_order(d):
    """Average linkage with end-leaf orientation, brute force on the ORIGINAL distances (O(N^3), tiny inputs)."""
    clusters = [[i] for i in range(d.shape[0])]
    while len(clusters) > 1:
        best = None
        for x in range(len(clusters)):
            for y in range(x + 1, len(clusters)):
                v = np.mean([d[i, j] for i in clusters[x] for j in clusters[y]])
                if best is None or v < best[0] - 1e-15:
                    best = (v, x, y)
        _, x, y = best
        lx, ly = clusters[x], clusters[y]
        cands = [(d[lx[-1], ly[0]], lx, ly), (d[lx[-1], ly[-1]], lx, ly[::-1]),
                 (d[lx[0], ly[0]], lx[::-1], ly), (d[lx[0], ly[-1]], lx[::-1], ly[::-1])]
        c = min(cands, key=lambda t: t[0])
        clusters[x] = c[1] + c[2]
        del clusters[y]
    return clusters[0]


def test_clustering_equals_brute_force_average_linkage():
    symbols, xyz = G.water_cluster_geometry(4, 11)
    basis = _basis(symbols, xyz)
    order, dist = K.ao_order(*basis, want_dist=True)
    ref = _reference_order(dist)
    assert list(order) == ref or list(order) == ref[::-1]


def test_chain_is_ordered_along_the_chain():
    """All-trans alkane: signatures change monotonically along the chain, so the leaf order walks the chain and keeps
    every carbon's hydrogens next to it."""
    symbols, xyz = G.alkane_geometry(24)
    order = K.ao_order(*_basis(symbols, xyz))
    x = xyz[order, 0]
    assert np.all(np.abs(np.diff(x)) <= 2.6 * 1.54 / 0.529177 * 0.9)       # consecutive atoms within ~ one C-C-C step
    assert abs(x[-1] - x[0]) >= 0.9 * (xyz[:, 0].max() - xyz[:, 0].min())   # one sweep from end to end
    carbons = [i for i, a in enumerate(order) if symbols[a] == "C"]
    cx = xyz[order[carbons], 0]
    assert np.all(np.diff(cx) > 0) or np.all(np.diff(cx) < 0)


def test_waters_stay_together_and_neighbours_are_near():
    symbols, xyz = G.water_cluster_geometry(32, 1001)
    order = K.ao_order(*_basis(symbols, xyz))
    assert np.array_equal(np.sort(order), np.arange(96))
    pos = np.empty(96, int)
    pos[order] = np.arange(96)
    for m in range(32):                      # O, H, H of a molecule are consecutive in the order
        p = pos[3 * m:3 * m + 3]
        assert p.max() - p.min() == 2
    step = np.linalg.norm(np.diff(xyz[order], axis=0), axis=1).mean()
    assert step < 0.6 * np.linalg.norm(np.diff(xyz, axis=0), axis=1).mean()
