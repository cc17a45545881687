"""CPU-side checks of the C-ABI library: it loads, exports every symbol include/kldi.h declares,
fails loudly without a GPU, and its host-side Morton key (Eq. 20) is the
bit interleave the paper defines."""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    import __graft_entry__ as g

    g.build()
    from paper_2605_10363_b200 import binding

    return binding.lib()


def test_every_declared_symbol_is_exported(lib):
    text = open(os.path.join(ROOT, "include", "kldi.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    declared = set(re.findall(r"\b(kldi_[a-z0-9_]+)\s*\(", text))
    assert {"kldi_plan_create", "kldi_eval_rho", "kldi_build_vxc", "kldi_exc"} <= declared
    from paper_2605_10363_b200 import binding

    assert declared == set(binding.EXPORTED)
    for name in declared:
        assert hasattr(lib, name), name


def test_stats_struct_layout_matches_header():
    """The ctypes mirror of kldi_stats must have the header's field order and types."""
    from paper_2605_10363_b200 import binding

    text = open(os.path.join(ROOT, "include", "kldi.h")).read()
    body = re.search(r"typedef struct \{([^}]*)\} kldi_stats;", text, flags=re.S).group(1)
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    fields = re.findall(r"(int64_t|int32_t|double)\s+([a-z_0-9]+)\s*;", body)
    cmap = {"int64_t": C.c_int64, "int32_t": C.c_int32, "double": C.c_double}
    assert [(n, cmap[t]) for t, n in fields] == list(binding.Stats._fields_)


def test_no_gpu_means_loud_failure(lib):
    import torch

    if torch.cuda.is_available():
        pytest.skip("GPU present")
    from paper_2605_10363_b200 import binding, workloads

    wl = workloads.named_config("cfg0")
    with pytest.raises(binding.KldiError):
        binding.Plan.from_workload(wl)
    # and directly at the C boundary: status KLDI_ECUDA (-3) with a message, no plan
    ax = np.zeros((1, 3)); sa = np.zeros(1, np.int32); sl = np.zeros(1, np.int32); so = np.array([0, 1], np.int32)
    al = np.ones(1); co = np.ones(1); gx = np.zeros((4, 3)); gw = np.ones(4)
    atoms = binding._Atoms(1, ax.ctypes.data)
    shells = binding._Shells(1, sa.ctypes.data, sl.ctypes.data, so.ctypes.data, al.ctypes.data, co.ctypes.data)
    grid = binding._Grid(4, gx.ctypes.data, gw.ctypes.data)
    h = C.c_void_p()
    rc = lib.kldi_plan_create(C.byref(atoms), C.byref(shells), C.byref(grid), 1e-12, 0, None, C.byref(h))
    assert rc == -3 and not h.value
    assert b"no CUDA device" in lib.kldi_last_error()


def test_invalid_arguments_are_rejected(lib):
    h = C.c_void_p()
    assert lib.kldi_plan_create(None, None, None, 1e-12, 0, None, C.byref(h)) == -1
    assert lib.kldi_plan_stats(None, None) == -1
    assert lib.kldi_plan_destroy(None) == 0
    assert lib.kldi_eval_rho(None, None, None, None) == -1
    assert lib.kldi_build_vxc(None, None, 0, None) == -1
    e = C.c_double()
    assert lib.kldi_exc(None, None, 0, C.byref(e), None) == -1


def _interleave_bruteforce(ix, iy, iz):
    m = 0
    for k in range(20):
        m |= ((iz >> k) & 1) << (3 * k)
        m |= ((iy >> k) & 1) << (3 * k + 1)
        m |= ((ix >> k) & 1) << (3 * k + 2)
    return m


def test_morton_key_is_eq20(lib):
    from paper_2605_10363_b200 import binding

    rng = np.random.default_rng(7)
    origin = np.array([-3.0, 2.5, -100.0])
    pts = origin + rng.uniform(0.0, 8000.0, size=(300, 3)) * rng.uniform(0, 1, size=(300, 1)) ** 3
    for p in pts:
        q = [int(np.trunc((p[c] - origin[c]) * 128.0)) for c in range(3)]
        q = [min(max(v, 0), 2 ** 20 - 1) for v in q]
        assert binding.morton_key(p, origin) == _interleave_bruteforce(*q)
    # single-axis unit steps land on the documented bit positions; x is the most significant
    assert binding.morton_key([1 / 128, 0, 0], [0, 0, 0]) == 4
    assert binding.morton_key([0, 1 / 128, 0], [0, 0, 0]) == 2
    assert binding.morton_key([0, 0, 1 / 128], [0, 0, 0]) == 1
    assert binding.morton_key([1e9, 1e9, 1e9], [0, 0, 0]) == 2 ** 60 - 1      # clamped to 20 bits per axis
    assert binding.morton_key([-5.0, -5.0, -5.0], [0, 0, 0]) == 0              # below the origin -> 0
    # locality: points inside one 1/128-bohr cell share a key
    assert binding.morton_key([0.5001, 0.2501, 0.1251], [0, 0, 0]) == binding.morton_key([0.5003, 0.2503, 0.1253], [0, 0, 0])


def test_grid_key_is_a_hilbert_curve(lib):
    """kldi_grid_key (the key the plan sorts by): a bijection of the 2^20-per-axis lattice onto
    60-bit indices whose successive cells are face neighbours (no jumps: what makes blocks of consecutive points
    compact), nested (the first 3 L index bits fix the cell at level L), clamped like Eq. 20."""
    from paper_2605_10363_b200 import binding

    for level in (1, 2, 3, 4):                     # the 2^level cube of cells, each 2^(20-level) lattice units wide
        n, side = 2 ** level, 2 ** (20 - level)
        cells = [(i, j, k) for i in range(n) for j in range(n) for k in range(n)]
        keys = {}
        for c in cells:
            lo = binding.grid_key([v * side / 128.0 for v in c], [0, 0, 0]) >> (60 - 3 * level)
            hi = binding.grid_key([((v + 1) * side - 1) / 128.0 + 1e-9 for v in c], [0, 0, 0]) >> (60 - 3 * level)
            assert lo == hi                        # nested: every lattice point of the cell shares the index prefix
            keys[lo] = c
        assert sorted(keys) == list(range(n ** 3))  # bijection at this level
        path = [keys[i] for i in range(n ** 3)]
        assert all(sum(abs(a - b) for a, b in zip(p, q)) == 1 for p, q in zip(path, path[1:]))
    # full-resolution neighbours along the curve, around an arbitrary point
    rng = np.random.default_rng(7)
    seen = set()
    for _ in range(200):
        q = rng.integers(0, 2 ** 20, 3)
        k = binding.grid_key([(v + 0.5) / 128.0 for v in q], [0, 0, 0])
        assert 0 <= k < 2 ** 60 and k not in seen
        seen.add(k)
        nb = [binding.grid_key([(v + 0.5 + d * (a == ax)) / 128.0 for a, v in enumerate(q)], [0, 0, 0])
              for ax in range(3) for d in (-1, 1) if 0 <= q[ax] + d < 2 ** 20]
        assert sum(abs(m - k) == 1 for m in nb) >= 1 or k in (0, 2 ** 60 - 1)   # predecessor or successor is a face neighbour
    assert binding.grid_key([-5.0, -5.0, -5.0], [0, 0, 0]) == binding.grid_key([0, 0, 0], [0, 0, 0]) == 0
    assert binding.grid_key([1e9, 1e9, 1e9], [0, 0, 0]) == binding.grid_key([8192.0, 8192.0, 8192.0], [0, 0, 0])


@pytest.mark.parametrize("square", [False, True])
def test_v_schedule_covers_every_unit_once(square):
    """Host logic of the V contraction (csrc/vsched.h): for every panel size the passes tile the (16-row strip,
    8-column block) units of the Gram matrix exactly once (LDA: blocks on and above the strip's diagonal; GGA:
    all), every item's operand columns lie inside the staged intervals, and no warp exceeds its slots x 4
    column blocks (its register-resident accumulators)."""
    from paper_2605_10363_b200 import binding as K

    for nb in list(range(1, 40)) + [47, 56, 64, 111]:
        passes, items = K.vsched(nb, square)
        ns = (nb + 1) // 2
        seen = np.zeros((ns, nb), dtype=np.int32)
        for P, I in zip(passes, items):
            c1_lo, c1_n, c2_lo, c2_n, max_load, units, smsp_load, shape = (int(v) for v in P[:8])
            n_warps, n_slots = shape & 0xFF, shape >> 8
            assert n_warps * n_slots <= 32
            assert c1_n + c2_n <= 256 and c1_lo % 8 == 0 and c2_lo % 8 == 0 and c1_n % 8 == 0 and c2_n % 8 == 0
            loads, tot = [], 0
            for w in range(n_warps):
                load = 0
                for k in range(n_slots):
                    a, b = int(I[w * n_slots + k, 0]), int(I[w * n_slots + k, 1])
                    nj, diag, a_slot, b_slot = (a >> 20) & 7, (a >> 24) & 1, a & 1023, (a >> 10) & 1023
                    if nj == 0:
                        continue
                    assert 1 <= nj <= 4
                    arow, bcol = b & 0xFFFF, b >> 16
                    assert arow % 16 == 0 and bcol % 8 == 0
                    # A rows come from interval 1; B columns from interval 1 (single interval) or interval 2
                    assert c1_lo + a_slot == arow and a_slot + 8 <= c1_n + (8 if nb % 2 else 0) + 8
                    if b_slot < c1_n and not square and c2_n == 0:
                        assert c1_lo + b_slot == bcol and b_slot + 8 * nj <= c1_n
                    else:
                        assert b_slot >= c1_n and c2_lo + (b_slot - c1_n) == bcol and b_slot - c1_n + 8 * nj <= c2_n
                    s = arow // 16
                    for j in range(bcol // 8, bcol // 8 + nj):
                        seen[s, j] += 1
                    # diag: the lower 8 rows of a strip's first block on the diagonal are not computed (LDA only)
                    assert diag == (0 if square else int(bcol == arow))
                    load += 2 * nj - diag
                loads.append(load)
                tot += load
            assert max(loads) == max_load <= 2 * 4 * n_slots and tot == units    # in 8x8 blocks
            # the balanced quantity: load per scheduler partition (warp % 4 shares one FP64 tensor pipe)
            assert max(sum(loads[q::4]) for q in range(4)) == smsp_load
            assert 4 * smsp_load <= units + 4 * 8 + 3
        want = np.ones((ns, nb), dtype=np.int32)
        if not square:
            for s in range(ns):
                want[s, : 2 * s] = 0
        assert np.array_equal(seen, want), (nb, square)


def test_v_layout_is_a_bijection_with_conflict_free_fragments():
    """kldi_vlayout_offset: a permutation of the panel's elements; a slab's columns are contiguous; the 16-byte
    chunks (2 r4 + j) of 8 adjacent columns fall into 8 different 16-byte bank groups for every quarter warp."""
    from paper_2605_10363_b200 import binding as K

    K8, po = 24, 40
    offs = np.array([[K.vlayout_offset(po, K8, c, r) for r in range(128)] for c in range(K8)])
    assert sorted(offs.ravel().tolist()) == list(range(po * 128, (po + K8) * 128))
    for rc in range(4):
        blk = offs[:, 32 * rc: 32 * rc + 32] - (po * 128 + rc * K8 * 32)
        assert blk.min() == 0 and blk.max() == K8 * 32 - 1
        for c in range(K8):
            assert blk[c].min() == 32 * c and blk[c].max() == 32 * c + 31      # column c is one 256-byte run
    for j in range(2):
        for h in range(2):
            for qpair in range(4):                                             # quarter warp: q4 in {2g, 2g+1}
                groups = set()
                for q4 in (2 * qpair, 2 * qpair + 1):
                    for r4 in range(4):
                        row = 2 * (2 * r4 + j + 8 * h)
                        o = K.vlayout_offset(0, K8, 8 + q4, row)
                        assert o % 2 == 0 and K.vlayout_offset(0, K8, 8 + q4, row + 1) == o + 1
                        groups.add((o * 8 // 16) % 8)
                assert len(groups) == 8
