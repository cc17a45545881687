"""Writes tests/golden/cfg3_oracle.npz: the dense CPU oracle on BASELINE.json configs[3] at FULL size
(256 waters, 6,400 AOs, 4,224,000 points, LDA Slater), for the full-size parity test and bench.py's eps leg.

Calls only oracle/ and the seeded input generator (no CUDA path).  The whole dense evaluation `O.exc(...)` is 0.7 PFLOP of
dgemm, two thirds of it the full 6400 x 6400 potential matrix — about 13 hours on 8 cores.  What is stored does not need
all of V, so the script walks the grid in chunks and takes the oracle's own steps, dense and unscreened, for every chunk:

    phi = O.ao_values(...)           all 6,400 AOs on the chunk's points
    rho = O.density(phi, D)          the full dense product Phi D (this is the 0.35 PFLOP that remains: ~1 h on 8 cores)
    e, v = O.slater(rho);  wv = w v;  E += fsum(w e)
    V[rows, :]  += O.vxc_lda_block_from_wv(phi, wv, rows, all)       16 full rows of V
    V[::97, ::89] += O.vxc_lda_block_from_wv(phi, wv, ::97, ::89)    a strided sample of V

(`vxc_lda_block_from_wv` is the definition of V restricted to rows / columns, pinned against the full V in
tests/test_oracle_pins.py.)  The Becke partition of the 4.2 M points (2.5e12 cell functions) is input generation, not
method arithmetic; pass the weights the same generator wrote on a GPU box with `--weights cfg3_w.npy` (workloads/becke.cu;
tests/test_gpu_parity.py::test_becke_cuda_equals_numpy holds it to the numpy recipe), or omit it to run the numpy Becke
(days).  The run is resumable: a checkpoint is written every `--sub` points and a later invocation continues from it;
`--lo/--hi` restrict a run to a range of points (every stored quantity is a sum over points or a per-point value), so that
disjoint ranges can run on different machines, and `--merge a.ckpt.npz b.ckpt.npz ...` adds finished ranges that tile
[0, n_pts) into the final file.

Stored (all float64): E; rho and wv on every 64th point; 16 full rows of V and the strided sample V[::97, ::89]; sum and
sum of squares of the weights (so that a test can tell that it runs on the same inputs).
Usage:  python tests/golden/make_cfg3_golden.py --weights baseline/_ref/cfg3_w.npy
"""
import argparse
import math
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

from oracle import exc_oracle as O  # noqa: E402
from paper_2605_10363_b200 import workloads as W  # noqa: E402

V_ROWS = [0, 1, 7, 14, 15, 19, 24, 25, 3199, 3200, 3207, 4242, 5001, 6385, 6398, 6399]
STRIDE_PTS = 64
STRIDE_V = (97, 89)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--weights", default=None, help="npy file of the config's grid_w written by the input generator")
    ap.add_argument("--config", default="cfg3")
    ap.add_argument("--out", default=os.path.join(ROOT, "tests", "golden", "cfg3_oracle.npz"))
    ap.add_argument("--chunk", type=int, default=8192)
    ap.add_argument("--sub", type=int, default=262144, help="points per checkpoint")
    ap.add_argument("--checkpoint", default=None, help="checkpoint file (default: <out>.ckpt.npz)")
    ap.add_argument("--budget", type=float, default=0.0, help="stop after this many seconds (0 = run to the end)")
    ap.add_argument("--lo", type=int, default=0, help="first point of this run's range")
    ap.add_argument("--hi", type=int, default=-1, help="end of this run's range (default: all points)")
    ap.add_argument("--merge", nargs="+", default=None, help="checkpoints of finished ranges that tile [0, n_pts)")
    a = ap.parse_args()
    gw = np.load(a.weights) if a.weights else None
    wl = W.named_config(a.config, grid_w=gw, becke_backend="numpy")
    assert wl.functional == "lda"
    basis = (wl.atom_xyz, wl.shell_atom, wl.shell_l, wl.shell_prim_off, wl.prim_alpha, wl.prim_coef)
    n, n_ao, sp = wl.n_pts, wl.n_ao, STRIDE_PTS
    rows = np.array([r for r in V_ROWS if r < n_ao])
    allc = np.arange(n_ao)
    sr, sc = np.arange(0, n_ao, STRIDE_V[0]), np.arange(0, n_ao, STRIDE_V[1])
    ck = a.checkpoint or (a.out + ".ckpt.npz")
    r_lo, r_hi = a.lo, (n if a.hi < 0 else min(n, a.hi))
    if a.merge:
        parts = [dict(np.load(f)) for f in a.merge]
        parts.sort(key=lambda d: int(d.get("lo", 0)))
        edge = 0
        for d in parts:   # the ranges must tile [0, n) without gap or overlap; `done` may be cut back to the next range's lo
            assert int(d["n_pts"]) == n and abs(float(d["w_sum"]) - wl.grid_w.sum()) <= 1e-9 * abs(wl.grid_w.sum())
            assert int(d.get("lo", 0)) == edge and int(d["done"]) > edge, (int(d.get("lo", 0)), edge)
            edge = int(d["done"])
        assert edge == n, (edge, n)
        st = {"done": np.int64(n), "seconds": np.float64(sum(float(d["seconds"]) for d in parts)),
              "E_parts": np.concatenate([d["E_parts"] for d in parts]),
              "rho_max": np.float64(max(float(d["rho_max"]) for d in parts))}
        for k in ("rho_strided", "wv_strided", "V_rows", "V_strided"):
            st[k] = sum(d[k] for d in parts)
    elif os.path.exists(ck):
        z = np.load(ck)
        st = {k: z[k] for k in z.files}
        assert int(st["n_pts"]) == n and abs(float(st["w_sum"]) - wl.grid_w.sum()) <= 1e-9 * abs(wl.grid_w.sum())
        print(f"resuming from {ck}: {int(st['done'])} of {n} points done", flush=True)
    else:
        st = {"done": np.int64(r_lo), "lo": np.int64(r_lo), "n_pts": np.int64(n), "w_sum": np.float64(wl.grid_w.sum()),
              "E_parts": np.zeros(0),
              "rho_strided": np.zeros((n + sp - 1) // sp), "wv_strided": np.zeros((n + sp - 1) // sp),
              "V_rows": np.zeros((len(rows), n_ao)), "V_strided": np.zeros((len(sr), len(sc))),
              "rho_max": np.float64(0.0), "seconds": np.float64(0.0)}
    t_start = time.time()
    while not a.merge and int(st["done"]) < r_hi and (a.budget <= 0 or time.time() - t_start < a.budget):
        lo = int(st["done"])
        hi = min(r_hi, lo + a.sub)
        t0 = time.time()
        e_terms = []
        for c0 in range(lo, hi, a.chunk):
            c1 = min(hi, c0 + a.chunk)
            phi = O.ao_values(*basis, wl.grid_xyz[c0:c1])
            rho = O.density(phi, wl.D)
            e, v = O.slater(rho)
            wv = wl.grid_w[c0:c1] * v
            e_terms.append(wl.grid_w[c0:c1] * e)
            st["V_rows"] += O.vxc_lda_block_from_wv(phi, wv, rows, allc)
            st["V_strided"] += O.vxc_lda_block_from_wv(phi, wv, sr, sc)
            idx = np.arange(((c0 + sp - 1) // sp) * sp, c1, sp)
            st["rho_strided"][idx // sp] = rho[idx - c0]
            st["wv_strided"][idx // sp] = wv[idx - c0]
            st["rho_max"] = np.float64(max(float(st["rho_max"]), float(rho.max())))
        st["E_parts"] = np.append(st["E_parts"], math.fsum(np.concatenate(e_terms).tolist()))
        st["seconds"] = np.float64(float(st["seconds"]) + time.time() - t0)
        st["done"] = np.int64(hi)
        np.savez(ck + ".tmp.npz", **st)
        os.replace(ck + ".tmp.npz", ck)
        print(f"  points {lo}..{hi} of {n}: {time.time() - t0:.0f} s", flush=True)
    if not a.merge and (int(st["done"]) < n or r_lo > 0):
        print(f"range {r_lo}..{r_hi}: {int(st['done'])} reached; checkpoint {ck} (run again to continue, or --merge)")
        return
    E = math.fsum(st["E_parts"].tolist())
    np.savez(a.out, E=np.float64(E), rho_strided=st["rho_strided"], wv_strided=st["wv_strided"],
             stride_pts=np.int64(STRIDE_PTS), v_rows=rows.astype(np.int64), V_rows=st["V_rows"],
             V_strided=st["V_strided"], stride_v=np.array(STRIDE_V, np.int64),
             w_sum=np.float64(wl.grid_w.sum()), w_sumsq=np.float64(np.sum(wl.grid_w ** 2)),
             n_pts=np.int64(wl.n_pts), n_ao=np.int64(wl.n_ao), seed=np.int64(wl.seed),
             oracle_seconds=st["seconds"],
             V_absmax=np.float64(max(np.abs(st["V_rows"]).max(), np.abs(st["V_strided"]).max())), rho_max=st["rho_max"])
    print(f"{a.config}: E = {E!r}, {float(st['seconds']):.0f} s, wrote {a.out}")


if __name__ == "__main__":
    main()
