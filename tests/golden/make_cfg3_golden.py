"""Writes tests/golden/cfg3_oracle.npz: the dense CPU oracle on BASELINE.json configs[3] at FULL size
(256 waters, 6,400 AOs, 4,224,000 points, LDA Slater), for the full-size parity test and bench.py's eps leg.

Calls only oracle/ and the seeded input generator (no CUDA path): `O.exc(...)` as it stands, dense and
unscreened, ~0.7 PFLOP of dgemm — about 70 minutes on 8 cores.  The Becke partition of the 4.2 M points
(2.5e12 cell functions) is input generation, not method arithmetic; pass the weights the same generator wrote
on a GPU box with `--weights cfg3_w.npy` (workloads/becke.cu; numerically the numpy recipe to rounding, which
tests/test_gpu_parity.py::test_becke_cuda_equals_numpy checks), or omit it to run the numpy Becke (days).

Stored (all float64): E; rho on every 64th point; wv on every 64th point; 16 full rows of V and the strided
sample V[::97, ::89]; sum and sum of squares of the weights (so that a test can tell that it runs on the same
inputs).  Usage:  python tests/golden/make_cfg3_golden.py --weights baseline/_ref/cfg3_w.npy
"""
import argparse
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
    ap.add_argument("--weights", default=None, help="npy file of cfg3's grid_w written by the input generator")
    ap.add_argument("--config", default="cfg3")
    ap.add_argument("--out", default=os.path.join(ROOT, "tests", "golden", "cfg3_oracle.npz"))
    ap.add_argument("--chunk", type=int, default=8192)
    a = ap.parse_args()
    gw = np.load(a.weights) if a.weights else None
    wl = W.named_config(a.config, grid_w=gw, becke_backend="numpy")
    basis = (wl.atom_xyz, wl.shell_atom, wl.shell_l, wl.shell_prim_off, wl.prim_alpha, wl.prim_coef)
    t0 = time.time()
    ref = O.exc(basis, wl.grid_xyz, wl.grid_w, wl.D, wl.functional, chunk=a.chunk)
    dt = time.time() - t0
    rows = [r for r in V_ROWS if r < wl.n_ao]
    np.savez(a.out, E=np.float64(ref["E"]), rho_strided=ref["rho"][::STRIDE_PTS], wv_strided=ref["wv"][::STRIDE_PTS],
             stride_pts=np.int64(STRIDE_PTS), v_rows=np.array(rows, np.int64), V_rows=ref["V"][rows, :],
             V_strided=ref["V"][::STRIDE_V[0], ::STRIDE_V[1]], stride_v=np.array(STRIDE_V, np.int64),
             w_sum=np.float64(wl.grid_w.sum()), w_sumsq=np.float64(np.sum(wl.grid_w ** 2)),
             n_pts=np.int64(wl.n_pts), n_ao=np.int64(wl.n_ao), seed=np.int64(wl.seed),
             oracle_seconds=np.float64(dt), V_absmax=np.float64(np.abs(ref["V"]).max()),
             rho_max=np.float64(ref["rho"].max()))
    print(f"{a.config}: E = {ref['E']!r}, {dt:.0f} s, wrote {a.out}")


if __name__ == "__main__":
    main()
