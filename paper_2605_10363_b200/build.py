"""In-tree build of the CUDA libraries with nvcc for sm_100a (no JIT cache, no torch extension).

  libkldi.so            — the product: csrc/*.cu behind the C ABI of include/kldi.h
  libkldi_workloads.so  — input generation helper (Becke weights), workloads/becke.cu

`python -m paper_2605_10363_b200.build` rebuilds both; __graft_entry__.build() calls build_all().
"""
from __future__ import annotations

import os
import shutil
import subprocess
import sys

PKG = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(PKG)
CSRC = os.path.join(PKG, "csrc")
LIB = os.path.join(PKG, "libkldi.so")
WL_LIB = os.path.join(PKG, "workloads", "libkldi_workloads.so")

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
    "-Xcompiler", "-fPIC", "--expt-relaxed-constexpr",
    "-cudart", "static",
]


def _nvcc() -> str:
    exe = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(exe):
        raise RuntimeError("nvcc not found")
    return exe


def _newer(target: str, sources: list) -> bool:
    if not os.path.exists(target):
        return False
    t = os.path.getmtime(target)
    return all(os.path.getmtime(s) <= t for s in sources)


def build_kldi(force: bool = False, verbose: bool = False) -> str:
    srcs = [os.path.join(CSRC, f) for f in ("api.cu", "plan.cu", "contract.cu", "vgram.cu", "pairsel.cu", "rho_i8.cu", "aoorder.cu", "xc_noalloc.cu")]
    deps = srcs + [os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith((".h", ".cuh"))]
    deps.append(os.path.join(ROOT, "include", "kldi.h"))
    if not force and _newer(LIB, deps):
        return LIB
    objs = []
    procs = []
    for s in srcs:
        o = s[:-3] + ".o"
        cmd = [_nvcc(), *NVCC_FLAGS, "-I", os.path.join(ROOT, "include"), "-I", CSRC, "-c", s, "-o", o]
        if verbose:
            cmd.insert(1, "-Xptxas=-v")
        procs.append((subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True), s))
        objs.append(o)
    for pr, s in procs:
        out, _ = pr.communicate()
        if pr.returncode != 0:
            raise RuntimeError(f"nvcc failed on {s}:\n{out}")
        if verbose:
            print(out)
    cmd = [_nvcc(), "-shared", "-cudart", "static", "-Xcompiler", "-fPIC", "-o", LIB, *objs]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError(f"link failed:\n{r.stdout}\n{r.stderr}")
    return LIB


def build_workloads(force: bool = False) -> str:
    src = os.path.join(PKG, "workloads", "becke.cu")
    if not force and _newer(WL_LIB, [src]):
        return WL_LIB
    cmd = [_nvcc(), *NVCC_FLAGS, "-shared", src, "-o", WL_LIB]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError(f"nvcc failed on {src}:\n{r.stdout}\n{r.stderr}")
    return WL_LIB


def build_all(force: bool = False, verbose: bool = False) -> None:
    build_kldi(force, verbose)
    build_workloads(force)


if __name__ == "__main__":
    build_all(force="--force" in sys.argv, verbose="-v" in sys.argv)
    print(LIB)
    print(WL_LIB)
