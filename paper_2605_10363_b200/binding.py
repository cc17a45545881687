"""ctypes binding of libkldi.so — argument marshalling only (include/kldi.h is the contract).

Every step of the path runs in the CUDA kernels behind the C ABI; PyTorch is used here for
device memory and the stream handle.  There is no CPU path: if libkldi.so is missing or no
CUDA device is present, calls raise.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional

import numpy as np

_PKG = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_PKG, "libkldi.so")

KLDI_LDA_SLATER = 0
KLDI_GGA_PBEX = 1

EXPORTED = [
    "kldi_plan_create", "kldi_plan_destroy", "kldi_plan_stats", "kldi_eval_rho", "kldi_build_vxc", "kldi_exc",
    "kldi_exc_host", "kldi_exc_grad", "kldi_eval_tau", "kldi_build_vtau", "kldi_last_timings", "kldi_plan_export", "kldi_plan_export_tile", "kldi_fp64_peak",
    "kldi_morton_key", "kldi_grid_key", "kldi_grid_keys", "kldi_last_error", "kldi_plan_set_option", "kldi_vsched_export",
    "kldi_vlayout_offset", "kldi_ao_order", "kldi_set_plan_default", "kldi_xc_lda_noalloc",
    "kldi_xc_lda_noalloc_max_pts",
]
KLDI_OPT_DETERMINISTIC_V = 1
KLDI_OPT_PAIR_TEST = 2
KLDI_OPT_RHO_DFMA = 3
KLDI_OPT_RHO_TC = 4
KLDI_OPT_HOST_V_TRIANGLE = 5


class KldiError(RuntimeError):
    pass


class _Atoms(C.Structure):
    _fields_ = [("n_atoms", C.c_int32), ("xyz", C.c_void_p)]


class _Shells(C.Structure):
    _fields_ = [("n_shells", C.c_int32), ("atom", C.c_void_p), ("l", C.c_void_p), ("nprim_off", C.c_void_p),
                ("alpha", C.c_void_p), ("coef", C.c_void_p)]


class _Grid(C.Structure):
    _fields_ = [("n_pts", C.c_int64), ("xyz", C.c_void_p), ("w", C.c_void_p)]


class Stats(C.Structure):
    _fields_ = [
        ("n_pts", C.c_int64), ("n_blocks", C.c_int64), ("n_blocks_nonempty", C.c_int64),
        ("n_ao", C.c_int32), ("n_shells", C.c_int32), ("n_atoms", C.c_int32), ("want_gradients", C.c_int32),
        ("retained_blocks", C.c_int64), ("candidate_blocks", C.c_int64), ("sum_k", C.c_int64),
        ("sum_k_pad", C.c_int64), ("max_k", C.c_int64), ("phi_bytes", C.c_int64), ("workspace_bytes", C.c_int64),
        ("flops_rho_useful", C.c_double), ("flops_rho_exec", C.c_double), ("flops_v_useful", C.c_double),
        ("flops_v_exec", C.c_double), ("flops_dense", C.c_double), ("plan_seconds", C.c_double), ("eps", C.c_double),
        ("flops_rho_useful_sym", C.c_double), ("flops_rho_exec_sym", C.c_double), ("flops_v_crit", C.c_double),
        ("pair_stages_total", C.c_int64), ("pair_stages_executed", C.c_int64),
        ("kernel_launches", C.c_int64), ("ops_rho_tc", C.c_double),
    ]

    def as_dict(self) -> dict:
        return {k: getattr(self, k) for k, _ in self._fields_}


_lib = None


def lib():
    """Load libkldi.so (built in-tree by paper_2605_10363_b200.build); raises if it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise KldiError(f"{LIB_PATH} not found: run `python -m paper_2605_10363_b200.build` "
                            "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        L.kldi_last_error.restype = C.c_char_p
        L.kldi_plan_create.argtypes = [C.POINTER(_Atoms), C.POINTER(_Shells), C.POINTER(_Grid), C.c_double, C.c_int,
                                       C.c_void_p, C.POINTER(C.c_void_p)]
        L.kldi_plan_destroy.argtypes = [C.c_void_p]
        L.kldi_plan_stats.argtypes = [C.c_void_p, C.POINTER(Stats)]
        L.kldi_eval_rho.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.kldi_build_vxc.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.c_void_p]
        L.kldi_exc.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.POINTER(C.c_double), C.c_void_p]
        L.kldi_exc_host.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.POINTER(C.c_double), C.c_void_p]
        L.kldi_exc_grad.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.POINTER(C.c_double), C.c_void_p]
        L.kldi_eval_tau.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.kldi_build_vtau.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.kldi_last_timings.argtypes = [C.c_void_p, C.POINTER(C.c_double)]
        L.kldi_plan_export.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_int64, C.POINTER(C.c_int64)]
        L.kldi_plan_export_tile.argtypes = [C.c_void_p, C.c_int64, C.c_int, C.c_void_p, C.c_int64,
                                            C.POINTER(C.c_int32)]
        L.kldi_fp64_peak.argtypes = [C.c_int, C.c_int, C.POINTER(C.c_double)]
        L.kldi_morton_key.argtypes = [C.POINTER(C.c_double), C.POINTER(C.c_double)]
        L.kldi_morton_key.restype = C.c_uint64
        L.kldi_grid_key.argtypes = [C.POINTER(C.c_double), C.POINTER(C.c_double)]
        L.kldi_grid_key.restype = C.c_uint64
        L.kldi_grid_keys.argtypes = [C.c_void_p, C.c_int64, C.POINTER(C.c_double), C.c_void_p]
        L.kldi_plan_set_option.argtypes = [C.c_void_p, C.c_int, C.c_int]
        L.kldi_ao_order.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.c_void_p, C.c_void_p]
        L.kldi_set_plan_default.argtypes = [C.c_int, C.c_int]
        L.kldi_xc_lda_noalloc.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p]
        L.kldi_xc_lda_noalloc_max_pts.argtypes = []
        L.kldi_xc_lda_noalloc_max_pts.restype = C.c_int64
        L.kldi_vsched_export.argtypes = [C.c_int, C.c_int, C.c_void_p, C.c_void_p, C.c_int64, C.POINTER(C.c_int64)]
        L.kldi_vlayout_offset.argtypes = [C.c_int64, C.c_int32, C.c_int32, C.c_int32]
        L.kldi_vlayout_offset.restype = C.c_int64
        for name in EXPORTED:
            if name not in ("kldi_last_error", "kldi_morton_key", "kldi_grid_key", "kldi_vlayout_offset",
                            "kldi_xc_lda_noalloc_max_pts"):
                getattr(L, name).restype = C.c_int
        _lib = L
    return _lib


def _check(rc: int, what: str):
    if rc != 0:
        raise KldiError(f"{what} failed (status {rc}): {lib().kldi_last_error().decode()}")


def _np(a, dtype):
    return np.ascontiguousarray(np.asarray(a), dtype=dtype)


_EXPORT_DTYPES = {0: np.int32, 1: np.int32, 2: np.int32, 3: np.int32, 4: np.int32, 5: np.int32, 6: np.int32,
                  7: np.int32, 8: np.uint64, 9: np.float64, 10: np.int64, 11: np.int32}
EXPORT_NAMES = {"perm_g": 0, "row_ptr": 1, "col_idx": 2, "col_ptr": 3, "row_idx": 4, "pos": 5, "shell_perm": 6,
                "ao_perm": 7, "grid_keys": 8, "morton_keys": 8, "block_amax": 9, "panel_off": 10, "blk_col0": 11}


class Plan:
    """kldi_plan: the once-per-geometry block-filtered representation."""

    def __init__(self, atom_xyz, shell_atom, shell_l, shell_prim_off, prim_alpha, prim_coef, grid_xyz, grid_w,
                 eps: float, want_gradients: bool = False, stream=None):
        import torch

        if not torch.cuda.is_available():
            raise KldiError("no CUDA device: libkldi has no CPU path")
        L = lib()
        ax = _np(atom_xyz, np.float64)
        sa, sl, so = _np(shell_atom, np.int32), _np(shell_l, np.int32), _np(shell_prim_off, np.int32)
        pa, pc = _np(prim_alpha, np.float64), _np(prim_coef, np.float64)
        gx, gw = _np(grid_xyz, np.float64), _np(grid_w, np.float64)
        atoms = _Atoms(ax.shape[0], ax.ctypes.data)
        shells = _Shells(sa.shape[0], sa.ctypes.data, sl.ctypes.data, so.ctypes.data, pa.ctypes.data, pc.ctypes.data)
        grid = _Grid(gx.shape[0], gx.ctypes.data, gw.ctypes.data)
        self._stream = stream if stream is not None else torch.cuda.current_stream()
        self._h = C.c_void_p()
        _check(L.kldi_plan_create(C.byref(atoms), C.byref(shells), C.byref(grid), float(eps),
                                  1 if want_gradients else 0, C.c_void_p(self._stream.cuda_stream),
                                  C.byref(self._h)), "kldi_plan_create")
        st = Stats()
        _check(L.kldi_plan_stats(self._h, C.byref(st)), "kldi_plan_stats")
        self.stats = st
        self.n_ao, self.n_pts = int(st.n_ao), int(st.n_pts)
        self.want_gradients = bool(want_gradients)
        self.device = torch.device("cuda", torch.cuda.current_device())

    @classmethod
    def from_workload(cls, wl, eps: Optional[float] = None, want_gradients: Optional[bool] = None, stream=None):
        return cls(wl.atom_xyz, wl.shell_atom, wl.shell_l, wl.shell_prim_off, wl.prim_alpha, wl.prim_coef,
                   wl.grid_xyz, wl.grid_w, wl.eps if eps is None else eps,
                   (wl.functional == "gga") if want_gradients is None else want_gradients, stream)

    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            lib().kldi_plan_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- helpers
    def _dev64(self, t, shape, name):
        import torch

        if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()
                and tuple(t.shape) == tuple(shape)):
            raise KldiError(f"{name}: expected a contiguous float64 CUDA tensor of shape {tuple(shape)}")
        return C.c_void_p(t.data_ptr())

    # ---- the calls of include/kldi.h
    def eval_rho(self, D, want_grad: bool = False):
        import torch

        rho = torch.empty(self.n_pts, dtype=torch.float64, device=self.device)
        drho = torch.empty((3, self.n_pts), dtype=torch.float64, device=self.device) if want_grad else None
        _check(lib().kldi_eval_rho(self._h, self._dev64(D, (self.n_ao, self.n_ao), "D"), C.c_void_p(rho.data_ptr()),
                                   C.c_void_p(drho.data_ptr()) if want_grad else None), "kldi_eval_rho")
        return (rho, drho) if want_grad else rho

    def build_vxc(self, wv, gga: bool = False, out=None):
        import torch

        shape = (4, self.n_pts) if gga else (self.n_pts,)
        V = out if out is not None else torch.empty((self.n_ao, self.n_ao), dtype=torch.float64, device=self.device)
        _check(lib().kldi_build_vxc(self._h, self._dev64(wv, shape, "wv"), 1 if gga else 0,
                                    self._dev64(V, (self.n_ao, self.n_ao), "V")), "kldi_build_vxc")
        return V

    def refresh_stats(self) -> "Stats":
        """Re-reads kldi_plan_stats (the pair-test counters change per call)."""
        st = Stats()
        _check(lib().kldi_plan_stats(self._h, C.byref(st)), "kldi_plan_stats")
        self.stats = st
        return st

    def set_option(self, option: int, value: int):
        _check(lib().kldi_plan_set_option(self._h, int(option), int(value)), "kldi_plan_set_option")

    def exc(self, D, functional: int = KLDI_LDA_SLATER, out=None, want_v: bool = True):
        import torch

        V = None
        if want_v:
            V = out if out is not None else torch.empty((self.n_ao, self.n_ao), dtype=torch.float64,
                                                        device=self.device)
        e = C.c_double(0.0)
        _check(lib().kldi_exc(self._h, self._dev64(D, (self.n_ao, self.n_ao), "D"), int(functional), C.byref(e),
                              self._dev64(V, (self.n_ao, self.n_ao), "V") if want_v else None), "kldi_exc")
        return e.value, V

    def eval_tau(self, D):
        """kldi_eval_tau: the kinetic-energy density on the caller's grid order, device tensor [n_pts]."""
        import torch

        tau = torch.empty(self.n_pts, dtype=torch.float64, device=self.device)
        _check(lib().kldi_eval_tau(self._h, self._dev64(D, (self.n_ao, self.n_ao), "D"), C.c_void_p(tau.data_ptr())),
               "kldi_eval_tau")
        return tau

    def build_vtau(self, wv_tau, out=None):
        """kldi_build_vtau: V = 1/2 sum_c (d_c Phi)^T diag(wv_tau) (d_c Phi)."""
        import torch

        V = out if out is not None else torch.empty((self.n_ao, self.n_ao), dtype=torch.float64, device=self.device)
        _check(lib().kldi_build_vtau(self._h, self._dev64(wv_tau, (self.n_pts,), "wv_tau"),
                                     self._dev64(V, (self.n_ao, self.n_ao), "V")), "kldi_build_vtau")
        return V

    def exc_grad(self, D, functional: int = KLDI_LDA_SLATER):
        """kldi_exc_grad: (E_xc, grad [n_atoms][3] device tensor, caller atom order)."""
        import torch

        g = torch.empty((int(self.stats.n_atoms), 3), dtype=torch.float64, device=self.device)
        e = C.c_double(0.0)
        _check(lib().kldi_exc_grad(self._h, self._dev64(D, (self.n_ao, self.n_ao), "D"), int(functional), C.byref(e),
                                   C.c_void_p(g.data_ptr())), "kldi_exc_grad")
        return e.value, g

    def exc_host(self, D_host, functional: int = KLDI_LDA_SLATER, V_host=None):
        """End-to-end form: D_host / V_host are host float64 arrays (numpy or pinned torch CPU tensors)."""
        def ptr(a):
            if a is None:
                return None
            if isinstance(a, np.ndarray):
                assert a.dtype == np.float64 and a.flags.c_contiguous and a.shape == (self.n_ao, self.n_ao)
                return C.c_void_p(a.ctypes.data)
            assert (not a.is_cuda) and a.is_contiguous() and tuple(a.shape) == (self.n_ao, self.n_ao)
            return C.c_void_p(a.data_ptr())

        e = C.c_double(0.0)
        _check(lib().kldi_exc_host(self._h, ptr(D_host), int(functional), C.byref(e), ptr(V_host)), "kldi_exc_host")
        return e.value

    def last_timings(self) -> dict:
        out = (C.c_double * 8)()
        _check(lib().kldi_last_timings(self._h, out), "kldi_last_timings")
        keys = ["permute_D", "rho", "xc", "wv_gather", "vxc", "finalise_V", "total"]
        return {k: out[i] for i, k in enumerate(keys)}

    def export(self, name: str) -> np.ndarray:
        which = EXPORT_NAMES[name]
        need = C.c_int64(0)
        _check(lib().kldi_plan_export(self._h, which, None, 0, C.byref(need)), "kldi_plan_export")
        dt = np.dtype(_EXPORT_DTYPES[which])
        buf = np.empty(need.value // dt.itemsize, dtype=dt)
        _check(lib().kldi_plan_export(self._h, which, C.c_void_p(buf.ctypes.data), need.value, C.byref(need)),
               "kldi_plan_export")
        return buf

    def export_tile(self, entry: int, comp: int = 0) -> np.ndarray:
        """Stored tile of BCS(R) entry `entry` as an array [width][128] (column-major tile)."""
        buf = np.empty((8, 128), dtype=np.float64)
        w = C.c_int32(0)
        _check(lib().kldi_plan_export_tile(self._h, int(entry), int(comp), C.c_void_p(buf.ctypes.data), buf.nbytes,
                                           C.byref(w)), "kldi_plan_export_tile")
        return buf[: w.value].copy()


def morton_key(xyz, origin) -> int:
    """Host evaluation of Eq. 20 as the plan applies it (no GPU needed)."""
    a = (C.c_double * 3)(*[float(v) for v in xyz])
    o = (C.c_double * 3)(*[float(v) for v in origin])
    return int(lib().kldi_morton_key(a, o))


def grid_key(xyz, origin) -> int:
    """Host evaluation of the key the plan sorts by (Hilbert index of Eq. 20's lattice coordinates)."""
    a = (C.c_double * 3)(*[float(v) for v in xyz])
    o = (C.c_double * 3)(*[float(v) for v in origin])
    return int(lib().kldi_grid_key(a, o))


KLDI_DEFAULT_AO_ORDER = 1
AO_ORDER_CURVE, AO_ORDER_OVERLAP, AO_ORDER_CALLER = 0, 1, 2


def set_plan_default(what: int, value: int) -> None:
    """Process-wide default of plans created afterwards (kldi_set_plan_default)."""
    _check(lib().kldi_set_plan_default(int(what), int(value)), "kldi_set_plan_default")


def ao_order(atom_xyz, shell_atom, shell_l, shell_prim_off, prim_alpha, prim_coef, want_dist: bool = False):
    """Host-only: overlap-signature order of the atoms (kldi_ao_order) -> order[, cosine distance matrix]."""
    ax = _np(atom_xyz, np.float64)
    sa, sl, so = _np(shell_atom, np.int32), _np(shell_l, np.int32), _np(shell_prim_off, np.int32)
    pa, pc = _np(prim_alpha, np.float64), _np(prim_coef, np.float64)
    atoms = _Atoms(ax.shape[0], ax.ctypes.data)
    shells = _Shells(sa.shape[0], sa.ctypes.data, sl.ctypes.data, so.ctypes.data, pa.ctypes.data, pc.ctypes.data)
    order = np.empty(ax.shape[0], dtype=np.int32)
    dist = np.empty((ax.shape[0], ax.shape[0])) if want_dist else None
    _check(lib().kldi_ao_order(C.byref(atoms), C.byref(shells), 1, C.c_void_p(order.ctypes.data),
                               C.c_void_p(dist.ctypes.data) if want_dist else None), "kldi_ao_order")
    return (order, dist) if want_dist else order


def xc_lda_noalloc(rho, w, wv_out, E_out, stream=None) -> None:
    """kldi_xc_lda_noalloc: wv_out = w v_rho(rho), E_out[0] = sum w e(rho); all four are float64 CUDA tensors the caller
    owns ([n], [n], [n], [1]); nothing is allocated.  Asynchronous on `stream` (default: torch's current stream)."""
    import torch

    n = rho.numel()
    for t, m in ((rho, n), (w, n), (wv_out, n), (E_out, 1)):
        if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()
                and t.numel() == m):
            raise KldiError("xc_lda_noalloc: expected contiguous float64 CUDA tensors of sizes n, n, n, 1")
    st = stream if stream is not None else torch.cuda.current_stream()
    _check(lib().kldi_xc_lda_noalloc(C.c_void_p(rho.data_ptr()), C.c_void_p(w.data_ptr()), n,
                                     C.c_void_p(wv_out.data_ptr()), C.c_void_p(E_out.data_ptr()),
                                     C.c_void_p(st.cuda_stream)), "kldi_xc_lda_noalloc")


def xc_lda_noalloc_max_pts() -> int:
    return int(lib().kldi_xc_lda_noalloc_max_pts())


def grid_keys(xyz, origin) -> np.ndarray:
    """Host evaluation of kldi_grid_key for an [n][3] array of points (no GPU needed)."""
    a = np.ascontiguousarray(xyz, dtype=np.float64).reshape(-1, 3)
    o = (C.c_double * 3)(*[float(v) for v in origin])
    out = np.empty(a.shape[0], dtype=np.uint64)
    _check(lib().kldi_grid_keys(C.c_void_p(a.ctypes.data), a.shape[0], o, C.c_void_p(out.ctypes.data)), "kldi_grid_keys")
    return out


def vsched(nb: int, square: bool = False):
    """Host-only: the V-contraction schedule of an nb-block panel -> (passes [n][8], items [n][32][2]) int32."""
    import numpy as np

    n = C.c_int64(0)
    _check(lib().kldi_vsched_export(int(nb), int(square), None, None, 0, C.byref(n)), "kldi_vsched_export")
    passes = np.zeros((n.value, 8), dtype=np.int32)
    items = np.zeros((n.value, 32, 2), dtype=np.int32)
    _check(lib().kldi_vsched_export(int(nb), int(square), passes.ctypes.data, items.ctypes.data, n.value,
                                    C.byref(n)), "kldi_vsched_export")
    return passes, items


def vlayout_offset(panel_off: int, K8: int, col: int, row: int) -> int:
    return int(lib().kldi_vlayout_offset(int(panel_off), int(K8), int(col), int(row)))


def fp64_peak(kind: str = "dmma", iters: int = 20000) -> float:
    t = C.c_double(0.0)
    _check(lib().kldi_fp64_peak({"dmma": 0, "dfma": 1, "mix": 2}[kind], int(iters), C.byref(t)), "kldi_fp64_peak")
    return t.value
