"""kldi_xc_lda_noalloc — the functional + energy step with its scratch in a static device array (no cudaMalloc: for
callers under CUDA graph capture or in harnesses that forbid allocation).  Checked against the existing path (the
functional stage inside kldi_exc, whose partial sums live in a plan-owned buffer) on two calls in a row; the second
call is smaller, so the array still holds stale partials of the first.  Collected last on purpose (file name)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL_V, TOL_E = 1e-9, 1e-8


def test_noalloc_entry_point_matches_existing_path_twice():
    import torch

    assert torch.cuda.is_available()
    from paper_2605_10363_b200 import binding as K
    from paper_2605_10363_b200 import workloads as W

    K.lib()
    for name, n in (("cfg1", 8), ("cfg1", 3)):          # two calls in a row, the second on fewer points
        wl = W.named_config(name, n_override=n)
        plan = K.Plan.from_workload(wl)
        D = torch.as_tensor(wl.D, device="cuda")
        E_ref, V_ref = plan.exc(D)                       # existing path: rho -> functional + energy -> V
        V_ref = V_ref.clone()
        rho = plan.eval_rho(D)                           # caller order
        w = torch.as_tensor(wl.grid_w, device="cuda")
        wv = torch.full_like(rho, float("nan"))
        E = torch.full((1,), float("nan"), dtype=torch.float64, device="cuda")
        torch.cuda.synchronize()
        before = torch.cuda.memory_allocated()
        K.xc_lda_noalloc(rho, w, wv, E)
        torch.cuda.synchronize()
        assert torch.cuda.memory_allocated() == before
        assert abs(float(E[0]) - E_ref) <= TOL_E, (float(E[0]), E_ref)
        assert abs(float(E[0]) - E_ref) <= 1e-12 * abs(E_ref)      # same arithmetic, only the summation tree differs
        V = plan.build_vxc(wv)                           # the new entry point's wv through the existing V contraction
        assert float((V - V_ref).abs().max()) <= TOL_V
        assert bool(torch.isfinite(wv).all())
        plan.close()


def test_noalloc_entry_point_rejects_oversize_and_bad_arguments():
    import torch

    from paper_2605_10363_b200 import binding as K

    mx = K.xc_lda_noalloc_max_pts()
    assert mx == 8388608
    L = K.lib()
    one = torch.zeros(1, dtype=torch.float64, device="cuda")
    rc = L.kldi_xc_lda_noalloc(one.data_ptr(), one.data_ptr(), mx + 1, one.data_ptr(), one.data_ptr(), None)
    assert rc == -1 and b"exceeds the static scratch" in L.kldi_last_error()
    assert L.kldi_xc_lda_noalloc(None, one.data_ptr(), 1, one.data_ptr(), one.data_ptr(), None) == -1
    with pytest.raises(K.KldiError):
        K.xc_lda_noalloc(one.cpu(), one, one, one)
    # exactly at the limit, and rho below the cutoff contributes nothing
    n = 1000
    rho = torch.zeros(n, dtype=torch.float64, device="cuda")
    rho[::2] = 1e-25
    w = torch.ones(n, dtype=torch.float64, device="cuda")
    wv, E = torch.empty_like(rho), torch.empty(1, dtype=torch.float64, device="cuda")
    K.xc_lda_noalloc(rho, w, wv, E)
    assert float(E[0]) == 0.0 and float(wv.abs().max()) == 0.0
