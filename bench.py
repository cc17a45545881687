#!/usr/bin/env python
"""bench.py — EXC evaluations/s of the block-filtered hot path on BASELINE.json configs[3]
(256 waters, 6,400 AOs, 4,224,000 grid points, LDA Slater, eps = 1e-12), one JSON line.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config cfg3] [--eps 1e-12]
  python bench.py --impl reference        # the CPU oracle, timed on the host cores (bounded sample)

A "step" is one whole kldi_exc call: D permute -> rho contraction -> functional + energy ->
V contraction -> V finalise, plan creation excluded (once per geometry,
PAPER.md:174) and reported beside it.  N > 1 (torchrun): the quadrature grid is sharded over the
ranks and V, E are all-reduced over NCCL; value = evaluations/s of the whole job.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

METRIC = "exc_evals_per_s"
UNIT = "evals/s"
N_SM, FMA_PER_CLK_SM = 148, 64          # B200: FP64 FMA lanes per SM per clock (DMMA.8x8x4 = 256 FMA / 4 clk)


def basis_of(wl):
    return (wl.atom_xyz, wl.shell_atom, wl.shell_l, wl.shell_prim_off, wl.prim_alpha, wl.prim_coef)


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        d["_source"] = "measured"
        return d
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0, "sm_max_mhz": 1965.0,
            "_source": "fallback"}


class ClockSampler:
    """nvidia-smi clocks and throttle reasons during the timed region (B200_PROFILING.md)."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self._stop, self._t = index, [], threading.Event(), None

    def _run(self):
        while not self._stop.is_set():
            try:
                out = subprocess.run(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                      "-i", str(self.index)], capture_output=True, text=True, timeout=5).stdout
                self.rows.append([c.strip() for c in out.strip().split(",")])
            except Exception:
                pass
            self._stop.wait(0.05)

    def __enter__(self):
        self._t = threading.Thread(target=self._run, daemon=True)
        self._t.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        self._t.join(timeout=6)

    def summary(self):
        sm, mx, reasons = [], 0.0, set()
        for r in self.rows:
            if len(r) < 7:
                continue
            try:
                sm.append(float(r[0]))
                mx = max(mx, float(r[1]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": mx or None,
                "reasons": sorted(reasons), "samples": len(sm)}


def cpu_oracle_sample(wl, n_sample: int):
    """The oracle as it stands on a bounded, strided sample of the workload's grid points."""
    from oracle import exc_oracle as O

    idx = np.arange(0, wl.n_pts, max(1, wl.n_pts // n_sample))[:n_sample]
    t0 = time.perf_counter()
    O.exc(basis_of(wl), wl.grid_xyz[idx], wl.grid_w[idx], wl.D, wl.functional)
    dt = time.perf_counter() - t0
    evals_per_s = (len(idx) / wl.n_pts) / dt
    try:
        cores = len(os.sched_getaffinity(0))
    except AttributeError:
        cores = os.cpu_count()
    try:                                   # the oracle is numpy: its dgemm threads are the BLAS pool's
        from threadpoolctl import threadpool_info
        blas = [int(p["num_threads"]) for p in threadpool_info() if p.get("user_api") == "blas"]
        cores = min(cores, max(blas)) if blas and cores else cores
    except Exception:
        pass
    return {"value": evals_per_s, "unit": UNIT, "cores": cores,
            "kind": "oracle",
            "sample": f"every {max(1, wl.n_pts // n_sample)}-th grid point ({len(idx)} of {wl.n_pts}), dense, "
                      f"{dt:.1f} s, extrapolated linearly in n_pts"}, dt


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from paper_2605_10363_b200 import workloads as W

    wl = W.named_config(args.config, eps=args.eps, becke_backend="auto")
    n_sample = args.ref_sample
    times = []
    base = None
    for i in range(args.warmup + args.steps):
        base, dt = cpu_oracle_sample(wl, n_sample)
        if i >= args.warmup:
            times.append(dt)
    dt = float(np.mean(times))
    val = (min(n_sample, wl.n_pts) / wl.n_pts) / dt
    base["value"] = val
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 / val, "higher_is_better": True,
            "scaling": "strong", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_name(args, wl)}, "cpu_baseline": base,
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))


def workload_name(args, wl):
    return (f"{args.config}: {wl.name}, {wl.n_atoms} atoms, {wl.n_ao} AOs, {wl.n_pts} grid points, "
            f"{wl.functional.upper()}, eps={args.eps:g}, D=2QQ^T")


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="kldi", choices=["kldi", "reference"])
    ap.add_argument("--config", default="cfg3")
    ap.add_argument("--eps", type=float, default=1e-12)
    ap.add_argument("--ref-sample", type=int, default=4096)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--pair-test", type=int, default=0, choices=[0, 1],
                    help="1: executable-pair selection a_pq*b_qr >= eps per call (Eq. 17-19)")
    ap.add_argument("--deterministic-v", type=int, default=2, choices=[0, 1, 2],
                    help="V accumulation: 2 (library default) = fixed-point integer atomics, bitwise reproducible; "
                         "1 = workspace partials + fixed-order reduce; 0 = FP64 atomics")
    ap.add_argument("--rho-tc", type=int, default=0, choices=[0, 1],
                    help="1: headline step with the tcgen05 int8 slice-product rho contraction (KLDI_OPT_RHO_TC); "
                         "0 times it as the extra leg tensor_core_rho")
    ap.add_argument("--rho-dfma", type=int, default=0, choices=[0, 1],
                    help="1: LDA rho contraction on the vector FP64 pipe (register tiles) instead of DMMA tiles")
    ap.add_argument("--grad", action="store_true",
                    help="also time kldi_exc_grad (LDA nuclear-gradient contraction) on a plan with gradient stores")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "kldi" else args.warmup

    if args.impl == "reference":
        return run_reference(args)

    import torch
    import torch.distributed as dist

    import __graft_entry__ as G

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the kldi path has no CPU fallback (use --impl reference)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    if local == 0:
        G.build()
    if world > 1:
        dist.barrier()

    from paper_2605_10363_b200 import binding as K
    from paper_2605_10363_b200 import sharding
    from paper_2605_10363_b200 import workloads as W

    t0 = time.perf_counter()
    if world == 1:
        wl_full = W.named_config(args.config, eps=args.eps)
    else:
        # the Becke partition (2.5e12 cell functions on cfg3) is evaluated once, on rank 0, and its weights broadcast;
        # geometry, basis, grid points and D are cheap and seeded, every rank builds them itself
        wl_full = W.named_config(args.config, eps=args.eps, becke_backend="auto" if rank == 0 else "none")
        gw = torch.as_tensor(wl_full.grid_w, device="cuda").contiguous()
        dist.broadcast(gw, src=0)
        wl_full.grid_w = gw.cpu().numpy()
        del gw
    gen_s = time.perf_counter() - t0
    wl = wl_full
    if world > 1:
        wl, _ = sharding.shard_workload(wl_full, rank, world)     # cost-balanced range of the plan's curve order
    gga = wl.functional == "gga"
    func = K.KLDI_GGA_PBEX if gga else K.KLDI_LDA_SLATER
    plan = K.Plan.from_workload(wl)
    plan.set_option(K.KLDI_OPT_DETERMINISTIC_V, args.deterministic_v)
    plan.set_option(K.KLDI_OPT_PAIR_TEST, args.pair_test)
    plan.set_option(K.KLDI_OPT_RHO_DFMA, args.rho_dfma)
    if not gga:
        plan.set_option(K.KLDI_OPT_RHO_TC, args.rho_tc)
    st = plan.stats.as_dict()
    D = torch.as_tensor(wl.D, device="cuda")
    V = torch.empty((wl.n_ao, wl.n_ao), dtype=torch.float64, device="cuda")

    def step():
        E, _ = plan.exc(D, func, out=V)
        if world > 1:
            E, _ = sharding.allreduce_exc(E, V)
        return E

    for _ in range(args.warmup):
        E = step()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    stage_ms = {}
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    with ClockSampler(torch.cuda.current_device()) as cs:
        ev0.record()
        for _ in range(args.steps):
            E = step()
        ev1.record()
        torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    n_stage = min(args.steps, 10)          # per-stage times from the library's own CUDA events: a separate, untimed pass
    for _ in range(n_stage):
        step()
        for k, v in plan.last_timings().items():
            stage_ms[k] = stage_ms.get(k, 0.0) + v / n_stage
    launches = int(plan.refresh_stats().kernel_launches)
    ms = ev0.elapsed_time(ev1)
    if world > 1:
        t = torch.tensor([ms], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms = float(t.item())
    ms_per_step = ms / args.steps
    value = 1e3 / ms_per_step

    # ---- end to end through the C ABI with HOST buffers (pinned): H2D of D and D2H of V inside the timed region.
    # D and V are symmetric: kldi_exc_host uploads the lower triangle of D, and with KLDI_OPT_HOST_V_TRIANGLE it
    # downloads only the lower triangle of V (row bands); the full-matrix download is timed beside it.
    e2e = None
    if world == 1:
        Dh = torch.as_tensor(wl.D).pin_memory()
        Vh = torch.empty((wl.n_ao, wl.n_ao), dtype=torch.float64).pin_memory()
        nn = wl.n_ao * wl.n_ao * 8
        bands = 1 if wl.n_ao < 1024 else 32
        tri = sum(8 * (wl.n_ao * (b + 1) // bands) * (wl.n_ao * (b + 1) // bands - wl.n_ao * b // bands)
                  for b in range(bands))
        res = {}
        for mode in (1, 0):
            plan.set_option(K.KLDI_OPT_HOST_V_TRIANGLE, mode)
            for _ in range(2):
                plan.exc_host(Dh, func, Vh)
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            for _ in range(args.steps):
                plan.exc_host(Dh, func, Vh)
            torch.cuda.synchronize()
            res[mode] = (time.perf_counter() - t0) / args.steps
        plan.set_option(K.KLDI_OPT_HOST_V_TRIANGLE, 0)
        e2e = {"value": 1.0 / res[1], "unit": UNIT, "h2d_bytes_per_step": tri, "d2h_bytes_per_step": tri + 8,
               "ms_per_step": res[1] * 1e3, "mode": "lower triangles of D (upload) and V (download), row bands",
               "full_v_download": {"value": 1.0 / res[0], "ms_per_step": res[0] * 1e3, "d2h_bytes_per_step": nn + 8}}

    # ---- the same step with the other V accumulation mode (0 = FP64 atomics; the default 2 = 64-bit fixed-point
    # integer atomics, bitwise reproducible) and, for LDA, with the tcgen05 int8 slice-product rho contraction
    def timed_leg(n):
        for _ in range(3):
            plan.exc(D, func, out=V)
        f0, f1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        f0.record()
        for _ in range(n):
            plan.exc(D, func, out=V)
        f1.record()
        torch.cuda.synchronize()
        return 1e3 * n / f0.elapsed_time(f1)

    fx_leg, tc_leg = None, None
    if world == 1:
        other = 0 if args.deterministic_v == 2 else 2
        Va = V.clone()
        plan.exc(D, func, out=V)
        same = bool(torch.equal(Va, V))
        plan.set_option(K.KLDI_OPT_DETERMINISTIC_V, other)
        fx_leg = {"headline_mode": args.deterministic_v, "headline_bitwise_equal_between_calls": same,
                  "other_mode": other, "other_mode_evals_per_s": timed_leg(args.steps),
                  "other_mode_vxc_ms": plan.last_timings()["vxc"],
                  "modes": "2 = fixed-point integer atomics (no FP64 atomics, reproducible), 0 = red.global.add.f64"}
        plan.set_option(K.KLDI_OPT_DETERMINISTIC_V, args.deterministic_v)
    if world == 1 and not gga:
        rho_ref = plan.eval_rho(D).clone()
        plan.set_option(K.KLDI_OPT_RHO_TC, 1 - args.rho_tc)
        evs = timed_leg(args.steps)
        tms = plan.last_timings()
        st_tc = plan.refresh_stats().as_dict()
        rho_tc = plan.eval_rho(D)
        which = "KLDI_OPT_RHO_TC=%d" % (1 - args.rho_tc)
        tc_leg = {"option": which, "evals_per_s": evs, "rho_ms": tms["rho"], "total_ms": tms["total"],
                  "max_abs_d_rho_between_paths": float((rho_tc - rho_ref).abs().max()),
                  "int8_ops_per_launch": st_tc["ops_rho_tc"], "kernel_launches": st_tc["kernel_launches"]}
        plan.set_option(K.KLDI_OPT_RHO_TC, args.rho_tc)
        del rho_ref, rho_tc

    # ---- BASELINE.json configs[3]: how the retained fraction, the throughput and the result move with eps.  The three
    # errors are taken against the stored result of the dense CPU oracle (tests/golden/cfg3_oracle.npz, written from
    # oracle/ alone): E_xc, rho on every 64th point, 16 full rows + a strided sample of V; without the file, against
    # this run's eps = 1e-12 result (GPU vs GPU: the screening increment only).
    eps_leg = None
    second_plan_s = None
    if world == 1 and args.config == "cfg3" and abs(args.eps - 1e-12) < 1e-20:
        gpath = os.path.join(ROOT, "tests", "golden", "cfg3_oracle.npz")
        gold = np.load(gpath) if os.path.exists(gpath) else None
        rho_a = plan.eval_rho(D).clone()
        Ea, _ = plan.exc(D, func, out=V)
        Va = V.clone()

        def errors(E_, rho_, V_):
            if gold is not None:
                sp, sv = int(gold["stride_pts"]), gold["stride_v"]
                rows = torch.as_tensor(gold["v_rows"], device="cuda")
                return {"reference": "dense CPU oracle (tests/golden/cfg3_oracle.npz)",
                        "max_abs_d_rho": float((rho_[::sp].cpu() - torch.as_tensor(gold["rho_strided"])).abs().max()),
                        "max_abs_d_V": max(float((V_[rows].cpu() - torch.as_tensor(gold["V_rows"])).abs().max()),
                                           float((V_[::int(sv[0]), ::int(sv[1])].cpu() - torch.as_tensor(gold["V_strided"])).abs().max())),
                        "abs_d_E": abs(E_ - float(gold["E"]))}
            return {"reference": "this run at eps = 1e-12 (GPU vs GPU)",
                    "max_abs_d_rho": float((rho_ - rho_a).abs().max()), "max_abs_d_V": float((V_ - Va).abs().max()),
                    "abs_d_E": abs(E_ - Ea)}

        eps_leg = [dict(eps=args.eps, evals_per_s=value, **errors(Ea, rho_a, Va))]
        for eps2 in (1e-10, 1e-8):
            p2 = K.Plan.from_workload(wl, eps=eps2)
            p2.set_option(K.KLDI_OPT_DETERMINISTIC_V, args.deterministic_v)
            if eps2 == 1e-10:
                second_plan_s = p2.stats.plan_seconds      # a plan after the first of the process: no module loading
            V2 = torch.empty_like(V)
            for _ in range(3):
                E2, _ = p2.exc(D, func, out=V2)
            q0, q1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize()
            q0.record()
            for _ in range(5):
                p2.exc(D, func, out=V2)
            q1.record()
            torch.cuda.synchronize()
            s2 = p2.stats.as_dict()
            eps_leg.append(dict(eps=eps2, evals_per_s=5e3 / q0.elapsed_time(q1),
                                retained_blocks_over_candidates=s2["retained_blocks"] / s2["candidate_blocks"],
                                sum_k=s2["sum_k"], phi_bytes=s2["phi_bytes"],
                                retained_over_dense_flops=(s2["flops_rho_useful_sym"] + s2["flops_v_useful"]) / (2 * s2["flops_dense"]),
                                **errors(E2, p2.eval_rho(D), V2)))
            p2.close()
        del rho_a, Va

    # ---- the LDA nuclear-gradient contraction on the same molecule (its own plan: Phi + grad Phi)
    grad_leg = None
    if args.grad and world == 1:
        plan_g = K.Plan.from_workload(wl, want_gradients=True)
        for _ in range(3):
            plan_g.exc_grad(D)
        tg = {}
        g0, g1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        g0.record()
        for _ in range(args.steps):
            plan_g.exc_grad(D)
            for k, v in plan_g.last_timings().items():
                tg[k] = tg.get(k, 0.0) + v / args.steps
        g1.record()
        torch.cuda.synchronize()
        gms = g0.elapsed_time(g1) / args.steps
        sg = plan_g.stats.as_dict()
        col_bytes = 4 * 8 * 128 * sg["sum_k"]           # X + three gradient stores, read once by k_grad_cols
        grad_leg = {"evals_per_s": 1e3 / gms, "ms_per_call": gms, "functional": "lda_slater",
                    "stage_ms": {"permute_D": tg["permute_D"], "x_and_rho_build": tg["rho"], "xc": tg["xc"],
                                 "grad_contraction": tg["vxc"]},
                    "x_build_tflops_issued": sg["flops_rho_exec"] / (tg["rho"] * 1e-3) / 1e12,
                    "grad_contraction_gbs": col_bytes / (tg["vxc"] * 1e-3) / 1e9,
                    "grad_contraction_frac_of_hbm": col_bytes / (tg["vxc"] * 1e-3) / 1e9 / peaks().get("hbm_gbs", 6650.0),
                    "sum_k": sg["sum_k"], "plan_create_s": sg["plan_seconds"]}
        tgg = []
        for i in range(3 + min(args.steps, 10)):
            plan_g.exc_grad(D, K.KLDI_GGA_PBEX)
            if i >= 3:
                tgg.append(plan_g.last_timings()["total"])
        grad_leg["gga_pbex_ms_per_call"] = float(np.median(tgg))
        # the same calls with KLDI_OPT_RHO_TC (X builds / tau builds as int8 slice products on tcgen05)
        plan_g.set_option(K.KLDI_OPT_RHO_TC, 1)
        tc_ms = {}
        for key, call in (("lda_slater", lambda: plan_g.exc_grad(D)), ("gga_pbex", lambda: plan_g.exc_grad(D, K.KLDI_GGA_PBEX)),
                          ("eval_tau", lambda: plan_g.eval_tau(D))):
            tt = []
            for i in range(6):
                call()
                if i >= 2:
                    tt.append(plan_g.last_timings()["total"])
            tc_ms[key] = float(np.median(tt))
        grad_leg["with_rho_tc_ms_per_call"] = tc_ms
        plan_g.set_option(K.KLDI_OPT_RHO_TC, 0)
        # the meta-GGA contractions on the same plan (three LDA-form builds each)
        wv_t = torch.as_tensor(wl.grid_w, device="cuda").clone()
        Vt = torch.empty((wl.n_ao, wl.n_ao), dtype=torch.float64, device="cuda")
        t_tau, t_vtau = [], []
        for i in range(3 + min(args.steps, 10)):
            plan_g.eval_tau(D)
            a = plan_g.last_timings()["rho"]
            plan_g.build_vtau(wv_t, out=Vt)
            b = plan_g.last_timings()["vxc"]
            if i >= 3:
                t_tau.append(a)
                t_vtau.append(b)
        grad_leg["meta_gga"] = {"eval_tau_ms": float(np.median(t_tau)), "build_vtau_ms": float(np.median(t_vtau)),
                                "tau_tflops_useful": 3 * sg["flops_rho_useful_sym"] / (np.median(t_tau) * 1e-3) / 1e12,
                                "vtau_tflops_useful": 3 * sg["flops_rho_useful_sym"] / (np.median(t_vtau) * 1e-3) / 1e12}
        plan_g.close()

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    pk = peaks()
    fp64_clock_peak = N_SM * FMA_PER_CLK_SM * 2 * pk.get("sm_max_mhz", 1965.0) * 1e6 / 1e12
    try:
        dmma_live = K.fp64_peak("dmma", 20000)
    except Exception:
        dmma_live = None
    # LDA: the rho build uses D = D^T (triangular D'), so its useful work is 128 K(K+1) per block;
    # GGA needs the full X = Phi D for grad rho.  The unsymmetrised 2*128*K^2 figure is reported beside it.
    f_rho = st["flops_rho_useful"] if gga else st["flops_rho_useful_sym"]
    f_rho_exec = st["flops_rho_exec"] if gga else st["flops_rho_exec_sym"]
    f_v = st["flops_v_useful"]
    f_total = f_rho + f_v
    f_total_unsym = st["flops_rho_useful"] + f_v
    t_rho = stage_ms["rho"] * 1e-3
    roof = {"bound": "tensor", "kernel": "k_rho (rho contraction, DMMA.8x8x4)",
            "achieved": f_rho / t_rho / 1e12, "peak": fp64_clock_peak, "unit": "TFLOP/s",
            "frac": f_rho / t_rho / 1e12 / fp64_clock_peak,
            "peak_source": "FP64 tensor peak derived from unit counts: 148 SMs x 64 FMA/clk x 2 x sm_max_mhz of "
                           f"MEASURED_PEAKS.json ({pk['_source']}); live DMMA microbenchmark "
                           f"{dmma_live and round(dmma_live, 2)} TFLOP/s; bf16-ratio rule would give "
                           f"{pk['bf16_tflops'] * 40.0 / 2250.0:.1f}",
            "flops_per_launch": f_rho, "exec_flops_per_launch": f_rho_exec,
            "exec_frac": f_rho_exec / t_rho / 1e12 / fp64_clock_peak,
            "launch_ms": stage_ms["rho"], "traffic": None,
            # DMMA.8x8x4 itself tops out below the FP64 unit rate (profiles/r1f_summary.md): issued FLOPs against it
            "dmma_instruction_cap_tflops": dmma_live,
            "exec_frac_of_dmma_cap": (f_rho_exec / t_rho / 1e12 / dmma_live) if dmma_live else None,
            "v_kernel": {"achieved": f_v / (stage_ms["vxc"] * 1e-3) / 1e12, "launch_ms": stage_ms["vxc"],
                         "frac": f_v / (stage_ms["vxc"] * 1e-3) / 1e12 / fp64_clock_peak,
                         "flops_per_launch": f_v, "exec_flops_per_launch": st["flops_v_exec"],
                         "exec_frac": st["flops_v_exec"] / (stage_ms["vxc"] * 1e-3) / 1e12 / fp64_clock_peak,
                         "schedule_critical_path_flops": st["flops_v_crit"],
                         "accumulation_mode": args.deterministic_v}}
    # DRAM bytes per launch come from an `ncu --set full` capture, which cannot run inside a timed benchmark: the
    # committed text file profiles/traffic.csv (config, kernel, bytes, round, source) is looked up and its provenance
    # reported; a kernel changed since that capture is the summary's to say.
    tr = os.path.join(ROOT, "profiles", "traffic.csv")
    kern = "k_rho_i8" if (args.rho_tc and not gga) else "k_rho"
    if os.path.exists(tr):
        with open(tr) as f:
            for ln in f:
                c = ln.strip().split(",")
                if len(c) >= 3 and c[0] == args.config and c[1] == kern and abs(args.eps - 1e-12) < 1e-20:
                    roof["traffic"] = int(c[2])
                    roof["traffic_source"] = "profiles/traffic.csv: " + ", ".join(c[3:])
    if args.rho_tc and not gga:
        # tensor-core path: int8 operations issued against the int8 peak (measured bf16 peak x the nominal 2:1 ratio)
        i8_peak = pk["bf16_tflops"] * 2.0
        ops = plan.refresh_stats().ops_rho_tc
        roof.update({"kernel": "k_rho_i8 (rho contraction, tcgen05 kind::i8 slice products)", "unit": "TOP/s (int8)",
                     "achieved": ops / t_rho / 1e12, "peak": i8_peak, "frac": ops / t_rho / 1e12 / i8_peak,
                     "peak_source": f"int8 tensor peak = measured bf16 {pk['bf16_tflops']} TFLOP/s ({pk['_source']}) x 2 "
                                    "(nominal 4.5 : 2.25 PFLOP/s)",
                     "retained_block_fp64_equivalent_tflops": f_rho / t_rho / 1e12,
                     "launch_ms_includes": "k_colmax + k_slice_D (D' digits) + k_rho_i8"})
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "strong", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_name(args, wl_full), "l2": "inputs_larger_than_l2 (Phi store "
                   f"{st['phi_bytes'] / 1e9:.1f} GB, D {wl.n_ao ** 2 * 8 / 1e6:.0f} MB)",
                   "parallelism": "single GPU" if world == 1 else f"grid sharded over {world} ranks + NCCL all-reduce of V,E"},
        "grid_points_per_s": wl_full.n_pts * value,
        "retained_block_tflops": f_total * world / (ms_per_step * 1e-3) / 1e12 if world == 1 else None,
        "retained_block_frac_of_fp64_peak": f_total / (ms_per_step * 1e-3) / 1e12 / fp64_clock_peak if world == 1 else None,
        "retained_block_frac_of_nominal_40tf": f_total / (ms_per_step * 1e-3) / 1e12 / 40.0 if world == 1 else None,
        "retained_block_tflops_without_rho_symmetry": f_total_unsym / (ms_per_step * 1e-3) / 1e12 if world == 1 else None,
        "flops": {"rho_useful": f_rho, "rho_useful_without_symmetry": st["flops_rho_useful"], "v_useful": f_v,
                  "rho_exec": f_rho_exec, "v_exec": st["flops_v_exec"], "rho_symmetry_halving": not gga,
                  "dense_one_product": st["flops_dense"], "retained_over_dense": f_total / (2 * st["flops_dense"]),
                  "v_symmetry_halving": not gga, "ao_partition": "one AO block per shell"},
        "stage_ms": stage_ms, "plan_create_s": st["plan_seconds"], "plan_create_note": "first plan of the process (includes one-time module loading)", "workload_gen_s": gen_s, "exc_energy": E,
        "plan": {k: st[k] for k in ("n_blocks", "n_blocks_nonempty", "retained_blocks", "candidate_blocks", "sum_k",
                                     "max_k", "phi_bytes")},
        "pair_test": {"enabled": bool(args.pair_test), "stages_total": plan.refresh_stats().pair_stages_total,
                      "stages_executed": plan.stats.pair_stages_executed},
        "gpu_launches": launches * args.steps, "gpu_launches_per_step": launches,
        "gpu_launches_note": "kernels of libkldi per kldi_exc, counted by the library (kldi_stats.kernel_launches); "
                             "the 4-5 cudaMemsetAsync nodes per call are not kernels of this library",
        "clocks": cs.summary(), "roofline": roof, "e2e": e2e,
        "nuclear_gradient": grad_leg, "v_accumulation": fx_leg, "tensor_core_rho": tc_leg, "eps_scaling": eps_leg,
        "plan_create_second_plan_s": second_plan_s,
    }
    if not args.no_cpu_baseline and world == 1:
        line["cpu_baseline"], _ = cpu_oracle_sample(wl_full, args.ref_sample)
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
