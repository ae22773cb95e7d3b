#!/usr/bin/env python
"""bench.py -- one JSON line for the hot path of arXiv:1405.4524 on B200 (contract: task prompt).

A step = one pass of the whole hot path over one batch of synthetic input at BASELINE.json configs[3]
(24^3x48, kappa 0.118, c_sw 1.5, links exp(i 0.4 H)): noise_fill of N_r = 32 Z4 sources, then clover_solve of all of
them in batches of 8 (fp32 BiCGStab with fp64 reliable updates, tol 1e-10), source prep, odd-site reconstruction,
fp64 full-lattice verification and layout reorders included.  metric = BiCGStab seconds/source; the Dslash GB/s half
of BASELINE.json's metric is the `roofline` object (the fused fp32 Dslash kernel of the iteration, timed launch by
launch with CUDA events inside the timed steps) plus `dslash` (the plain hop kernel timed alone).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config i]
"""
import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "BiCGStab seconds/source at 24^3x48 (clover Dslash GB/s, % of HBM peak: see roofline)"
UNIT = "s/source"


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        return json.load(open(p)), "measured"
    return {"hbm_gbs": 6650.0}, "fallback"


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons with NVML during the timed region."""

    def __init__(self, index=0, period=0.05):
        super().__init__(daemon=True)
        self.index, self.period, self.samples, self.reasons, self.stop_flag = index, period, [], set(), False
        self.max_mhz = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def run(self):
        if not self.nv:
            return
        nv = self.nv
        names = {nv.nvmlClocksThrottleReasonSwPowerCap: "sw_power_cap", nv.nvmlClocksThrottleReasonHwSlowdown: "hw_slowdown",
                 nv.nvmlClocksThrottleReasonHwThermalSlowdown: "hw_thermal_slowdown",
                 nv.nvmlClocksThrottleReasonSwThermalSlowdown: "sw_thermal_slowdown",
                 nv.nvmlClocksThrottleReasonHwPowerBrakeSlowdown: "hw_power_brake"}
        while not self.stop_flag:
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, name in names.items():
                    if r & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            time.sleep(self.period)

    def summary(self):
        s = sorted(self.samples)
        return {"sm_mhz": s[len(s) // 2] if s else None, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": len(s)}


def oracle_sample(cfg, iters_sample, U=None):
    """Time the CPU oracle as it stands on a bounded sample: `iters_sample` BiCGStab iterations of one source on the full
    lattice, scaled by the iteration count the same oracle needs to reach 1e-10 with the same parameters on 8^3x16
    (iteration counts are volume independent for these uncorrelated links)."""
    import numpy as np
    import oracle
    from paper_1405_4524_b200 import workloads as wl
    small = (8, 8, 8, 16)
    Us = wl.gauge_links(small, cfg["eps"], cfg["gauge_seed"])
    As = oracle.clover_matrix(Us, cfg["kappa"], cfg["csw"])
    _, info = oracle.bicgstab(Us, As, wl.BC, cfg["kappa"], oracle.noise_fill(small, cfg["noise_seed"], 1, scale=wl.INV_SQRT2)[0], tol=wl.TOL)
    n_it = info["iters"]
    if U is None:
        U = wl.gauge_links(cfg["dims"], cfg["eps"], cfg["gauge_seed"])
    A = oracle.clover_matrix(U, cfg["kappa"], cfg["csw"])
    eta = oracle.noise_fill(cfg["dims"], cfg["noise_seed"], 1, scale=wl.INV_SQRT2)[0]

    def run():
        t0 = time.perf_counter()
        oracle.bicgstab(U, A, wl.BC, cfg["kappa"], eta, tol=1e-30, max_iter=iters_sample)
        return (time.perf_counter() - t0) / iters_sample * n_it   # seconds per source
    return run, n_it, oracle.threads()


def run_reference(args, cfg):
    """--impl reference: the oracle on the host cores (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    iters_sample = 2
    run, n_it, cores = oracle_sample(cfg, iters_sample)
    for _ in range(args.warmup):
        run()
    vals = [run() for _ in range(args.steps)]
    v = sum(vals) / len(vals)
    sample = (f"{iters_sample} BiCGStab iterations (2 D applies each + true residual) of 1 source on {cfg['name']}, "
              f"scaled to the {n_it} iterations the oracle needs for 1e-10 at these parameters on 8^3x16")
    print(json.dumps({"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
                      "warmup": args.warmup, "ms_per_step": v * 1e3, "higher_is_better": False, "scaling": "weak", "vs_baseline": None,
                      "dtype": "f64", "data": "synthetic", "config": {"workload": cfg["name"], "n_rhs": 1, "solver": "oracle BiCGStab, unpreconditioned"},
                      "cpu_baseline": {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
                      "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3)
    ap.add_argument("--recon", type=int, default=0, choices=[0, 12, 18], help="override the workload's link storage of the fp32 operator (0: as configured)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--kernel-bench", action="store_true", help="only time the three Dslash kernels alone (fp32/fp64, B = 1 and batch) and print them")
    ap.add_argument("--reps", type=int, default=20)
    ap.add_argument("--kb-filter", default="", help="comma-separated substrings; with --kernel-bench only time kernels whose name contains one")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup

    from paper_1405_4524_b200 import workloads as wl
    cfg = dict(wl.CONFIGS[args.config])
    if args.recon:
        cfg["recon"] = args.recon
    if args.impl == "reference":
        return run_reference(args, cfg)

    import numpy as np
    import torch
    from paper_1405_4524_b200 import binding as B   # fails loudly if the CUDA library is missing

    rank, world, local = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")), int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl")

    def barrier():
        if dist:
            dist.barrier()
        torch.cuda.synchronize()

    from paper_1405_4524_b200 import sharding

    def max_over_ranks(x):
        return sharding.max_over_ranks(x, device="cuda")

    dims, n_rhs, batch = cfg["dims"], cfg["n_rhs"], cfg["batch"]
    X, Y, Z, T = dims
    V, Vh = X * Y * Z * T, X * Y * Z * T // 2
    U = wl.gauge_links(dims, cfg["eps"], cfg["gauge_seed"])
    ctx = B.Clover(torch.from_numpy(U).cuda(), cfg["kappa"], cfg["csw"], bc=wl.BC, recon=cfg["recon"], max_rhs=8)
    if args.kernel_bench:
        peaks, _ = measured_peaks()
        res = {}
        for prec, b in ((32, 4), (64, 8)):
            g = cfg["recon"] if prec == 32 else 18
            for nr in sorted({1, batch}):
                for k, name, fl in ((B.KERNEL_HOP, "hop", 1320), (B.KERNEL_AINV_HOP, "ainv_hop", 1824), (B.KERNEL_A_MINUS_HOP, "a_minus_hop", 1872),
                                    (B.KERNEL_A_MINUS_HOP_S, "a_minus_hop_s", 1872), (B.KERNEL_A_MINUS_HOP_XW, "a_minus_hop_xw", 1872)):
                    if args.kb_filter and not any(f in f"fp{prec}_{name}_b{nr}" for f in args.kb_filter.split(",")):
                        continue
                    t = ctx.bench_kernel(k, prec, nr, reps=args.reps, flush_l2=True) * 1e-3
                    bm = (8 * g * b + (72 * b if k else 0)) / nr + 24 * b * {B.KERNEL_A_MINUS_HOP: 3, B.KERNEL_A_MINUS_HOP_S: 4, B.KERNEL_A_MINUS_HOP_XW: 4}.get(k, 2)
                    res[f"fp{prec}_{name}_b{nr}"] = {"us": round(t * 1e6, 2), "bytes_per_site_rhs": bm, "gbs": round(bm * Vh * nr / t / 1e9, 1),
                                                     "frac_hbm": round(bm * Vh * nr / t / 1e9 / peaks["hbm_gbs"], 4), "gflops": round(fl * Vh * nr / t / 1e9, 1)}
        print(json.dumps({"kernel_bench": cfg["name"], "peak_gbs": peaks["hbm_gbs"], "kernels": res}))
        ctx.close()
        return
    # weak scaling: every rank solves its own n_rhs sources (distinct noise streams), replicas of the operator, no collective
    offset = sharding.source_offset(rank, n_rhs)
    eta = torch.empty((n_rhs, T, Z, Y, X, 4, 3), dtype=torch.complex128, device="cuda")
    psi = torch.empty_like(eta)
    launches = 0
    kstats = {"n_ainv_hop": 0, "n_a_minus_hop": 0, "ms_ainv_hop": 0.0, "ms_a_minus_hop": 0.0, "n_a_minus_hop_s": 0, "ms_a_minus_hop_s": 0.0}
    phases = {k: 0.0 for k in ("ms_total", "ms_reorder", "ms_prep", "ms_iterate", "ms_reliable", "ms_finish")}
    last = {}

    def step(count):
        nonlocal launches
        B.noise_fill(dims, cfg["noise_seed"], n_rhs, rhs_offset=offset, time_dilution=cfg["dilution"], scale=wl.INV_SQRT2, out=eta)
        _, infos, bad = ctx.solve(eta, tol=wl.TOL, batch=batch, mixed=bool(cfg["mixed"]), out=psi)
        if bad:
            raise RuntimeError(f"{bad} sources did not converge: {infos}")
        last["infos"] = infos
        if count:
            s = ctx.stats()
            launches += s["kernel_launches"] + 1
            for k in kstats:
                kstats[k] += s[k]
            for k in phases:
                phases[k] += s[k]

    for _ in range(args.warmup):
        step(False)
    sampler = ClockSampler(local)
    barrier()
    sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(args.steps):
        step(True)
    e1.record()
    barrier()
    sampler.stop_flag = True
    ms = max_over_ranks(e0.elapsed_time(e1))
    value = sharding.whole_job_seconds_per_source(ms, args.steps, n_rhs, world)   # world * n_rhs sources per step

    # ---- roofline of the dominant kernel: the fused fp32 Dslash y_e = A x_e - kappa^2 H_eo t_o (+dots) of the iteration ----
    peaks, peak_kind = measured_peaks()
    b = 4 if cfg["mixed"] else 8
    g = cfg["recon"] if cfg["mixed"] else 18
    merged = kstats["n_a_minus_hop_s"] > 0   # merged iteration (solver.cu): both fused Dslash variants also read w (r or r0) at the own site
    bytes_a_minus = (8 * g * b + 72 * b) / batch + 24 * b * (4 if merged else 3)   # links + clover shared by the batch; in, x, (w,) out per rhs
    bytes_ainv = (8 * g * b + 72 * b) / batch + 24 * b * 2
    prec = 32 if cfg["mixed"] else 64
    timed = "CUDA events around every launch inside the timed steps"
    if kstats["n_a_minus_hop"]:
        t_a_minus = kstats["ms_a_minus_hop"] / kstats["n_a_minus_hop"] * 1e-3
        t_ainv = kstats["ms_ainv_hop"] / kstats["n_ainv_hop"] * 1e-3
    else:   # launch-bound lattice: the iteration ran as a CUDA graph, without per-launch events; time the kernels alone
        t_a_minus = ctx.bench_kernel(B.KERNEL_A_MINUS_HOP, prec, batch, reps=20) * 1e-3
        t_ainv = ctx.bench_kernel(B.KERNEL_AINV_HOP, prec, batch, reps=20) * 1e-3
        timed = "kernel timed alone (the solve replays its iteration as a CUDA graph on this lattice; fields fit L2)"
    ach = bytes_a_minus * Vh * batch / t_a_minus / 1e9
    traffic = None
    tp = os.path.join(ROOT, "profiles", "traffic.json")   # DRAM bytes per launch from the committed ncu --set full capture
    if os.path.exists(tp):
        traffic = json.load(open(tp)).get(f"a_minus_hop{'_xw' if merged else ''}_{cfg['name']}_b{batch}")
    epi = "t = A s - k^2 H tmp, +<t,s>,<t,t>,<r0,t>,<r0,s>" if merged else "A x - k^2 H t,+dots"
    roofline = {"bound": "hbm", "kernel": (f"dslash2_kernel<B={batch},recon={g},{epi}> (fp32, one thread per site and rhs pair)" if cfg["mixed"] and batch >= 2
                           else f"dslash_kernel<{'float' if cfg['mixed'] else 'double'},B={batch},recon={g},{epi}>"),
                "achieved": ach, "timed": timed, "peak": peaks["hbm_gbs"], "peak_kind": peak_kind, "unit": "GB/s", "frac": ach / peaks["hbm_gbs"],
                "traffic": traffic, "algorithmic_bytes_per_site_rhs": bytes_a_minus, "us_per_launch": t_a_minus * 1e6,
                "gflops": 1872.0 * Vh * batch / t_a_minus / 1e9,
                "other_kernels": {"ainv_hop": {"achieved": bytes_ainv * Vh * batch / t_ainv / 1e9, "us_per_launch": t_ainv * 1e6,
                                               "frac": bytes_ainv * Vh * batch / t_ainv / 1e9 / peaks["hbm_gbs"],
                                               "algorithmic_bytes_per_site_rhs": bytes_ainv}}}
    if merged:   # the other fused variant of the iteration: s = r - alpha (A p - k^2 H tmp), same bytes, no reduction
        t_s = kstats["ms_a_minus_hop_s"] / kstats["n_a_minus_hop_s"] * 1e-3
        roofline["other_kernels"]["a_minus_hop_s"] = {"achieved": bytes_a_minus * Vh * batch / t_s / 1e9, "us_per_launch": t_s * 1e6,
                                                      "frac": bytes_a_minus * Vh * batch / t_s / 1e9 / peaks["hbm_gbs"],
                                                      "algorithmic_bytes_per_site_rhs": bytes_a_minus}

    # ---- the plain Wilson hop kernel timed alone (BASELINE.json: "clover Dslash GB/s"), fields larger than L2 or L2 flushed ----
    dslash = {}
    if rank == 0:
        for nr in (1, batch):
            t = ctx.bench_kernel(B.KERNEL_HOP, 32, nr, reps=20, flush_l2=True) * 1e-3
            bm = 8 * cfg["recon"] * 4 / nr + 24 * 4 * 2
            dslash[f"fp32_hop_b{nr}"] = {"us": t * 1e6, "gbs": bm * Vh * nr / t / 1e9, "pct_hbm": 100 * bm * Vh * nr / t / 1e9 / peaks["hbm_gbs"],
                                         "gflops": 1320.0 * Vh * nr / t / 1e9, "bytes_per_site_rhs": bm}

    # ---- e2e: the same step through clover_solve_host (pinned host sources in, propagators out, copies inside) ----
    e2e = None
    if not args.no_e2e:
        per = V * 24 * 8
        h_eta = torch.empty((n_rhs, T, Z, Y, X, 4, 3), dtype=torch.complex128).pin_memory()
        h_psi = torch.empty_like(h_eta).pin_memory()
        h_eta.copy_(eta)
        for _ in range(2):
            ctx.solve_host(h_eta, tol=wl.TOL, batch=batch, mixed=bool(cfg["mixed"]), out=h_psi)
        barrier()
        t0 = time.perf_counter()
        e0.record()
        for _ in range(args.steps):
            ctx.solve_host(h_eta, tol=wl.TOL, batch=batch, mixed=bool(cfg["mixed"]), out=h_psi)
        e1.record()
        barrier()
        ems = max_over_ranks(e0.elapsed_time(e1))
        e2e = {"value": ems * 1e-3 / (args.steps * n_rhs) / world, "unit": UNIT, "h2d_bytes_per_step": per * n_rhs, "d2h_bytes_per_step": per * n_rhs,
               "wall_s_per_step": (time.perf_counter() - t0) / args.steps}
        del h_eta, h_psi

    # ---- H1 noise fill alone (a pure write stream: 192 B per site and source in fp64) ----
    noise = None
    if rank == 0:
        B.noise_fill(dims, cfg["noise_seed"], n_rhs, rhs_offset=offset, time_dilution=cfg["dilution"], scale=wl.INV_SQRT2, out=eta)
        torch.cuda.synchronize()
        n0, n1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        n0.record()
        for _ in range(5):
            B.noise_fill(dims, cfg["noise_seed"], n_rhs, rhs_offset=offset, time_dilution=cfg["dilution"], scale=wl.INV_SQRT2, out=eta)
        n1.record()
        torch.cuda.synchronize()
        tn = n0.elapsed_time(n1) / 5 * 1e-3
        noise = {"ms": tn * 1e3, "write_gbs": n_rhs * V * 192 / tn / 1e9, "frac_hbm": n_rhs * V * 192 / tn / 1e9 / peaks["hbm_gbs"]}

    # ---- NEXT row (S 8(f) rank 1): stochastic-operator contraction O_ij(t) of the step's sources and solutions ----
    contraction = None
    if rank == 0:
        o = B.stochastic_operators(eta, psi)
        torch.cuda.synchronize()
        c0, c1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        c0.record()
        for _ in range(5):
            o = B.stochastic_operators(eta, psi)
        c1.record()
        torch.cuda.synchronize()
        tc = c0.elapsed_time(c1) / 5 * 1e-3
        cbytes = 2 * n_rhs * V * 24 * 8
        cflop = 8.0 * n_rhs * n_rhs * 12 * V
        fp64_peak = 148 * 64 * 2 * 1.965e9     # fp64 FMA lanes per SM x SMs x 2 flop x max clock
        contraction = {"what": "O_ij(t) = sum_y eta_i^* gamma5 X_j, all t, N_r = %d (paper eq. 7.6)" % n_rhs, "ms": tc * 1e3,
                       "gbs": cbytes / tc / 1e9, "frac_hbm": cbytes / tc / 1e9 / peaks["hbm_gbs"], "tflops_fp64": cflop / tc / 1e12,
                       "frac_fp64_alu": cflop / tc / fp64_peak, "bound": "alu (fp64 FMA) ~ hbm", "dtype": "f64"}
        del o

    # ---- NEXT row (S 8(f) rank 2): outer-product fill S and S^dagger at the paper's Table II size (L = 8: 8^3x16) ----
    fill_res = None
    if rank == 0 and args.config == 3:
        fd = (8, 8, 8, 16)
        fe = B.noise_fill(fd, 2001, n_rhs, scale=wl.INV_SQRT2)
        fx = B.noise_fill(fd, 977, n_rhs, scale=1.0)
        fs = torch.empty((16, 512, 12, 512, 12), dtype=torch.complex128, device="cuda")
        times = {}
        for dag in (0, 1):
            B.stochastic_fill(fx, fe, t0=0, scale=wl.INV_SQRT2, dagger=bool(dag), out=fs.view((512, 12, 16, 512, 12)) if dag else fs)
            torch.cuda.synchronize()
            c0, c1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            c0.record()
            for _ in range(3):
                B.stochastic_fill(fx, fe, t0=0, scale=wl.INV_SQRT2, dagger=bool(dag), out=fs.view((512, 12, 16, 512, 12)) if dag else fs)
            c1.record()
            torch.cuda.synchronize()
            times[dag] = c0.elapsed_time(c1) / 3 * 1e-3
        B.timeslice_norm2(fs, 1, 16)
        torch.cuda.synchronize()
        c0.record()
        for _ in range(3):
            B.timeslice_norm2(fs, 1, 16)
        c1.record()
        torch.cuda.synchronize()
        t_trace = c0.elapsed_time(c1) / 3 * 1e-3
        # the two-source-set trace: a second fill from an independent noise set, then sum Tr[S1 S2^+] per timeslice
        fs2 = torch.empty_like(fs)
        B.stochastic_fill(B.noise_fill(fd, 978, n_rhs, scale=1.0), B.noise_fill(fd, 2002, n_rhs, scale=wl.INV_SQRT2), t0=0, scale=wl.INV_SQRT2, out=fs2)
        B.timeslice_inner(fs, fs2, 1, 16)
        torch.cuda.synchronize()
        c0.record()
        for _ in range(3):
            B.timeslice_inner(fs, fs2, 1, 16)
        c1.record()
        torch.cuda.synchronize()
        t_inner = c0.elapsed_time(c1) / 3 * 1e-3
        del fs2
        fbytes = fs.numel() * 16
        fflop = 8.0 * fs.numel() * n_rhs
        fp64_peak = 148 * 64 * 2 * 1.965e9
        fill_res = {"what": "S and S^dagger fill (paper eq. 7.3), 8^3x16, N_r = %d in one pass, 9.66 GB each" % n_rhs,
                    "ms_fill": times[0] * 1e3, "ms_fill_dagger": times[1] * 1e3, "write_gbs": fbytes / times[0] / 1e9,
                    "tflops_fp64": fflop / times[0] / 1e12, "frac_fp64_alu": fflop / times[0] / fp64_peak,
                    "frac_hbm_write": fbytes / times[0] / 1e9 / peaks["hbm_gbs"], "ms_per_source_both": (times[0] + times[1]) * 1e3 / n_rhs,
                    "trace": {"what": "sum_x sum_z Tr S_s S_s^+ for all 16 timeslices (Table I last row)", "ms": t_trace * 1e3,
                              "read_gbs": fbytes / t_trace / 1e9, "frac_hbm": fbytes / t_trace / 1e9 / peaks["hbm_gbs"],
                              "paper_table1_s_per_timeslice": 43.3},
                    "trace_two_sets": {"what": "sum_x sum_z Tr S_s1 S_s2^+ for all 16 timeslices, fills from two independent source sets (P:L303)",
                                       "ms": t_inner * 1e3, "read_gbs": 2 * fbytes / t_inner / 1e9, "frac_hbm": 2 * fbytes / t_inner / 1e9 / peaks["hbm_gbs"]},
                    "paper_table2_s_per_source": {"cpu": 100.8, "gpu": 8.8, "hardware": "unnamed", "cite": "PAPER.md L340-344"}}
        del fs, fe, fx

    if rank != 0:
        return
    out = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
           "ms_per_step": ms / args.steps, "higher_is_better": False, "scaling": "weak", "vs_baseline": None,
           "dtype": "f32" if cfg["mixed"] else "f64", "data": "synthetic",
           "config": {"workload": cfg["name"], "n_rhs_per_gpu": n_rhs, "batch": batch, "tol": wl.TOL, "kappa": cfg["kappa"], "c_sw": cfg["csw"],
                      "eps": cfg["eps"], "recon": cfg["recon"], "time_dilution": cfg["dilution"],
                      "solver": "even-odd BiCGStab, fp32 iteration + fp64 reliable updates" if cfg["mixed"] else "even-odd BiCGStab fp64",
                      "l2": ("one fp32 field of the batch is %.0f MB; " % (Vh * batch * 96 / 1e6)) +
                            ("fields per sweep exceed the 126 MB L2; " if Vh * batch * 96 * 3 > 126e6 else "the sweeps FIT the 126 MB L2 (parity-size lattice: HBM fractions are not meaningful here); ") +
                            "the stand-alone hop timing flushes L2 between launches"},
           "clocks": sampler.summary(), "gpu_launches": launches, "roofline": roofline, "dslash": dslash, "e2e": e2e, "noise_fill": noise, "next_contraction": contraction, "next_fill": fill_res,
           "solve": {"iters": [i["iters"] for i in last["infos"]][::batch], "reliable_updates": [i["reliable_updates"] for i in last["infos"]][::batch],
                     "max_true_resid": max(i["true_resid"] for i in last["infos"]),
                     "phase_ms_per_step": {k: v / args.steps for k, v in phases.items()}}}
    if not args.no_cpu_baseline and world == 1:
        run, n_it, cores = oracle_sample(cfg, 2, U)
        v = run()
        out["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle",
                               "sample": f"2 oracle BiCGStab iterations of 1 source on {cfg['name']} (unpreconditioned fp64, OpenMP over sites), "
                                         f"scaled to the {n_it} iterations the oracle needs for 1e-10 at these parameters on 8^3x16"}
    print(json.dumps(out))
    ctx.close()


if __name__ == "__main__":
    main()
