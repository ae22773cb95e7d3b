#!/usr/bin/env python
"""bench.py -- one JSON line for the hot path of arXiv:1405.4524 on B200 (contract: task prompt).

A step = one pass of the whole hot path over one batch of synthetic input at BASELINE.json configs[3]
(24^3x48, kappa 0.118, c_sw 1.5, links exp(i 0.4 H)): noise_fill of N_r = 32 Z4 sources, then clover_solve of all of
them in batches of 8 (fp32 BiCGStab with fp64 reliable updates, tol 1e-10), source prep, odd-site reconstruction,
fp64 full-lattice verification and layout reorders included.  metric = BiCGStab seconds/source; the Dslash GB/s half
of BASELINE.json's metric is the `roofline` object (the kernel of the iteration with the largest summed device time, every
launch timed with CUDA events inside the timed steps; the other kernels under `other_kernels`) plus `dslash` (the plain hop
kernel timed alone).

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


def oracle_setup(cfg, U=None):
    import oracle
    from paper_1405_4524_b200 import workloads as wl
    if U is None:
        U = wl.gauge_links(cfg["dims"], cfg["eps"], cfg["gauge_seed"])
    A = oracle.clover_matrix(U, cfg["kappa"], cfg["csw"])
    eta = oracle.noise_fill(cfg["dims"], cfg["noise_seed"], 1, time_dilution=cfg["dilution"], scale=wl.INV_SQRT2)[0]
    return oracle, wl, U, A, eta


def oracle_full_solve(cfg, U=None):
    """cpu_baseline: ONE full solve of one source of the workload by the oracle as it stands (unpreconditioned fp64 BiCGStab to
    the workload's tolerance, all host cores), measured, plus the oracle's D-apply rate on all cores and on one thread."""
    oracle, wl, U, A, eta = oracle_setup(cfg, U)
    cores = oracle.threads()
    t0 = time.perf_counter()
    _, info = oracle.bicgstab(U, A, wl.BC, cfg["kappa"], eta, tol=wl.TOL)
    t_solve = time.perf_counter() - t0
    sites = eta.size // 12

    def d_rate(threads, reps):
        oracle.set_threads(threads)
        oracle.apply_D(U, A, wl.BC, cfg["kappa"], eta)
        t = time.perf_counter()
        for _ in range(reps):
            oracle.apply_D(U, A, wl.BC, cfg["kappa"], eta)
        dt = (time.perf_counter() - t) / reps
        oracle.set_threads(cores)
        return {"threads": threads, "s_per_apply": dt, "sites_per_s": sites / dt, "gflops": 1872.0 * sites / dt / 1e9}
    return {"value": t_solve, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"full solve of 1 source of {cfg['name']} to {wl.TOL:g}: {info['iters']} iterations of the oracle's unpreconditioned fp64 BiCGStab "
                      f"(2 D applies each), true residual {info['true_resid']:.2e}, measured not projected",
            "iters": info["iters"], "true_resid": info["true_resid"], "extrapolated": False,
            "d_apply": {"flop_per_site": 1872, "all_cores": d_rate(cores, 3), "one_thread": d_rate(1, 1)}}


def run_reference(args, cfg):
    """--impl reference: the oracle on the host cores (rank 0 only).  One full solve first (its iteration count N and measured
    time are reported in cpu_baseline); every timed step then measures the oracle's cost per BiCGStab iteration on the same
    source as the difference between a 10-iteration and a 2-iteration call (so the set-up and the trailing true-residual apply
    of a call cancel) and reports N x that: a bounded sample of the same work, kept in line with the full solve."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    base = oracle_full_solve(cfg)
    oracle, wl, U, A, eta = oracle_setup(cfg)
    n_it, lo, hi = base["iters"], 2, 10

    def call(n):
        t0 = time.perf_counter()
        oracle.bicgstab(U, A, wl.BC, cfg["kappa"], eta, tol=1e-30, max_iter=n)
        return time.perf_counter() - t0

    def run():
        return (call(hi) - call(lo)) / (hi - lo) * n_it   # seconds per source
    for _ in range(args.warmup):
        run()
    vals = [run() for _ in range(args.steps)]
    v = sum(vals) / len(vals)
    base["per_iteration_s_full_solve"] = base["value"] / n_it
    base["per_iteration_s_sampled"] = v / n_it
    base["sample"] += (f"; each timed step of this arm = ({hi}-iteration call - {lo}-iteration call) / {hi - lo} x {n_it} iterations on the same source")
    base["value"] = v
    print(json.dumps({"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
                      "warmup": args.warmup, "ms_per_step": v * 1e3, "higher_is_better": False, "scaling": "weak", "vs_baseline": None,
                      "dtype": "f64", "data": "synthetic", "config": {"workload": cfg["name"], "n_rhs": 1, "solver": "oracle BiCGStab, unpreconditioned"},
                      "cpu_baseline": base,
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
    kstats = {"n_ainv_hop": 0, "n_a_minus_hop": 0, "ms_ainv_hop": 0.0, "ms_a_minus_hop": 0.0, "n_a_minus_hop_s": 0, "ms_a_minus_hop_s": 0.0,
              "n_xrp_update": 0, "ms_xrp_update": 0.0}
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

    # ---- roofline of the DOMINANT kernel: the kernel of the solve with the largest summed device time inside the timed steps
    # (clover_get_stats: CUDA events around every launch on the solve's stream); the others are listed under other_kernels ----
    peaks, peak_kind = measured_peaks()
    b = 4 if cfg["mixed"] else 8
    g = cfg["recon"] if cfg["mixed"] else 18
    merged = kstats["n_a_minus_hop_s"] > 0   # merged iteration (solver.cu): both fused Dslash variants also read w (r or r0) at the own site
    bytes_a_minus = (8 * g * b + 72 * b) / batch + 24 * b * (4 if merged else 3)   # links + clover shared by the batch; in, x, (w,) out per rhs
    bytes_ainv = (8 * g * b + 72 * b) / batch + 24 * b * 2
    bytes_xrp = 24 * b * 9      # one sweep: reads x, p, s, t, r, q0, writes x, r, p
    prec = 32 if cfg["mixed"] else 64
    rt, pair = ("float" if cfg["mixed"] else "double"), (cfg["mixed"] and batch >= 2)
    if cfg["mixed"] and batch == 8:
        kname = lambda what: f"dslash3_kernel<B=8,recon={g},{what}> (fp32, persistent one-warp CTAs, one thread per site and rhs pair, operator records by cp.async.bulk)"
    elif pair:
        kname = lambda what: f"dslash2_kernel<B={batch},recon={g},{what}> (fp32, one thread per site and rhs pair)"
    else:
        kname = lambda what: f"dslash_kernel<{rt},B={batch},recon={g},{what}>"
    timed = "CUDA events around every launch inside the timed steps"
    table = {}   # name -> (kernel, launches, summed ms, algorithmic bytes / site / rhs, flop / site / rhs, traffic key)
    if kstats["n_a_minus_hop"]:
        table["ainv_hop"] = (kname("tmp = A^-1 H x"), kstats["n_ainv_hop"], kstats["ms_ainv_hop"], bytes_ainv, 1824.0, "ainv_hop")
        table["a_minus_hop"] = (kname("t = A s - k^2 H tmp, +<t,s>,<t,t>,<r0,t>,<r0,s>" if merged else "A x - k^2 H t,+dots"), kstats["n_a_minus_hop"],
                                kstats["ms_a_minus_hop"], bytes_a_minus, 1872.0, "a_minus_hop_xw" if merged else "a_minus_hop")
        if merged:
            table["a_minus_hop_s"] = (kname("s = r - alpha (A p - k^2 H tmp)"), kstats["n_a_minus_hop_s"], kstats["ms_a_minus_hop_s"], bytes_a_minus, 1872.0,
                                      "a_minus_hop_s")
            if kstats["n_xrp_update"]:
                table["xrp_update"] = (f"xrp_update_kernel<{rt}> (x, r, p updates + <q0,p>, ||r||^2: 9 vector passes)", kstats["n_xrp_update"],
                                       kstats["ms_xrp_update"], bytes_xrp, 0.0, "xrp_update")
    else:   # launch-bound lattice: the iteration ran as a CUDA graph, without per-launch events; time the kernels alone
        timed = "kernel timed alone (the solve replays its iteration as a CUDA graph on this lattice; fields fit L2)"
        table["ainv_hop"] = (kname("tmp = A^-1 H x"), 20, ctx.bench_kernel(B.KERNEL_AINV_HOP, prec, batch, reps=20) * 20, bytes_ainv, 1824.0, "ainv_hop")
        table["a_minus_hop"] = (kname("A x - k^2 H t,+dots"), 20, ctx.bench_kernel(B.KERNEL_A_MINUS_HOP, prec, batch, reps=20) * 20, bytes_a_minus, 1872.0, "a_minus_hop")
    traffic_db, tp = {}, os.path.join(ROOT, "profiles", "traffic.json")   # DRAM bytes per launch from the committed ncu --set full capture
    if os.path.exists(tp):
        traffic_db = json.load(open(tp))

    def entry(name):
        kernel, n, ms_sum, bts, fl, tkey = table[name]
        t = ms_sum / n * 1e-3
        ach = bts * Vh * batch / t / 1e9
        e = {"kernel": kernel, "achieved": ach, "frac": ach / peaks["hbm_gbs"], "us_per_launch": t * 1e6, "launches": n,
             "algorithmic_bytes_per_site_rhs": bts, "algorithmic_bytes_per_launch": bts * Vh * batch,
             "share_of_step": ms_sum / phases["ms_total"] if phases["ms_total"] else None,
             "traffic": traffic_db.get(f"{tkey}_{cfg['name']}_b{batch}")}
        if fl:
            e["gflops"] = fl * Vh * batch / t / 1e9
        return e
    dominant = max(table, key=lambda k: table[k][2])
    roofline = {"bound": "hbm", "name": dominant, "unit": "GB/s", "peak": peaks["hbm_gbs"], "peak_kind": peak_kind, "timed": timed,
                "dominance": "largest summed device time of one kernel inside the timed steps (share_of_step = its launches' time / solve time)",
                "traffic_source": traffic_db.get("source", "none: no ncu capture committed for this configuration")}
    roofline.update(entry(dominant))
    roofline["other_kernels"] = {k: entry(k) for k in table if k != dominant}

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

    def loop_seconds(fn, reps):
        """Device time per call of fn(): one warm-up call, then `reps` calls back to back between two CUDA events, done twice; the faster
        of the two loops (one stalled loop -- e.g. behind the release of the e2e leg's pinned buffers -- must not skew a 2 ms kernel)."""
        fn()
        torch.cuda.synchronize()
        best = None
        for _ in range(2):
            a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a0.record()
            for _ in range(reps):
                fn()
            a1.record()
            a1.synchronize()
            t = a0.elapsed_time(a1) / reps
            best = t if best is None else min(best, t)
        return best * 1e-3

    # ---- H1 noise fill alone (a pure write stream: 192 B per site and source in fp64) ----
    noise = None
    if rank == 0:
        tn = loop_seconds(lambda: B.noise_fill(dims, cfg["noise_seed"], n_rhs, rhs_offset=offset, time_dilution=cfg["dilution"], scale=wl.INV_SQRT2, out=eta), 5)
        noise = {"ms": tn * 1e3, "write_gbs": n_rhs * V * 192 / tn / 1e9, "frac_hbm": n_rhs * V * 192 / tn / 1e9 / peaks["hbm_gbs"]}

    # ---- NEXT row (S 8(f) rank 1): stochastic-operator contraction O_ij(t) of the step's sources and solutions ----
    contraction = None
    if rank == 0:
        tc = loop_seconds(lambda: B.stochastic_operators(eta, psi), 5)
        cbytes = 2 * n_rhs * V * 24 * 8
        cflop = 8.0 * n_rhs * n_rhs * 12 * V
        fp64_peak = 148 * 64 * 2 * 1.965e9     # fp64 FMA lanes per SM x SMs x 2 flop x max clock
        contraction = {"what": "O_ij(t) = sum_y eta_i^* gamma5 X_j, all t, N_r = %d (paper eq. 7.6)" % n_rhs, "ms": tc * 1e3,
                       "gbs": cbytes / tc / 1e9, "frac_hbm": cbytes / tc / 1e9 / peaks["hbm_gbs"], "tflops_fp64": cflop / tc / 1e12,
                       "flop_counting": "tflops_fp64 counts 8 flop per complex multiply-add (the textbook count); the kernel executes 6 (three real products, Gauss' form): frac_fp64_alu is of the EXECUTED rate",
                       "executed_tflops_fp64": 0.75 * cflop / tc / 1e12, "frac_fp64_alu": 0.75 * cflop / tc / fp64_peak, "bound": "alu (fp64 tensor pipe, DMMA) ~ hbm", "dtype": "f64"}

    # ---- NEXT row (S 8(f) rank 2): outer-product fill S and S^dagger at the paper's Table II size (L = 8: 8^3x16) ----
    fill_res = None
    if rank == 0 and args.config == 3:
        fd = (8, 8, 8, 16)
        fe = B.noise_fill(fd, 2001, n_rhs, scale=wl.INV_SQRT2)
        fx = B.noise_fill(fd, 977, n_rhs, scale=1.0)
        fs = torch.empty((16, 512, 12, 512, 12), dtype=torch.complex128, device="cuda")
        times = {}
        for dag in (0, 1):
            times[dag] = loop_seconds(lambda: B.stochastic_fill(fx, fe, t0=0, scale=wl.INV_SQRT2, dagger=bool(dag), out=fs.view((512, 12, 16, 512, 12)) if dag else fs), 3)
        t_trace = loop_seconds(lambda: B.timeslice_norm2(fs, 1, 16), 3)
        # the two-source-set trace: a second fill from an independent noise set, then sum Tr[S1 S2^+] per timeslice
        fs2 = torch.empty_like(fs)
        B.stochastic_fill(B.noise_fill(fd, 978, n_rhs, scale=1.0), B.noise_fill(fd, 2002, n_rhs, scale=wl.INV_SQRT2), t0=0, scale=wl.INV_SQRT2, out=fs2)
        t_inner = loop_seconds(lambda: B.timeslice_inner(fs, fs2, 1, 16), 3)
        del fs2
        fbytes = fs.numel() * 16
        fflop = 8.0 * fs.numel() * n_rhs
        fp64_peak = 148 * 64 * 2 * 1.965e9
        fill_res = {"what": "S and S^dagger fill (paper eq. 7.3), 8^3x16, N_r = %d in one pass, 9.66 GB each" % n_rhs,
                    "ms_fill": times[0] * 1e3, "ms_fill_dagger": times[1] * 1e3, "write_gbs": fbytes / times[0] / 1e9,
                    "tflops_fp64": fflop / times[0] / 1e12, "executed_tflops_fp64": 0.75 * fflop / times[0] / 1e12, "frac_fp64_alu": 0.75 * fflop / times[0] / fp64_peak,
                    "flop_counting": "tflops_fp64 counts 8 flop per complex multiply-add; the kernel executes 6 (Gauss' three-multiplication form): frac_fp64_alu is of the EXECUTED rate",
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
        out["cpu_baseline"] = oracle_full_solve(cfg, U)
    print(json.dumps(out))
    ctx.close()


if __name__ == "__main__":
    main()
