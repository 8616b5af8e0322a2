#!/usr/bin/env python
"""bench.py -- throughput of the HQMC pseudofermion hot path on B200.

A STEP is one pass of the whole hot path on one lattice:
    phi = M^+(theta) eta                         (S8, pseudofermion refresh)
    one leapfrog step of the MD trajectory       (S13): 2 fixed-count PCG solves of M^+M x = phi
        (S5-S7: fused M^+M, preconditioner, fused axpy/dot), force + boson force + momentum kicks
        (S9, S10), drift + phase table (S11, S1), energies H0, H1 (S12)
with the paper's fixed-iteration CG protocol: --cg-iters iterations per solve.
`value` = M^+M applications x sites / time, in Gsite/s (BASELINE.json's metric), for the WHOLE step,
i.e. it charges the preconditioner, the vector updates, the force and the energies to the M^+M count.
The other BASELINE quantities ride along in the same JSON line: CG-solve ms (`cg_ms_per_solve`,
`cg_us_per_iter`), achieved HBM GB/s against the measured peak (`roofline`), ms per trajectory step.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--cg-iters I] [--config 4]
    python -m torch.distributed.run --nproc-per-node N ... bench.py --gpus N ...   (replicas, weak scaling)
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "MdagM_Gsite_per_s"
UNIT = "Gsite/s"
# algorithmic bytes per site (complex128): read v (16) + 2 link phases as theta (16) + write (16)
BYTES_PER_SITE = {"mdagm": 48.0, "cg_axpy": 96.0, "precond": 32.0, "cg_dupdate": 48.0}
# dram__bytes_read.sum + dram__bytes_write.sum per launch from the committed `ncu --set full` captures (profiles/), L=48, c128
TRAFFIC_NCU = {"mdagm": 35.5e6}


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
            except Exception:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def dist_env():
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    return rank, world, local


# --------------------------------------------------------------------------------------------------
# reference arm / cpu_baseline: the oracle as it stands, on the host cores, on a bounded sample
# --------------------------------------------------------------------------------------------------
def oracle_step_sample(L, Ntau, seed, cg_iters, nsteps_md=1, threads=None):
    """One hot-path step with the CPU oracle (same structure as the GPU step, cg_iters per solve).
    -> (seconds, MdagM applications, threads used)."""
    from oracle import oracle as orc
    from paper_2508_16298_b200 import inputs
    orc.build()
    # torchrun exports OMP_NUM_THREADS=1 for its ranks; only one rank ever runs the oracle, so it takes the cores it may use
    threads = threads or max(orc.max_threads(), len(os.sched_getaffinity(0)))
    orc.set_threads(threads)
    theta = inputs.theta_uniform(L, Ntau, seed)
    eta = inputs.complex_gaussian((Ntau, L, L), seed)
    p = inputs.momenta(L, Ntau, seed)
    o = orc.Oracle(L, Ntau)
    t0 = time.perf_counter()
    phi = o.apply_Mdag(theta, eta)
    r = o.trajectory(theta, p, phi, nsteps_md, 0.05, cg_tol=0.0, cg_max_iter=cg_iters)
    dt = time.perf_counter() - t0
    return dt, r["cg_iters"], orc.get_threads()


def run_reference(args):
    rank, world, _ = dist_env()
    if rank != 0:
        return 0
    from paper_2508_16298_b200 import inputs
    c = inputs.CONFIGS[args.config]
    L, Ntau, N = c["L"], c["Ntau"], c["L"] * c["L"] * c["Ntau"]
    iters = args.ref_cg_iters
    times, apps, threads = [], 0, 1
    for i in range(args.warmup + args.steps):
        dt, a, threads = oracle_step_sample(L, Ntau, c["seed"], iters)
        if i >= args.warmup:
            times.append(dt); apps += a
    total = sum(times)
    value = apps * N / total / 1e9
    sample = (f"bounded sample of the workload: same lattice (L={L}, Ntau={Ntau}), same step structure, each fixed-count solve cut to "
              f"{iters} of its {args.cg_iters} PCG iterations ({2 * iters} M^+M per step); the metric is per M^+M application")
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * total / max(1, len(times)), "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": workload_config(args, L, Ntau, args.cg_iters),     # the workload; `sample` says what was run of it
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))
    return 0


def workload_config(args, L, Ntau, cg_iters):
    return {"workload": f"BASELINE config {args.config}: L={L}, Ntau={Ntau}, theta uniform[-pi,pi) (seeded), complex128; "
                        f"step = M^+ refresh + 1 leapfrog step (2 fixed-count PCG solves, W=6 preconditioner, force, kicks, "
                        f"drift, energies)",
            "L": L, "Ntau": Ntau, "sites": L * L * Ntau, "cg_iters_per_solve": cg_iters, "precond_W": 6,
            "l2": "no flush inside a step: a step is 2 x cg_iters_per_solve PCG iterations over the same vectors, and the solver "
                  "keeps that loop's live set (r, d, Od|z, packed phases = 71 MB at L=48, x streamed evict-first) L2-resident "
                  "on purpose -- the reuse is the algorithm's own, not a benchmark artefact; the whole step (7 fermion vectors "
                  "+ phases + theta, p, force) exceeds the 126 MB L2, and the separate M^+M kernel sweep rotates 8 input/output "
                  "buffer pairs (cold) next to the same-buffer (warm) figure"}


# --------------------------------------------------------------------------------------------------
# GPU arm
# --------------------------------------------------------------------------------------------------
def run_gpu(args):
    import torch
    import torch.distributed as dist
    from paper_2508_16298_b200 import hqmc, inputs, replicas

    rank, world, local = dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    c = inputs.CONFIGS[args.config]
    L, Ntau = c["L"], c["Ntau"]
    N = L * L * Ntau
    seed = replicas.replica_seed(c["seed"], rank)          # one independent lattice (Markov chain) per rank
    prec = args.prec
    cdt = np.complex128 if prec == "c128" else np.complex64
    theta0 = inputs.theta_uniform(L, Ntau, seed)
    eta = inputs.complex_gaussian((Ntau, L, L), seed).astype(cdt)
    p0 = inputs.momenta(L, Ntau, seed)

    g = hqmc.HQMC(L, Ntau, prec=prec, device=str(dev))
    to_dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)
    d_theta0, d_p0, d_eta = to_dev(theta0), to_dev(p0), to_dev(eta)
    d_theta, d_p, d_phi = torch.empty_like(d_theta0), torch.empty_like(d_p0), g.new_vec()
    I = args.cg_iters

    def step_device():
        d_theta.copy_(d_theta0); d_p.copy_(d_p0)
        g.set_theta(d_theta)
        g.apply_Mdag(d_eta, d_phi)
        return g.trajectory(d_theta, d_p, d_phi, 1, 0.05, cg_tol=0.0, cg_max_iter=I)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        r = step_device()
    g.reset_stats()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    apps = 0
    e0.record()
    for _ in range(args.steps):
        r = step_device()
        apps += r["cg_iters"]
    e1.record()
    barrier()
    ms_local = e0.elapsed_time(e1)
    stats = g.kernel_stats()
    launches = sum(v[0] for v in stats.values())

    # ---- end to end through the host-buffer entry points (pinned host memory, copies inside the timed region)
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    h_theta0, h_p0, h_eta = pin(theta0), pin(p0), pin(eta)
    h_theta, h_p, h_phi = torch.empty_like(h_theta0).pin_memory(), torch.empty_like(h_p0).pin_memory(), torch.empty_like(h_eta).pin_memory()
    n_theta, n_p, n_phi, n_eta = h_theta.numpy(), h_p.numpy(), h_phi.numpy(), h_eta.numpy()

    def step_host():
        h_theta.copy_(h_theta0); h_p.copy_(h_p0)
        g.refresh_host(n_theta, n_eta, n_phi)                       # H2D theta, eta; phi = M^+ eta; D2H phi
        return g.trajectory_host(n_theta, n_p, n_phi, 1, 0.05, cg_tol=0.0, cg_max_iter=I)   # H2D theta, p, phi; D2H theta, p

    e2e_steps = max(1, min(args.steps, args.e2e_steps))
    step_host()
    barrier()
    t0 = time.perf_counter()
    e2e_apps = 0
    for _ in range(e2e_steps):
        e2e_apps += step_host()["cg_iters"]
    torch.cuda.synchronize()
    e2e_s_local = time.perf_counter() - t0
    barrier()
    vb, tb = N * (16 if prec == "c128" else 8), 2 * N * 8
    h2d, d2h = (tb + vb) + (2 * tb + vb), vb + 2 * tb

    # ---- per-kernel cost INSIDE the graph-replayed PCG iteration, by leave-one-out: the same fixed-count solve is timed
    # (CUDA events on the library's stream) with all kernels and with one kernel class not launched; the difference is
    # that kernel's cost in the launch configuration the step uses.  The class that carries the iteration bookkeeping
    # cannot be left out: it gets the remainder.  (Per-launch events would add the launch gaps of a non-replayed run.)
    kern = None
    if rank == 0:
        kern = pcg_kernel_costs(g, torch, d_phi, I)

    # ---- M^+M kernel alone, cold (rotating 8 buffer pairs > L2) and warm (same buffers)
    sweep = None
    if rank == 0 and not args.no_sweep:
        sweep = mdagm_sweep(g, torch, dev, L, Ntau, prec)

    clocks = sampler.stop() if rank == 0 else None

    # ---- aggregate over ranks: max time, summed work
    ms, total_apps = replicas.aggregate(ms_local, apps, world)
    e2e_s, total_e2e_apps = replicas.aggregate(e2e_s_local, e2e_apps, world)
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0

    value = total_apps * N / (ms * 1e-3) / 1e9
    e2e_value = total_e2e_apps * N / e2e_s / 1e9
    peak, peak_src = measured_peaks()
    bps = dict(BYTES_PER_SITE)
    if prec != "c128":
        bps = {k: v / 2 for k, v in bps.items()}
    per_kernel = {}
    for name, us in kern["us"].items():
        per_kernel[name] = {"us_in_graph": us, "share_of_iteration": us / kern["iter_us"],
                            "alg_bytes_per_site": bps[name], "alg_GBps": bps[name] * N / us / 1e3}
    dom = max(per_kernel, key=lambda k: per_kernel[k]["us_in_graph"])
    achieved = per_kernel[dom]["alg_GBps"]
    roofline = {"bound": "hbm", "kernel": dom, "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                "traffic": TRAFFIC_NCU.get(dom), "traffic_source": "dram__bytes_read.sum + dram__bytes_write.sum of the committed ncu --set full capture (profiles/r02_summary.md); not measured by this run",
                "peak_source": peak_src, "alg_bytes_per_site": bps[dom],
                "how": "leave-one-out CUDA-event timing of the graph-replayed fixed-count PCG solve (bench.py pcg_kernel_costs)"}
    # the whole PCG iteration against the same peak: algorithmic bytes of all its kernels / the iteration time.  The vector
    # kernels are served largely from L2 (their alg_GBps can exceed the HBM peak), so this is a figure of merit against the
    # HBM-streaming model of the iteration, not a DRAM-traffic claim (in-situ DRAM bytes: profiles/).
    it_bytes = sum(bps.values()) * N
    roofline["iteration"] = {"alg_bytes_per_site": sum(bps.values()), "achieved": it_bytes / kern["iter_us"] / 1e3, "unit": "GB/s",
                             "frac": it_bytes / kern["iter_us"] / 1e3 / peak}
    # the same kernel against the fp64 issue rate, the roof it actually sits under (DRAM 16 % busy): ~150
    # flop per site and M^+M (two B products of 28 FMA per site, the link decode, the two axpys, the dot), peak = SMs x 64
    # fp64 lanes x 2 flop x the SM clock sampled during the run
    if dom == "mdagm" and prec == "c128":
        sm_mhz = (clocks or {}).get("sm_mhz") or 1965.0
        alu_peak = torch.cuda.get_device_properties(0).multi_processor_count * 64 * 2 * sm_mhz * 1e6 / 1e12
        alu_ach = 150.0 * N / (per_kernel[dom]["us_in_graph"] * 1e-6) / 1e12
        roofline["alu"] = {"bound": "alu", "flops_per_site": 150, "achieved": alu_ach, "peak": alu_peak, "unit": "TFLOP/s",
                           "frac": alu_ach / alu_peak, "peak_source": "SMs x 64 fp64 lanes x 2 x sampled SM clock (guide: unit counts)"}
    ms_per_step = ms / args.steps
    us_per_iter = kern["iter_us"]
    cb_dt, cb_apps, cb_threads = oracle_step_sample(L, Ntau, c["seed"], args.ref_cg_iters)
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64" if prec == "c128" else "f32", "data": "synthetic", "config": workload_config(args, L, Ntau, I),
            "clocks": clocks,
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h, "steps": e2e_steps},
            "gpu_launches": launches, "roofline": roofline,
            "cpu_baseline": {"value": cb_apps * N / cb_dt / 1e9, "unit": UNIT, "cores": cb_threads, "kind": "oracle",
                             "sample": f"one step on the same lattice with fixed-count CG cut to {args.ref_cg_iters} iterations per solve "
                                       f"({cb_apps} M^+M), {cb_dt:.1f} s"},
            "cg_us_per_iter": us_per_iter, "cg_iters_per_s": 1e6 / us_per_iter, "cg_ms_per_solve_fixed": us_per_iter * I * 1e-3,
            "ms_per_trajectory_step": ms_per_step, "kernels": per_kernel, "mdagm_sweep": sweep,
            # BASELINE's first figure, for the M^+M kernel itself (`value` charges the whole step to the M^+M count)
            "mdagm_kernel": {"us_in_graph": per_kernel["mdagm"]["us_in_graph"], "Gsite_per_s": N / per_kernel["mdagm"]["us_in_graph"] / 1e3,
                             "alg_GBps": per_kernel["mdagm"]["alg_GBps"], "frac_of_peak": per_kernel["mdagm"]["alg_GBps"] / peak},
            "dH_fixed_count_unconverged": r["H1"] - r["H0"]}
    if world == 1 and not args.no_extras:
        try:
            line.update(contract_numbers(args, torch, hqmc, inputs, theta0, inputs.complex_gaussian((Ntau, L, L), seed)))
        except Exception as e:                                           # never lose the metric line over the extra keys
            line["contract_numbers_error"] = repr(e)[:300]
    if world == 1 and not args.no_small:
        line["batched_chains"] = small_lattice_chains(torch, hqmc, inputs, args.cg_iters)
    print(json.dumps(line))
    g.close()
    if world > 1:
        dist.destroy_process_group()
    return 0


def contract_numbers(args, torch, hqmc, inputs, theta_cfg, eta_cfg):
    """The figures BASELINE.json's metric and configs name beyond the timed step, measured in the same run (rank 0, N = 1):
    `cg_solve`  -- config 4's "preconditioned CG to 1e-10, with iteration count and ms per solve": on BASELINE's uniform field
                   and on a paper-regime field (c_tau = 80, K = 1), with the recurrence residual and the residual of the
                   GPU solution under the ORACLE's operator (one CPU M^+M after the timed region; reading C16 i);
    `c64`       -- the complex64 variant "timed separately": M^+M and PCG iteration in the replayed graph;
    `config5`   -- L=64, Ntau=640 on its seeded heat-bath field: ms per 20-step trajectory (fixed-count protocol), M^+M us;
    `md_graph`  -- leapfrog step replayed as one CUDA graph against plain launches (the paper reports
                   2-5 x from CUDA graphs for L < 30 and 1-2 x above, on its GPU, for whole sweeps) at L = 12, 24, 48."""
    from oracle import oracle as orc
    out = {}
    c = inputs.CONFIGS[args.config]
    L, Ntau, N = c["L"], c["Ntau"], c["L"] * c["L"] * c["Ntau"]
    orc.build(); orc.set_threads(max(orc.max_threads(), len(os.sched_getaffinity(0))))
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()

    def solve_on(theta, label, **kw):
        g = hqmc.HQMC(L, Ntau, **kw)
        g.set_theta(dev(theta))
        phi = g.apply_Mdag(dev(eta_cfg))
        x = g.new_vec()
        g.cg_solve(phi, 0.0, 64, x=x)                               # graph capture outside the timed solve
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(); x, it, rel, ok = g.cg_solve(phi, args.tol, args.max_iter, x=x); e1.record(); torch.cuda.synchronize()
        ms = e0.elapsed_time(e1)
        phi_h, x_h = phi.cpu().numpy(), x.cpu().numpy()
        o = orc.Oracle(L, Ntau, **kw)
        res_orc = float(np.linalg.norm((phi_h - o.apply_MdagM(theta, x_h)).ravel()) / np.linalg.norm(phi_h.ravel()))
        g.close()
        return {"field": label, "tol": args.tol, "iterations": it, "converged": bool(ok), "ms_per_solve": ms, "us_per_iter": 1e3 * ms / max(1, it),
                "recurrence_relres": rel, "oracle_operator_relres": res_orc}

    if not args.no_solve:
        out["cg_solve"] = {
            "baseline_field": solve_on(theta_cfg, "BASELINE config 4: theta uniform[-pi,pi)"),
            "paper_regime_field": solve_on(inputs.theta_paper_regime(L, Ntau, c["seed"], sweeps=20),
                                           "paper regime: heat bath at c_tau = 1/(J dtau^2) = 80, K = 1 (PAPER.md:107), cold start, 20 sweeps",
                                           c_tau=80.0, K=1.0)}
        # the sampler in the regime the paper runs it: whole trajectories on the paper-regime field at config
        # 4's size, 3 leapfrog steps (eps = 0.02), every solve converged to --tol; ms per trajectory, best of 3
        th_pr = inputs.theta_paper_regime(L, Ntau, c["seed"], sweeps=20)
        g = hqmc.HQMC(L, Ntau, c_tau=80.0, K=1.0)
        g.set_theta(dev(th_pr))
        phi = g.apply_Mdag(dev(eta_cfg))
        p_pr = inputs.momenta(L, Ntau, c["seed"])
        best, rr = 1e30, None
        for k in range(4):
            d_th, d_p = dev(th_pr), dev(p_pr)
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(); rr = g.trajectory(d_th, d_p, phi, 3, 0.02, cg_tol=args.tol, cg_max_iter=args.max_iter); e1.record(); torch.cuda.synchronize()
            if k:
                best = min(best, e0.elapsed_time(e1))
        g.close()
        out["paper_regime_trajectory"] = {"protocol": "L=48, Ntau=480, c_tau=80, K=1 pure-gauge heat-bath field (not equilibrated under the fermion action: a timing protocol, dH is not a physics figure), 3 leapfrog steps of eps 0.02, 4 PCG solves to tol",
                                          "tol": args.tol, "ms_per_trajectory": best, "cg_iters": rr["cg_iters"], "converged": rr["converged"],
                                          "dH": rr["H1"] - rr["H0"], "MdagM_Gsite_per_s_all_in": rr["cg_iters"] * N / (best * 1e-3) / 1e9}
    # complex64 variant (BASELINE config 4: "with a complex64 variant timed separately")
    g = hqmc.HQMC(L, Ntau, prec="c64")
    g.set_theta(dev(theta_cfg))
    phi = g.apply_Mdag(dev(eta_cfg.astype(np.complex64)))
    k64 = pcg_kernel_costs(g, torch, phi, args.cg_iters)
    out["c64"] = {"mdagm_us_in_graph": k64["us"]["mdagm"], "mdagm_Gsite_per_s": N / k64["us"]["mdagm"] / 1e3,
                  "mdagm_alg_GBps": 24.0 * N / k64["us"]["mdagm"] / 1e3, "cg_us_per_iter": k64["iter_us"], "kernels_us": k64["us"]}
    g.close()
    # config 5 on its own field
    if not args.no_config5:
        c5 = inputs.CONFIGS[5]
        L5, Nt5, N5 = c5["L"], c5["Ntau"], c5["L"] * c5["L"] * c5["Ntau"]
        th5 = inputs.make_theta(5)
        g = hqmc.HQMC(L5, Nt5)
        d_th0 = dev(th5)
        g.set_theta(d_th0)
        phi = g.apply_Mdag(dev(inputs.complex_gaussian((Nt5, L5, L5), c5["seed"])))
        k5 = pcg_kernel_costs(g, torch, phi, args.cg_iters)
        ms = []
        for k in range(2):                                          # first trajectory is warm-up
            d_th, d_p = d_th0.clone(), dev(inputs.momenta(L5, Nt5, c5["seed"] + k))
            g.set_theta(d_th)
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(); r = g.trajectory(d_th, d_p, phi, 20, 0.05, cg_tol=0.0, cg_max_iter=args.cg_iters); e1.record(); torch.cuda.synchronize()
            ms.append(e0.elapsed_time(e1))
        peak, _ = measured_peaks()
        out["config5"] = {"L": L5, "Ntau": Nt5, "sites": N5, "theta": "seeded heat bath at 1/g^2 = 1 + pi flux (BASELINE config 5)",
                          "protocol": f"20 leapfrog steps, eps 0.05, {args.cg_iters} fixed PCG iterations per solve (PAPER.md:348), 21 solves",
                          "ms_per_trajectory": ms[1], "cg_iters_per_trajectory": r["cg_iters"], "us_per_cg_iter_all_in": 1e3 * ms[1] / r["cg_iters"],
                          "MdagM_Gsite_per_s_all_in": r["cg_iters"] * N5 / (ms[1] * 1e-3) / 1e9,
                          "hbm_fraction_alg": 224.0 * N5 * r["cg_iters"] / (ms[1] * 1e-3) / 1e9 / peak,
                          "mdagm_us_in_graph": k5["us"]["mdagm"], "mdagm_Gsite_per_s": N5 / k5["us"]["mdagm"] / 1e3,
                          "mdagm_alg_GBps": 48.0 * N5 / k5["us"]["mdagm"] / 1e3, "cg_us_per_iter": k5["iter_us"], "kernels_us": k5["us"]}
        g.close()
    # leapfrog step as one CUDA graph vs plain launches
    mg = {"protocol": "3 leapfrog steps, eps 0.01, 100 fixed PCG iterations per solve, uniform theta; ms per trajectory, best of 5",
          "paper": "PAPER.md:334-350: CUDA graphs give 2-5 x for L < 30 and 1-2 x for larger lattices (its GPU, whole sweeps) -- context"}
    for Lg in (12, 24, 48):
        Ng = 10 * Lg
        th, p0 = inputs.theta_uniform(Lg, Ng, 7), inputs.momenta(Lg, Ng, 7)
        res, fin = {}, {}
        for on in (True, False, "persistent"):
            g = hqmc.HQMC(Lg, Ng)
            if on == "persistent":                      # the whole solve as one persistent kernel (small lattices only)
                try:
                    g.set_cg_persistent(hqmc.PERSIST_ON)
                except hqmc.HqmcError:
                    g.close()
                    continue
            else:
                g.set_cg_persistent(hqmc.PERSIST_OFF)
                g.set_md_graph(on)
            g.set_theta(dev(th))
            phi = g.apply_Mdag(dev(inputs.complex_gaussian((Ng, Lg, Lg), 7)))
            best = 1e30
            for k in range(6):
                d_th, d_p = dev(th), dev(p0)
                torch.cuda.synchronize()
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(); g.trajectory(d_th, d_p, phi, 3, 0.01, cg_tol=0.0, cg_max_iter=100); e1.record(); torch.cuda.synchronize()
                if k:
                    best = min(best, e0.elapsed_time(e1))
            res[on if on == "persistent" else ("graph" if on else "plain")] = best
            fin[on] = (d_th, d_p)
            g.close()
        mg[f"L{Lg}"] = {"ms_graph": res["graph"], "ms_plain": res["plain"], "speedup": res["plain"] / res["graph"],
                        "bitwise_identical": bool(torch.equal(fin[True][0], fin[False][0]) and torch.equal(fin[True][1], fin[False][1]))}
        if "persistent" in res:
            mg[f"L{Lg}"]["ms_persistent_kernel"] = res["persistent"]
            mg[f"L{Lg}"]["max_abs_diff_theta_persistent"] = float((fin["persistent"][0] - fin[True][0]).abs().max())
    out["md_graph"] = mg
    # one chain of a small lattice (PAPER.md:350's launch-bound regime): the four-kernel graph-replayed loop against the
    # one-launch persistent kernel (pcg_persist.cuh), us per PCG iteration over 2000 fixed iterations
    pp = {"protocol": "uniform theta, Ntau = 10 L, 2000 fixed iterations, wall clock around hqmc_cg_solve; us per iteration"}
    for Lp in (8, 12, 16, 20):
        Np = 10 * Lp
        g = hqmc.HQMC(Lp, Np)
        g.set_theta(dev(inputs.theta_uniform(Lp, Np, 7)))
        phi = g.apply_Mdag(dev(inputs.complex_gaussian((Np, Lp, Lp), 7)))
        row = {}
        for name, mode in (("loop", hqmc.PERSIST_OFF), ("persistent", hqmc.PERSIST_ON)):
            g.set_cg_persistent(mode)
            g.cg_solve(phi, 0.0, 200)
            torch.cuda.synchronize(); t0 = time.perf_counter()
            g.cg_solve(phi, 0.0, 2000)
            torch.cuda.synchronize()
            row[name] = 1e6 * (time.perf_counter() - t0) / 2000
        pp[f"L{Lp}"] = row
        g.close()
    out["pcg_persistent"] = pp
    return out


def small_lattice_chains(torch, hqmc, inputs, cg_iters, L=16, n_chain=40, md_steps=3, eps=0.01):
    """Extra key of the JSON line (not the metric): a lattice that cannot fill the GPU on its own (L=16, N_tau=160) run as one
    chain (hqmc_leapfrog_trajectory) and as n_chain independent chains advanced together (hqmc_leapfrog_trajectory_batched);
    same protocol as the main step (uniform theta, fixed-count PCG).  Trajectories per second and all-in Gsite/s."""
    try:
        Ntau, N = 10 * L, L * L * 10 * L
        g = hqmc.HQMC(L, Ntau)
        th0 = np.stack([inputs.theta_uniform(L, Ntau, 100 + b) for b in range(n_chain)])
        p0 = np.stack([inputs.momenta(L, Ntau, 100 + b) for b in range(n_chain)])
        eta = torch.from_numpy(np.stack([inputs.complex_gaussian((Ntau, L, L), 100 + b) for b in range(n_chain)])).cuda()
        out = {"L": L, "Ntau": Ntau, "md_steps": md_steps, "cg_iters_per_solve": cg_iters}
        for n in (1, n_chain):
            ms = []
            for k in range(3):                                           # first one is warm-up
                th, p = torch.from_numpy(th0[:n].copy()).cuda(), torch.from_numpy(p0[:n].copy()).cuda()
                torch.cuda.synchronize()
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record()
                if n == 1:
                    g.set_theta(th[0])
                    r = g.trajectory(th[0], p[0], g.apply_Mdag(eta[0].contiguous()), md_steps, eps, cg_tol=0.0, cg_max_iter=cg_iters)
                    its = r["cg_iters"]
                else:
                    r = g.trajectory_batched(th, p, g.refresh_batched(th, eta[:n].contiguous()), md_steps, eps, cg_tol=0.0, cg_max_iter=cg_iters)
                    its = sum(r["cg_iters"])
                e1.record(); torch.cuda.synchronize()
                if k:
                    ms.append(e0.elapsed_time(e1))
            t = float(np.mean(ms))
            out[f"chains_{n}"] = {"ms_per_batch": t, "trajectories_per_s": n / (t * 1e-3), "MdagM_Gsite_per_s": its * N / (t * 1e-3) / 1e9}
        g.close()
        return out
    except Exception as e:                                               # never lose the metric line over the extra key
        return {"error": repr(e)[:200]}


def pcg_kernel_costs(g, torch, d_phi, iters):
    """-> {"iter_us": us per PCG iteration, "us": {kernel class: us per launch inside the replayed graph}}."""
    from paper_2508_16298_b200 import hqmc
    x = g.new_vec()
    iters = max(64, (iters // 32) * 32)

    def run():
        g.cg_solve(d_phi, 0.0, iters, x=x)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(); g.cg_solve(d_phi, 0.0, iters, x=x); e1.record()
        torch.cuda.synchronize()
        return 1e3 * e0.elapsed_time(e1) / iters

    g.set_debug_skip(0)
    full = run()
    g.reset_stats(); g.cg_solve(d_phi, 0.0, 32, x=x); torch.cuda.synchronize()
    used = [k for k in ("mdagm", "cg_axpy", "precond", "cg_dupdate") if g.kernel_stats()[k][0] >= 32]
    keeper = "precond"                                                # the class that counts iterations / sets `done`
    out = {}
    for k in used:
        if k == keeper:
            continue
        g.set_debug_skip(1 << hqmc.KERNEL_CLASSES.index(k))
        out[k] = full - run()
    g.set_debug_skip(0)
    out[keeper] = full - sum(out.values())
    return {"iter_us": full, "us": out}


def run_solve(args):
    """--mode solve: one preconditioned CG solve to --tol on the chosen config (BASELINE.json: "CG-solve ms ... iteration
    count and ms per solve reported"), plus the same solve without the preconditioner capped at the same iteration count."""
    import torch
    from paper_2508_16298_b200 import hqmc, inputs
    c = inputs.CONFIGS[args.config]
    L, Ntau = c["L"], c["Ntau"]
    theta = inputs.theta_paper_regime(L, Ntau, c["seed"]) if args.theta == "paper" else inputs.make_theta(args.config)
    eta = inputs.complex_gaussian((Ntau, L, L), c["seed"])
    out = {"mode": "solve", "config": args.config, "L": L, "Ntau": Ntau, "tol": args.tol,
           "theta": "paper regime (c_tau=80, K=1 heat bath, cold start)" if args.theta == "paper" else c["theta"]}
    for W in (6, 0):
        g = hqmc.HQMC(L, Ntau, W=W)
        g.set_theta(torch.from_numpy(theta).cuda())
        phi = g.apply_Mdag(torch.from_numpy(eta).cuda())
        cap = args.max_iter if W else out["W6"]["iters"]
        torch.cuda.synchronize(); t0 = time.perf_counter()
        x, it, rel, ok = g.cg_solve(phi, args.tol, cap)
        torch.cuda.synchronize(); dt = time.perf_counter() - t0
        true_res = float(torch.linalg.vector_norm(phi - g.apply_MdagM(x)) / torch.linalg.vector_norm(phi))
        out[f"W{W}"] = {"iters": it, "converged": ok, "recurrence_relres": rel, "true_relres": true_res, "ms_per_solve": 1e3 * dt,
                        "us_per_iter": 1e6 * dt / max(1, it), "SF_minus_eta2": float((torch.vdot(phi.ravel(), x.ravel()).real
                                                                                     - (abs(torch.from_numpy(eta)) ** 2).sum()))}
        g.close()
    print(json.dumps(out))
    return 0


def run_slab(args):
    """--mode slab: the tau-slab path (paper_2508_16298_b200/slab.py) -- us per PCG iteration with
    the lattice cut into S slabs, fixed iteration count.  One process: S = 1, 2, 4 slabs on the one GPU, slab after
    slab (what sharding costs in halo slices, extra launches and host time, with no link in the way).  Under torchrun with N
    ranks: one slab per rank, halos and sums over NCCL, time = max over ranks."""
    import torch
    from paper_2508_16298_b200 import hqmc, inputs
    from paper_2508_16298_b200.slab import CudaSlabOps, SlabLayout, SlabSolver
    rank, world, local = dist_env()
    torch.cuda.set_device(local)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    c = inputs.CONFIGS[args.config]
    L, Ntau = (args.L, 10 * args.L) if args.L else (c["L"], c["Ntau"])
    iters = args.cg_iters
    theta = inputs.theta_uniform(L, Ntau, c["seed"])
    eta = inputs.complex_gaussian((Ntau, L, L), c["seed"])
    out = {"mode": "slab", "L": L, "Ntau": Ntau, "iters": iters, "n_gpus": world, "theta": "uniform", "slabs": {}}
    dev = torch.device("cuda", local)
    if rank == 0:
        g = hqmc.HQMC(L, Ntau, device=dev)
        g.set_theta(torch.from_numpy(theta).to(dev))
        phi1 = g.apply_Mdag(torch.from_numpy(eta).to(dev))
        g.cg_solve(phi1, 0.0, iters)
        torch.cuda.synchronize(); t0 = time.perf_counter()
        x1, _, rel1, _ = g.cg_solve(phi1, 0.0, iters)
        torch.cuda.synchronize()
        out["one_context"] = {"us_per_iter": 1e6 * (time.perf_counter() - t0) / iters, "relres": rel1}
        phi_h = phi1.cpu().numpy()
        x1_h = x1.cpu().numpy()
        g.close()
    else:
        phi_h = None
    if world > 1:
        import torch.distributed as dist
        box = [phi_h]
        dist.broadcast_object_list(box, src=0)
        phi_h = box[0]
    for S in ([world] if world > 1 else [1, 2, 4]):
        lay = SlabLayout(L, Ntau, S, W=6, world=world, rank=rank)
        ops = CudaSlabOps(lay, device=dev)
        sol = SlabSolver(lay, ops)
        part = lambda a: [torch.from_numpy(np.ascontiguousarray(a[lay.bounds[gg]:lay.bounds[gg + 1]])).to(dev) for gg in lay.owned]
        sol.set_theta(part(theta))
        rhs = sol.extend(part(phi_h), ops.new_vec)
        xs = [ops.new_vec(i) for i in range(len(lay.owned))]
        res = {}
        for graph in (False, True):
            try:
                sol.solve(rhs, xs, 0.0, min(iters, 20), graph=graph)
            except Exception as e:          # e.g. a communicator that cannot be captured into a CUDA graph
                res["graph" if graph else "plain"] = {"error": repr(e)[:200]}
                continue
            torch.cuda.synchronize()
            if world > 1:
                torch.distributed.barrier()
            t0 = time.perf_counter()
            it, rel, _ = sol.solve(rhs, xs, 0.0, iters, graph=graph)
            torch.cuda.synchronize()
            dt = time.perf_counter() - t0
            if world > 1:
                t = torch.tensor([dt], dtype=torch.float64, device=dev)
                torch.distributed.all_reduce(t, op=torch.distributed.ReduceOp.MAX)
                dt = float(t)
            res["graph" if graph else "plain"] = {"us_per_iter": 1e6 * dt / it, "relres": rel}
        if rank == 0 and world == 1:
            x = np.concatenate([sol.own(v, i).cpu().numpy() for i, v in enumerate(xs)], axis=0)
            res["max_rel_diff_vs_one_context"] = float(np.abs(x - x1_h).max() / np.abs(x1_h).max())
        res["halo_slices_per_slab"] = 2 * lay.H
        res["owned_slices"] = [lay.nt(gg) for gg in range(S)]
        out["slabs"][str(S)] = res
        ops.close()
    if rank == 0:
        print(json.dumps(out))
    if world > 1:
        torch.distributed.destroy_process_group()
    return 0


def run_trajectory(args):
    """--mode trajectory: BASELINE config 5's protocol ("5 HMC trajectories of 20 leapfrog steps each, reporting ms per
    trajectory and HBM fraction") on the chosen config.  The PCG runs the paper's fixed iteration count per solve
    (--cg-iters): on BASELINE's rough fields a solve to 1e-10 needs 3-6 x 10^5 iterations (`--mode solve`),
    i.e. half an hour per trajectory, so tolerance-stopped trajectories are timed on the paper-regime field (--theta paper,
    --tol) instead.  Not the timed metric of the JSON contract."""
    import torch
    from paper_2508_16298_b200 import hqmc, inputs
    c = inputs.CONFIGS[args.config]
    L, Ntau = c["L"], c["Ntau"]
    if args.L:                                               # the paper's shape at another size: V_s = L^2, N_tau = 10 L
        L, Ntau = args.L, 10 * args.L
    if args.chains:
        return run_chains(args, L, Ntau, c["seed"])
    N = L * L * Ntau
    paper = args.theta == "paper"
    theta0 = inputs.theta_paper_regime(L, Ntau, c["seed"]) if paper else inputs.make_theta(args.config)
    kw = dict(c_tau=80.0, K=1.0) if paper else {}
    g = hqmc.HQMC(L, Ntau, **kw)
    tol, cap = (args.tol, args.max_iter) if paper else (0.0, args.cg_iters)
    d_theta0 = torch.from_numpy(theta0).cuda()
    times, iters, dH = [], [], []
    for k in range(args.n_traj + 1):                              # first one is warm-up
        d_theta = d_theta0.clone()
        d_p = torch.from_numpy(inputs.momenta(L, Ntau, c["seed"] + k)).cuda()
        g.set_theta(d_theta)
        d_phi = g.apply_Mdag(torch.from_numpy(inputs.complex_gaussian((Ntau, L, L), c["seed"] + k)).cuda())
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        r = g.trajectory(d_theta, d_p, d_phi, args.md_steps, args.eps, cg_tol=tol, cg_max_iter=cap)
        e1.record(); torch.cuda.synchronize()
        if k:
            times.append(e0.elapsed_time(e1)); iters.append(r["cg_iters"]); dH.append(r["H1"] - r["H0"])
    ms = float(np.mean(times))
    it = float(np.mean(iters))
    peak, peak_src = measured_peaks()
    bps = 224.0                                                   # algorithmic bytes per site per PCG iteration
    print(json.dumps({"mode": "trajectory", "config": args.config, "L": L, "Ntau": Ntau, "sites": N,
                      "theta": "paper regime (c_tau=80, K=1 heat bath, cold start)" if paper else c["theta"],
                      "md_steps": args.md_steps, "eps": args.eps, "trajectories": args.n_traj,
                      "cg": f"to {tol:g}" if paper else f"fixed {cap} iterations per solve (PAPER.md:348)",
                      "ms_per_trajectory": ms, "ms_min": float(np.min(times)), "ms_max": float(np.max(times)),
                      "cg_iters_per_trajectory": it, "us_per_cg_iter_all_in": 1e3 * ms / it,
                      "MdagM_Gsite_per_s": it * N / (ms * 1e-3) / 1e9,
                      "hbm_fraction_alg": bps * N * it / (ms * 1e-3) / 1e9 / peak, "peak_GBps": peak, "peak_source": peak_src,
                      "dH": dH}))
    g.close()
    return 0


def run_chains(args, L, Ntau, seed):
    """--mode trajectory --chains n1,n2,...: n independent Markov chains advanced together on one GPU
    (hqmc_leapfrog_trajectory_batched), paper-regime fields (4 distinct heat-bath fields cycled over the chains; momenta and
    pseudofermions differ per chain), PCG to --tol.  Reports ms per batch of trajectories and trajectories per second for
    every chain count, next to the one-chain path (chains = 1 runs hqmc_leapfrog_trajectory)."""
    import torch
    from paper_2508_16298_b200 import hqmc, inputs
    N = L * L * Ntau
    counts = [int(x) for x in args.chains.split(",")]
    nmax = max(counts)
    fields = [inputs.theta_paper_regime(L, Ntau, seed + 17 * k) for k in range(min(4, nmax))]
    g = hqmc.HQMC(L, Ntau, c_tau=80.0, K=1.0)
    out = {}
    for n in counts:
        times, iters = [], []
        for k in range(args.n_traj + 1):                          # first one is warm-up
            th = torch.from_numpy(np.stack([fields[b % len(fields)] for b in range(n)])).cuda()
            p = torch.from_numpy(np.stack([inputs.momenta(L, Ntau, seed + 1000 * k + b) for b in range(n)])).cuda()
            eta = torch.from_numpy(np.stack([inputs.complex_gaussian((Ntau, L, L), seed + 1000 * k + b) for b in range(n)])).cuda()
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            if n == 1:
                g.set_theta(th[0])
                phi = g.apply_Mdag(eta[0].contiguous())
                r = g.trajectory(th[0], p[0], phi, args.md_steps, args.eps, cg_tol=args.tol, cg_max_iter=args.max_iter)
                its = r["cg_iters"]
            else:
                phi = g.refresh_batched(th, eta)
                r = g.trajectory_batched(th, p, phi, args.md_steps, args.eps, cg_tol=args.tol, cg_max_iter=args.max_iter)
                its = sum(r["cg_iters"])
            e1.record(); torch.cuda.synchronize()
            assert r["converged"]
            if k:
                times.append(e0.elapsed_time(e1)); iters.append(its)
        ms, it = float(np.mean(times)), float(np.mean(iters))
        out[str(n)] = {"ms_per_batch": ms, "trajectories_per_s": n / (ms * 1e-3), "cg_iters_all_chains": it,
                       "MdagM_Gsite_per_s": it * N / (ms * 1e-3) / 1e9}
    print(json.dumps({"mode": "trajectory", "chains": out, "L": L, "Ntau": Ntau, "sites": N, "md_steps": args.md_steps, "eps": args.eps,
                      "theta": "paper regime (c_tau=80, K=1 heat bath, cold start), 4 fields cycled", "cg": f"to {args.tol:g}",
                      "trajectories_timed": args.n_traj}))
    g.close()
    return 0


def run_measure(args):
    """--mode measure: the stochastic estimator (widening row NEXT-2) on a paper-regime field of the chosen
    config: n_rv noise vectors -> G xi by PCG -> the pair correlator over binom(n_rv, 2) pairs through Eq.19 (cuFFT).  Not the
    timed metric; reports time per stage."""
    import torch
    from paper_2508_16298_b200 import hqmc, inputs
    c = inputs.CONFIGS[args.config]
    L, Ntau, n_rv = c["L"], c["Ntau"], args.n_rv
    if args.L:                                               # the paper's shape at another size: V_s = L^2, N_tau = 10 L
        L, Ntau = args.L, 10 * args.L
    theta = inputs.theta_paper_regime(L, Ntau, c["seed"])
    g = hqmc.HQMC(L, Ntau)
    g.set_theta(torch.from_numpy(theta).cuda())
    xi = torch.from_numpy(np.stack([inputs.complex_gaussian((Ntau, L, L), c["seed"] + 10 * k, inputs.STREAM_VEC) for k in range(n_rv)])).cuda()
    gv = torch.empty_like(xi)
    out = g.new_vec()

    def timed(fn):
        fn(); torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(); r = fn(); e1.record(); torch.cuda.synchronize()
        return r, e0.elapsed_time(e1)

    # vectors per launch of the multi-right-hand-side PCG: 0 = library default (by L2 footprint), 1 = one at a time
    by_batch = {}
    for bs in [int(b) for b in args.green_batch.split(",")][::-1]:
        g.set_green_batch(bs)
        (_, iters, ok), ms_solve = timed(lambda: g.green_apply(xi, args.tol, args.max_iter, out=gv))
        by_batch[str(bs)] = {"ms_green_apply": ms_solve, "cg_iters_total": iters, "converged": ok}
    _, ms_2pt = timed(lambda: g.green_2pt(gv, xi, out=out))
    _, ms_pair = timed(lambda: g.pair_correlator(gv, xi, out=out))
    back = g.apply_M(gv[0].contiguous())
    res = float(torch.linalg.vector_norm(back - xi[0]) / torch.linalg.vector_norm(xi[0]))
    npair = n_rv * (n_rv - 1) // 2
    print(json.dumps({"mode": "measure", "config": args.config, "L": L, "Ntau": Ntau, "n_rv": n_rv, "tol": args.tol,
                      "theta": "paper regime (c_tau=80, K=1 heat bath, cold start)", "converged": ok, "cg_iters_total": iters,
                      "green_batch": int(args.green_batch.split(",")[0]), "ms_green_apply": ms_solve, "ms_per_vector": ms_solve / n_rv, "by_green_batch": by_batch, "relres_M_Gxi_minus_xi": res,
                      "ms_green_2pt": ms_2pt, "pairs": npair, "ms_pair_correlator": ms_pair, "us_per_pair": 1e3 * ms_pair / npair}))
    g.close()
    return 0


def mdagm_sweep(g, torch, dev, L, Ntau, prec, nbuf=8, reps=25):
    """M^+M alone: cold = rotate nbuf distinct (in, out) pairs so every launch streams from HBM; warm = one pair."""
    N = L * L * Ntau
    ins = [g.new_vec() for _ in range(nbuf)]
    outs = [g.new_vec() for _ in range(nbuf)]
    for v in ins:
        v.copy_(torch.randn(v.shape, dtype=v.dtype, device=dev))
    res = {}
    for mode in ("cold", "warm"):
        for i in range(nbuf):
            g.apply_MdagM(ins[i], outs[i])
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        n = 0
        for _ in range(reps):
            for i in range(nbuf):
                j = i if mode == "cold" else 0
                g.apply_MdagM(ins[j], outs[j]); n += 1
        e1.record()
        torch.cuda.synchronize()
        us = 1e3 * e0.elapsed_time(e1) / n
        bps = 48.0 if prec == "c128" else 24.0
        res[mode] = {"us": us, "Gsite_per_s": N / us / 1e3, "alg_GBps": bps * N / us / 1e3}
    return res


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--config", type=int, default=4, help="BASELINE.json config number (1-5); 4 = L=48, Ntau=480")
    ap.add_argument("--cg-iters", type=int, default=500, help="fixed PCG iterations per solve (PAPER.md:348)")
    ap.add_argument("--ref-cg-iters", type=int, default=60, help="PCG iterations per solve of the CPU-oracle sample")
    ap.add_argument("--e2e-steps", type=int, default=2)
    ap.add_argument("--prec", default="c128", choices=["c128", "c64"])
    ap.add_argument("--no-sweep", action="store_true")
    ap.add_argument("--no-small", action="store_true", help="skip the extra small-lattice batched-chains key of the JSON line")
    ap.add_argument("--no-extras", action="store_true", help="skip cg_solve / c64 / config5 / md_graph keys (converged solves, second lattice)")
    ap.add_argument("--no-solve", action="store_true", help="skip the converged config-4 solves (about 20 s of GPU time)")
    ap.add_argument("--no-config5", action="store_true", help="skip the L=64 lattice (its heat-bath field costs 40 s of host time)")
    ap.add_argument("--mode", default="step", choices=["step", "solve", "measure", "trajectory", "slab"],
                    help="solve: one full PCG solve to --tol; measure: the stochastic estimator on a paper-regime field (neither is the timed metric)")
    ap.add_argument("--n-traj", type=int, default=5, help="trajectory mode: timed trajectories (BASELINE config 5: 5)")
    ap.add_argument("--md-steps", type=int, default=20, help="trajectory mode: leapfrog steps per trajectory (BASELINE config 5: 20)")
    ap.add_argument("--eps", type=float, default=0.05, help="trajectory mode: leapfrog step size")
    ap.add_argument("--n-rv", type=int, default=40, help="measure mode: number of noise vectors (PAPER.md:244)")
    ap.add_argument("--green-batch", default="0", help="measure mode: vectors per launch of the batched PCG, comma list to compare "
                    "(0 = library default, 1 = one at a time); the first entry is the one the other stages run after")
    ap.add_argument("--L", type=int, default=0, help="measure / trajectory modes: lattice size override (N_tau = 10 L)")
    ap.add_argument("--chains", default="", help="trajectory mode: comma list of chain counts advanced together (paper-regime fields)")
    ap.add_argument("--tol", type=float, default=1e-10)
    ap.add_argument("--theta", default="config", choices=["config", "paper"], help="solve / trajectory modes: the config's field or a paper-regime field")
    ap.add_argument("--max-iter", type=int, default=3000000)
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "b200":
        args.warmup = 3
    if args.mode == "solve":
        return run_solve(args)
    if args.mode == "measure":
        return run_measure(args)
    if args.mode == "trajectory":
        return run_trajectory(args)
    if args.mode == "slab":
        return run_slab(args)
    return run_reference(args) if args.impl == "reference" else run_gpu(args)


if __name__ == "__main__":
    sys.exit(main())
