#!/usr/bin/env python
"""bench.py — headline benchmark of the SEM hot path on B200 (BASELINE.json metric).

A "step" is one pass of the whole hot path over the synthetic batch: ONE Jacobi-PCG pressure iteration
(axhelm with the fused x / Jacobi + direction updates and p.Ap -> Dirichlet mask -> gather-scatter, done as an
in-place sum over the edge/corner classes plus a partner gather folded into the r update -> ||r||^2 and r.z reductions) on the 64^3-element deformed box of BASELINE.json configs[3]
(N = 7, fp64, 134 217 728 local nodes, lambda = 0).  K steps = one semb_pcg_solve call with maxit = K and
rtol = 0 (it cannot stop early), bracketed by CUDA events on the launching stream.

    value     = local nodes processed per second by the whole step (GDOF/s), all ranks
    roofline  = the dominant kernel (the PCG-fused axhelm launch): 104 B/node algorithmic bytes / its mean device
                time measured with CUDA event pairs around its launches INSIDE the timed solve, against
                MEASURED_PEAKS.json hbm_gbs; axhelm_sweep = the stand-alone operator at 64 / 72 B/node
    pcg_iter  = the whole iteration against the fixed 171.6 B/node model
    e2e       = the same K iterations through semb_pcg_solve_host: b from pinned host memory, x back to it
    cpu_baseline = the oracle (oracle/semoracle.c, as it stands) timed on this box's host cores

`--impl reference` times the oracle alone, same metric/unit/config.  Multi-GPU: replicas only:
each rank runs the same workload on its own GPU, value = sum over ranks / max-over-ranks time.
"""
import argparse
import json
import os
import subprocess
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_2501_13240_b200 import inputs as I  # noqa: E402

METRIC = "SEM Jacobi-PCG pressure-iteration throughput (axhelm+gather-scatter+mask+Jacobi+fused updates), N=7 fp64"
UNIT = "GDOF/s"
B_AXHELM = 64.0          # algorithmic bytes per node, Poisson axhelm
B_AXHELM_HELM = 72.0
B_AXHELM_PCG = 104.0     # the PCG-fused launch: reads r, dinv, p, x (32) + G (48), writes p, x, q (24)
NCU_TRAFFIC_AXHELM_PCG = 13.943e9   # dram read + write bytes of one launch on cfg3, ncu --set full (profiles/r1_v4_axhelm_full.md)
B_ITER = 171.6           # algorithmic bytes per node per Jacobi-PCG iteration, N = 7, Poisson
WORKLOADS = {            # name -> elements per direction of the deformed box (BASELINE.json configs[3] / configs[1]),
    "cfg3_box64_deformed_N7": 64,     # or ("ogrid", cfg): the cylinder O-grids of configs[2] / configs[4]
    "cfg1_box16_deformed_N7": 16,
    "box32_deformed_N7": 32,
    "cfg2_ogrid_N7": ("ogrid", 2),
    "cfg4_ogrid_N9": ("ogrid", 4),
}


def model_bytes_per_iteration(N):
    """64 (axhelm) + 20 * n_shared/n (gather-scatter) + 64 + 32, n_shared/n = 1 - ((N-1)/(N+1))^3."""
    return 64.0 + 20.0 * (1.0 - ((N - 1.0) / (N + 1.0)) ** 3) + 64.0 + 32.0


def measured_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 100 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.p = index, None

    def start(self):
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                       "--format=csv,noheader,nounits", "-lms", "100"],
                                      stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.p = None

    def stop(self):
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.p.terminate()
        try:
            out, _ = self.p.communicate(timeout=5)
        except subprocess.TimeoutExpired:
            self.p.kill(); out, _ = self.p.communicate()
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in out.strip().splitlines():
            f = [t.strip() for t in line.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for nme, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nme)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


def aggregate(ms_local, nodes_local, steps, dist=None, device=None):
    """Whole-job figure from per-rank device times (replicas only): every rank processed
    nodes_local x steps node updates in ms_local milliseconds; the job took the MAX over ranks and processed the
    SUM over ranks.  Returns (ms, value in GDOF/s).  `dist` = an initialised torch.distributed module or None."""
    import torch
    ms, total = float(ms_local), float(nodes_local) * steps
    if dist is not None and dist.is_initialized() and dist.get_world_size() > 1:
        t = torch.tensor([ms], dtype=torch.float64, device=device)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        c = torch.tensor([total], dtype=torch.float64, device=device)
        dist.all_reduce(c, op=dist.ReduceOp.SUM)
        ms, total = float(t.item()), float(c.item())
    return ms, total / (ms * 1e-3) / 1e9


def build_problem(torch, semb, ne):
    """64^3 (or ne^3) deformed box, N = 7, or an O-grid of configs[2] / [4]: mesh on the host, coordinates to the device, setup."""
    if isinstance(ne, tuple):
        m, _ = I.config_mesh(ne[1], lambda N: semb.gll(N)[0])
    else:
        xi = semb.gll(7)[0]
        m = I.box_mesh(ne, ne, ne, 7, xi, deform=0.05, name=f"box{ne}_deformed")
    x, y, z = (torch.from_numpy(a).cuda() for a in (m.x, m.y, m.z))
    G = semb.Mesh(m.E, m.N, x, y, z, m.face_tag, m.period)
    del x, y, z
    torch.cuda.empty_cache()
    return m, G


def oracle_sample(steps, warmup):
    """The oracle's Jacobi-PCG iteration on the 16^3-element member of the same deformed-box family."""
    from oracle import semoracle as O
    O.build()
    ne = 16
    xi = O.gll(7)[0]
    m = I.box_mesh(ne, ne, ne, 7, xi, deform=0.05)
    P = O.Problem(m.E, m.N, m.x, m.y, m.z, m.face_tag, m.period, lam=0.0, dirichlet_tags=0b10)
    b = P.assemble_rhs(I.uniform(I.seed_for(3, 2), m.n))
    if warmup > 0:
        P.pcg(b, precond=1, rtol=0.0, maxit=warmup)
    t0 = time.perf_counter()
    r = P.pcg(b, precond=1, rtol=0.0, maxit=steps)
    dt = time.perf_counter() - t0
    assert r["iters"] == steps
    return dict(n=m.n, seconds=dt, steps=steps, cores=O.num_threads(),
                sample=f"{steps} Jacobi-PCG iterations of oracle/semoracle.c on the 16^3-element deformed box "
                       f"(N=7, {m.n} local nodes = 1/64 of the workload), OpenMP over elements in axhelm only")


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    s = oracle_sample(max(args.steps, 1), args.warmup)
    val = s["n"] * s["steps"] / s["seconds"] / 1e9
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * s["seconds"] / s["steps"], "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": args.workload, "sample": s["sample"]},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": s["cores"], "kind": "oracle", "sample": s["sample"]},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg3_box64_deformed_N7", choices=list(WORKLOADS))
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-export", action="store_true")
    ap.add_argument("--no-cfg1", action="store_true", help="skip the configs[1] batched axhelm + gather-scatter section")
    ap.add_argument("--solve-maxit", type=int, default=20000, help="iteration cap of the time-to-solution solves (profiling runs)")
    ap.add_argument("--no-solve", action="store_true", help="skip the time-to-solution section (full pressure solves)")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)

    import torch
    from paper_2501_13240_b200 import semb
    semb.lib()                                         # fails loudly if the CUDA library is missing
    rank = int(os.environ.get("RANK", "0")); world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    K, W = max(args.steps, 1), max(args.warmup, 0)
    peak, peak_src = measured_peak()

    ne = WORKLOADS[args.workload]
    m, G = build_problem(torch, semb, ne)
    n = m.n
    b_iter = B_ITER if m.N == 7 else model_bytes_per_iteration(m.N)
    f = torch.from_numpy(I.uniform(I.seed_for(3, 2), n)).cuda()
    b = torch.empty_like(f)
    G.assemble_rhs(f, b, 0b10)
    x = torch.zeros_like(b)
    del f
    solve = dict(lam=0.0, tags=0b10, precond=1, rtol=0.0, atol=0.0)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- warm-up, then exactly K timed steps
    if W > 0:
        G.pcg_solve(b, x, maxit=W, check_every=W, **solve)
    sampler = ClockSampler(local)
    barrier()
    sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    st = G.pcg_solve(b, x, maxit=K, check_every=K, profile=True, **solve)
    e1.record()
    barrier()
    clocks = sampler.stop()
    ms = e0.elapsed_time(e1)
    assert st["iters"] == K, st
    ms, value = aggregate(ms, n, K, dist, "cuda")
    ms_step = ms / K
    ax_ms = st["axhelm_ms"]
    ax_gbs = B_AXHELM_PCG * n / (ax_ms * 1e-3) / 1e9

    # ---- axhelm alone, Poisson and Helmholtz (BASELINE.json configs[3] "roofline sweep"); not the headline
    u = torch.from_numpy(I.uniform(I.seed_for(3, 1), n)).cuda()
    w = torch.empty_like(u)
    sweep = {}
    for name, lam, nbytes in (("poisson", 0.0, B_AXHELM), ("helmholtz", 1e4, B_AXHELM_HELM)):
        for _ in range(5):
            G.apply_axhelm(u, w, lam=lam)
        reps = 20
        a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize(); a0.record()
        for _ in range(reps):
            G.apply_axhelm(u, w, lam=lam)
        a1.record(); torch.cuda.synchronize()
        t = a0.elapsed_time(a1) / reps
        sweep[name] = {"ms": t, "gdofs": n / (t * 1e-3) / 1e9, "gbs": nbytes * n / (t * 1e-3) / 1e9,
                       "frac_of_measured_peak": nbytes * n / (t * 1e-3) / 1e9 / peak,
                       "frac_of_8TBs": nbytes * n / (t * 1e-3) / 8e12}
    del u, w

    # ---- time to solution of the pressure solve on the same mesh and right-hand side, rtol 1e-10: Jacobi-PCG (the
    #      north_star path) and the p-multigrid V-cycle preconditioner of PAPER.md:L102.  Context for
    #      the per-iteration headline above, not part of it.
    solve_tts = None
    if not args.no_solve and world == 1:
        solve_tts = {}
        for name, kw in (("pmg_pcg", dict(precond=3, mg_smooth=1, mg_coarse=64, mg_coarse_frac=0.003)),
                         ("pmg_fp32_pcg", dict(precond=3, mg_smooth=1, mg_coarse=64, mg_coarse_frac=0.003, mg_fp32=True)),
                         ("jacobi_pcg", dict(precond=1))):
            xs = torch.zeros_like(b)
            if name.startswith("pmg"):
                G.pcg_solve(b, xs, lam=0.0, tags=0b10, rtol=1e-10, maxit=2, **kw)        # builds the levels, estimates the bounds
                xs.zero_()
            s0, s1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize(); s0.record()
            sst = G.pcg_solve(b, xs, lam=0.0, tags=0b10, rtol=1e-10, maxit=args.solve_maxit, **kw)
            s1.record(); torch.cuda.synchronize()
            solve_tts[name] = {"iters": sst["iters"], "status": sst["status"], "seconds": s0.elapsed_time(s1) * 1e-3,
                               "rel_residual": sst["r_norm"] / sst["b_norm"]}
            del xs
        solve_tts["speedup"] = solve_tts["jacobi_pcg"]["seconds"] / solve_tts["pmg_pcg"]["seconds"]
        solve_tts["speedup_fp32_levels"] = solve_tts["jacobi_pcg"]["seconds"] / solve_tts["pmg_fp32_pcg"]["seconds"]

    # ---- configs[3]: zero-copy export of temperature and velocity magnitude to the in-device min/max/256-bin histogram
    #      consumer (PAPER.md:L138-159 hand-off; overhead formula of PAPER.md:L375 against the PCG iteration time)
    export = None
    if not args.no_export and world == 1:
        T = torch.from_numpy((1.0 - m.z) + 0.05 * I.uniform(I.seed_for(3, 31), n)).cuda()
        vel = [torch.from_numpy(3.0 * I.uniform(I.seed_for(3, 32 + c), n)).cuda() for c in range(3)]
        G.publish_field("temperature", T)
        for nm, t in zip(("velocity_x", "velocity_y", "velocity_z"), vel):
            G.publish_field(nm, t)
        mm = torch.zeros(2, dtype=torch.float64, device="cuda"); hist = torch.zeros(256, dtype=torch.int64, device="cuda")

        def analysis_step(cycle):
            G.publish_state(cycle, 1e-3 * cycle)                     # refreshes |v| (one kernel: 24 B read + 8 B written per node)
            dT = G.export_field("temperature"); dV = G.export_field("velocity_magnitude")
            semb.field_minmax_hist(dT, 256, 0.0, 1.0, mm, hist)      # one pass: 8 B/node
            semb.field_minmax_hist(dV, 256, 0.0, 0.0, mm, hist)      # range found on the device: two passes, 16 B/node
            return dT
        dT = analysis_step(0)
        torch.cuda.synchronize()
        free0 = torch.cuda.mem_get_info()[0]
        x0, x1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        reps = 10
        x0.record()
        for c in range(reps):
            analysis_step(c + 1)
        x1.record(); torch.cuda.synchronize()
        t_an = x0.elapsed_time(x1) / reps
        nbytes = (24 + 8 + 8 + 16) * n
        export = {"ms_per_analysis_step": t_an, "bytes_per_node": 56, "gbs": nbytes / (t_an * 1e-3) / 1e9,
                  "pointer_identity": bool(dT.ptr == T.data_ptr()), "bytes_allocated": int(free0 - torch.cuda.mem_get_info()[0]),
                  "overhead_vs_pcg_iteration_pct": {str(nv): 100.0 * ((t_an + nv * ms_step) / (nv * ms_step) - 1.0) for nv in (1, 10, 100)},
                  "note": "overhead = (t_vis + (n_vis - 1) t_novis) / (n_vis t_novis) - 1 with t_vis = t_novis + analysis step, "
                          "t_novis = one PCG iteration (PAPER.md:L375)"}
        del T, vel

    # ---- configs[1]: batched axhelm + gather-scatter on the 16^3 deformed box, Helmholtz lambda = 10/dt = 1e4, nfields = 3,
    #      100 applications timed.  Its working set (~150 MB + 3 x 2 x 17 MB) is about the size of the L2: reported, but no
    #      roofline claim is made from it.
    cfg1 = None
    if not args.no_cfg1 and world == 1:
        m1, G1 = build_problem(torch, semb, 16)
        U = torch.from_numpy(I.uniform(I.seed_for(1, 1), 3 * m1.n)).cuda()
        Wv = torch.empty_like(U)
        for _ in range(5):
            G1.apply_axhelm(U, Wv, lam=1e4, nfields=3); G1.gather_scatter(Wv, nfields=3)
        c0, c1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize(); c0.record()
        for _ in range(100):
            G1.apply_axhelm(U, Wv, lam=1e4, nfields=3); G1.gather_scatter(Wv, nfields=3)
        c1.record(); torch.cuda.synchronize()
        t1 = c0.elapsed_time(c1) / 100
        cfg1 = {"ms_per_application": t1, "nfields": 3, "local_nodes": m1.n, "gdofs": 3 * m1.n / (t1 * 1e-3) / 1e9,
                "note": "axhelm (72 B/node) + stand-alone gather-scatter on 3 fields; working set about the size of L2"}
        G1.close(); del U, Wv

    # ---- configs[4]: 10 synthetic time steps, each one pressure Poisson solve + 3 velocity + 1 temperature Helmholtz solves
    #      (lambda = 1.5/dt = 3000) through ONE semb_step_solve call, right-hand sides perturbed per step, warm starts
    #      (R12).  Only on the cfg4 workload; every solve with Jacobi-PCG (as configs[4] words it), then every solve
    #      with the p-multigrid preconditioner on FP32-storage levels.
    steps10 = None
    if args.workload.startswith("cfg4") and not args.no_solve and world == 1:
        lam_h = 1.5 / 5e-4
        kinds = [(0.0, 0b10), (lam_h, 0b110), (lam_h, 0b110), (lam_h, 0b110), (lam_h, 0b10)]
        f0 = [I.divergence_source(m, I.seed_for(4, 30 + i)) for i in range(5)]
        rms = [float(np.sqrt(np.mean(v ** 2))) for v in f0]
        f0d = [torch.from_numpy(v).cuda() for v in f0]
        steps10 = {}
        for pname, pkw in (("jacobi_pcg_all_solves", dict(precond=1)), ("pmg_fp32_pcg_all_solves", dict(precond=3, mg_fp32=True))):
            xs = [torch.zeros(n, dtype=torch.float64, device="cuda") for _ in range(5)]
            bs = [torch.empty(n, dtype=torch.float64, device="cuda") for _ in range(5)]
            secs, iters = [], []
            for step in range(10):
                for i in range(5):
                    eta = torch.from_numpy(I.uniform(I.seed_for(4, 100 * (step + 1) + i), n)).cuda()
                    eta.mul_(0.1 * rms[i]).add_(f0d[i])
                    G.assemble_rhs(eta, bs[i], kinds[i][1])
                    del eta
                solves = [dict(b=bs[i], x=xs[i], lam=kinds[i][0], tags=kinds[i][1], rtol=1e-10, x0_is_zero=(step == 0),
                               **pkw) for i in range(5)]
                t0e, t1e = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                torch.cuda.synchronize(); t0e.record()
                rcs, sts = G.step_solve(solves)
                t1e.record(); torch.cuda.synchronize()
                secs.append(t0e.elapsed_time(t1e) * 1e-3); iters.append([q["iters"] for q in sts])
            steps10[pname] = {"seconds_per_step_mean": float(np.mean(secs)), "seconds_first_step": secs[0],
                              "seconds_per_step_after_first": float(np.mean(secs[1:])),
                              "iterations_last_step": iters[-1], "status": rcs}
            del xs, bs
        del f0d

    # ---- end to end through the C ABI with HOST buffers (pinned): b H2D, K iterations, x D2H
    e2e = None
    if not args.no_e2e:
        bh = b.cpu().pin_memory(); xh = torch.empty_like(bh).pin_memory()
        G.pcg_solve_host(bh, xh, maxit=1, check_every=1, **solve)                      # warm-up (allocates staging)
        barrier()
        h0, h1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        h0.record()
        G.pcg_solve_host(bh, xh, maxit=K, check_every=K, **solve)
        h1.record(); barrier()
        hms = h0.elapsed_time(h1)
        hms, e2e_value = aggregate(hms, n, K, dist, "cuda")
        e2e = {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": 8 * n / K,
               "d2h_bytes_per_step": 8 * n / K, "note": "one call = b host->device, K iterations, x device->host"}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": args.workload, "E": m.E, "N": m.N, "local_nodes": n, "lambda": 0.0,
                   "parallelism": "replicas only" if world > 1 else "single GPU",
                   "l2": "inputs larger than L2 (every vector is %.2f GB)" % (8 * n / 1e9)},
        "roofline": {"bound": "hbm", "kernel": f"k_axhelm_line<{m.N + 1},4,*>: axhelm (Poisson) with the fused PCG prologue (x += alpha p, p = dinv r + beta p) and p.Ap epilogue", "achieved": ax_gbs, "peak": peak,
                     "unit": "GB/s", "frac": ax_gbs / peak, "traffic": NCU_TRAFFIC_AXHELM_PCG if args.workload.startswith("cfg3") else None, "peak_source": peak_src,
                     "bytes_per_node": B_AXHELM_PCG, "ms": ax_ms, "timed_launches": st["profiled"],
                     "frac_of_8TBs": ax_gbs / 8000.0, "gdofs": n / (ax_ms * 1e-3) / 1e9},
        "pcg_iter": {"ms": ms_step, "model_bytes_per_node": b_iter, "gbs": b_iter * n / (ms_step * 1e-3) / 1e9,
                     "frac_of_measured_peak": b_iter * n / (ms_step * 1e-3) / 1e9 / peak,
                     "frac_of_8TBs": b_iter * n / (ms_step * 1e-3) / 8e12},
        "axhelm_sweep": sweep,
        "time_to_solution": solve_tts,
        "export": export,
        "cfg1_batched_axhelm_gs": cfg1,
        "cfg4_ten_steps": steps10,
        "e2e": e2e, "gpu_launches": st["launches"], "clocks": clocks,
    }
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        s = oracle_sample(60, 2)
        line["cpu_baseline"] = {"value": s["n"] * s["steps"] / s["seconds"] / 1e9, "unit": UNIT, "cores": s["cores"],
                                "kind": "oracle", "sample": s["sample"]}
    if rank == 0:
        print(json.dumps(line))
    G.close()
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
