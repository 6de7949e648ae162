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

Further sections of the same JSON line (single GPU only), so that every quoted number is driver-run: `configs` = the
Jacobi-PCG iteration, the stand-alone axhelm and the time to solution on the O-grids of BASELINE.json configs[2] and
configs[4] (build -> 20 iterations -> destroy), `cfg4_ten_steps` = the first steps of configs[4]'s ten-step recipe through
semb_step_solve, `e2e_single` = ONE semb_apply_axhelm_host call (nothing amortised), `stream_ceiling` = what HBM delivers
for a pure 7 : 1 read : write stream on this device.

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


import hashlib  # noqa: E402

UNIT = "GDOF/s"
B_AXHELM = 64.0          # algorithmic bytes per node, Poisson axhelm
B_AXHELM_HELM = 72.0
B_ITER = 171.6           # algorithmic bytes per node per Jacobi-PCG iteration, N = 7, Poisson (the fixed denominator)
B_AXHELM_PCG = 104.0     # the PCG-fused launch: reads r, dinv, p, x (32) + G (48), writes p, x, q (24)
WORKLOADS = {            # name -> elements per direction of the deformed box (BASELINE.json configs[3] / configs[1]),
    "cfg3_box64_deformed_N7": 64,     # or ("ogrid", cfg): the cylinder O-grids of configs[2] / configs[4]
    "cfg1_box16_deformed_N7": 16,
    "box32_deformed_N7": 32,
    "cfg2_ogrid_N7": ("ogrid", 2),
    "cfg4_ogrid_N9": ("ogrid", 4),
}
TRAFFIC_JSON = os.path.join(ROOT, "profiles", "r2_traffic.json")
KERNEL_SOURCES = ["axhelm_kernels.cuh", "axhelm_launch.cuh", "axhelm.cu", "reduce.cuh"]     # what the dominant kernel is compiled from


def metric_name(N):
    return ("SEM Jacobi-PCG pressure-iteration throughput (axhelm+gather-scatter+mask+Jacobi+fused updates), "
            f"N={N} fp64")


def model_bytes_per_iteration(N):
    """64 (axhelm) + 20 * n_shared/n (gather-scatter) + 64 + 32, n_shared/n = 1 - ((N-1)/(N+1))^3;
    N = 7: 171.6 B/node."""
    return 64.0 + 20.0 * (1.0 - ((N - 1.0) / (N + 1.0)) ** 3) + 64.0 + 32.0


def iter_bytes(N):
    return B_ITER if N == 7 else model_bytes_per_iteration(N)


def measured_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs: a 1:1 copy)"
    return 6650.0, "fallback (B200_PROFILING.md)"


def kernel_source_hash():
    h = hashlib.sha256()
    for f in KERNEL_SOURCES:
        with open(os.path.join(ROOT, "paper_2501_13240_b200", "csrc", f), "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()


def recorded_traffic(workload):
    """dram read + write bytes per launch of the dominant kernel from the tracked ncu record (profiles/r2_traffic.json),
    or None when the record was captured from other kernel sources than the ones in the tree (stale) or does not exist."""
    try:
        with open(TRAFFIC_JSON) as f:
            rec = json.load(f)["entries"].get(workload)
    except (OSError, ValueError, KeyError):
        return None, "no record"
    if not rec:
        return None, "no record for this workload"
    if rec.get("kernel_sources_sha256") != kernel_source_hash():
        return None, "record is stale: kernel sources changed since the capture"
    return float(rec["dram_bytes_per_launch"]), f"{os.path.relpath(TRAFFIC_JSON, ROOT)} (ncu --set full, commit {rec.get('commit', '?')})"


def record_traffic(args):
    """`bench.py --record-traffic RAW.csv --workload W`: read `ncu -i X.ncu-rep --page raw --csv` output, take the launches
    of the PCG-fused axhelm kernel (k_axhelm_line<..,4|5,..>), and write their median dram bytes into profiles/r2_traffic.json
    together with the hash of the kernel sources and the commit they were captured at."""
    import csv
    with open(args.record_traffic, newline="") as f:
        rows = list(csv.reader(f))
    hdr = rows[0]
    ik, ir, iw, it = (hdr.index(c) for c in ("Kernel Name", "dram__bytes_read.sum", "dram__bytes_write.sum", "gpu__time_duration.sum"))
    units = rows[1]
    mult = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}
    tot, ns = [], []
    for r in rows[2:]:
        name = r[ik]
        if "k_axhelm_line" not in name:
            continue
        targs = name[name.index("<") + 1:].split(",")
        if int(targs[1]) & 4 == 0:
            continue
        tot.append(float(r[ir].replace(",", "")) * mult[units[ir]] + float(r[iw].replace(",", "")) * mult[units[iw]])
        ns.append(float(r[it].replace(",", "")) * {"ns": 1.0, "us": 1e3, "ms": 1e6}.get(units[it], 1.0))
        kname = name
    assert tot, "no PCG-fused axhelm launch in the capture"
    try:
        with open(TRAFFIC_JSON) as f:
            rec = json.load(f)
    except OSError:
        rec = {"what": "dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel, ncu --set full; "
                       "written by `python bench.py --record-traffic <raw csv> --workload <W>`", "entries": {}}
    commit = subprocess.run(["git", "rev-parse", "--short", "HEAD"], cwd=ROOT, capture_output=True, text=True).stdout.strip()
    rec["entries"][args.workload] = {"kernel": kname, "launches_captured": len(tot), "dram_bytes_per_launch": float(np.median(tot)),
                                     "duration_ns_under_ncu": float(np.median(ns)), "kernel_sources": KERNEL_SOURCES,
                                     "kernel_sources_sha256": kernel_source_hash(), "commit": commit or "unknown",
                                     "command": args.traffic_command}
    with open(TRAFFIC_JSON, "w") as f:
        json.dump(rec, f, indent=1)
    print(json.dumps(rec["entries"][args.workload]))


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 100 ms from start() to stop(): the WHOLE GPU part of the run.
    sm_mhz = median over the samples taken while the GPU was busy (utilisation >= 50 %), all samples if there are none."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,utilization.gpu,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

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
        return self.parse(out)

    @staticmethod
    def parse(out):
        sm, busy, mx, pw, reasons = [], [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in out.strip().splitlines():
            f = [t.strip() for t in line.split(",")]
            if len(f) < 8:
                continue
            try:
                c, m, p = float(f[0]), float(f[1]), float(f[2])
            except ValueError:
                continue
            sm.append(c); mx.append(m); pw.append(p)
            try:
                if float(f[3]) >= 50.0:
                    busy.append(c)
            except ValueError:
                pass
            for nme, v in zip(names, f[4:8]):
                if v.lower().startswith("active"):
                    reasons.add(nme)
        use = busy if busy else sm
        return {"sm_mhz": float(np.median(use)) if use else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "samples_under_load": len(busy),
                "reasons": sorted(reasons), "window": "the whole GPU part of the run (all sections)"}


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


def timed(torch, fn, reps, warm=0):
    """mean device milliseconds of fn() over reps back-to-back calls on the current stream (CUDA events)"""
    for _ in range(warm):
        fn()
    a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize(); a0.record()
    for _ in range(reps):
        fn()
    a1.record(); torch.cuda.synchronize()
    return a0.elapsed_time(a1) / reps


def axhelm_sweep(torch, G, n, peak, lam_h, seed):
    """the stand-alone operator, Poisson (64 B/node) and Helmholtz (72 B/node), 20 timed applications after 5 warm-ups"""
    u = torch.from_numpy(I.uniform(seed, n)).cuda()
    w = torch.empty_like(u)
    out = {}
    for name, lam, nbytes in (("poisson", 0.0, B_AXHELM), ("helmholtz", lam_h, B_AXHELM_HELM)):
        t = timed(torch, lambda: G.apply_axhelm(u, w, lam=lam), 20, warm=5)
        gbs = nbytes * n / (t * 1e-3) / 1e9
        out[name] = {"ms": t, "gdofs": n / (t * 1e-3) / 1e9, "gbs": gbs, "frac_of_measured_peak": gbs / peak,
                     "frac_of_8TBs": gbs / 8000.0}
    del u, w
    return out


def iteration_numbers(torch, G, m, b, K, W, peak, precond=1, **kw):
    """K iterations of one semb_pcg_solve (rtol = 0: cannot stop early) after W warm-up iterations; CUDA events on the
    launching stream; the fused axhelm launches are bracketed by event pairs inside the solve (opts.profile)."""
    n = m.n
    x = torch.zeros_like(b)
    solve = dict(lam=0.0, tags=0b10, precond=precond, rtol=0.0, atol=0.0, **kw)
    if W > 0:
        G.pcg_solve(b, x, maxit=W, check_every=W, **solve)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize(); e0.record()
    st = G.pcg_solve(b, x, maxit=K, check_every=K, profile=True, **solve)
    e1.record(); torch.cuda.synchronize()
    assert st["iters"] == K, st
    ms = e0.elapsed_time(e1) / K
    b_iter = iter_bytes(m.N)
    gbs = b_iter * n / (ms * 1e-3) / 1e9
    ax_gbs = B_AXHELM_PCG * n / (st["axhelm_ms"] * 1e-3) / 1e9 if st["axhelm_ms"] > 0 else None
    del x
    return {"ms": ms, "iterations_timed": K, "model_bytes_per_node": b_iter, "gbs": gbs, "frac_of_measured_peak": gbs / peak,
            "frac_of_8TBs": gbs / 8000.0, "gdofs": n / (ms * 1e-3) / 1e9,
            "fused_axhelm": {"ms": st["axhelm_ms"], "bytes_per_node": B_AXHELM_PCG, "gbs": ax_gbs,
                             "frac_of_8TBs": ax_gbs / 8000.0 if ax_gbs else None, "share_of_iteration": st["axhelm_ms"] / ms},
            "launches_per_iteration": st["launches"] / K}


def time_to_solution(torch, G, b, variants, maxit):
    """full pressure solves to rtol 1e-10 on the same right-hand side (wall = device time around the call)"""
    out = {}
    for name, kw in variants:
        xs = torch.zeros_like(b)
        if kw.get("precond") == 3:
            G.pcg_solve(b, xs, lam=0.0, tags=0b10, rtol=1e-10, maxit=2, **kw)        # builds the levels, estimates the bounds
            xs.zero_()
        s0, s1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize(); s0.record()
        sst = G.pcg_solve(b, xs, lam=0.0, tags=0b10, rtol=1e-10, maxit=maxit, **kw)
        s1.record(); torch.cuda.synchronize()
        out[name] = {"iters": sst["iters"], "status": sst["status"], "seconds": s0.elapsed_time(s1) * 1e-3,
                     "rel_residual": sst["r_norm"] / sst["b_norm"]}
        del xs
    return out


def ten_steps(torch, G, m, nsteps, variants):
    """configs[4]: per time step one pressure Poisson solve + 3 velocity + 1 temperature Helmholtz solves (lambda = 1.5/dt =
    3000) through ONE semb_step_solve call, right-hand sides perturbed per step, warm starts from the previous step
    (R12).  nsteps <= 10 of the recipe's ten steps are run (the default bench run keeps to the first ones)."""
    n = m.n
    lam_h = 1.5 / 5e-4
    kinds = [(0.0, 0b10), (lam_h, 0b110), (lam_h, 0b110), (lam_h, 0b110), (lam_h, 0b10)]
    f0 = [I.divergence_source(m, I.seed_for(4, 30 + i)) for i in range(5)]
    rms = [float(np.sqrt(np.mean(v ** 2))) for v in f0]
    f0d = [torch.from_numpy(v).cuda() for v in f0]
    out = {"steps_run": nsteps, "of": 10, "solves_per_step": 5}
    for pname, pkw in variants:
        xs = [torch.zeros(n, dtype=torch.float64, device="cuda") for _ in range(5)]
        bs = [torch.empty(n, dtype=torch.float64, device="cuda") for _ in range(5)]
        secs, iters, rcs = [], [], 0
        for step in range(nsteps):
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
        out[pname] = {"seconds_per_step": secs, "seconds_per_step_mean": float(np.mean(secs)),
                      "seconds_per_step_after_first": float(np.mean(secs[1:])) if len(secs) > 1 else None,
                      "iterations_per_step": iters, "status": rcs,
                      "note": "step 1 includes building the multigrid levels and estimating their bounds" if pkw.get("precond") == 3 else ""}
        del xs, bs
    del f0d
    return out


def image_section(torch, semb, G, m, ms_step):
    """SURVEY.md §8 f-4 / PAPER.md:L371-373: the parts of the paper's overview scene as CUDA kernels on the exported
    temperature field, each a 4096 x 2048 image: two slices next to the walls, two vertical slices, one isocontour."""
    n = m.n
    T = torch.from_numpy((1.0 - m.z) + 0.05 * I.uniform(I.seed_for(3, 31), n)).cuda()
    G.publish_field("temperature", T)
    G.publish_state(1, 0.0)
    d = G.export_field("temperature")
    W, H = 4096, 2048
    key = torch.zeros(W * H, dtype=torch.int64, device="cuda"); rgba = torch.zeros(W * H, dtype=torch.int32, device="cuda")
    cw = [(59, 76, 192), (141, 176, 254), (221, 221, 221), (244, 154, 123), (180, 4, 38)]
    cm = semb.colormap(0.0, 1.0, cw)
    lo = [float(min(a.min() for a in (m.x, m.y))), float(m.z.min())]
    ext = float(max(m.x.max(), m.y.max())) - lo[0]
    views = {"slice_horizontal_lower_boundary_layer": semb.image_view(W, H, (lo[0], lo[0], 0.02), (1, 0, 0), (0, 1, 0), ext / W, ext / H),
             "slice_horizontal_upper_boundary_layer": semb.image_view(W, H, (lo[0], lo[0], 0.98), (1, 0, 0), (0, 1, 0), ext / W, ext / H),
             "slice_vertical_x": semb.image_view(W, H, (lo[0] + 0.5 * ext, lo[0], 0.0), (0, 1, 0), (0, 0, 1), ext / W, 1.0 / H),
             "slice_vertical_y": semb.image_view(W, H, (lo[0], lo[0] + 0.5 * ext, 0.0), (1, 0, 0), (0, 0, 1), ext / W, 1.0 / H)}
    out = {"pixels": [W, H]}
    total = 0.0
    for name, vw in views.items():
        t = timed(torch, lambda: G.image_slice(d, vw, cm, key, rgba), 5, warm=1)
        hit = int(((key >> 32) != 0xffffffff).sum().item())
        out[name] = {"ms": t, "pixels_hit": hit}
        total += t
    # isocontour T = 0.5 seen from above at an angle, coloured by the temperature
    u = np.array([1.0, 0.0, 0.0]); v = np.array([0.0, 0.8, 0.6]); w = np.cross(u, v)
    o = np.array([lo[0] - 0.1 * ext, lo[0] - 0.3 * ext, -0.2]) - 2.0 * w
    vw = semb.image_view(W, H, o, u, v, 1.2 * ext / W, 1.6 * ext / H, 0.0, 6.0)
    t = timed(torch, lambda: G.image_isosurface(d, 0.5, d, vw, cm, (0.0, 0.6, 0.8), key, rgba), 5, warm=1)
    out["isocontour_T_0.5"] = {"ms": t, "pixels_hit": int(((key >> 32) != 0xffffffff).sum().item())}
    total += t
    out["overview_scene_ms"] = total
    out["overhead_vs_pcg_iteration_pct"] = {str(nv): 100.0 * ((total + nv * ms_step) / (nv * ms_step) - 1.0) for nv in (10, 100, 1000)}
    out["note"] = ("five 4096 x 2048 partial images of the paper's overview scene (PAPER.md:L371: two wall slices, two vertical slices, one "
                   "isocontour) from the zero-copy exported field; the paper's ASCENT/VTK-m pipeline takes 4-5 s per part on 3360 A100 "
                   "(Table 5, L412-424: context, other hardware and a 350x larger mesh)")
    del T, key, rgba
    return out


def geometry_section(torch, semb, G3, m3, peak):
    """the same operator from fewer bytes.  (a) the float-stored factors on the cfg3 mesh (curved
    elements); (b) a 64^3, N = 7 box with tanh-stretched layers -- the paper's own mesh class, every
    element an affine brick -- applied from the stored factors, from 7 constants per element and from the trilinear
    coefficients; plus the Jacobi-PCG iteration on that mesh in the stored and the affine representation."""
    n = m3.n
    u = torch.from_numpy(I.uniform(I.seed_for(3, 1), n)).cuda(); w = torch.empty_like(u)
    out = {"note": "bytes_per_node = what the representation streams per node (u, w and the factors); modes 2, 3 are bound by the "
                   "SM (shared-memory transposes + fp64 pipe), not by HBM: their frac_of_8TBs is reported for the byte model only"}

    def sweep(G, label, byts):
        r = {}
        for nm, lam, bb in (("poisson", 0.0, byts[0]), ("helmholtz", 1e4, byts[1])):
            t = timed(torch, lambda: G.apply_axhelm(u, w, lam=lam), 20, warm=5)
            r[nm] = {"ms": t, "gdofs": n / (t * 1e-3) / 1e9, "bytes_per_node": bb, "gbs": bb * n / (t * 1e-3) / 1e9,
                     "frac_of_8TBs": bb * n / (t * 1e-3) / 8e12}
        out[label] = r
    G3.set_geometry_mode(1)
    sweep(G3, "cfg3_float_stored_factors", (40.0, 44.0))
    G3.set_geometry_mode(0)
    return out, u, w, sweep


def geometry_section_affine(torch, semb, out, u, w, sweep, peak):
    xi = semb.gll(7)[0]
    m = I.box_mesh(64, 64, 64, 7, xi, zstretch=2.0, name="box64_stretched_affine")
    x, y, z = (torch.from_numpy(a).cuda() for a in (m.x, m.y, m.z))
    G = semb.Mesh(m.E, m.N, x, y, z, m.face_tag, m.period)
    del x, y, z
    Np = 512.0
    sweep(G, "affine_box_stored", (64.0, 72.0))
    dev = G.set_geometry_mode(2)
    sweep(G, "affine_box_element_constants", (16.0 + 64.0 / Np, 16.0 + 64.0 / Np))
    f = torch.from_numpy(I.uniform(I.seed_for(3, 2), m.n)).cuda()
    b = torch.empty_like(f)
    G.assemble_rhs(f, b, 0b10)
    del f
    it2 = iteration_numbers(torch, G, m, b, 20, 3, peak)
    G.set_geometry_mode(3)
    sweep(G, "affine_box_trilinear_on_the_fly", (16.0 + 192.0 / Np, 16.0 + 192.0 / Np))
    G.set_geometry_mode(0)
    it0 = iteration_numbers(torch, G, m, b, 20, 3, peak)
    out["affine_box_jacobi_pcg_iteration_ms"] = {"stored": it0["ms"], "element_constants": it2["ms"],
                                                 "fused_axhelm_ms": {"stored": it0["fused_axhelm"]["ms"], "element_constants": it2["fused_axhelm"]["ms"]}}
    out["affine_box_measured_deviation_from_affine"] = dev[1]
    del b
    G.close()
    torch.cuda.empty_cache()
    return out


def boussinesq_section(torch, semb, G, m, nsteps):
    """configs[4] as a REAL time step (Eqs. (1)-(3)): no-slip walls, isothermal plates T(z=0) = 1,
    T(z=1) = 0, adiabatic side wall, started from the conduction state plus a seeded perturbation of theta,
    dt = 5e-4 (configs[4]), Ra = 1e8, Pr = 0.7; pressure by p-multigrid PCG on FP32 levels with Chebyshev-Schwarz smoothing, Helmholtz solves by Jacobi-PCG."""
    n = m.n
    st = semb.FlowState(n)
    th0 = torch.from_numpy(0.05 * I.uniform(I.seed_for(4, 7), n) * np.sin(np.pi * m.z)).cuda()
    G.gather_scatter(th0)                       # continuous start field: QQ^T, then the inverse multiplicity through a unit field
    ones = torch.ones(n, dtype=torch.float64, device="cuda"); G.gather_scatter(ones)
    th0.div_(ones); G.apply_mask(th0, 0b10)
    st.theta.copy_(th0)
    del th0, ones
    secs, its = [], []
    for s in range(nsteps):
        t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize(); t0.record()
        rc, it = G.boussinesq_step(st, 1e8, 0.7, 5e-4, 0b110, 0b10, rtol=1e-10, mg_fp32=True, mg_schwarz=True)
        t1.record(); torch.cuda.synchronize()
        secs.append(t0.elapsed_time(t1) * 1e-3); its.append(it)
    umax = max(float(c.abs().max()) for c in st.u)
    out = {"steps_run": nsteps, "seconds_per_step": secs, "iterations_per_step_p_ux_uy_uz_theta": its, "status": rc, "max_abs_velocity": umax,
           "points_per_second_per_gpu": n / secs[-1],
           "note": "one full Boussinesq step (explicit terms, curl-curl pressure Poisson with mean projection, 3 velocity + 1 temperature "
                   "Helmholtz solves); step 1 builds the multigrid levels and the metrics.  Paper context: 34-36 M points per second per "
                   "A100 for the whole NekRS step at p = 7, 9 (Table 4, L279-285; other hardware, other preconditioner)"}
    del st
    return out


def config_section(torch, semb, name, peak, args):
    """build -> 20 Jacobi-PCG iterations -> stand-alone axhelm -> time to solution (-> ten steps on cfg4) -> destroy"""
    m, G = build_problem(torch, semb, WORKLOADS[name])
    n = m.n
    cfg = WORKLOADS[name][1]
    f = torch.from_numpy(I.divergence_source(m, I.seed_for(cfg, 3))).cuda()
    b = torch.empty_like(f)
    G.assemble_rhs(f, b, 0b10)
    del f
    sec = {"E": m.E, "N": m.N, "local_nodes": n,
           "jacobi_pcg_iteration": iteration_numbers(torch, G, m, b, 20, 3, peak),
           "axhelm_sweep": axhelm_sweep(torch, G, n, peak, 1e4 if cfg == 2 else 3000.0, I.seed_for(cfg, 1))}
    if cfg == 2:
        sec["chebyshev2_jacobi_pcg_iteration_ms"] = iteration_numbers(torch, G, m, b, 20, 3, peak, precond=2, cheb_degree=2)["ms"]
    steps = None
    if not args.no_solve:
        variants = [("pmg_fp32_pcg", dict(precond=3, mg_fp32=True)),
                    ("pmg_fp32_schwarz_pcg", dict(precond=3, mg_fp32=True, mg_schwarz=True, mg_smooth=1, mg_kind=4))]
        if args.full_solves:
            variants += [("pmg_pcg", dict(precond=3)), ("jacobi_pcg", dict(precond=1))]
        sec["time_to_solution"] = time_to_solution(torch, G, b, variants, args.solve_maxit)
        if cfg == 4 and args.cfg4_steps > 0:
            sv = [("pmg_fp32_schwarz_pcg_all_solves", dict(precond=3, mg_fp32=True, mg_schwarz=True, mg_smooth=1, mg_kind=4))]
            if args.full_solves:
                sv += [("pmg_fp32_pcg_all_solves", dict(precond=3, mg_fp32=True)), ("jacobi_pcg_all_solves", dict(precond=1))]
            steps = ten_steps(torch, G, m, args.cfg4_steps, sv)
            sec["boussinesq_steps"] = boussinesq_section(torch, semb, G, m, 3)
    del b
    G.close()
    torch.cuda.empty_cache()
    return sec, steps


def export_section(torch, semb, G, m, ms_step):
    """one analysis step = publish_state + export of temperature and velocity magnitude + min/max/256-bin histogram of both"""
    n = m.n
    T = torch.from_numpy((1.0 - m.z) + 0.05 * I.uniform(I.seed_for(3, 31), n)).cuda()
    vel = [torch.from_numpy(3.0 * I.uniform(I.seed_for(3, 32 + c), n)).cuda() for c in range(3)]
    G.publish_field("temperature", T)
    for nm, t in zip(("velocity_x", "velocity_y", "velocity_z"), vel):
        G.publish_field(nm, t)
    mm = torch.zeros(2, dtype=torch.float64, device="cuda"); hist = torch.zeros(256, dtype=torch.int64, device="cuda")

    def analysis_step(cycle):
        G.publish_state(cycle, 1e-3 * cycle)                     # no kernel: nobody asked for the derived field's buffer
        dT = G.export_field("temperature")
        dv = [G.export_field(nm) for nm in ("velocity_x", "velocity_y", "velocity_z")]
        semb.field_minmax_hist(dT, 256, 0.0, 1.0, mm, hist)      # range given: one pass, 8 B/node
        semb.vector_magnitude_minmax_hist(dv[0], dv[1], dv[2], 256, 0.0, 5.2, mm, hist)   # |v| on the fly, range given: one pass, 24 B/node
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
    nbytes = (8 + 24) * n
    out = {"ms_per_analysis_step": t_an, "bytes_per_node": 32, "gbs": nbytes / (t_an * 1e-3) / 1e9,
           "pointer_identity": bool(dT.ptr == T.data_ptr()), "bytes_allocated": int(free0 - torch.cuda.mem_get_info()[0]),
           "overhead_vs_pcg_iteration_pct": {str(nv): 100.0 * ((t_an + nv * ms_step) / (nv * ms_step) - 1.0) for nv in (1, 10, 100)},
           "note": "min / max / 256-bin histogram of T (8 B/node) and of |v| computed on the fly from its components (24 B/node), each one "
                   "pass with a given range; overhead = (t_vis + (n_vis - 1) t_novis) / (n_vis t_novis) - 1 with t_vis = t_novis + analysis "
                   "step, t_novis = one PCG iteration (PAPER.md:L375)"}
    del T, vel
    return out


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
    line = {"impl": "reference", "metric": metric_name(7), "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
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
    ap.add_argument("--no-geometry", action="store_true", help="skip the geometry-representation section (row f-3)")
    ap.add_argument("--no-configs", action="store_true", help="skip the configs[2] / configs[4] O-grid sections")
    ap.add_argument("--cfg4-steps", type=int, default=2, help="how many of configs[4]'s ten time steps to run (default 2)")
    ap.add_argument("--full-solves", action="store_true", help="also run the fp64 p-multigrid and the Jacobi-PCG solves / steps on the O-grids")
    ap.add_argument("--solve-maxit", type=int, default=20000, help="iteration cap of the time-to-solution solves (profiling runs)")
    ap.add_argument("--no-solve", action="store_true", help="skip the time-to-solution sections (full pressure solves)")
    ap.add_argument("--record-traffic", default=None, metavar="RAW.csv", help="write profiles/r2_traffic.json from an `ncu --page raw --csv` dump and exit")
    ap.add_argument("--traffic-command", default="", help="the ncu command line the dump came from (stored in the record)")
    args = ap.parse_args()
    if args.record_traffic:
        return record_traffic(args)
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
    b_iter = iter_bytes(m.N)
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

    # ---- warm-up, then exactly K timed steps; the clock sampler runs from here to the end of the GPU sections
    sampler = ClockSampler(local)
    sampler.start()
    if W > 0:
        G.pcg_solve(b, x, maxit=W, check_every=W, **solve)
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    st = G.pcg_solve(b, x, maxit=K, check_every=K, profile=True, **solve)
    e1.record()
    barrier()
    ms = e0.elapsed_time(e1)
    assert st["iters"] == K, st
    ms, value = aggregate(ms, n, K, dist, "cuda")
    ms_step = ms / K
    ax_ms = st["axhelm_ms"]
    ax_gbs = B_AXHELM_PCG * n / (ax_ms * 1e-3) / 1e9
    single = world == 1

    # ---- axhelm alone, Poisson and Helmholtz (BASELINE.json configs[3] "roofline sweep"); not the headline
    sweep = axhelm_sweep(torch, G, n, peak, 1e4, I.seed_for(3, 1))

    # ---- what HBM delivers for a pure 7 : 1 read : write stream (axhelm's mix) and for a 1 : 1 copy, this device, this run
    ceiling = None
    if single:
        n_pr = min(n, 1 << 27) & ~1
        src = torch.empty(7 * n_pr, dtype=torch.float64, device="cuda").normal_()
        dst = torch.empty(n_pr, dtype=torch.float64, device="cuda")
        t7 = timed(torch, lambda: semb.stream_probe(src, dst, 7), 10, warm=3)
        t1 = timed(torch, lambda: semb.stream_probe(src, dst, 1), 10, warm=3)
        ceiling = {"read7_write1_gbs": 64.0 * n_pr / (t7 * 1e-3) / 1e9, "copy_gbs": 16.0 * n_pr / (t1 * 1e-3) / 1e9,
                   "note": "semb_stream_probe: dst = sum of 7 (1) input streams, one block per 16 KB tile, 128-bit loads, all issued before use, "
                           "bulk L2 prefetch 8 MB ahead (the axhelm kernels' memory schedule without their arithmetic)"}
        del src, dst

    # ---- time to solution of the pressure solve on the same mesh and right-hand side, rtol 1e-10: Jacobi-PCG (the
    #      north_star path) and the p-multigrid V-cycle preconditioner of PAPER.md:L102.
    solve_tts = None
    if not args.no_solve and single:
        variants = [("pmg_pcg", dict(precond=3, mg_smooth=1, mg_coarse=64, mg_coarse_frac=0.003)),
                    ("pmg_fp32_pcg", dict(precond=3, mg_smooth=1, mg_coarse=64, mg_coarse_frac=0.003, mg_fp32=True))]
        if isinstance(ne, tuple):
            variants = [("pmg_pcg", dict(precond=3)), ("pmg_fp32_pcg", dict(precond=3, mg_fp32=True)),
                        ("pmg_fp32_schwarz_pcg", dict(precond=3, mg_fp32=True, mg_schwarz=True, mg_smooth=1, mg_kind=4))]
        if args.full_solves:                  # ~4200 iterations, 14 s on cfg3: not in the default run
            variants.append(("jacobi_pcg", dict(precond=1)))
        solve_tts = time_to_solution(torch, G, b, variants, args.solve_maxit)
        if args.full_solves:
            solve_tts["speedup"] = solve_tts["jacobi_pcg"]["seconds"] / solve_tts["pmg_pcg"]["seconds"]
            solve_tts["speedup_fp32_levels"] = solve_tts["jacobi_pcg"]["seconds"] / solve_tts["pmg_fp32_pcg"]["seconds"]
        else:
            solve_tts["jacobi_pcg_seconds_at_the_measured_iteration_time"] = "iterations x ms_per_step; run with --full-solves to measure (4196 iterations, 13.97 s at r2 start)"

    # ---- configs[3]: zero-copy export of temperature and velocity magnitude to the in-device min/max/256-bin histogram
    #      consumer (PAPER.md:L138-159 hand-off; overhead formula of PAPER.md:L375 against the PCG iteration time)
    export = None
    if not args.no_export and single:
        export = export_section(torch, semb, G, m, ms_step)

    # ---- configs[1]: batched axhelm + gather-scatter on the 16^3 deformed box, Helmholtz lambda = 10/dt = 1e4, nfields = 3,
    #      100 applications timed.  Its working set (~150 MB + 3 x 2 x 17 MB) is about the size of the L2: reported, but no
    #      roofline claim is made from it.
    cfg1 = None
    if not args.no_cfg1 and single:
        m1, G1 = build_problem(torch, semb, 16)
        U = torch.from_numpy(I.uniform(I.seed_for(1, 1), 3 * m1.n)).cuda()
        Wv = torch.empty_like(U)

        def app():
            G1.apply_axhelm(U, Wv, lam=1e4, nfields=3); G1.gather_scatter(Wv, nfields=3)
        t1 = timed(torch, app, 100, warm=5)
        cfg1 = {"ms_per_application": t1, "nfields": 3, "local_nodes": m1.n, "gdofs": 3 * m1.n / (t1 * 1e-3) / 1e9,
                "note": "axhelm (72 B/node) + stand-alone gather-scatter on 3 fields; working set about the size of L2"}
        G1.close(); del U, Wv

    # ---- configs[0] (64 elements, N = 7, 32 768 nodes): the latency regime.  One persistent cooperative kernel runs the whole solve
    #      (csrc/pcg_persist.cu); SEMB_PCG_PERSIST=0 selects the launch-per-phase loop for comparison.
    cfg0 = None
    if not args.no_cfg1 and single:
        m0, _ = I.config_mesh(0, lambda N: semb.gll(N)[0])
        G0 = semb.Mesh(m0.E, m0.N, *(torch.from_numpy(a).cuda() for a in (m0.x, m0.y, m0.z)), m0.face_tag, m0.period)
        f0 = torch.from_numpy(I.uniform(I.seed_for(0, 2), m0.n)).cuda(); b0 = torch.empty_like(f0); G0.assemble_rhs(f0, b0, 0b10)
        x0 = torch.zeros_like(b0)
        cfg0 = {"local_nodes": m0.n, "elements": m0.E, "N": m0.N}
        for key, env in (("launch_per_phase", "0"), ("persistent_kernel", "1")):
            os.environ["SEMB_PCG_PERSIST"] = env
            G0.pcg_solve(b0, x0, tags=0b10, precond=1, rtol=0.0, maxit=20, check_every=20)
            x0.zero_()
            t0 = timed(torch, lambda: G0.pcg_solve(b0, x0, tags=0b10, precond=1, rtol=0.0, maxit=500, check_every=500), 1)
            x0.zero_()
            e0_, e1_ = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize(); e0_.record()
            st0 = G0.pcg_solve(b0, x0, tags=0b10, precond=1, rtol=1e-10, maxit=5000)
            e1_.record(); torch.cuda.synchronize()
            cfg0[key] = {"us_per_iteration": 1e3 * t0 / 500,
                         "solve_to_1e-10": {"iters": st0["iters"], "ms": e0_.elapsed_time(e1_), "launches": st0["launches"]}}
            x0.zero_()
        os.environ.pop("SEMB_PCG_PERSIST", None)
        G0.close(); del f0, b0, x0

    # ---- end to end through the C ABI with HOST buffers (pinned): b H2D, K iterations, x D2H
    e2e = e2e_single = None
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
               "d2h_bytes_per_step": 8 * n / K, "ms_total": hms,
               "note": "one call = b host->device, K iterations, x device->host: the two copies are amortised over K steps"}
        if single:
            # one axhelm application through semb_apply_axhelm_host: u from pinned host memory, w back to it, nothing amortised
            uh, wh = bh.numpy(), xh.numpy()
            G.apply_axhelm_host(uh, wh, lam=0.0)
            t0 = time.perf_counter()
            reps = 3
            for _ in range(reps):
                G.apply_axhelm_host(uh, wh, lam=0.0)
            dt = (time.perf_counter() - t0) / reps
            e2e_single = {"call": "semb_apply_axhelm_host", "seconds": dt, "gdofs": n / dt / 1e9, "h2d_bytes": 8 * n, "d2h_bytes": 8 * n,
                          "effective_copy_gbs": 16 * n / dt / 1e9,
                          "note": "ONE operator application with host buffers: bound by the two PCIe copies (8 B/node each way), "
                                  "the kernel itself is %.1f %% of the call" % (100.0 * sweep["poisson"]["ms"] * 1e-3 / dt)}
        del bh, xh

    # ---- the in-situ image consumer on the exported field
    images = None
    if single and not args.no_export:
        images = image_section(torch, semb, G, m, ms_step)

    # ---- reduced-traffic geometry representations (part on this mesh, part on an affine box built below)
    geo_modes = geo_state = None
    if single and not args.no_geometry and args.workload.startswith("cfg3"):
        geo_state = geometry_section(torch, semb, G, m, peak)

    # ---- configs[4] ten-step recipe when cfg4 IS the workload (otherwise inside the configs section below)
    steps10 = None
    if args.workload.startswith("cfg4") and not args.no_solve and single and args.cfg4_steps > 0:
        sv = [("pmg_fp32_schwarz_pcg_all_solves", dict(precond=3, mg_fp32=True, mg_schwarz=True, mg_smooth=1, mg_kind=4))]
        if args.full_solves:
            sv += [("pmg_fp32_pcg_all_solves", dict(precond=3, mg_fp32=True)), ("jacobi_pcg_all_solves", dict(precond=1))]
        steps10 = ten_steps(torch, G, m, args.cfg4_steps, sv)
    bq_main = None
    if args.workload.startswith("cfg4") and not args.no_solve and single:
        bq_main = boussinesq_section(torch, semb, G, m, 3)

    launches = st["launches"]
    del b, x
    G.close()
    torch.cuda.empty_cache()

    if geo_state is not None:
        geo_modes = geometry_section_affine(torch, semb, *geo_state, peak)
        geo_state = None

    # ---- the other configurations: O-grids of configs[2] and configs[4], each build -> measure -> destroy
    configs = None
    if single and not args.no_configs:
        configs = {}
        for name in ("cfg2_ogrid_N7", "cfg4_ogrid_N9"):
            if name == args.workload:
                continue
            sec, steps = config_section(torch, semb, name, peak, args)
            configs[name] = sec
            if steps is not None:
                steps10 = steps
    clocks = sampler.stop()

    traffic, traffic_src = recorded_traffic(args.workload)
    frac = ax_gbs / peak
    line = {
        "metric": metric_name(m.N), "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": args.workload, "E": m.E, "N": m.N, "local_nodes": n, "lambda": 0.0,
                   "parallelism": "replicas only" if world > 1 else "single GPU",
                   "l2": "inputs larger than L2 (every vector is %.2f GB)" % (8 * n / 1e9)},
        "roofline": {"bound": "hbm", "kernel": f"k_axhelm_line<{m.N + 1},4,*>: axhelm (Poisson) with the fused PCG prologue (x += alpha p, p = dinv r + beta p) and p.Ap epilogue",
                     "achieved": ax_gbs, "peak": peak, "unit": "GB/s", "frac": frac, "traffic": traffic, "traffic_source": traffic_src,
                     "peak_source": peak_src, "bytes_per_node": B_AXHELM_PCG, "ms": ax_ms, "timed_launches": st["profiled"],
                     "frac_of_8TBs": ax_gbs / 8000.0, "gdofs": n / (ax_ms * 1e-3) / 1e9,
                     "frac_of_stream_ceiling": ax_gbs / ceiling["read7_write1_gbs"] if ceiling else None,
                     "peak_is_a_ceiling": bool(frac <= 1.0),
                     "note": ("frac > 1: the 1:1 copy bandwidth in MEASURED_PEAKS.json is NOT an upper bound for this read-heavy kernel "
                              "(it pays a read/write bus turnaround per 16 bytes where this kernel pays one per 104); read frac_of_8TBs "
                              "(north_star's denominator) and frac_of_stream_ceiling instead") if frac > 1.0 else ""},
        "stream_ceiling": ceiling,
        "pcg_iter": {"ms": ms_step, "model_bytes_per_node": b_iter, "gbs": b_iter * n / (ms_step * 1e-3) / 1e9,
                     "frac_of_measured_peak": b_iter * n / (ms_step * 1e-3) / 1e9 / peak,
                     "frac_of_8TBs": b_iter * n / (ms_step * 1e-3) / 8e12},
        "axhelm_sweep": sweep,
        "time_to_solution": solve_tts,
        "export": export,
        "image_consumer": images,
        "cfg1_batched_axhelm_gs": cfg1,
        "cfg0_small_mesh_pcg": cfg0,
        "geometry_modes": geo_modes,
        "configs": configs,
        "cfg4_ten_steps": steps10,
        "boussinesq_steps": bq_main if bq_main is not None else (configs or {}).get("cfg4_ogrid_N9", {}).get("boussinesq_steps"),
        "e2e": e2e, "e2e_single": e2e_single, "gpu_launches": launches, "clocks": clocks,
    }
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        s = oracle_sample(60, 2)
        line["cpu_baseline"] = {"value": s["n"] * s["steps"] / s["seconds"] / 1e9, "unit": UNIT, "cores": s["cores"],
                                "kind": "oracle", "sample": s["sample"]}
    if rank == 0:
        print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
