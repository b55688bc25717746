#!/usr/bin/env python
"""bench.py — FP64 N=7 Ax+gs throughput on BASELINE.json config 2 (20x20x18 = 7200 hex elements, ~2.47 M points).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--leg headline|sweep|...]

A "step" is one pass of the whole hot path: w = QQ^T (D^T G D) u over the full mesh (sem_ax_gs through the C ABI).
metric  = Ax+gs GDOF/s with DOF = E N^3 (the paper's n); value = whole-job DOF/s with inputs resident in HBM.
e2e     = same metric with u copied from pinned host memory and w copied back inside every timed step (two lanes,
          each its own context and stream, take alternate steps so that H2D and D2H overlap on the full-duplex link).
roofline= the dominant kernel (the local Ax) timed alone with CUDA events: 64 B x nL algorithmic bytes per launch
          against the measured HBM copy bandwidth of MEASURED_PEAKS.json; DRAM bytes from the committed ncu capture
          (profiles/r2_dram_traffic.txt, steady state, --cache-control none) are printed beside the algorithmic bytes.
N > 1   = independent replicas, one per GPU (the path has no inter-GPU exchange in the headline; DESIGN.md Multi-GPU).
--impl reference times the CPU oracle (oracle/) on the host cores, rank 0 only.
--leg   the other evidence tables of profiles/ (one GPU): sweep (config 3), levels (config 4 + transfers + smoother),
        config5, proj, gs_many, fdm, peaks.  The default leg "headline" prints the driver's JSON line.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "Ax+gs GDOF/s (FP64, N=7, E=7200)"
UNIT = "GDOF/s"
WORKLOAD = "config2: 20x20x18=7200 hex, N=7, smooth deformation 0.05, stored G, u~U[-1,1] seed 0"
MIN_TIMED_STEPS = 1000          # BASELINE.json config 2: "1000 applications timed"; a 20-step region is a 1 ms sample


def measured_peak_gbs():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md)"


def ncu_traffic():
    """Per-launch DRAM bytes (read + write) per kernel from the committed steady-state ncu capture
    (profiles/r2_dram_traffic.txt: `kernel_key=bytes` lines), {} if the file is missing."""
    out = {}
    try:
        with open(os.path.join(ROOT, "profiles", "r2_dram_traffic.txt")) as f:
            for line in f:
                if "=" in line and not line.startswith("#"):
                    k, v = line.strip().split("=", 1)
                    out[k] = float(v)
    except Exception:
        pass
    return out


class ClockSampler:
    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_id: str):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", gpu_id, f"--query-gpu={self.FIELDS}",
                                       "--format=csv,noheader,nounits", "-lms", "20"], stdout=self.f,
                                      stderr=subprocess.DEVNULL)
        except Exception:
            self.p = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.p is None:
            return out
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except Exception:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.f:
            parts = [s.strip() for s in line.split(",")]
            if len(parts) < 7:
                continue
            try:
                sm.append(float(parts[0])); mx.append(float(parts[1])); pw.append(float(parts[2]))
            except ValueError:
                continue
            for nm, v in zip(names, parts[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        self.f.close()
        os.unlink(self.f.name)
        if sm:
            out.update(sm_mhz=float(np.median(sm)), sm_max_mhz=float(max(mx)), power_w_max=float(max(pw)),
                       reasons=sorted(reasons), samples=len(sm))
        return out


# ------------------------------------------------------------------------------------------------------------------
# The CPU oracle as a timed baseline.  ONE estimator for both the cpu_baseline object of our arm and the
# --impl reference arm: `warm` untimed applications, then `steps` applications timed as one region, mean per step.
# (Round 1 reported a median of 400 in one leg and a mean of 20 in the other and they were 2x apart.)
# ------------------------------------------------------------------------------------------------------------------
def oracle_ax_gs_timer(mesh, Es=None):
    import oracle
    oracle.build()
    from paper_2110_01716_b200 import inputs
    G, _, rc = oracle.geom_trilinear(mesh.vert, mesh.N)
    assert rc == 0
    u = inputs.field_uniform(mesh.gid, 0)
    gid = mesh.gid
    if Es is not None and Es < mesh.E:                  # bounded sample: the first Es elements of the same mesh
        G, u, gid = np.ascontiguousarray(G[:Es]), np.ascontiguousarray(u[:Es]), mesh.gid[:Es]
    om = oracle.Maps(gid)

    def run(warm, steps):
        for _ in range(warm):
            oracle.gs(oracle.ax(G, u, mesh.N).ravel(), om)
        t0 = time.perf_counter()
        for _ in range(steps):
            oracle.gs(oracle.ax(G, u, mesh.N).ravel(), om)
        return (time.perf_counter() - t0) / steps
    return run, oracle.num_threads()


def cpu_oracle_baseline(mesh, budget_s: float):
    """The oracle as it stands, timed on the host cores: full Ax+gs applications of config 2."""
    run, cores = oracle_ax_gs_timer(mesh)
    t1 = run(5, 5)                                              # 5 warm-up applications, then a first estimate
    steps = int(max(5, min(400, budget_s / max(t1, 1e-6))))
    t = run(0, steps)
    return {"value": mesh.dofs / t / 1e9, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"{steps} full Ax+gs applications of config 2 (all 7200 elements) after 10 warm-up applications, "
                      "mean per application (the same estimator as --impl reference)", "ms_per_step": t * 1e3}


def cpu_oracle_pcg_config5(n: int, iters: int = 5):
    """BASELINE.md's plan for config 5 on the CPU: the oracle's PCG timed for a few iterations, reported per iteration,
    on a down-sized replica of config 5 (n^3 elements instead of 100^3: the full size needs ~45 GB of host memory)."""
    import oracle
    oracle.build()
    from paper_2110_01716_b200 import inputs
    mesh = inputs.config5(n)
    G, _, rc = oracle.geom_trilinear(mesh.vert, mesh.N)
    assert rc == 0
    om = oracle.Maps(mesh.gid)
    mask_u = oracle.mask_unique(mesh.dirichlet, om)
    rng_b = inputs.field_uniform(mesh.gid, 5).ravel()
    b_u = np.zeros(om.U)
    b_u[om.l2u] = rng_b
    b_u[mask_u != 0] = 0.0
    oracle.pcg(G, mesh.N, om, mask_u, b_u, tol=1e-30, maxit=1)                 # warm-up
    t0 = time.perf_counter()
    oracle.pcg(G, mesh.N, om, mask_u, b_u, tol=1e-30, maxit=iters)
    dt = (time.perf_counter() - t0) / iters
    return {"iters_per_s": 1.0 / dt, "ms_per_iter": dt * 1e3, "elements": mesh.E, "cores": oracle.num_threads(),
            "kind": "oracle", "sample": f"{iters} PCG iterations of the oracle on a {n}^3-element replica of config 5 "
                                        f"({mesh.E} of 1 000 000 elements), mean per iteration incl. its setup pass",
            "scaled_to_config5_iters_per_s": 1.0 / dt * mesh.E / 1.0e6}


def run_reference(args):
    """--impl reference: the CPU oracle on the host cores (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    from paper_2110_01716_b200 import inputs
    mesh = inputs.config2()
    run, cores = oracle_ax_gs_timer(mesh)
    t_full = run(2, 2)
    total = args.steps + args.warmup
    budget = 150.0
    Es = mesh.E
    if total * t_full > budget:                       # bounded sample: the first Es elements of the same mesh
        Es = max(16, int(mesh.E * budget / (total * t_full)))
        run, cores = oracle_ax_gs_timer(mesh, Es)
    t = run(args.warmup, args.steps)
    val = Es * mesh.N ** 3 / t / 1e9
    sample = (f"each step = Ax+gs on the first {Es} of {mesh.E} elements of config 2; {args.warmup} warm-up steps, then "
              f"{args.steps} steps timed as one region, mean per step")
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": t * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": WORKLOAD, "sample": sample},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def max_over_ranks(ms: float, world: int, device: str) -> float:
    """Device time of a timed region for the whole job: the maximum over the ranks (replicas run independently)."""
    if world <= 1:
        return ms
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(units_per_rank_per_step: float, world: int, steps: int, ms: float) -> float:
    """Whole-job throughput in 1e9 units/s: every rank processed `units_per_rank_per_step` per step (weak scaling)."""
    return world * units_per_rank_per_step * steps / (ms * 1e-3) / 1e9


def event_time_us(torch, fn, reps, warm=3):
    """CUDA-event time per call in microseconds, on torch's current stream (the one every context here runs on)."""
    for _ in range(warm):
        fn()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record()
    for _ in range(reps):
        fn()
    e1.record()
    torch.cuda.synchronize()
    return e0.elapsed_time(e1) * 1e3 / reps


# ------------------------------------------------------------------------------------------------------------------
# config 5 (BASELINE.json configs[4]): the full Jacobi-PCG Poisson solve on n^3 elements (100^3 at full size)
# ------------------------------------------------------------------------------------------------------------------
def run_config5(torch, binding, inputs, n: int, peak: float, tol: float = 1e-8, maxit: int = 20000):
    """n^3 elements, N = 7, random +-10 % vertices (seed 3), scrambled element order (seed 4), homogeneous Dirichlet,
    b = M Q^T(B f), f = 3 pi^2 sin(pi x) sin(pi y) sin(pi z), Jacobi-PCG to `tol`; error against the analytic solution."""
    t0 = time.perf_counter()
    mesh = inputs.config5(n)
    t_mesh = time.perf_counter() - t0
    t0 = time.perf_counter()
    sem = binding.Sem(mesh.E, mesh.N, mesh.vert, mesh.gid, mesh.dirichlet)
    sem.geom(with_mass=True)
    torch.cuda.synchronize()
    t_setup = time.perf_counter() - t0
    cnt = sem.counts()
    nL, S = cnt["nL"], cnt["S"]
    # node coordinates on the device: trilinear blend of the element vertices at the GLL points (S5)
    xi = torch.from_numpy(sem.gll()[0]).cuda()
    p = mesh.p
    V = torch.from_numpy(mesh.vert).cuda()                                  # [E, 8, 3]
    w1 = torch.stack([(1 - xi) / 2, (1 + xi) / 2])                           # [2, p]
    exact = torch.ones(mesh.E, p, p, p, device="cuda", dtype=torch.float64)
    for d in range(3):                                                       # one coordinate at a time: 4 GB each
        xd = torch.zeros(mesh.E, p, p, p, device="cuda", dtype=torch.float64)
        for v in range(8):
            ia, ib, ic = v & 1, (v >> 1) & 1, (v >> 2) & 1
            wgt = w1[ic][:, None, None] * w1[ib][None, :, None] * w1[ia][None, None, :]
            xd += wgt[None] * V[:, v, d][:, None, None, None]
        exact *= torch.sin(np.pi * xd)
        del xd
    exact = exact.reshape(-1)
    # b = M Q Q^T (B f):  (A + 1 B) f - A f = B f with the library's own mass factor
    f = 3 * np.pi ** 2 * exact
    t1, t2 = torch.empty_like(f), torch.empty_like(f)
    sem.ax(f, t1, 1.0)
    sem.ax(f, t2, 0.0)
    t1 -= t2
    del t2, f
    sem.gs(t1)
    mask = torch.from_numpy(mesh.dirichlet.ravel()).cuda() != 0
    t1[mask] = 0.0
    del mask
    x = torch.zeros_like(t1)
    sem.pcg(t1, x, 1e-30, 3)                                                 # warm-up: allocates the work vectors
    x.zero_()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    it, rel = sem.pcg(t1, x, tol, maxit)
    torch.cuda.synchronize()
    dt = time.perf_counter() - t0
    err = float((x - exact).abs().max())
    bytes_it = (64.0 + 56.0 + 32.0) * nL + 16.0 * S
    out = {"workload": f"config5: {n}^3 = {mesh.E} hex, N=7, random +-10% vertices (seed 3), element order permuted "
                       f"(seed 4), Dirichlet, b = M Q^T(B f), Jacobi-PCG to {tol:g}",
           "E": mesh.E, "nL": nL, "U": cnt["U"], "S": S, "iters": it, "relres": rel, "solve_s": dt,
           "iters_per_s": it / dt, "ms_per_iter": dt / it * 1e3, "algorithmic_bytes_per_iter": bytes_it,
           "algorithmic_GBs": bytes_it * it / dt / 1e9, "frac_of_measured_peak": bytes_it * it / dt / 1e9 / peak,
           "max_err_vs_analytic": err, "mesh_s": t_mesh, "setup_s": t_setup,
           "timed": "wall clock around one sem_pcg call"}
    sem.close()
    # a9: the same iteration with the geometric factors recomputed in the operator (no 48 B per node of G traffic; the
    # operator is then bound by the FP64 pipe): 60 iterations from x = 0, ms per iteration only
    x.zero_()
    torch.cuda.empty_cache()
    sr = binding.Sem(mesh.E, mesh.N, mesh.vert, mesh.gid, mesh.dirichlet)
    sr.geom(mode=binding.SEM_G_RECOMPUTE, with_mass=True)
    sr.pcg(t1, x, 1e-30, 3)
    x.zero_()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    it_r, _ = sr.pcg(t1, x, 1e-30, 64)
    torch.cuda.synchronize()
    dt_r = time.perf_counter() - t0
    out["recomputed_G"] = {"ms_per_iter": dt_r / it_r * 1e3, "iters_timed": it_r, "speedup_vs_stored": (dt / it) / (dt_r / it_r),
                           "what": "SEM_G_RECOMPUTE: sem_ax = ax_dmma_rg (factors recomputed in registers from the 8 "
                                   "vertices, tensor-core contractions); no stored G (24.6 GB at 100^3)"}
    sr.close()
    del x, t1, exact
    torch.cuda.empty_cache()
    return out


# ------------------------------------------------------------------------------------------------------------------
# the other legs (evidence tables under profiles/); each prints markdown
# ------------------------------------------------------------------------------------------------------------------
def leg_sweep_case(torch, binding, inputs, mesh, dtype, peak, fp_peak, label):
    esize = 8 if dtype == torch.float64 else 4
    u = torch.from_numpy(inputs.field_uniform(mesh.gid, 1).ravel()).cuda().to(dtype)
    w = torch.empty_like(u)
    row = {}
    for mode in (binding.SEM_G_STORED, binding.SEM_G_RECOMPUTE):
        with binding.Sem(mesh.E, mesh.N, mesh.vert, mesh.gid) as sem:
            sem.geom(mode=mode)
            cnt = sem.counts()
            nL, S = cnt["nL"], cnt["S"]
            reps = max(20, min(2000, int(2e9 / (nL * 64))))
            t_ax = event_time_us(torch, lambda: sem.ax(u, w), reps)
            if mode == binding.SEM_G_STORED:
                t_gs = event_time_us(torch, lambda: sem.gs(w), reps)
                t_axgs = event_time_us(torch, lambda: sem.ax_gs(u, w), reps)
                b_ax = 8.0 * esize * nL
                row.update(nL=nL, S=S, ax=t_ax, gs=t_gs, axgs=t_axgs, ax_gbs=b_ax / t_ax / 1e3,
                           axgs_gbs=(b_ax + 2.0 * esize * S) / t_axgs / 1e3, gdofs=mesh.dofs / t_axgs / 1e3)
            else:
                row.update(ax_re=t_ax, re_tflops=(12 * mesh.p + 15 + 125) * nL / t_ax / 1e6)
    print(f"| {label} | {mesh.E} | {mesh.N} | {row['nL']} | {row['ax']:.1f} | {row['ax_gbs']:.0f} | "
          f"{row['ax_gbs'] / peak:.2f} | {row['gs']:.1f} | {row['axgs']:.1f} | {row['axgs_gbs']:.0f} | "
          f"{row['axgs_gbs'] / peak:.2f} | {row['gdofs']:.1f} | {row['ax_re']:.1f} | {row['re_tflops']:.1f} | "
          f"{row['re_tflops'] / fp_peak:.2f} |", flush=True)


def run_leg(args):
    import torch

    from paper_2110_01716_b200 import binding, build, inputs
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(0)
    torch.cuda.set_stream(torch.cuda.Stream())
    build.build()
    binding.lib()
    peak, _ = measured_peak_gbs()
    leg = args.leg
    if leg == "ncu":
        # a short eager run for ncu captures (profiles/): the legacy default stream cannot be captured, so every
        # sem_ax_gs is two plain kernel launches; 30 applications at config 2, then 10 PCG iterations
        torch.cuda.set_stream(torch.cuda.default_stream())
        mesh = inputs.config2()
        with binding.Sem(mesh.E, mesh.N, mesh.vert, mesh.gid, mesh.dirichlet) as sem:
            sem.geom(mode=args.gmode)                # --gmode 1: the recomputed-G operator (a9)
            sem.set_variant(args.variant)
            u = torch.from_numpy(inputs.field_uniform(mesh.gid, 0).ravel()).cuda()
            w = torch.empty_like(u)
            for _ in range(30):
                sem.ax_gs(u, w)
            x = torch.zeros_like(u)
            sem.pcg(w, x, 1e-30, 10)
            torch.cuda.synchronize()
        print("ncu leg done")
        return
    if leg == "peaks":
        for k, name in ((0, "FP64 FMA"), (1, "FP32 FMA"), (2, "FP64 DMMA m8n8k4")):
            print(f"{name}: {binding.measure_peak(k):.2f} TFLOP/s")
        return
    if leg == "config5":
        print(json.dumps(run_config5(torch, binding, inputs, args.config5_n, peak)))
        return
    if leg in ("sweep", "levels"):
        fp64, fp32 = binding.measure_peak(0), binding.measure_peak(1)
        print(f"HBM peak = {peak:.0f} GB/s (MEASURED_PEAKS.json hbm_gbs, else the profiling guide's fallback); "
              f"FP64 FMA peak = {fp64:.1f} TFLOP/s, FP32 = {fp32:.1f} TFLOP/s (sem_measure_peak, this run)")
        print("| case | E | N | nL | Ax us | Ax GB/s | frac of HBM peak | gs us | Ax+gs us | Ax+gs GB/s | Ax+gs frac | "
              "GDOF/s (E N^3) | Ax recomputed-G us | recomputed TFLOP/s | frac of FMA peak |")
        print("|---|---|---|---|---|---|---|---|---|---|---|---|---|---|---|")
        if leg == "sweep":
            for N in [int(x) for x in args.orders.split(",")]:
                n = 8
                while n <= args.max_n:
                    leg_sweep_case(torch, binding, inputs, inputs.config3(n, N), torch.float64, peak, fp64,
                                   f"cfg3 {n}^3 f64")
                    n *= 2
            return
        for N in (7, 3, 1):
            leg_sweep_case(torch, binding, inputs, inputs.config4(N), torch.float32, peak, fp32, "cfg4 20x20x18 f32")
        print()
        print("| transfer (FP32, E = 7200) | us | GB/s | frac of peak |")
        print("|---|---|---|---|")
        sems = {N: binding.Sem(m.E, N, m.vert, m.gid) for N, m in ((N, inputs.config4(N)) for N in (7, 3, 1))}
        for Nc, Nf in ((3, 7), (1, 3)):
            sc, sf = sems[Nc], sems[Nf]
            vc = torch.randn(sc.nL, device="cuda", dtype=torch.float32)
            vf = torch.randn(sf.nL, device="cuda", dtype=torch.float32)
            for name, fn in ((f"prolong {Nc}->{Nf}", lambda: sc.transfer(sf, vc, vf, binding.SEM_PROLONG)),
                             (f"restrict {Nf}->{Nc}", lambda: sc.transfer(sf, vf, vc, binding.SEM_RESTRICT))):
                t = event_time_us(torch, fn, 2000)
                gbs = 4.0 * (sc.nL + sf.nL) / t / 1e3
                print(f"| {name} | {t:.2f} | {gbs:.0f} | {gbs / peak:.2f} |", flush=True)
        print()
        print("| smoother (FP32, E = 7200, zero guess) | us | us per operator application |")
        print("|---|---|---|")
        for N in (7, 3, 1):
            m = inputs.config4(N)
            with binding.Sem(m.E, N, m.vert, m.gid, m.dirichlet) as sd:
                sd.geom()
                b = torch.randn(sd.nL, device="cuda", dtype=torch.float32)
                x = torch.zeros_like(b)
                for order in (2, 4):
                    t = event_time_us(torch, lambda: sd.cheby(b, x, order, 0.2, 2.2, True), 500)
                    print(f"| N = {N}, order {order} | {t:.1f} | {t / (order - 1):.1f} |", flush=True)
        for s_ in sems.values():
            s_.close()
        return
    if leg == "proj":
        mesh = inputs.config2()
        with binding.Sem(mesh.E, mesh.N, mesh.vert, mesh.gid, mesh.dirichlet) as sem:
            sem.geom()
            nL = sem.nL
            fields = [torch.from_numpy(inputs.field_uniform(mesh.gid, 40 + k).ravel()).cuda() for k in range(4)]
            rhs = [torch.empty_like(fields[0]) for _ in range(4)]
            for f_, r_ in zip(fields, rhs):
                sem.ax_gs(f_, r_)
            xbar, bred, x = (torch.empty_like(rhs[0]) for _ in range(3))
            print("| step | PCG iterations without projection | with projection (L) | reduced / full right-hand side norm |")
            print("|---|---|---|---|")
            with binding.Proj(sem, 30) as pj:
                for m_ in range(12):
                    t = 0.05 * m_
                    b = rhs[0] + t * rhs[1] + t * t * rhs[2] + np.sin(3 * t) * 0.1 * rhs[3]
                    it0, _ = sem.pcg(b, x.zero_(), 1e-8, 5000)
                    pj.guess(b, xbar, bred)
                    ratio = float(bred.norm() / b.norm())
                    it1, _ = sem.pcg(bred, x.zero_(), 1e-8 * float(b.norm() / max(float(bred.norm()), 1e-300)), 5000)
                    L_before = pj.size()
                    pj.update(x)
                    print(f"| {m_} | {it0} | {it1} ({L_before}) | {ratio:.2e} |", flush=True)
            with binding.Proj(sem, 30) as pj:
                for k in range(30):
                    pj.update(torch.from_numpy(inputs.field_uniform(mesh.gid, 200 + k).ravel()).cuda())
                assert pj.size() == 30
                t_g = event_time_us(torch, lambda: pj.guess(rhs[0], xbar, bred), 50)
                gb = 8.0 * nL * (31 + 61 + 2) / t_g / 1e3
                print(f"\nsem_proj_guess with L = 30 at config 2: {t_g:.0f} us = {gb:.0f} GB/s ({gb / peak:.2f} of peak; "
                      f"31 vectors read by the multi-dot, 61 read + 2 written by the update pass)")
        return
    if leg == "gs_many":
        mesh = inputs.config2()
        print("| fields | precision | sem_gs x fields us | sem_gs_many us | speed-up |")
        print("|---|---|---|---|---|")
        with binding.Sem(mesh.E, mesh.N, mesh.vert, mesh.gid) as sem:
            for dt, name in ((torch.float64, "FP64"), (torch.float32, "FP32")):
                for nf in (2, 3, 4, 6):
                    w = torch.randn(nf, sem.nL, device="cuda", dtype=dt)

                    def separate():
                        for f in range(nf):
                            sem.gs(w[f])
                    t1 = event_time_us(torch, separate, 300)
                    t2 = event_time_us(torch, lambda: sem.gs_many(w), 300)
                    print(f"| {nf} | {name} | {t1:.1f} | {t2:.1f} | {t1 / t2:.2f} |", flush=True)
        return
    if leg == "fdm":
        fp = {torch.float32: binding.measure_peak(1), torch.float64: binding.measure_peak(0)}
        print("| E | m | precision | us | GB/s | frac of HBM peak | TFLOP/s | frac of FMA peak |")
        print("|---|---|---|---|---|---|---|---|")
        for E, m in ((7200, 10), (7200, 8), (7200, 7), (7200, 6), (7200, 5), (7200, 4), (7200, 12), (3573, 11),
                     (3573, 9), (3573, 7)):
            mesh = inputs.box_mesh(E, 1, 1, 1)
            with binding.Sem(mesh.E, 1, mesh.vert, mesh.gid) as sem:
                sem.set_variant(args.variant if args.variant >= 100 else 100)      # 101: the FP32 tensor-core kernel
                A, B = inputs.fdm_pairs(E, m, 7)
                S, invL = binding.fdm_setup(A, B)
                for dt, name in ((torch.float32, "FP32"), (torch.float64, "FP64")):
                    dS, dL = (torch.from_numpy(a.ravel()).cuda().to(dt) for a in (S, invL))
                    b = torch.randn(E * m ** 3, device="cuda", dtype=dt)
                    u = torch.empty_like(b)
                    t = event_time_us(torch, lambda: sem.fdm_apply(m, dS, dL, b, u), 500)
                    nbytes = b.element_size() * E * (3 * m ** 3 + 3 * m * m)
                    tf = 12.0 * m ** 4 * E / t / 1e6
                    print(f"| {E} | {m} | {name} | {t:.2f} | {nbytes / t / 1e3:.0f} | {nbytes / t / 1e3 / peak:.2f} | "
                          f"{tf:.2f} | {tf / fp[dt]:.2f} |", flush=True)
        return
    raise SystemExit(f"unknown --leg {leg}")


def run_sharded(args):
    """--sharded-n n: NEXT-4, operator and Jacobi-PCG with the ELEMENTS partitioned over the ranks (contiguous blocks of
    a config-5 style mesh of n^3 elements, scrambled order unless --sharded-lex), interface exchange and all-reduces
    through the hooks of paper_2110_01716_b200/sharded.py.  Strong scaling: the total work is fixed.  Not the default
    multi-GPU mode (north_star scopes the headline to replicas).  Under torchrun: one rank per GPU over NCCL.  With
    --emulate-ranks R (one process, one GPU): R ranks on R host threads sharing the GPU, which serialises them -- the
    time is the SUM over ranks and shows what the partition costs (split launches, pack / add kernels, hook calls)
    against the single-context call on the same mesh, not a speed-up."""
    import torch
    import torch.distributed as dist

    from paper_2110_01716_b200 import binding, build, inputs, sharded
    emu = args.emulate_ranks
    world = emu if emu > 0 else int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    if emu == 0:
        if not dist.is_initialized():
            if world == 1:
                os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
                os.environ.setdefault("MASTER_PORT", "29531")
            dist.init_process_group("nccl", rank=rank, world_size=world, device_id=torch.device("cuda", local))
        if rank == 0:
            build.build()
        dist.barrier()
    else:
        build.build()
    n = args.sharded_n
    mesh = inputs.box_mesh(n, n, n, 7, "random", seed=3, name=f"lex{n}") if args.sharded_lex else inputs.config5(n)
    # the scrambled order has no locality: contiguous blocks would put every element on the interface -> bisection
    part = ([np.arange(lo, hi) for lo, hi in zip(sharded.partition_bounds(mesh.E, world)[:-1],
                                                 sharded.partition_bounds(mesh.E, world)[1:])]
            if args.sharded_lex else sharded.partition_rcb(mesh.vert, world))
    K, W = max(args.steps, 20), max(args.warmup, 3)
    pcg_its = 50
    side = torch.cuda.Stream()
    torch.cuda.set_stream(side)

    def make(r, comm):
        sl = part[r]
        sh = sharded.ShardedSem(comm, len(sl), mesh.N, mesh.vert[sl], mesh.gid[sl], mesh.dirichlet[sl],
                                stream=side).geom()
        u = torch.from_numpy(sh.to_local(inputs.field_uniform(mesh.gid[sl], 0)).ravel()).cuda()
        return sh, u, torch.empty_like(u), torch.zeros_like(u)

    def timed(fn):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        if emu == 0:
            dist.barrier()
            torch.cuda.synchronize()
        e0.record(side)
        fn()
        e1.record(side)
        torch.cuda.synchronize()
        return e0.elapsed_time(e1)

    if emu > 0:
        gath = sharded.local_gathers(mesh.N, [mesh.gid[part[r]] for r in range(world)],
                                     [mesh.dirichlet[part[r]] for r in range(world)])
        tw = sharded.ThreadWorld(world, timeout=600.0)
        parts = [make(r, sharded.ThreadComm(tw, r, *gath)) for r in range(world)]

        def apply_all(k):
            sharded.run_ranks(world, lambda r: [parts[r][0].ax_gs(parts[r][1], parts[r][2]) for _ in range(k)], tw)

        def pcg_all():
            return sharded.run_ranks(world, lambda r: parts[r][0].pcg(parts[r][1], parts[r][3].zero_(), 1e-30, pcg_its), tw)

        apply_all(W)
        ms = timed(lambda: apply_all(K))
        pcg_all()
        ms_pcg = timed(pcg_all)
        with binding.Sem(mesh.E, mesh.N, mesh.vert, mesh.gid, mesh.dirichlet, stream=side) as one:
            one.geom()
            u1 = torch.from_numpy(inputs.field_uniform(mesh.gid, 0).ravel()).cuda()
            w1, x1 = torch.empty_like(u1), torch.zeros_like(u1)
            for _ in range(W):
                one.ax_gs(u1, w1)
            ms_one = timed(lambda: [one.ax_gs(u1, w1) for _ in range(K)])
            one.pcg(u1, x1, 1e-30, pcg_its)
            ms_pcg_one = timed(lambda: one.pcg(u1, x1.zero_(), 1e-30, pcg_its))
        shs = [p[0] for p in parts]
        ib = float(sum(s.interface_bytes() for s in shs))
        extra = {"emulated_ranks_on_one_gpu": world, "time_is": "sum over ranks (they share the GPU)",
                 "single_context_ms_per_step": ms_one / K, "single_context_pcg_ms_per_iter": ms_pcg_one / pcg_its,
                 "interface_elements_per_rank": [s.n_iface for s in shs], "elements_per_rank": [s.E for s in shs],
                 "chunks_per_rank": [len(s.sem.chunks()[0]) - 1 for s in shs]}
        launches = K * sum(2 * (len(s.sem.chunks()[0]) - 1) + 2 * len(s.uniq) for s in shs)
    else:
        sh, u, w, x = make(rank, sharded.DistComm())
        for _ in range(W):
            sh.ax_gs(u, w)
        ms = max_over_ranks(timed(lambda: [sh.ax_gs(u, w) for _ in range(K)]), world, "cuda")
        sh.pcg(u, x, 1e-30, pcg_its)
        ms_pcg = max_over_ranks(timed(lambda: sh.pcg(u, x.zero_(), 1e-30, pcg_its)), world, "cuda")
        t = torch.tensor([sh.interface_bytes()], device="cuda", dtype=torch.float64)
        dist.all_reduce(t)
        ib = float(t.item())
        shs = [sh]
        extra = {"interface_elements_this_rank": sh.n_iface, "elements_this_rank": sh.E}
        launches = K * (2 * (len(sh.sem.chunks()[0]) - 1) + 2 * len(sh.uniq))
    if rank == 0:
        print(json.dumps({
            "metric": "Ax+gs GDOF/s (FP64, N=7), elements partitioned over the ranks", "value": mesh.dofs * K / (ms * 1e-3) / 1e9,
            "unit": UNIT, "n_gpus": 1 if emu else world, "steps": K, "warmup": W, "ms_per_step": ms / K, "higher_is_better": True,
            "scaling": "strong", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"{'lexicographic' if args.sharded_lex else 'config5-style scrambled'} {n}^3 hex, N=7, "
                                   "random +-10 % vertices, Dirichlet; "
                                   f"{'contiguous element blocks' if args.sharded_lex else 'coordinate bisection'} per rank, interface "
                                   "elements first, exchange started after the interface chunk",
                       "E": mesh.E, "interface_bytes_sent_per_step_all_ranks": ib, **extra},
            "pcg_sharded": {"iters": pcg_its, "ms_per_iter": ms_pcg / pcg_its, "allreduces_per_iter": 2},
            "gpu_launches": launches}))
    for s in shs:
        s.close()
    if emu == 0:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5000)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--leg", default="headline",
                    choices=["headline", "sweep", "levels", "config5", "proj", "gs_many", "fdm", "peaks", "ncu"])
    ap.add_argument("--e2e-steps", type=int, default=50)
    ap.add_argument("--cpu-seconds", type=float, default=12.0)
    ap.add_argument("--variant", type=int, default=0)
    ap.add_argument("--gmode", type=int, default=0, help="--leg ncu: 0 = stored G, 1 = SEM_G_RECOMPUTE")
    ap.add_argument("--pcg-iters", type=int, default=300)
    ap.add_argument("--config5-n", type=int, default=100, help="elements per direction of the config-5 leg (0 = skip)")
    ap.add_argument("--emulate-ranks", type=int, default=0,
                    help="with --sharded-n, one process: this many ranks on host threads sharing one GPU")
    ap.add_argument("--sharded-lex", action="store_true", help="with --sharded-n: lexicographic element order (slabs)")
    ap.add_argument("--sharded-n", type=int, default=0,
                    help="NEXT-4: > 0 runs the element-partitioned operator on a config-5 style mesh of n^3 elements")
    ap.add_argument("--max-n", type=int, default=64)
    ap.add_argument("--orders", default="3,5,7,8,9")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    if args.sharded_n > 0:
        return run_sharded(args)
    if args.leg != "headline":
        return run_leg(args)
    args.warmup = max(args.warmup, 3)

    import torch
    import torch.distributed as dist

    from paper_2110_01716_b200 import binding, build, inputs

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    # a non-default stream: repeated sem_ax_gs calls and the V-cycle replay CUDA graphs, which the legacy default stream
    # cannot record; every context created below runs on it and the timing events are recorded on it
    torch.cuda.set_stream(torch.cuda.Stream())
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    if rank == 0:
        build.build()
    if world > 1:
        dist.barrier()
    binding.lib()

    mesh = inputs.config2()
    sem = binding.Sem(mesh.E, mesh.N, mesh.vert, mesh.gid)
    sem.geom()
    sem.set_variant(args.variant)
    cnt = sem.counts()
    nL, S = cnt["nL"], cnt["S"]
    u = torch.from_numpy(inputs.field_uniform(mesh.gid, 0).ravel()).cuda()
    w = torch.empty_like(u)
    # The headline region is never shorter than BASELINE.json's 1000 applications: the driver's --steps 20 would be a
    # 1 ms sample (round 1: 56.5 us per step at 20 steps against 53.4 us at 5000).  `steps` in the line is what was timed.
    K, W = max(args.steps, MIN_TIMED_STEPS), max(args.warmup, 50)

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    def timed(fn, steps, side_streams=()):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        e0.record()
        for s_ in side_streams:
            s_.wait_event(e0)
        for j in range(steps):
            fn(j) if side_streams else fn()
        for s_ in side_streams:                      # the end event must come after the work of every lane
            torch.cuda.current_stream().wait_stream(s_)
        e1.record()
        barrier()
        return max_over_ranks(e0.elapsed_time(e1), world, "cuda")

    for _ in range(W):
        sem.ax_gs(u, w)
    try:
        gpu_id = str(torch.cuda.get_device_properties(local).uuid)
        gpu_id = gpu_id if gpu_id.startswith("GPU-") else "GPU-" + gpu_id
    except Exception:
        gpu_id = str(local)
    sampler = ClockSampler(gpu_id) if rank == 0 else None
    time.sleep(0.05)
    # ---- the metric: K applications of the whole path, inputs resident in HBM ----
    ms_total = timed(lambda: sem.ax_gs(u, w), K)
    # ---- kernel shares: the local operator alone, the gather-scatter alone ----
    # (bursts of 500 launches: MEASURED_PEAKS.json's hbm_gbs is a burst figure, "best of 10", and 5000 launches of one
    # kernel alone run into the power cap, which the whole-step loop above already reflects)
    Kk = 500
    ms_ax = timed(lambda: sem.ax(u, w), Kk)
    wz = torch.zeros_like(u)
    ms_gs = timed(lambda: sem.gs(wz), Kk)
    clocks = sampler.stop() if sampler else None

    # ---- e2e: host buffers, H2D of u and D2H of w inside every timed step.  Two lanes (context + stream + device
    # buffers each) take alternate steps, so one lane's H2D overlaps the other's D2H on the full-duplex link; every step
    # still copies its own input in and its own result out.
    Ke = max(2, min(args.e2e_steps, K))
    u_h = torch.from_numpy(inputs.field_uniform(mesh.gid, 0).ravel()).pin_memory()
    lanes = []
    for _ in range(2):
        st_ = torch.cuda.Stream()
        with torch.cuda.stream(st_):
            sl = binding.Sem(mesh.E, mesh.N, mesh.vert, mesh.gid)
            sl.geom()
        lanes.append((st_, sl, torch.empty_like(u), torch.empty_like(u), torch.empty_like(u_h).pin_memory()))

    def e2e_step(j):
        st_, sl, ud, wd, wh = lanes[j % 2]
        with torch.cuda.stream(st_):
            ud.copy_(u_h, non_blocking=True)
            sl.ax_gs(ud, wd)
            wh.copy_(wd, non_blocking=True)

    for j in range(4):
        e2e_step(j)
    ms_e2e = timed(e2e_step, Ke, side_streams=[l[0] for l in lanes])
    sem.ax_gs(u, w)                                  # the device-resident path's result for the same input
    torch.cuda.synchronize()
    e2e_ok = bool(torch.equal(lanes[0][4], lanes[1][4]) and torch.equal(lanes[0][4], w.cpu()))
    w_h = lanes[0][4]
    for l in lanes:
        l[1].close()
    extras = rank == 0 and world == 1 and args.pcg_iters > 0
    peak, peak_src = measured_peak_gbs()

    # ---- PCG iterations/s (second half of BASELINE.json's metric): config 2 with the Dirichlet mask, fixed count ----
    pcg = None
    if extras:
        semd = binding.Sem(mesh.E, mesh.N, mesh.vert, mesh.gid, mesh.dirichlet)
        semd.geom()
        rhs = torch.empty_like(u)
        semd.ax_gs(u, rhs)                               # an assembled, masked right-hand side
        x = torch.zeros_like(u)
        semd.pcg(rhs, x, 1e-30, 20)                      # warm-up (allocates the work vectors)
        x.zero_()
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        nit, rel = semd.pcg(rhs, x, 1e-30, args.pcg_iters)
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        # Ax 64 + gs 16 S/nL + update 56 + direction 32 bytes per local node per iteration
        pcg_bytes = (64.0 + 56.0 + 32.0) * nL + 16.0 * S
        pcg = {"iters_per_s": nit / dt, "us_per_iter": dt / nit * 1e6, "iters": nit, "relres": rel,
               "algorithmic_GBs": pcg_bytes * nit / dt / 1e9,
               "frac_of_measured_peak": pcg_bytes * nit / dt / 1e9 / peak,
               "timed": "wall clock around one sem_pcg call (host polls a device flag every 16 iterations)"}
        semd.close()

    # ---- NEXT-1: the same Poisson problem solved to 1e-8 by Jacobi-PCG and by flexible PCG + FP32 p-multigrid V-cycle
    solve = None
    if extras:
        side = torch.cuda.Stream()                       # the V-cycle replays a CUDA graph on a non-default stream
        with torch.cuda.stream(side):
            lv = []
            for N in (7, 3, 1):
                mN = inputs.config4(N)
                sN = binding.Sem(mN.E, N, mN.vert, mN.gid, mN.dirichlet)
                sN.geom()
                lv.append(sN)
            lam = [1.1 * s_.lambda_max(30) for s_ in lv]
            rhs = torch.empty_like(u)
            lv[0].ax_gs(u, rhs)
            x = torch.zeros_like(u)

            def wall(fn):
                side.synchronize()
                t0 = time.perf_counter()
                out = fn()
                side.synchronize()
                return out, (time.perf_counter() - t0) * 1e3

            with binding.Pmg(lv, [0.1 * l for l in lam], lam, 2, 8, binding.SEM_F32) as mg:
                mg.fpcg(rhs, x, 1e-8, 3)                 # warm-up: allocations, graph capture
                (it_m, rel_m), ms_m = wall(lambda: mg.fpcg(rhs, x, 1e-8, 200))
                # NEXT-2b: the same cycle with Chebyshev-accelerated overlapping Schwarz smoothing on N = 7 and N = 3
                t0 = time.perf_counter()
                for s_ in lv[:2]:
                    s_.schwarz_setup()
                ms_setup = (time.perf_counter() - t0) * 1e3
                lams = [1.1 * lv[0].lambda_max_schwarz(0, 30), 1.1 * lv[1].lambda_max_schwarz(0, 30), lam[2]]
                mg.set_smoother(binding.SEM_SMOOTH_CHEBY_SCHWARZ, [0.1 * l for l in lams], lams)
                mg.fpcg(rhs, x, 1e-8, 3)
                (it_s, rel_s), ms_s = wall(lambda: mg.fpcg(rhs, x, 1e-8, 200))
                # the restricted variant: one fused kernel per application, no exchange after the local solve
                lamr = [1.1 * lv[0].lambda_max_schwarz(1, 30), 1.1 * lv[1].lambda_max_schwarz(1, 30), lam[2]]
                mg.set_smoother(binding.SEM_SMOOTH_CHEBY_RAS, [0.1 * l for l in lamr], lamr)
                mg.fpcg(rhs, x, 1e-8, 3)
                (it_r, rel_r), ms_r = wall(lambda: mg.fpcg(rhs, x, 1e-8, 200))
            # Schwarz is the stronger smoother: one Chebyshev step per smoothing (order 1) is its best cycle here
            with binding.Pmg(lv, [0.1 * l for l in lam], lam, 1, 16, binding.SEM_F32) as mg1:
                mg1.set_smoother(binding.SEM_SMOOTH_CHEBY_RAS, [0.1 * l for l in lamr], lamr)
                mg1.fpcg(rhs, x, 1e-8, 3)
                (it_r1, rel_r1), ms_r1 = wall(lambda: mg1.fpcg(rhs, x, 1e-8, 200))
            r32 = rhs.float()
            z32 = torch.empty_like(r32)
            us_sw = event_time_us(torch, lambda: lv[0].schwarz(r32, z32), 300)
            us_ras = event_time_us(torch, lambda: lv[0].schwarz(r32, z32, binding.SEM_SCHWARZ_RAS), 300)
            lv[0].pcg(rhs, x.zero_(), 1e-8, 20)
            (it_j, rel_j), ms_j = wall(lambda: lv[0].pcg(rhs, x.zero_(), 1e-8, 5000))
            m10 = mesh.N + 3
            # algorithmic bytes of one Schwarz application, FP32: read r (4), write + read the block b~ around Eq. (3)
            # (2 x 4 m^3/p^3), Lambda^-1 and S, write + read-modify-write z (gs counted as 8 S/nL)
            sw_bytes = 4.0 * (nL + mesh.E * (5 * m10 ** 3 + 3 * m10 * m10) + nL) + 8.0 * S
            solve = {"tol": 1e-8, "levels": "N = 7-3-1, smoother order 2, FP32 V-cycle, FP64 flexible PCG",
                     "pmg_fcg": {"smoother": "Chebyshev-Jacobi", "iters": it_m, "relres": rel_m, "ms": ms_m},
                     "pmg_fcg_schwarz": {"smoother": "Chebyshev-accelerated additive Schwarz (NEXT-2b) on N = 7, 3",
                                         "iters": it_s, "relres": rel_s, "ms": ms_s, "setup_ms": ms_setup},
                     "pmg_fcg_ras": {"smoother": "Chebyshev-accelerated restricted additive Schwarz on N = 7, 3 (fused: "
                                                 "gather, Eq. (3), weighted own part in one kernel)",
                                     "iters": it_r, "relres": rel_r, "ms": ms_r},
                     "pmg_fcg_ras_order1": {"smoother": "the same with smoother order 1 (one RAS application before and "
                                                        "after the coarse correction) and 16 coarse steps on the "
                                                        "assembled N = 1 operator",
                                            "iters": it_r1, "relres": rel_r1, "ms": ms_r1},
                     "schwarz_apply_f32": {"us_asm": us_sw, "us_ras": us_ras, "algorithmic_GBs": sw_bytes / us_sw / 1e3,
                                           "frac_of_measured_hbm_peak": sw_bytes / us_sw / 1e3 / peak,
                                           "what": "sem_schwarz at E = 7200, N = 7 (10^3 blocks): extension gather, "
                                                   "Eq. (3), weighted combination, gather-scatter"},
                     "jacobi_pcg": {"iters": it_j, "relres": rel_j, "ms": ms_j}}
            for s_ in lv:
                s_.close()

    # ---- arithmetic peaks of this device (sem_measure_peak) and the kernels quoted against them ----
    peaks = a9 = None
    if extras:
        peaks = {"fp64_fma_TFLOPs": binding.measure_peak(0), "fp32_fma_TFLOPs": binding.measure_peak(1),
                 "fp64_dmma_TFLOPs": binding.measure_peak(2),
                 "how": "sem_measure_peak: register-resident FMA / mma.sync m8n8k4 chains, best of 5 launches, CUDA events"}
        # a9: the operator with G recomputed from the 8 trilinear vertices (FP64-ALU bound: 12p+15+125 flops per node)
        with binding.Sem(mesh.E, mesh.N, mesh.vert, mesh.gid) as sr:
            sr.geom(mode=binding.SEM_G_RECOMPUTE)
            for _ in range(3):
                sr.ax(u, w)
            ms_r = timed(lambda: sr.ax(u, w), 200)
        tf = (12 * mesh.p + 15 + 125) * nL / (ms_r / 200 * 1e-3) / 1e12
        a9 = {"kernel": "sem_ax, SEM_G_RECOMPUTE (a9)", "us": ms_r / 200 * 1e3, "TFLOPs_fp64": tf, "bound": "alu",
              "frac_of_measured_fp64_fma_peak": tf / peaks["fp64_fma_TFLOPs"],
              "algorithmic_GBs": (16.0 + 192.0 / mesh.p ** 3) * nL / (ms_r / 200 * 1e-3) / 1e9}

    # ---- NEXT-2a: the Schwarz smoothers' fast-diagonalisation local solve (Eq. (3)) on config 2's 7200 elements,
    # extended blocks of m = N + 3 = 10 points per direction, FP32 (the paper's preconditioner precision) and FP64
    fdm = None
    if extras:
        m_ = mesh.N + 3
        S_h, iL_h = binding.fdm_setup(*inputs.fdm_pairs(mesh.E, m_, 7))
        fdm = {"workload": f"E = {mesh.E} blocks of {m_}^3, seeded 1-D operator pairs", "m": m_,
               "timed": "500 back-to-back launches of sem_fdm_apply, CUDA events"}
        for dt_, name, pk in ((torch.float32, "f32", "fp32_fma_TFLOPs"), (torch.float64, "f64", "fp64_fma_TFLOPs")):
            dS, dL = (torch.from_numpy(a.ravel()).cuda().to(dt_) for a in (S_h, iL_h))
            b_ = torch.randn(mesh.E * m_ ** 3, device="cuda", dtype=dt_)
            u_ = torch.empty_like(b_)
            for _ in range(3):
                sem.fdm_apply(m_, dS, dL, b_, u_)
            ms_f = timed(lambda: sem.fdm_apply(m_, dS, dL, b_, u_), 500)
            nbytes = b_.element_size() * mesh.E * (3 * m_ ** 3 + 3 * m_ * m_)
            tfl = 12.0 * m_ ** 4 * mesh.E / (ms_f / 500 * 1e-3) / 1e12
            fdm[name] = {"us": ms_f / 500 * 1e3, "TFLOPs": tfl, "frac_of_measured_fma_peak": tfl / peaks[pk],
                         "algorithmic_GBs": nbytes / (ms_f / 500 * 1e-3) / 1e9,
                         "frac_of_measured_hbm_peak": nbytes / (ms_f / 500 * 1e-3) / 1e9 / peak}

    dofs = mesh.dofs
    value = whole_job_value(dofs, world, K, ms_total)
    e2e_value = whole_job_value(dofs, world, Ke, ms_e2e)
    ax_s = ms_ax * 1e-3 / Kk
    gs_s = ms_gs * 1e-3 / Kk
    step_s = ms_total * 1e-3 / K
    ax_bytes = 64.0 * nL                                     # 64 B per local node, FP64, stored G
    achieved = ax_bytes / ax_s / 1e9
    whole_bytes = 64.0 * nL + 16.0 * S
    tr = ncu_traffic()
    ax_dram, gs_dram = tr.get("ax_dram_bytes_per_launch"), tr.get("gs_dram_bytes_per_launch")
    sem.set_variant(0)
    ax_kernel = "ax_dmma<3,12> (local D^T G D u, FP64 p=8, DMMA m8n8k4)" if args.variant == 0 else f"variant {args.variant}"
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": ms_total / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": WORKLOAD, "E": mesh.E, "N": mesh.N, "nL": nL, "U": cnt["U"], "S": S, "dofs_EN3": dofs,
                   "parallelism": "1 GPU" if world == 1 else f"{world} independent replicas",
                   "l2": "no explicit flush: G (177 MB, read evict-first) exceeds the 126 MB L2 and streams from HBM "
                         "every step; u and w (29.5 MB each) stay L2-resident by design (u is loaded evict-last, w is "
                         "re-read by the gather-scatter), as they do between the kernels of a PCG iteration -- DRAM "
                         "bytes per launch are printed beside the algorithmic bytes (roofline.traffic)",
                   "steps_requested": args.steps, "warmup_requested": args.warmup,
                   "min_timed_steps": MIN_TIMED_STEPS, "ax_variant": args.variant},
        "clocks": clocks,
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": int(u_h.numel() * 8),
                "d2h_bytes_per_step": int(w_h.numel() * 8), "steps": Ke, "ms_per_step": ms_e2e / Ke,
                "lanes": 2, "result_matches_device_path": e2e_ok},
        "gpu_launches": 2 * K,
        "roofline": {"bound": "hbm", "kernel": ax_kernel, "achieved": achieved,
                     "peak": peak, "unit": "GB/s", "frac": achieved / peak, "traffic": ax_dram,
                     "achieved_dram_GBs": (ax_dram / ax_s / 1e9) if ax_dram else None,
                     "frac_dram": (ax_dram / ax_s / 1e9 / peak) if ax_dram else None,
                     "traffic_source": tr.get("_source", "profiles/r2_dram_traffic.txt (ncu --cache-control none, "
                                                          "steady state; constant from the committed capture)"),
                     "peak_source": peak_src, "algorithmic_bytes_per_launch": ax_bytes,
                     "us_per_launch": ax_s * 1e6, "timed": f"{Kk} back-to-back launches of sem_ax alone, CUDA events",
                     "frac_of_nominal_8TBs": achieved / 8000.0},
        "breakdown": {"ax_us": ax_s * 1e6, "gs_us": gs_s * 1e6, "ax_gs_us": step_s * 1e6,
                      "ax_gs_algorithmic_GBs": whole_bytes / step_s / 1e9,
                      "ax_gs_frac_of_measured_peak": whole_bytes / step_s / 1e9 / peak,
                      "ax_gs_frac_of_nominal_8TBs": whole_bytes / step_s / 1e9 / 8000.0,
                      "ax_gs_dram_GBs": ((ax_dram + gs_dram) / step_s / 1e9) if ax_dram and gs_dram else None,
                      "gs_algorithmic_GBs": 16.0 * S / gs_s / 1e9,
                      "gs_dram_bytes_per_launch": gs_dram,
                      "ax_TFLOPs_fp64": (12 * mesh.p + 15) * nL / ax_s / 1e12,
                      "G_local_nodes_per_s": nL * K / (ms_total * 1e-3) / 1e9},
    }
    if peaks is not None:
        line["peaks"] = peaks
        line["breakdown"]["ax_frac_of_measured_fp64_fma_peak"] = line["breakdown"]["ax_TFLOPs_fp64"] / peaks["fp64_fma_TFLOPs"]
        line["a9_recomputed_G"] = a9
    if solve is not None:
        line["poisson_solve"] = solve
    if fdm is not None:
        line["fdm"] = fdm
    if pcg is not None:
        line["pcg"] = pcg
    sem.close()
    del u, w, wz
    torch.cuda.empty_cache()
    if extras and args.config5_n > 0:
        line["pcg_config5"] = run_config5(torch, binding, inputs, args.config5_n, peak)
    if rank == 0 and world == 1 and args.cpu_seconds > 0:
        line["cpu_baseline"] = cpu_oracle_baseline(mesh, args.cpu_seconds)
        if args.config5_n > 0:
            line["pcg_config5_cpu_baseline"] = cpu_oracle_pcg_config5(min(args.config5_n, 40))
    if rank == 0:
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
