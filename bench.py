#!/usr/bin/env python
"""bench.py — FP64 N=7 Ax+gs throughput on BASELINE.json config 2 (20x20x18 = 7200 hex elements, ~2.47 M points).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]

A "step" is one pass of the whole hot path: w = QQ^T (D^T G D) u over the full mesh (sem_ax_gs through the C ABI).
metric  = Ax+gs GDOF/s with DOF = E N^3 (the paper's n); value = whole-job DOF/s with inputs resident in HBM.
e2e     = same metric with u copied from pinned host memory and w copied back inside every timed step (two lanes,
          each its own context and stream, take alternate steps so that H2D and D2H overlap on the full-duplex link).
roofline= the dominant kernel (the local Ax) timed alone with CUDA events: 64 B x nL algorithmic bytes per launch
          against the measured HBM copy bandwidth of MEASURED_PEAKS.json.
N > 1   = independent replicas, one per GPU (the path has no inter-GPU exchange in this build).
--impl reference times the CPU oracle (oracle/) on the host cores, rank 0 only.
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


def measured_peak_gbs():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md)"


def ncu_traffic_bytes():
    """Per-launch DRAM bytes (read + write) of the Ax kernel from the committed ncu capture, else None."""
    try:
        with open(os.path.join(ROOT, "profiles", "ax_traffic.txt")) as f:
            for line in f:
                if line.startswith("dram_bytes_per_launch="):
                    return float(line.split("=", 1)[1])
    except Exception:
        pass
    return None


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


def cpu_oracle_baseline(mesh, budget_s: float, max_reps: int = 400):
    """The oracle as it stands, timed on the host cores: full Ax+gs applications of config 2."""
    import oracle
    oracle.build()
    from paper_2110_01716_b200 import inputs
    G, _, rc = oracle.geom_trilinear(mesh.vert, mesh.N)
    assert rc == 0
    om = oracle.Maps(mesh.gid)
    u = inputs.field_uniform(mesh.gid, 0)
    oracle.gs(oracle.ax(G, u, mesh.N).ravel(), om)          # warm-up
    times = []
    t_start = time.perf_counter()
    while len(times) < max_reps and (time.perf_counter() - t_start < budget_s or len(times) < 5):
        t0 = time.perf_counter()
        oracle.gs(oracle.ax(G, u, mesh.N).ravel(), om)
        times.append(time.perf_counter() - t0)
    med = float(np.median(times))
    return {"value": mesh.dofs / med / 1e9, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
            "sample": f"{len(times)} full Ax+gs applications of config 2 (all 7200 elements), median", "ms_per_step": med * 1e3}


def run_reference(args):
    """--impl reference: the CPU oracle on the host cores (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    import oracle
    oracle.build()
    from paper_2110_01716_b200 import inputs
    mesh = inputs.config2()
    G, _, rc = oracle.geom_trilinear(mesh.vert, mesh.N)
    u = inputs.field_uniform(mesh.gid, 0)
    om = oracle.Maps(mesh.gid)
    t0 = time.perf_counter()
    oracle.gs(oracle.ax(G, u, mesh.N).ravel(), om)
    t_full = time.perf_counter() - t0
    t0 = time.perf_counter()
    oracle.gs(oracle.ax(G, u, mesh.N).ravel(), om)
    t_full = min(t_full, time.perf_counter() - t0)
    total = args.steps + args.warmup
    budget = 150.0
    Es = mesh.E
    if total * t_full > budget:                       # bounded sample: the first Es elements of the same mesh
        Es = max(16, int(mesh.E * budget / (total * t_full)))
        G, u = np.ascontiguousarray(G[:Es]), np.ascontiguousarray(u[:Es])
        om = oracle.Maps(mesh.gid[:Es])
    for _ in range(args.warmup):
        oracle.gs(oracle.ax(G, u, mesh.N).ravel(), om)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle.gs(oracle.ax(G, u, mesh.N).ravel(), om)
    dt = time.perf_counter() - t0
    val = Es * mesh.N ** 3 * args.steps / dt / 1e9
    sample = f"each step = Ax+gs on the first {Es} of {mesh.E} elements of config 2"
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": WORKLOAD, "sample": sample},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle", "sample": sample},
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


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5000)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--e2e-steps", type=int, default=50)
    ap.add_argument("--cpu-seconds", type=float, default=12.0)
    ap.add_argument("--variant", type=int, default=0)
    ap.add_argument("--pcg-iters", type=int, default=300)
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
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
    K, W = args.steps, args.warmup

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
    # ---- the metric: K applications of the whole path, inputs resident in HBM (working set 236 MB > 126 MB L2) ----
    ms_total = timed(lambda: sem.ax_gs(u, w), K)
    # ---- kernel shares: the local operator alone, the gather-scatter alone ----
    # (bursts of at most 500 launches: MEASURED_PEAKS.json's hbm_gbs is a burst figure, "best of 10", and 5000 launches
    # of one kernel alone run into the power cap, which the whole-step loop above already reflects)
    Kk = min(K, 500)
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

    # ---- PCG iterations/s (second half of BASELINE.json's metric): config 2 with the Dirichlet mask, fixed count ----
    pcg = None
    if rank == 0 and world == 1 and args.pcg_iters > 0:
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
               "timed": "wall clock around one sem_pcg call (host polls a device flag every 16 iterations)"}
        semd.close()

    # ---- NEXT-1: the same Poisson problem solved to 1e-8 by Jacobi-PCG and by flexible PCG + FP32 p-multigrid V-cycle
    solve = None
    if rank == 0 and world == 1 and args.pcg_iters > 0:
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
            lv[0].pcg(rhs, x.zero_(), 1e-8, 20)
            (it_j, rel_j), ms_j = wall(lambda: lv[0].pcg(rhs, x.zero_(), 1e-8, 5000))
            solve = {"tol": 1e-8, "levels": "N = 7-3-1, Chebyshev-Jacobi order 2, FP32 V-cycle, FP64 flexible PCG",
                     "pmg_fcg": {"iters": it_m, "relres": rel_m, "ms": ms_m},
                     "jacobi_pcg": {"iters": it_j, "relres": rel_j, "ms": ms_j}}
            for s_ in lv:
                s_.close()

    # ---- NEXT-2a: the Schwarz smoothers' fast-diagonalisation local solve (Eq. (3)) on config 2's 7200 elements,
    # extended blocks of m = N + 3 = 10 points per direction, FP32 (the paper's preconditioner precision) and FP64
    fdm = None
    if rank == 0 and world == 1 and args.pcg_iters > 0:
        m_ = mesh.N + 3
        S_h, iL_h = binding.fdm_setup(*inputs.fdm_pairs(mesh.E, m_, 7))
        fdm = {"workload": f"E = {mesh.E} blocks of {m_}^3, seeded 1-D operator pairs", "m": m_,
               "timed": "500 back-to-back launches of sem_fdm_apply, CUDA events"}
        for dt_, name in ((torch.float32, "f32"), (torch.float64, "f64")):
            dS, dL = (torch.from_numpy(a.ravel()).cuda().to(dt_) for a in (S_h, iL_h))
            b_ = torch.randn(mesh.E * m_ ** 3, device="cuda", dtype=dt_)
            u_ = torch.empty_like(b_)
            for _ in range(3):
                sem.fdm_apply(m_, dS, dL, b_, u_)
            ms_f = timed(lambda: sem.fdm_apply(m_, dS, dL, b_, u_), 500)
            nbytes = b_.element_size() * mesh.E * (3 * m_ ** 3 + 3 * m_ * m_)
            fdm[name] = {"us": ms_f / 500 * 1e3, "TFLOPs": 12.0 * m_ ** 4 * mesh.E / (ms_f / 500 * 1e-3) / 1e12,
                         "algorithmic_GBs": nbytes / (ms_f / 500 * 1e-3) / 1e9}

    dofs = mesh.dofs
    value = whole_job_value(dofs, world, K, ms_total)
    e2e_value = whole_job_value(dofs, world, Ke, ms_e2e)
    peak, peak_src = measured_peak_gbs()
    ax_s = ms_ax * 1e-3 / Kk
    ax_bytes = 64.0 * nL                                     # 64 B per local node, FP64, stored G
    achieved = ax_bytes / ax_s / 1e9
    whole_bytes = 64.0 * nL + 16.0 * S
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": ms_total / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": WORKLOAD, "E": mesh.E, "N": mesh.N, "nL": nL, "U": cnt["U"], "S": S, "dofs_EN3": dofs,
                   "parallelism": "1 GPU" if world == 1 else f"{world} independent replicas",
                   "l2": "inputs (u+G+w = 236 MB) larger than the 126 MB L2; no explicit flush",
                   "ax_variant": args.variant},
        "clocks": clocks,
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": int(u_h.numel() * 8),
                "d2h_bytes_per_step": int(w_h.numel() * 8), "steps": Ke, "ms_per_step": ms_e2e / Ke,
                "lanes": 2, "result_matches_device_path": e2e_ok},
        "gpu_launches": 2 * K,
        "roofline": {"bound": "hbm", "kernel": "ax_stream<double,8,5,8> (local D^T G D u)", "achieved": achieved,
                     "peak": peak, "unit": "GB/s", "frac": achieved / peak, "traffic": ncu_traffic_bytes(),
                     "peak_source": peak_src, "algorithmic_bytes_per_launch": ax_bytes,
                     "us_per_launch": ax_s * 1e6, "timed": f"{Kk} back-to-back launches of sem_ax alone, CUDA events",
                     "frac_of_nominal_8TBs": achieved / 8000.0},
        "breakdown": {"ax_us": ms_ax / Kk * 1e3, "gs_us": ms_gs / Kk * 1e3, "ax_gs_us": ms_total / K * 1e3,
                      "ax_gs_algorithmic_GBs": whole_bytes / (ms_total * 1e-3 / K) / 1e9,
                      "ax_gs_frac_of_measured_peak": whole_bytes / (ms_total * 1e-3 / K) / 1e9 / peak,
                      "ax_gs_frac_of_nominal_8TBs": whole_bytes / (ms_total * 1e-3 / K) / 1e9 / 8000.0,
                      "ax_TFLOPs_fp64": (12 * mesh.p + 15) * nL / ax_s / 1e12,
                      "G_local_nodes_per_s": nL * K / (ms_total * 1e-3) / 1e9},
    }
    if solve is not None:
        line["poisson_solve"] = solve
    if fdm is not None:
        for name in ("f32", "f64"):
            fdm[name]["frac_of_measured_hbm_peak"] = fdm[name]["algorithmic_GBs"] / peak
        line["fdm"] = fdm
    if pcg is not None:
        pcg["frac_of_measured_peak"] = pcg["algorithmic_GBs"] / peak
        line["pcg"] = pcg
    if rank == 0 and world == 1 and args.cpu_seconds > 0:
        line["cpu_baseline"] = cpu_oracle_baseline(mesh, args.cpu_seconds)
    sem.close()
    if rank == 0:
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
