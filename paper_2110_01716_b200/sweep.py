"""Bandwidth sweep (BASELINE.json config 3) and mixed-precision levels (config 4) through the C ABI.

    python -m paper_2110_01716_b200.sweep [--max-n 64] [--orders 3,5,7,9] [--levels]

Box meshes of n^3 elements (n = 8, 16, 32, 64), random +-10 % interior-vertex perturbation (seed 1), FP64, stored G and
G recomputed from the 8 trilinear vertices; with --levels also config 4 (20x20x18, N = 7, 3, 1, FP32).  Every case is
timed with CUDA events over back-to-back launches after warm-up and printed as one markdown table row:
algorithmic bytes are 64 B (FP64) / 32 B (FP32) per local node for Ax with stored G, 16 + 192/p^3 B recomputed, and
16 B (8 B) per shared copy for gs.  Needs a CUDA device; there is no CPU fallback.
"""
from __future__ import annotations

import argparse
import json
import os
import sys

import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2110_01716_b200 import binding, inputs  # noqa: E402


def _peak():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"])
    except Exception:
        return 6650.0


def _time(fn, reps):
    for _ in range(3):
        fn()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record()
    for _ in range(reps):
        fn()
    e1.record()
    torch.cuda.synchronize()
    return e0.elapsed_time(e1) * 1e3 / reps          # us


def run_case(mesh, dtype, peak, label):
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
            t_ax = _time(lambda: sem.ax(u, w), reps)
            if mode == binding.SEM_G_STORED:
                t_gs = _time(lambda: sem.gs(w), reps)
                t_axgs = _time(lambda: sem.ax_gs(u, w), reps)
                b_ax = 8.0 * esize * nL
                row.update(nL=nL, S=S, ax=t_ax, gs=t_gs, axgs=t_axgs, ax_gbs=b_ax / t_ax / 1e3,
                           axgs_gbs=(b_ax + 2.0 * esize * S) / t_axgs / 1e3,
                           gdofs=mesh.dofs / t_axgs / 1e3)
            else:
                p3 = mesh.p ** 3
                row.update(ax_re=t_ax, re_gbs=(2.0 * esize + 192.0 / p3) * nL / t_ax / 1e3,
                           re_tflops=(12 * mesh.p + 15 + 125) * nL / t_ax / 1e6)
    print(f"| {label} | {mesh.E} | {mesh.N} | {row['nL']} | {row['ax']:.1f} | {row['ax_gbs']:.0f} | "
          f"{row['ax_gbs'] / peak:.2f} | {row['gs']:.1f} | {row['axgs']:.1f} | {row['axgs_gbs']:.0f} | "
          f"{row['gdofs']:.1f} | {row['ax_re']:.1f} | {row['re_tflops']:.1f} |", flush=True)


def run_config5(n: int, peak: float):
    """BASELINE.json config 5: n^3 elements (100 at full size), N = 7, random +-10 % vertices (seed 3), scrambled element
    order (seed 4), homogeneous Dirichlet, b = M Q^T(B f), f = 3 pi^2 sin(pi x) sin(pi y) sin(pi z), Jacobi-PCG to 1e-8.
    The right-hand side and the node coordinates are built with torch on the device from sem_get-free data: B = the
    7th geometric factor is not exported at this size, so b is assembled as A applied to nothing -- instead we use the
    discrete identity b = A u_h-free form: b = Q Q^T (B f) with B f evaluated by the library's own mass factor."""
    import time

    import numpy as np
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
    a = (1 - xi) / 2
    bb = (1 + xi) / 2
    w1 = torch.stack([a, bb])                                                # [2, p]
    xyz = torch.zeros(mesh.E, p, p, p, 3, device="cuda", dtype=torch.float64)
    for v in range(8):
        ia, ib, ic = v & 1, (v >> 1) & 1, (v >> 2) & 1
        wgt = w1[ic][:, None, None] * w1[ib][None, :, None] * w1[ia][None, None, :]
        xyz += wgt[None, :, :, :, None] * V[:, v][:, None, None, None, :]
    exact = (torch.sin(np.pi * xyz[..., 0]) * torch.sin(np.pi * xyz[..., 1]) * torch.sin(np.pi * xyz[..., 2])).reshape(-1)
    del xyz
    # b = M Q Q^T (B f): lambda B u with the Helmholtz term only is not exposed, so use  (A + 1 B) f - A f  = B f
    f = 3 * np.pi ** 2 * exact
    t1, t2 = torch.empty_like(f), torch.empty_like(f)
    sem.ax(f, t1, 1.0)
    sem.ax(f, t2, 0.0)
    t1 -= t2                                                                 # B f, local
    del t2
    sem.gs(t1)
    mask = torch.from_numpy(mesh.dirichlet.ravel()).cuda() != 0
    t1[mask] = 0.0
    x = torch.zeros_like(t1)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    it, rel = sem.pcg(t1, x, 1e-8, 20000)
    torch.cuda.synchronize()
    dt = time.perf_counter() - t0
    err = float((x - exact).abs().max())
    bytes_it = (64.0 + 56.0 + 32.0) * nL + 16.0 * S
    print(f"config 5 with {n}^3 elements: E = {mesh.E}, nL = {nL}, U = {cnt['U']}, S = {S}; mesh {t_mesh:.1f} s, "
          f"setup {t_setup:.1f} s; PCG {it} iterations, relres {rel:.2e}, {dt:.2f} s = {it / dt:.1f} iterations/s, "
          f"{bytes_it * it / dt / 1e9:.0f} GB/s algorithmic = {bytes_it * it / dt / 1e9 / peak:.2f} of peak; "
          f"max |x - sin sin sin| = {err:.2e}", flush=True)
    sem.close()


def run_projection(peak: float):
    """NEXT-3 at config 2: bandwidth of the tall-skinny kernels with L = 30 stored solutions, and what the projection
    buys over a sequence of slowly evolving right-hand sides (Jacobi-PCG iterations to 1e-8 with and without it)."""
    import numpy as np
    mesh = inputs.config2()
    with binding.Sem(mesh.E, mesh.N, mesh.vert, mesh.gid, mesh.dirichlet) as sem:
        sem.geom()
        nL = sem.nL
        fields = [torch.from_numpy(inputs.field_uniform(mesh.gid, 40 + k).ravel()).cuda() for k in range(4)]
        rhs = [torch.empty_like(fields[0]) for _ in range(4)]
        for f_, r_ in zip(fields, rhs):
            sem.ax_gs(f_, r_)                                   # assembled, masked right-hand sides A f_k
        xbar, bred, x = (torch.empty_like(rhs[0]) for _ in range(3))
        print("| step | PCG iterations without projection | with projection (L) | reduced / full right-hand side norm |")
        print("|---|---|---|---|")
        with binding.Proj(sem, 30) as pj:
            for m_ in range(12):
                t = 0.05 * m_
                b = rhs[0] + t * rhs[1] + t * t * rhs[2] + np.sin(3 * t) * 0.1 * rhs[3]
                it0, _ = sem.pcg(b, x.zero_(), 1e-8 , 5000)
                pj.guess(b, xbar, bred)
                ratio = float(bred.norm() / b.norm())
                it1, _ = sem.pcg(bred, x.zero_(), 1e-8 * float(b.norm() / max(float(bred.norm()), 1e-300)), 5000)
                L_before = pj.size()
                pj.update(x)
                print(f"| {m_} | {it0} | {it1} ({L_before}) | {ratio:.2e} |", flush=True)
        with binding.Proj(sem, 30) as pj:                       # fill the space, then time the two kernels' passes
            for k in range(30):
                pj.update(torch.from_numpy(inputs.field_uniform(mesh.gid, 200 + k).ravel()).cuda())
            assert pj.size() == 30
            t_g = _time(lambda: pj.guess(rhs[0], xbar, bred), 50)
            gb = 8.0 * nL * (31 + 61 + 2) / t_g / 1e3
            print(f"\nsem_proj_guess with L = 30 at config 2: {t_g:.0f} us = {gb:.0f} GB/s ({gb / peak:.2f} of peak; "
                  f"31 vectors read by the multi-dot, 61 read + 2 written by the update pass)")


def run_gs_many(peak: float):
    """NEXT-4, first piece: sem_gs_many (gatherScatterMany) on config 2 against nf separate sem_gs calls."""
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
                t1 = _time(separate, 300)
                t2 = _time(lambda: sem.gs_many(w), 300)
                print(f"| {nf} | {name} | {t1:.1f} | {t2:.1f} | {t1 / t2:.2f} |", flush=True)


def run_fdm(peak: float):
    """NEXT-2a: sem_fdm_apply (Eq. (3)) at the paper's per-GPU element count, m = N + 3 for N = 7, 5, 3, 1 and
    the paper's 8-5-1 / 8-6-4-1 schedules.  Bytes = b, Lambda^-1, u (m^3 each) + S (3 m^2) per element; flops = 12 m^4."""
    print("| E | m | precision | us | GB/s | frac of HBM peak | TFLOP/s |")
    print("|---|---|---|---|---|---|---|")
    # E = 7200: config 2's element count; (3573, 11): the paper's Table 2 case (E/P = 3573, N = 8, FP32: 171 us on V100)
    for E, m in ((7200, 10), (7200, 8), (7200, 7), (7200, 6), (7200, 5), (7200, 4), (7200, 12), (3573, 11), (3573, 9), (3573, 7)):
        mesh = inputs.box_mesh(E, 1, 1, 1)
        with binding.Sem(mesh.E, 1, mesh.vert, mesh.gid) as sem:
            A, B = inputs.fdm_pairs(E, m, 7)
            S, invL = binding.fdm_setup(A, B)
            for dt, name in ((torch.float32, "FP32"), (torch.float64, "FP64")):
                dS, dL = (torch.from_numpy(a.ravel()).cuda().to(dt) for a in (S, invL))
                b = torch.randn(E * m ** 3, device="cuda", dtype=dt)
                u = torch.empty_like(b)
                t = _time(lambda: sem.fdm_apply(m, dS, dL, b, u), 500)
                nbytes = b.element_size() * E * (3 * m ** 3 + 3 * m * m)
                print(f"| {E} | {m} | {name} | {t:.2f} | {nbytes / t / 1e3:.0f} | {nbytes / t / 1e3 / peak:.2f} | "
                      f"{12.0 * m ** 4 * E / t / 1e6:.2f} |", flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gs-many", action="store_true", help="NEXT-4: gather-scatter of several fields in one pass")
    ap.add_argument("--fdm", action="store_true", help="NEXT-2a: fast-diagonalisation local solve (Eq. (3)) at E = 7200")
    ap.add_argument("--proj", action="store_true", help="NEXT-3: projection onto previous solutions at config 2")
    ap.add_argument("--config5", type=int, default=0, help="run config 5 with this many elements per direction")
    ap.add_argument("--max-n", type=int, default=64)
    ap.add_argument("--orders", default="3,5,7,9")
    ap.add_argument("--levels", action="store_true")
    args = ap.parse_args()
    if not torch.cuda.is_available():
        raise SystemExit("sweep needs a CUDA device: the product path has no CPU fallback")
    peak = _peak()
    if args.config5 > 0:
        return run_config5(args.config5, peak)
    if args.proj:
        return run_projection(peak)
    if args.fdm:
        return run_fdm(peak)
    if args.gs_many:
        return run_gs_many(peak)
    print(f"peak = {peak:.0f} GB/s (MEASURED_PEAKS.json hbm_gbs, else the profiling guide's fallback)")
    print("| case | E | N | nL | Ax us | Ax GB/s | frac of peak | gs us | Ax+gs us | Ax+gs GB/s | GDOF/s (E N^3) | "
          "Ax recomputed-G us | recomputed TFLOP/s |")
    print("|---|---|---|---|---|---|---|---|---|---|---|---|---|")
    for N in [int(x) for x in args.orders.split(",")]:
        n = 8
        while n <= args.max_n:
            run_case(inputs.config3(n, N), torch.float64, peak, f"cfg3 {n}^3 f64")
            n *= 2
    if args.levels:
        for N in (7, 3, 1):
            run_case(inputs.config4(N), torch.float32, peak, "cfg4 20x20x18 f32")
        # NEXT-1: transfers between config 4's levels, FP32; bytes = one read of the input + one write of the output
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
                t = _time(fn, 2000)
                gbs = 4.0 * (sc.nL + sf.nL) / t / 1e3
                print(f"| {name} | {t:.2f} | {gbs:.0f} | {gbs / peak:.2f} |", flush=True)
        # NEXT-1: Chebyshev-Jacobi smoother, FP32, zero initial guess: order - 1 operator applications + order fused
        # vector kernels; bytes = (order-1) x (Ax+gs) + vector traffic (init 16, step 32, final 12 B/node incl. Minv FP64)
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
                    t = _time(lambda: sd.cheby(b, x, order, 0.2, 2.2, True), 500)
                    print(f"| N = {N}, order {order} | {t:.1f} | {t / (order - 1):.1f} |", flush=True)
        for s_ in sems.values():
            s_.close()


if __name__ == "__main__":
    main()
