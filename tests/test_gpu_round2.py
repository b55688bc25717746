"""GPU parity tests added in round 2 (through the C ABI, against the CPU oracle): the stated sizes VERDICT r1 found
missing (config 4's FP32 coarse levels at E = 7200; config 5 at its full 10^6 elements, where G offsets pass 2^31),
the tensor-core operator kernel, and the regression tests of the round-1 advisor findings."""
import os

import numpy as np
import pytest

from paper_2110_01716_b200 import inputs

pytestmark = pytest.mark.gpu

TOL64, TOL32, TOLPCG = 1e-12, 1e-5, 1e-9


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("gpu-marked test needs a CUDA device (run with -m 'not gpu' on CPU boxes)")
    return torch


@pytest.fixture(scope="module")
def binding():
    from paper_2110_01716_b200 import binding as b, build
    build.build()
    b.lib()
    return b


def relerr(a, b):
    return float(np.max(np.abs(np.asarray(a, np.float64) - b)) / np.max(np.abs(b)))


def to_dev(torch, a, dtype=None):
    t = torch.from_numpy(np.ascontiguousarray(a)).cuda()
    return t if dtype is None else t.to(dtype)


def _ax_gs_oracle(oracle_mod, mesh, u, masked):
    oG, _, rc = oracle_mod.geom_trilinear(mesh.vert, mesh.N)
    assert rc == 0
    om = oracle_mod.Maps(mesh.gid)
    w = oracle_mod.gs(oracle_mod.ax(oG, u, mesh.N).ravel(), om)
    if masked:
        w = np.where(oracle_mod.mask_unique(mesh.dirichlet, om)[om.l2u] != 0, 0.0, w)
    return w


# --------------------------------------------------------------------------- config 4 at its stated size (E = 7200)
@pytest.mark.parametrize("N", [3, 1])
def test_ax_gs_f32_levels_config4_full_size(torch_cuda, binding, oracle_mod, N):
    """BASELINE.json configs[3]: FP32 Ax+gs on the 20x20x18 mesh at the p-multigrid coarse levels N = 3 and N = 1,
    u ~ N(0,1) per unique node (seed 2), against the FP64 oracle at 1e-5 -- the launch shape bench.py's poisson_solve
    runs (1800 / 450 element groups: the persistent CTAs of ax_stream<float,4,..> wrap their ring more than once)."""
    m = inputs.config4(N)
    assert m.E == 7200
    u = inputs.field_normal(m.gid, 2)
    for masked in (False, True):
        ow = _ax_gs_oracle(oracle_mod, m, u, masked)
        with binding.Sem(m.E, m.N, m.vert, m.gid, m.dirichlet if masked else None) as sem:
            sem.geom()
            du = to_dev(torch_cuda, u.ravel(), torch_cuda.float32)
            dw = torch_cuda.full_like(du, float("nan"))
            for _ in range(3):                               # eager, captured, replayed
                sem.ax_gs(du, dw)
            torch_cuda.cuda.synchronize()
            assert relerr(dw.cpu().numpy(), ow) <= TOL32, (N, masked)
            d64 = to_dev(torch_cuda, u.ravel())
            w64 = torch_cuda.full_like(d64, float("nan"))
            sem.ax_gs(d64, w64)
            assert relerr(w64.cpu().numpy(), ow) <= TOL64, (N, masked)


# --------------------------------------------------------------------------- the tensor-core operator (FP64, p = 8)
@pytest.mark.parametrize("variant", [0, 2, 3])
def test_ax_dmma_vs_scalar_kernels(torch_cuda, binding, oracle_mod, variant):
    """FP64 p = 8: the DMMA kernel (variants 0 and 3) and the scalar streaming kernel (variant 2) against the oracle on a
    mesh with more elements than resident warps (every warp walks its ring several times: mbarrier phase wrap-around),
    with and without the Helmholtz term, and with the fused p.q dot of the PCG loop (through sem_pcg below)."""
    m = inputs.box_mesh(22, 22, 23, 7, "random", seed=1)       # 11132 elements > 148 x 12 warps x 6
    oG, _, rc = oracle_mod.geom_trilinear(m.vert, m.N)
    assert rc == 0
    u = inputs.field_uniform(m.gid, 4)
    for lam in (0.0, 12.5):
        ow = oracle_mod.ax(oG, u, m.N, lam)
        with binding.Sem(m.E, m.N, m.vert, m.gid) as sem:
            sem.geom(with_mass=lam != 0.0)
            sem.set_variant(variant)
            du = to_dev(torch_cuda, u.ravel())
            dw = torch_cuda.full_like(du, float("nan"))
            sem.ax(du, dw, lam)
            torch_cuda.cuda.synchronize()
            assert relerr(dw.cpu().numpy().reshape(ow.shape), ow) <= TOL64, (variant, lam)


@pytest.mark.parametrize("variant", [0, 2])
def test_ax_tf32_vs_scalar_kernel(torch_cuda, binding, oracle_mod, variant):
    """FP32 p = 8: the TF32 x 3 tensor-core kernel (variant 0: hi*hi + lo*hi + hi*lo, FP32 accumulation) and the scalar
    streaming kernel (variant 2) against the FP64 oracle at 1e-5 (S16), more elements than resident warps, with and
    without the Helmholtz term, inputs spanning six orders of magnitude (the split must not lose the small ones)."""
    m = inputs.box_mesh(22, 22, 23, 7, "random", seed=1)
    oG, _, rc = oracle_mod.geom_trilinear(m.vert, m.N)
    assert rc == 0
    u = inputs.field_normal(m.gid, 4) * (10.0 ** (6.0 * inputs.hash_uniform01(3, 7, m.gid) - 3.0))
    for lam in (0.0, 12.5):
        ow = oracle_mod.ax(oG, u, m.N, lam)
        with binding.Sem(m.E, m.N, m.vert, m.gid) as sem:
            sem.geom(with_mass=lam != 0.0)
            sem.set_variant(variant)
            du = to_dev(torch_cuda, u.ravel(), torch_cuda.float32)
            dw = torch_cuda.full_like(du, float("nan"))
            sem.ax(du, dw, lam)
            torch_cuda.cuda.synchronize()
            assert relerr(dw.cpu().numpy().reshape(ow.shape), ow) <= TOL32, (variant, lam)


def test_ax_dmma_bit_repeatable(torch_cuda, binding):
    """The default FP64 p = 8 path (DMMA operator + record gather-scatter) has no atomics on data: repeated applications
    give bit-identical results, eager or replayed from the CUDA graph."""
    m = inputs.config2()
    side = torch_cuda.cuda.Stream()
    with torch_cuda.cuda.stream(side):
        with binding.Sem(m.E, m.N, m.vert, m.gid, m.dirichlet) as sem:
            sem.geom()
            du = to_dev(torch_cuda, inputs.field_uniform(m.gid, 9).ravel())
            outs = []
            for _ in range(5):
                dw = torch_cuda.full_like(du, float("nan"))
                sem.ax_gs(du, dw)
                side.synchronize()
                outs.append(dw)
            dw = torch_cuda.full_like(du, float("nan"))
            for _ in range(4):                               # same arguments: eager, captured, replayed
                sem.ax_gs(du, dw)
            side.synchronize()
            outs.append(dw)
            for o in outs[1:]:
                assert torch_cuda.equal(o, outs[0])


# --------------------------------------------------------------------------- config 5 at its full size, sampled
@pytest.mark.slow
def test_config5_full_size_sampled_parity(torch_cuda, binding, oracle_mod):
    """BASELINE.json configs[4] at full size: 100^3 = 10^6 elements, 512 M local nodes, 24.6 GB of G -- the only workload
    whose G entry index exceeds 2^31 (64-bit offsets) -- in the launch configuration bench.py's pcg_config5 leg
    runs.  The oracle cannot do 512 M nodes in seconds, so outputs are SAMPLED: for 48 elements (the first, the last,
    elements on both sides of the 2^31 boundary, seeded random ones) the oracle computes w = M QQ^T A_L u from the
    element's whole 27-element neighbourhood (every copy of every node of the sampled element lies in it), and all 512
    outputs of each sampled element are compared at 1e-12.  Counts are checked against SURVEY's table."""
    n = 100
    m = inputs.config5(n)
    assert m.E == 1_000_000
    p3 = m.p ** 3
    u = inputs.field_uniform(m.gid, 6)                        # [E, 512], continuous (per unique node)
    # ---- sampled elements and their lexicographic 27-neighbourhoods ----
    first_big = (2 ** 31) // (6 * p3) + 1                     # first element whose G entries start beyond 2^31
    sample = [0, 1, m.E - 1, m.E - 2, first_big - 2, first_big - 1, first_big, first_big + 1, 500_000, 999_000]
    sample += [int(s) for s in (inputs.hash_uniform01(77, 0, np.arange(38)) * m.E).astype(np.int64)]
    sample = sorted(set(sample))
    inv = np.empty(m.E, dtype=np.int64)
    inv[m.perm] = np.arange(m.E)                              # lexicographic element -> index in this mesh
    ow = {}
    for e in sample:
        lex = int(m.perm[e])
        ex, ey, ez = lex % n, (lex // n) % n, lex // (n * n)
        nb = []
        for dz in (-1, 0, 1):
            for dy in (-1, 0, 1):
                for dx in (-1, 0, 1):
                    x, y, z = ex + dx, ey + dy, ez + dz
                    if 0 <= x < n and 0 <= y < n and 0 <= z < n:
                        nb.append(int(inv[x + n * (y + n * z)]))
        nb = np.array(sorted(nb))
        oG, _, rc = oracle_mod.geom_trilinear(m.vert[nb], m.N)
        assert rc == 0
        wl = oracle_mod.ax(oG, u[nb], m.N).reshape(len(nb), p3)
        om = oracle_mod.Maps(m.gid[nb])                       # canonical maps of the neighbourhood
        ws = oracle_mod.gs(wl.ravel(), om).reshape(len(nb), p3)
        me = int(np.searchsorted(nb, e))
        ow[e] = np.where(m.dirichlet[e] != 0, 0.0, ws[me])
    # ---- the CUDA path on the whole mesh ----
    with binding.Sem(m.E, m.N, m.vert, m.gid, m.dirichlet) as sem:
        c = sem.counts()
        assert (c["nL"], c["U"], c["S"], c["Us"]) == (512_000_000, 344_472_101, 293_832_792, 126_304_893)
        sem.geom()
        du = to_dev(torch_cuda, u.reshape(-1))
        del u
        dw = torch_cuda.full_like(du, float("nan"))
        sem.ax_gs(du, dw)
        torch_cuda.cuda.synchronize()
        scale = max(float(np.max(np.abs(v))) for v in ow.values())   # max |w_orc| over the sample (<= the global max)
        worst = 0.0
        for e in sample:
            got = dw[e * p3:(e + 1) * p3].cpu().numpy()
            worst = max(worst, float(np.max(np.abs(got - ow[e]))) / scale)
        assert worst <= TOL64, worst
        # recomputed-G and scalar-kernel variants on the same input agree on the sampled elements too
        sem.set_variant(2)
        dw2 = torch_cuda.full_like(du, float("nan"))
        sem.ax_gs(du, dw2)
        torch_cuda.cuda.synchronize()
        for e in sample[:12]:
            got = dw2[e * p3:(e + 1) * p3].cpu().numpy()
            assert float(np.max(np.abs(got - ow[e]))) / scale <= TOL64, e


# --------------------------------------------------------------------------- advisor r1: stale interpolation matrix
def test_transfer_between_graph_replays_keeps_J(torch_cuda, binding, oracle_mod):
    """a recorded V-cycle / flexible-PCG graph bakes in the device pointer of the interpolation
    matrix.  An FP64 sem_transfer (and one with another coarse partner) on the same fine context between two solves of
    an FP32 sem_fpcg must not change what the replayed graph reads: iteration count and solution stay the oracle's."""
    orders = (5, 2)
    meshes = [inputs.box_mesh(4, 4, 3, N, "random", seed=5) for N in orders]
    m_other = inputs.box_mesh(4, 4, 3, 3, "random", seed=5)
    olv = [oracle_mod.Level(m) for m in meshes]
    L0 = olv[0]
    xs = np.where(L0.mask_u != 0, 0.0, inputs.field_normal(L0.maps.uniq_gid, 17))
    b_u = L0.A(xs)
    ores = oracle_mod.fpcg(L0, lambda r: oracle_mod.vcycle(olv, r, 2, 6), b_u, tol=1e-8, maxit=60)
    side = torch_cuda.cuda.Stream()
    with torch_cuda.cuda.stream(side):
        sems = [binding.Sem(m.E, m.N, m.vert, m.gid, m.dirichlet).geom() for m in meshes]
        s_other = binding.Sem(m_other.E, m_other.N, m_other.vert, m_other.gid, m_other.dirichlet).geom()
        try:
            with binding.Pmg(sems, [l.lmin for l in olv], [l.lmax for l in olv], 2, 6, binding.SEM_F32) as mg:
                b = to_dev(torch_cuda, b_u[L0.maps.l2u])
                x = torch_cuda.empty_like(b)
                its = []
                for solve in range(4):
                    x.fill_(float("nan"))
                    it, rel = mg.fpcg(b, x, 1e-8, 60)
                    its.append(it)
                    assert rel <= 1e-8 and abs(it - ores["iters"]) <= 2, solve
                    assert relerr(x.cpu().numpy(), ores["x"][L0.maps.l2u]) <= 1e-6, solve
                    # between the solves: the same level pair in FP64, and another coarse partner in FP32
                    vc = torch_cuda.randn(sems[1].nL, device="cuda", dtype=torch_cuda.float64)
                    vf = torch_cuda.empty(sems[0].nL, device="cuda", dtype=torch_cuda.float64)
                    sems[1].transfer(sems[0], vc, vf, binding.SEM_PROLONG)
                    ref = oracle_mod.prolong(vc.cpu().numpy(), orders[1], orders[0])
                    assert relerr(vf.cpu().numpy(), ref.ravel()) <= TOL64
                    vo = torch_cuda.randn(s_other.nL, device="cuda", dtype=torch_cuda.float32)
                    vf32 = torch_cuda.empty(sems[0].nL, device="cuda", dtype=torch_cuda.float32)
                    s_other.transfer(sems[0], vo, vf32, binding.SEM_PROLONG)
                assert max(its) - min(its) <= 1
        finally:
            for s_ in sems + [s_other]:
                s_.close()


def test_measure_peak(torch_cuda, binding):
    """sem_measure_peak returns plausible rates (B200: ~36 TFLOP/s FP64 FMA = DMMA, ~68 FP32) and rejects a bad kind."""
    f64, f32, dm = (binding.measure_peak(k) for k in (0, 1, 2))
    assert 10.0 < f64 < 80.0 and 20.0 < f32 < 160.0 and 10.0 < dm < 80.0
    assert 0.8 < dm / f64 < 1.25
    with pytest.raises(binding.SemError):
        binding.measure_peak(7)


# --------------------------------------------------------------------------- NEXT-2b: overlapping Schwarz smoother
def _schwarz_case(N, masked, permute):
    return inputs.box_mesh(4, 3, 3, N, "random", seed=11 + N, permute_seed=5 if permute else None)


@pytest.mark.parametrize("N,masked,permute", [(7, True, True), (7, False, False), (3, True, False), (2, True, True),
                                              (5, False, True), (4, True, False)])
def test_schwarz_setup_and_apply_parity(torch_cuda, binding, oracle_mod, N, masked, permute):
    """sem_schwarz_setup / sem_schwarz against the oracle's Schwarz (reading S29): face neighbours bit-exact, 1-D operator
    pairs 1e-13, weights 1e-14, and z = S r for the additive and the restricted variant in FP64 (1e-10: the library's
    Jacobi eigen-solver and scipy's differ in the last digits of S) and FP32 (1e-5), on a deformed mesh, with and without
    the Dirichlet mask, in lexicographic and in scrambled element order."""
    m = _schwarz_case(N, masked, permute)
    maps = oracle_mod.Maps(m.gid)
    mask_u = oracle_mod.mask_unique(m.dirichlet, maps) if masked else np.zeros(maps.U, np.uint8)
    r_u = np.where(mask_u != 0, 0.0, inputs.field_normal(maps.uniq_gid, 21))
    with binding.Sem(m.E, m.N, m.vert, m.gid, m.dirichlet if masked else None) as sem:
        sem.geom()
        with pytest.raises(binding.SemError) as err:
            sem.schwarz(to_dev(torch_cuda, r_u[maps.l2u]), torch_cuda.empty(sem.nL, device="cuda", dtype=torch_cuda.float64))
        assert err.value.code == binding.SEM_ESTATE
        sem.schwarz_setup()
        for kind, restricted in ((binding.SEM_SCHWARZ_ASM, False), (binding.SEM_SCHWARZ_RAS, True)):
            sw = oracle_mod.Schwarz(m, maps, mask_u, restricted)
            nbr, A, B, W = sem.get_schwarz(kind)
            assert np.array_equal(nbr, sw.nbr)
            assert np.max(np.abs(A - sw.A1)) <= 1e-13 * np.max(np.abs(sw.A1))
            assert np.max(np.abs(B - sw.B1)) <= 1e-13 * np.max(np.abs(sw.B1))
            Wo = (sw.W if restricted else np.sqrt(sw.W))[maps.l2u]
            assert np.max(np.abs(W.ravel() - Wo)) <= 1e-14
            oz = sw.apply(r_u)[maps.l2u]
            for dt, tol in ((torch_cuda.float64, 1e-10), (torch_cuda.float32, TOL32)):
                dr = to_dev(torch_cuda, r_u[maps.l2u], dt)
                dz = torch_cuda.full_like(dr, float("nan"))
                sem.schwarz(dr, dz, kind)
                torch_cuda.cuda.synchronize()
                assert relerr(dz.cpu().numpy(), oz) <= tol, (N, kind, dt)
                sem.schwarz(dr, dr, kind)                      # in place
                assert torch_cuda.equal(dr, dz)


def test_schwarz_needs_an_interior_face_node(torch_cuda, binding):
    m = inputs.box_mesh(3, 3, 3, 1, "affine")
    with binding.Sem(m.E, m.N, m.vert, m.gid) as sem:
        sem.geom()
        with pytest.raises(binding.SemError) as err:
            sem.schwarz_setup()
        assert err.value.code == binding.SEM_EINVAL


@pytest.mark.parametrize("N,order,zero_guess,kind", [(7, 2, True, 0), (5, 3, False, 0), (3, 1, True, 0), (4, 2, False, 1)])
def test_cheby_schwarz_parity(torch_cuda, binding, oracle_mod, N, order, zero_guess, kind):
    """sem_cheby_schwarz against the oracle's cheby_pc with the Schwarz operator, and sem_lambda_max_schwarz against the
    dense-free power iteration of the oracle (same start-independent limit: compared loosely)."""
    m = _schwarz_case(N, True, False)
    L = oracle_mod.Level(m, power_its=5)
    L.use_schwarz(m, restricted=bool(kind), power_its=40)
    b_u = L.A(np.where(L.mask_u != 0, 0.0, inputs.field_normal(L.maps.uniq_gid, 3)))
    x0_u = None if zero_guess else np.where(L.mask_u != 0, 0.0, inputs.field_normal(L.maps.uniq_gid, 4))
    ox = oracle_mod.cheby_pc(L.A, L.schwarz.apply, b_u, x0_u, order, L.slmin, L.slmax)[L.maps.l2u]
    with binding.Sem(m.E, m.N, m.vert, m.gid, m.dirichlet) as sem:
        sem.geom()
        sem.schwarz_setup()
        lam = sem.lambda_max_schwarz(kind, 40)
        assert abs(1.1 * lam - L.slmax) <= 0.05 * L.slmax
        for dt, tol in ((torch_cuda.float64, 1e-9), (torch_cuda.float32, 5e-5)):
            db = to_dev(torch_cuda, b_u[L.maps.l2u], dt)
            dx = torch_cuda.full_like(db, float("nan")) if zero_guess else to_dev(torch_cuda, x0_u[L.maps.l2u], dt)
            sem.cheby_schwarz(db, dx, order, L.slmin, L.slmax, zero_guess, kind)
            torch_cuda.cuda.synchronize()
            assert relerr(dx.cpu().numpy(), ox) <= tol, (N, order, dt)


def test_vcycle_and_fpcg_with_schwarz_smoothing(torch_cuda, binding, oracle_mod):
    """The V-cycle with Chebyshev-Schwarz smoothing on the levels with N >= 2 (sem_pmg_set_smoother) against the oracle's
    cycle with the same smoother, FP64 1e-9 / FP32 1e-4, and flexible PCG around it: the oracle's iteration count,
    which is below the Chebyshev-Jacobi cycle's on the same problem."""
    orders = (7, 3, 1)
    meshes = [inputs.box_mesh(4, 3, 3, N, "random", seed=3) for N in orders]
    olv = [oracle_mod.Level(m) for m in meshes]
    ojac = [oracle_mod.Level(m) for m in meshes]
    for L, m in zip(olv[:-1], meshes[:-1]):
        L.use_schwarz(m)
    L0 = olv[0]
    xs = np.where(L0.mask_u != 0, 0.0, inputs.field_normal(L0.maps.uniq_gid, 17))
    b_u = L0.A(xs)
    oz = oracle_mod.vcycle(olv, b_u, 2, 8)
    ores = oracle_mod.fpcg(L0, lambda r: oracle_mod.vcycle(olv, r, 2, 8), b_u, tol=1e-8, maxit=60)
    ojres = oracle_mod.fpcg(ojac[0], lambda r: oracle_mod.vcycle(ojac, r, 2, 8), b_u, tol=1e-8, maxit=60)
    assert ores["iters"] < ojres["iters"]
    side = torch_cuda.cuda.Stream()
    with torch_cuda.cuda.stream(side):
        sems = [binding.Sem(m.E, m.N, m.vert, m.gid, m.dirichlet).geom() for m in meshes]
        try:
            slmin = [getattr(l, "slmin", l.lmin) for l in olv]
            slmax = [getattr(l, "slmax", l.lmax) for l in olv]
            for prec, dt, tol in ((binding.SEM_F64, torch_cuda.float64, 1e-9), (binding.SEM_F32, torch_cuda.float32, 1e-4)):
                with binding.Pmg(sems, [l.lmin for l in olv], [l.lmax for l in olv], 2, 8, prec) as mg:
                    mg.set_smoother(binding.SEM_SMOOTH_CHEBY_SCHWARZ, slmin, slmax)
                    dr = to_dev(torch_cuda, b_u[L0.maps.l2u], dt)
                    dz = torch_cuda.full_like(dr, float("nan"))
                    for _ in range(3):                           # eager, captured, replayed
                        mg.vcycle(dr, dz)
                    side.synchronize()
                    assert relerr(dz.cpu().numpy(), oz[L0.maps.l2u]) <= tol, prec
                    b = to_dev(torch_cuda, b_u[L0.maps.l2u])
                    x = torch_cuda.full_like(b, float("nan"))
                    it, rel = mg.fpcg(b, x, 1e-8, 60)
                    assert rel <= 1e-8 and abs(it - ores["iters"]) <= (0 if prec == binding.SEM_F64 else 1)
                    assert relerr(x.cpu().numpy(), ores["x"][L0.maps.l2u]) <= 1e-6
        finally:
            for s_ in sems:
                s_.close()


@pytest.mark.slow
def test_schwarz_config2_full_size_f32(torch_cuda, binding, oracle_mod):
    """VERDICT r1 item 5's bar: the Schwarz smoother at E = 7200, N = 7 in FP32 (the paper's preconditioner precision,
    P:109) against the FP64 oracle at 1e-5, and the flexible-PCG iteration count of the 7-3-1 cycle with Chebyshev-Schwarz
    smoothing at config 2 below the Chebyshev-Jacobi cycle's."""
    m = inputs.config2()
    maps = oracle_mod.Maps(m.gid)
    mask_u = oracle_mod.mask_unique(m.dirichlet, maps)
    sw = oracle_mod.Schwarz(m, maps, mask_u)
    r_u = np.where(mask_u != 0, 0.0, inputs.field_normal(maps.uniq_gid, 2))
    oz = sw.apply(r_u)[maps.l2u]
    side = torch_cuda.cuda.Stream()
    with torch_cuda.cuda.stream(side):
        lv = []
        for N in (7, 3, 1):
            mN = inputs.config4(N)
            lv.append(binding.Sem(mN.E, N, mN.vert, mN.gid, mN.dirichlet).geom())
        try:
            lv[0].schwarz_setup()
            dr = to_dev(torch_cuda, r_u[maps.l2u], torch_cuda.float32)
            dz = torch_cuda.full_like(dr, float("nan"))
            lv[0].schwarz(dr, dz)
            side.synchronize()
            assert relerr(dz.cpu().numpy(), oz) <= TOL32
            lv[1].schwarz_setup()
            lamj = [1.1 * s_.lambda_max(30) for s_ in lv]
            lams = [1.1 * lv[0].lambda_max_schwarz(0, 30), 1.1 * lv[1].lambda_max_schwarz(0, 30), lamj[2]]
            u = to_dev(torch_cuda, inputs.field_uniform(m.gid, 0).ravel())
            rhs = torch_cuda.empty_like(u)
            lv[0].ax_gs(u, rhs)
            x = torch_cuda.zeros_like(u)
            with binding.Pmg(lv, [0.1 * l for l in lamj], lamj, 2, 8, binding.SEM_F32) as mg:
                it_j, rel_j = mg.fpcg(rhs, x, 1e-8, 100)
                mg.set_smoother(binding.SEM_SMOOTH_CHEBY_SCHWARZ, [0.1 * l for l in lams], lams)
                it_s, rel_s = mg.fpcg(rhs, x, 1e-8, 100)
            assert rel_j <= 1e-8 and rel_s <= 1e-8 and it_s < it_j, (it_s, it_j)
        finally:
            for s_ in lv:
                s_.close()


# --------------------------------------------------------------------------- NEXT-4: several fields sharing the geometry
@pytest.mark.parametrize("N,nf,pad,dtype,lam", [(7, 3, 0, "f64", 0.0), (7, 3, 64, "f64", 7.5), (7, 2, 0, "f64", 0.0),
                                                (7, 5, 16, "f64", 0.0), (7, 4, 0, "f64", 3.0), (7, 1, 0, "f64", 0.0),
                                                (5, 3, 8, "f64", 0.0), (7, 3, 0, "f32", 0.0), (3, 3, 4, "f32", 2.0)])
def test_ax_gs_many_parity(torch_cuda, binding, oracle_mod, N, nf, pad, dtype, lam):
    """sem_ax_gs_many (the three velocity components share the geometry): every field against the oracle's
    independent M QQ^T (A_L + lambda B) u_f at 1e-12 / 1e-5.  FP64 N = 7 takes the fused kernel (groups of 3 and 2 fields
    read G once); other orders and FP32 run field by field.  More elements than resident warps; padded field stride."""
    m = inputs.box_mesh(13, 12, 11, N, "random", seed=2) if N == 7 else inputs.box_mesh(6, 5, 4, N, "random", seed=2)
    oG, _, rc = oracle_mod.geom_trilinear(m.vert, m.N)
    assert rc == 0
    om = oracle_mod.Maps(m.gid)
    msk = oracle_mod.mask_unique(m.dirichlet, om)[om.l2u] != 0
    tdt = torch_cuda.float64 if dtype == "f64" else torch_cuda.float32
    tol = TOL64 if dtype == "f64" else TOL32
    us = [inputs.field_uniform(m.gid, 30 + f) for f in range(nf)]
    ows = [np.where(msk, 0.0, oracle_mod.gs(oracle_mod.ax(oG, u, m.N, lam).ravel(), om)) for u in us]
    with binding.Sem(m.E, m.N, m.vert, m.gid, m.dirichlet) as sem:
        sem.geom(with_mass=lam != 0.0)
        stride = sem.nL + pad
        du = torch_cuda.zeros(nf, stride, device="cuda", dtype=tdt)
        for f in range(nf):
            du[f, :sem.nL] = to_dev(torch_cuda, us[f].ravel(), tdt)
        dw = torch_cuda.full_like(du, float("nan"))
        sem.ax_gs_many(du, dw, lam)
        torch_cuda.cuda.synchronize()
        for f in range(nf):
            assert relerr(dw[f, :sem.nL].cpu().numpy(), ows[f]) <= tol, (N, nf, f)
        if pad:
            assert bool(torch_cuda.isnan(dw[:, sem.nL:]).all())          # the padding is not touched
        # each field equals what sem_ax_gs gives for it alone (same arithmetic, same summation order in the gs)
        if dtype == "f64":
            w1 = torch_cuda.empty(sem.nL, device="cuda", dtype=tdt)
            sem.ax_gs(du[0, :sem.nL].contiguous(), w1, lam)
            assert relerr(w1.cpu().numpy(), ows[0]) <= tol


def test_pcg_many_matches_independent_solves(torch_cuda, binding, oracle_mod):
    """sem_pcg_many: three right-hand sides in lockstep, each with its own alpha / beta / stopping test -- every field
    reproduces the oracle's Jacobi-PCG on it alone (iteration count, relres, solution at 1e-9), although the fields
    converge at different iterations and one right-hand side is zero (0 iterations); Helmholtz shift lambda > 0 as in
    the velocity solves."""
    m = inputs.box_mesh(5, 4, 4, 7, "smooth")
    lam = 40.0
    oG, _, rc = oracle_mod.geom_trilinear(m.vert, m.N)
    om = oracle_mod.Maps(m.gid)
    mask_u = oracle_mod.mask_unique(m.dirichlet, om)
    xs = [np.where(mask_u != 0, 0.0, inputs.field_normal(om.uniq_gid, 50 + f)) for f in range(3)]
    xs[1] = xs[1] * 0.0
    xyz = oracle_mod.node_xyz(m.vert, m.N).reshape(-1, 3)
    smooth = np.zeros(om.U)
    smooth[om.l2u] = np.sin(np.pi * xyz[:, 0]) * np.sin(np.pi * xyz[:, 1]) * np.sin(np.pi * xyz[:, 2])
    xs[2] = np.where(mask_u != 0, 0.0, smooth)                       # a smooth solution: stops at another iteration
    bs = [oracle_mod.apply_Ag(oG, m.N, om, mask_u, x, lam) for x in xs]
    ores = [oracle_mod.pcg(oG, m.N, om, mask_u, b, tol=1e-9, maxit=400, lam=lam) for b in bs]
    assert ores[1]["iters"] == 0 and ores[2]["iters"] != ores[0]["iters"]
    with binding.Sem(m.E, m.N, m.vert, m.gid, m.dirichlet) as sem:
        sem.geom(with_mass=True)
        sem.set_lambda(lam)
        stride = sem.nL + 32
        b = torch_cuda.zeros(3, stride, device="cuda", dtype=torch_cuda.float64)
        for f in range(3):
            b[f, :sem.nL] = to_dev(torch_cuda, bs[f][om.l2u])
        x = torch_cuda.zeros_like(b)
        its, rels = sem.pcg_many(b, x, 1e-9, 400)
        for f in range(3):
            assert its[f] == ores[f]["iters"], (f, its, [o["iters"] for o in ores])
            assert abs(rels[f] - ores[f]["relres"]) <= 1e-4 * ores[f]["relres"] + 1e-30      # recurrence residual after ~140 iterations
            if ores[f]["iters"]:
                xo = ores[f]["x"][om.l2u]
                assert relerr(x[f, :sem.nL].cpu().numpy(), xo) <= TOLPCG, f
            else:
                assert float(x[f].abs().max()) == 0.0
        # maxit reached: every field reports maxit iterations
        x.zero_()
        its, _ = sem.pcg_many(b, x, 1e-30, 7)
        assert its[0] == 7 and its[1] == 0 and its[2] == 7


# --------------------------------------------------------------------------- NEXT-4: elements partitioned over ranks
@pytest.mark.parametrize("world,masked,dtype", [(2, True, "f64"), (3, False, "f64"), (4, True, "f32")])
def test_sharded_apply_emulated_on_one_gpu(torch_cuda, binding, oracle_mod, world, masked, dtype):
    """The sharded operator of paper_2110_01716_b200/sharded.py with all ranks' contexts on ONE GPU, phase by phase (local
    sem_ax_gs + sem_iface_pack on every rank, buffer hand-over, sem_iface_add on every rank; no kernel waits on another):
    every rank's result equals the single-context sem_ax_gs -- bit for bit on the nodes that live on one rank only, to
    round-off on interface nodes -- and the oracle.  Scrambled element order, so the interfaces are ragged and nodes are
    shared by up to `world` ranks."""
    from paper_2110_01716_b200 import sharded
    m = inputs.box_mesh(6, 5, 4, 7, "random", seed=8, permute_seed=2)
    tdt = torch_cuda.float64 if dtype == "f64" else torch_cuda.float32
    tol = TOL64 if dtype == "f64" else TOL32
    u = inputs.field_uniform(m.gid, 12)
    ow = _ax_gs_oracle(oracle_mod, m, u, masked).reshape(m.E, -1)
    with binding.Sem(m.E, m.N, m.vert, m.gid, m.dirichlet if masked else None) as one:
        one.geom()
        du = to_dev(torch_cuda, u.ravel(), tdt)
        w1 = torch_cuda.empty_like(du)
        one.ax_gs(du, w1)
        w1 = w1.cpu().numpy().reshape(m.E, -1)
    b = sharded.partition_bounds(m.E, world)
    gath = sharded.local_gathers(m.N, [m.gid[b[r]:b[r + 1]] for r in range(world)],
                                 [m.dirichlet[b[r]:b[r + 1]] if masked else None for r in range(world)])
    shards = []
    try:
        for r in range(world):
            sl = slice(b[r], b[r + 1])
            s = sharded.ShardedSem(sharded.LocalComm(r, world, *gath), b[r + 1] - b[r], m.N, m.vert[sl], m.gid[sl],
                                   m.dirichlet[sl] if masked else None, dtype=tdt)
            shards.append(s.geom())
        us = [to_dev(torch_cuda, shards[r].to_local(u[b[r]:b[r + 1]]).ravel(), tdt) for r in range(world)]
        ws = [torch_cuda.full_like(x, float("nan")) for x in us]
        sharded.emulated_ax_gs(shards, us, ws)
        torch_cuda.cuda.synchronize()
        n_shared = 0
        for r, s in enumerate(shards):
            got = ws[r].cpu().numpy().reshape(b[r + 1] - b[r], -1)
            maps = s.sem.maps()
            shared_u = np.zeros(maps["uniq_gid"].size, bool)
            for q in s.uniq.values():
                shared_u[q.cpu().numpy()] = True
            shared = s.from_local(shared_u[maps["l2u"]].reshape(got.shape))
            got = s.from_local(got)
            assert relerr(got, ow[b[r]:b[r + 1]]) <= tol * max(1.0, np.max(np.abs(ow)) / np.max(np.abs(ow[b[r]:b[r + 1]])))
            n_shared += int(shared.sum())
            assert np.array_equal(got[~shared], w1[b[r]:b[r + 1]][~shared])          # one rank only: bit-identical
            assert np.max(np.abs(got - w1[b[r]:b[r + 1]])) <= tol * np.max(np.abs(w1))
            for q, lst in s.plan.items():                                             # symmetric plan, same order
                assert np.array_equal(lst, shards[q].plan[r])
        assert n_shared > 0
    finally:
        for s in shards:
            s.close()


# --------------------------------------------------------------------------- fields larger than L2: chunked Ax / gs
@pytest.mark.parametrize("N,dtype", [(7, "f64"), (3, "f32"), (4, "f64"), (2, "f64")])
def test_chunked_ax_gs_is_bit_identical(torch_cuda, binding, oracle_mod, monkeypatch, N, dtype):
    """When the field does not fit in L2, sem_ax_gs alternates operator and gather-scatter chunk by chunk (records are
    sorted by the owner group of a node's last copy).  Forced here on a small scrambled mesh through SEM_CHUNK_GROUPS:
    the result is bit-identical to the un-chunked path, equals the oracle, and the PCG loop (fused dot, skip flag) runs
    through it unchanged."""
    import os
    m = inputs.box_mesh(6, 5, 4, N, "random", seed=4, permute_seed=9)
    u = inputs.field_uniform(m.gid, 5)
    ow = _ax_gs_oracle(oracle_mod, m, u, True)
    tdt = torch_cuda.float64 if dtype == "f64" else torch_cuda.float32
    outs, its, xs = [], [], []
    for chunk in (None, "3", "7"):
        if chunk is None:
            monkeypatch.delenv("SEM_CHUNK_GROUPS", raising=False)
        else:
            monkeypatch.setenv("SEM_CHUNK_GROUPS", chunk)
        with binding.Sem(m.E, m.N, m.vert, m.gid, m.dirichlet) as sem:
            sem.geom()
            du = to_dev(torch_cuda, u.ravel(), tdt)
            dw = torch_cuda.full_like(du, float("nan"))
            sem.ax_gs(du, dw)
            torch_cuda.cuda.synchronize()
            outs.append(dw.clone())
            if dtype == "f64":
                b = dw.clone()
                x = torch_cuda.zeros_like(b)
                its.append(sem.pcg(b, x, 1e-10, 300)[0])
                xs.append(x.cpu().numpy())
    assert relerr(outs[0].cpu().numpy(), ow) <= (TOL64 if dtype == "f64" else TOL32)
    assert torch_cuda.equal(outs[1], outs[0]) and torch_cuda.equal(outs[2], outs[0])
    assert len(set(its)) <= 1 and all(relerr(x, xs[0]) <= 1e-9 for x in xs[1:])


# --------------------------------------------------------------------------- element renumbering inside sem_pcg
@pytest.mark.parametrize("iso", [False, True])
def test_pcg_through_the_inner_renumbered_context(torch_cuda, binding, oracle_mod, monkeypatch, iso):
    """Large meshes in an element order without locality get a second context over the same elements sorted by their
    smallest global id, and sem_pcg runs there (b, x gathered / scattered in 4 KB blocks).  Forced here with SEM_INNER=1 on
    a small scrambled mesh: iteration count, residual history and solution equal the oracle's, with trilinear and with
    isoparametric (node_xyz) geometry, a non-zero initial guess and the Helmholtz shift; a lexicographic mesh of the same
    size gets no inner context even when large (checked through the unchanged result with SEM_INNER unset)."""
    m = inputs.box_mesh(5, 4, 4, 5, "random", seed=7, permute_seed=11)
    lam = 3.0
    om = oracle_mod.Maps(m.gid)
    xyz = oracle_mod.node_xyz(m.vert, m.N)
    if iso:
        oG, _, rc = oracle_mod.geom_iso(xyz, m.N)
    else:
        oG, _, rc = oracle_mod.geom_trilinear(m.vert, m.N)
    assert rc == 0
    mask_u = oracle_mod.mask_unique(m.dirichlet, om)
    xs = np.where(mask_u != 0, 0.0, inputs.field_normal(om.uniq_gid, 9))
    x0 = np.where(mask_u != 0, 0.0, 0.3 * inputs.field_normal(om.uniq_gid, 10))
    b_u = oracle_mod.apply_Ag(oG, m.N, om, mask_u, xs, lam)
    ores = oracle_mod.pcg(oG, m.N, om, mask_u, b_u, x0_u=x0, tol=1e-10, maxit=300, lam=lam)
    results = []
    for inner in ("1", None):
        if inner is None:
            monkeypatch.delenv("SEM_INNER", raising=False)
        else:
            monkeypatch.setenv("SEM_INNER", inner)
        with binding.Sem(m.E, m.N, m.vert, m.gid, m.dirichlet) as sem:
            sem.geom(node_xyz=xyz if iso else None, with_mass=True)
            sem.set_lambda(lam)
            b = to_dev(torch_cuda, b_u[om.l2u])
            x = to_dev(torch_cuda, x0[om.l2u])
            it, rel = sem.pcg(b, x, 1e-10, 300)
            assert it == ores["iters"], (inner, it, ores["iters"])
            assert relerr(x.cpu().numpy(), ores["x"][om.l2u]) <= TOLPCG
            h = sem.pcg_history(it + 1)
            assert np.max(np.abs(h - ores["hist"]) / ores["hist"]) <= 1e-5
            results.append(x.cpu().numpy())
            # the operator on the caller's vectors is untouched by the inner context
            du = to_dev(torch_cuda, inputs.field_uniform(m.gid, 3).ravel())
            dw = torch_cuda.empty_like(du)
            sem.ax_gs(du, dw, lam)
            ow = oracle_mod.gs(oracle_mod.ax(oG, inputs.field_uniform(m.gid, 3), m.N, lam).ravel(), om)
            assert relerr(dw.cpu().numpy(), np.where(mask_u[om.l2u] != 0, 0.0, ow)) <= TOL64
    assert relerr(results[0], results[1]) <= 1e-9


def test_recompute_mode_keeps_no_stored_G_and_handles_helmholtz_in_fp32(torch_cuda, binding, oracle_mod):
    """SEM_G_RECOMPUTE (a9): no stored G is kept, yet the Jacobi diagonal, sem_get_geom and the PCG loop work
    (G is rebuilt for the duration of those calls), and the FP32 operator with lambda > 0 finds its mass factor."""
    m = inputs.box_mesh(5, 4, 3, 7, "random", seed=6)
    lam = 4.0
    oG, odJ, rc = oracle_mod.geom_trilinear(m.vert, m.N)
    om = oracle_mod.Maps(m.gid)
    mask_u = oracle_mod.mask_unique(m.dirichlet, om)
    u = inputs.field_uniform(m.gid, 2)
    ow = oracle_mod.ax(oG, u, m.N, lam)
    with binding.Sem(m.E, m.N, m.vert, m.gid, m.dirichlet) as sem:
        sem.geom(mode=binding.SEM_G_RECOMPUTE, with_mass=True)
        sem.set_lambda(lam)
        for dt, tol in ((torch_cuda.float64, TOL64), (torch_cuda.float32, TOL32)):
            du = to_dev(torch_cuda, u.ravel(), dt)
            dw = torch_cuda.full_like(du, float("nan"))
            sem.ax(du, dw, lam)
            assert relerr(dw.cpu().numpy().reshape(ow.shape), ow) <= tol, dt
        G, dJ = sem.get_geom()
        assert np.max(np.abs(G - oG)) <= 1e-12 * np.max(np.abs(oG)) and np.max(np.abs(dJ - odJ)) <= 1e-12 * np.max(np.abs(odJ))
        xs = np.where(mask_u != 0, 0.0, inputs.field_normal(om.uniq_gid, 5))
        b_u = oracle_mod.apply_Ag(oG, m.N, om, mask_u, xs, lam)
        ores = oracle_mod.pcg(oG, m.N, om, mask_u, b_u, tol=1e-9, maxit=200, lam=lam)
        b = to_dev(torch_cuda, b_u[om.l2u])
        x = torch_cuda.zeros_like(b)
        it, _ = sem.pcg(b, x, 1e-9, 200)
        assert it == ores["iters"] and relerr(x.cpu().numpy(), ores["x"][om.l2u]) <= TOLPCG


@pytest.mark.parametrize("m,E", [(10, 900), (8, 700), (6, 500), (12, 300), (7, 450)])
def test_fdm_apply_tensor_core_variant(torch_cuda, binding, oracle_mod, m, E):
    """The FP32 tensor-core variant of the local solve (sem_set_variant(101): TF32 m16n8k8 in three passes, lines padded
    to MMA tiles) against the oracle's Eq. (3) at 1e-5, in place and out of place."""
    mesh = inputs.box_mesh(E, 1, 1, 1)
    A, B = inputs.fdm_pairs(E, m, seed=70 + m)
    S = np.empty_like(A)
    lam = []
    for e in range(E):
        le = []
        for d in range(3):
            S[e, d], l = oracle_mod.fdm_eig(A[e, d], B[e, d])
            le.append(l)
        lam.append(oracle_mod.fdm_inv_lambda(*le))
    iL = np.stack(lam)
    b = 2.0 * inputs.hash_uniform01(9, 12, np.arange(E * m ** 3)).reshape(E, m, m, m) - 1.0
    ou = oracle_mod.fdm_apply(S, iL, b)
    with binding.Sem(mesh.E, 1, mesh.vert, mesh.gid) as sem:
        sem.set_variant(101)
        dS, dL, db = (to_dev(torch_cuda, a.ravel(), torch_cuda.float32) for a in (S, iL, b))
        du = torch_cuda.full_like(db, float("nan"))
        sem.fdm_apply(m, dS, dL, db, du)
        torch_cuda.cuda.synchronize()
        assert relerr(du.cpu().numpy(), ou.ravel()) <= TOL32
        sem.fdm_apply(m, dS, dL, db, db)
        assert torch_cuda.equal(db, du)


def test_pcg_graph_replay_on_side_stream(torch_cuda, binding, oracle_mod):
    """On a non-default stream sem_pcg replays one CUDA graph of 16 iterations (iteration number and p.q kept on the
    device): the config-1 trajectory after 20 iterations (maxit ends inside the second batch), a converged solve
    (iteration count, history, solution) and a zero right-hand side equal the oracle's, as on the default stream."""
    m = inputs.config1()
    om = oracle_mod.Maps(m.gid)
    oG, _, rc = oracle_mod.geom_trilinear(m.vert, m.N)
    mask_u = oracle_mod.mask_unique(m.dirichlet, om)
    xyz = oracle_mod.node_xyz(m.vert, m.N).reshape(-1, 3)
    us = np.zeros(om.U)
    us[om.l2u] = np.sin(np.pi * xyz[:, 0]) * np.sin(np.pi * xyz[:, 1]) * np.sin(np.pi * xyz[:, 2])
    us[mask_u != 0] = 0.0
    b_u = oracle_mod.apply_Ag(oG, m.N, om, mask_u, us)
    o20 = oracle_mod.pcg(oG, m.N, om, mask_u, b_u, tol=1e-30, maxit=20)
    ofull = oracle_mod.pcg(oG, m.N, om, mask_u, b_u, tol=1e-10, maxit=400)
    side = torch_cuda.cuda.Stream()
    with torch_cuda.cuda.stream(side):
        with binding.Sem(m.E, m.N, m.vert, m.gid, m.dirichlet) as sem:
            sem.geom()
            b = to_dev(torch_cuda, b_u[om.l2u])
            for _ in range(2):                                   # the second call builds its graph anew
                x = torch_cuda.zeros_like(b)
                it, rel = sem.pcg(b, x, 1e-30, 20)
                assert it == 20 and abs(rel - o20["relres"]) <= 1e-9 * o20["relres"]
                assert relerr(x.cpu().numpy(), o20["x"][om.l2u]) <= TOLPCG
            x = torch_cuda.zeros_like(b)
            it, rel = sem.pcg(b, x, 1e-10, 400)
            assert it == ofull["iters"] and rel <= 1e-10
            assert relerr(x.cpu().numpy(), ofull["x"][om.l2u]) <= TOLPCG
            h = sem.pcg_history(it + 1)
            big = ofull["hist"] >= 1e-4                          # below that the recurrence residual drifts by round-off
            assert np.max(np.abs(h - ofull["hist"])[big] / ofull["hist"][big]) <= 1e-5
            xz = torch_cuda.ones_like(b)
            itz, relz = sem.pcg(torch_cuda.zeros_like(b), xz.zero_(), 1e-8, 50)
            assert itz == 0


# --------------------------------------------------------------------------- arbitrary element orientations
@pytest.mark.parametrize("N", [7, 4, 3])
def test_reoriented_elements(torch_cuda, binding, oracle_mod, N):
    """Every element's local frame rotated by a seeded proper rotation (inputs.reorient), scrambled element order:
    neighbours meet with arbitrary relative orientation, as in an unstructured hexahedral mesh.  Maps bit-exact, Ax+gs
    1e-12, Jacobi-PCG at equal iteration count 1e-9, and the Schwarz smoother -- whose face links (base, two strides,
    axis and side of the neighbour's face) now take every value -- setup bit-exact / 1e-13 and both variants 1e-10 / 1e-5;
    the sharded operator over 3 emulated ranks equals the single-context one."""
    from paper_2110_01716_b200 import sharded
    m = inputs.reorient(inputs.box_mesh(4, 3, 3, N, "random", seed=21, permute_seed=6), 13)
    om = oracle_mod.Maps(m.gid)
    oG, _, rc = oracle_mod.geom_trilinear(m.vert, m.N)
    assert rc == 0
    mask_u = oracle_mod.mask_unique(m.dirichlet, om)
    u = inputs.field_uniform(m.gid, 8)
    ow = np.where(mask_u[om.l2u] != 0, 0.0, oracle_mod.gs(oracle_mod.ax(oG, u, m.N).ravel(), om))
    xs = np.where(mask_u != 0, 0.0, inputs.field_normal(om.uniq_gid, 9))
    b_u = oracle_mod.apply_Ag(oG, m.N, om, mask_u, xs)
    ores = oracle_mod.pcg(oG, m.N, om, mask_u, b_u, tol=1e-9, maxit=400)
    with binding.Sem(m.E, m.N, m.vert, m.gid, m.dirichlet) as sem:
        mp = sem.maps()
        for k in ("l2u", "mult", "seg_off", "seg_idx", "uniq_gid"):
            assert np.array_equal(mp[k], getattr(om, k)), k
        sem.geom()
        du = to_dev(torch_cuda, u.ravel())
        dw = torch_cuda.full_like(du, float("nan"))
        sem.ax_gs(du, dw)
        assert relerr(dw.cpu().numpy(), ow) <= TOL64
        w1 = dw.cpu().numpy()
        b = to_dev(torch_cuda, b_u[om.l2u])
        x = torch_cuda.zeros_like(b)
        it, _ = sem.pcg(b, x, 1e-9, 400)
        assert it == ores["iters"] and relerr(x.cpu().numpy(), ores["x"][om.l2u]) <= TOLPCG
        sem.schwarz_setup()
        r_u = np.where(mask_u != 0, 0.0, inputs.field_normal(om.uniq_gid, 21))
        for kind, restricted in ((binding.SEM_SCHWARZ_ASM, False), (binding.SEM_SCHWARZ_RAS, True)):
            sw = oracle_mod.Schwarz(m, om, mask_u, restricted)
            nbr, A, B, W = sem.get_schwarz(kind)
            assert np.array_equal(nbr, sw.nbr)
            assert np.max(np.abs(A - sw.A1)) <= 1e-13 * np.max(np.abs(sw.A1))
            assert np.max(np.abs(B - sw.B1)) <= 1e-13 * np.max(np.abs(sw.B1))
            oz = sw.apply(r_u)[om.l2u]
            for dt, tol in ((torch_cuda.float64, 1e-10), (torch_cuda.float32, TOL32)):
                dr = to_dev(torch_cuda, r_u[om.l2u], dt)
                dz = torch_cuda.full_like(dr, float("nan"))
                sem.schwarz(dr, dz, kind)
                assert relerr(dz.cpu().numpy(), oz) <= tol, (N, kind, dt)
    world = 3
    bnd = sharded.partition_bounds(m.E, world)
    gath = sharded.local_gathers(m.N, [m.gid[bnd[r]:bnd[r + 1]] for r in range(world)],
                                 [m.dirichlet[bnd[r]:bnd[r + 1]] for r in range(world)])
    shards = []
    try:
        for r in range(world):
            sl = slice(bnd[r], bnd[r + 1])
            shards.append(sharded.ShardedSem(sharded.LocalComm(r, world, *gath), bnd[r + 1] - bnd[r], m.N, m.vert[sl],
                                             m.gid[sl], m.dirichlet[sl]).geom())
        us = [to_dev(torch_cuda, shards[r].to_local(u.reshape(m.E, -1)[bnd[r]:bnd[r + 1]]).ravel()) for r in range(world)]
        ws = [torch_cuda.full_like(v, float("nan")) for v in us]
        sharded.emulated_ax_gs(shards, us, ws)
        got = np.concatenate([s.from_local(w.cpu().numpy().reshape(s.E, -1)).ravel() for s, w in zip(shards, ws)])
        assert np.max(np.abs(got - w1)) <= TOL64 * np.max(np.abs(w1))
    finally:
        for s in shards:
            s.close()


def test_vcycle_ras_on_reoriented_levels(torch_cuda, binding, oracle_mod):
    """The 7-3-1 V-cycle with Chebyshev-RAS smoothing (order 1) on levels whose elements are all rotated the same seeded
    way (the transfers are element-local tensor products, so every level must use the same frames): the cycle equals the
    oracle's (FP64 1e-9) and flexible PCG takes the oracle's iteration count."""
    orders = (7, 3, 1)
    meshes = [inputs.reorient(inputs.box_mesh(4, 3, 3, N, "random", seed=3), 5) for N in orders]
    olv = [oracle_mod.Level(m) for m in meshes]
    for L, m in zip(olv[:-1], meshes[:-1]):
        L.use_schwarz(m, restricted=True)
    L0 = olv[0]
    xs = np.where(L0.mask_u != 0, 0.0, inputs.field_normal(L0.maps.uniq_gid, 17))
    b_u = L0.A(xs)
    oz = oracle_mod.vcycle(olv, b_u, 1, 8)
    ores = oracle_mod.fpcg(L0, lambda r: oracle_mod.vcycle(olv, r, 1, 8), b_u, tol=1e-8, maxit=60)
    side = torch_cuda.cuda.Stream()
    with torch_cuda.cuda.stream(side):
        sems = [binding.Sem(m.E, m.N, m.vert, m.gid, m.dirichlet).geom() for m in meshes]
        try:
            slmin = [getattr(l, "slmin", l.lmin) for l in olv]
            slmax = [getattr(l, "slmax", l.lmax) for l in olv]
            with binding.Pmg(sems, [l.lmin for l in olv], [l.lmax for l in olv], 1, 8, binding.SEM_F64) as mg:
                mg.set_smoother(binding.SEM_SMOOTH_CHEBY_RAS, slmin, slmax)
                dr = to_dev(torch_cuda, b_u[L0.maps.l2u])
                dz = torch_cuda.full_like(dr, float("nan"))
                for _ in range(3):
                    mg.vcycle(dr, dz)
                side.synchronize()
                assert relerr(dz.cpu().numpy(), oz[L0.maps.l2u]) <= 1e-9
                x = torch_cuda.full_like(dr, float("nan"))
                it, rel = mg.fpcg(dr, x, 1e-8, 60)
                assert rel <= 1e-8 and it == ores["iters"]
                assert relerr(x.cpu().numpy(), ores["x"][L0.maps.l2u]) <= 1e-7
        finally:
            for s_ in sems:
                s_.close()


@pytest.mark.parametrize("masked,lam,order,zero_guess", [(True, 0.0, 8, True), (False, 2.5, 5, False), (True, 1.0, 1, True),
                                                         (True, 0.0, 2, False)])
def test_assembled_coarse_operator(torch_cuda, binding, oracle_mod, monkeypatch, masked, lam, order, zero_guess):
    """N = 1: sem_cheby runs on the assembled operator (one kernel per Chebyshev step, no gather-scatter).  Against the
    oracle's Chebyshev-Jacobi and against the matrix-free path (SEM_COARSE=0), FP64 1e-11 and FP32 1e-5, masked and not,
    Helmholtz, zero and non-zero guess, re-oriented scrambled elements; the result stays continuous bit for bit."""
    m = inputs.reorient(inputs.box_mesh(6, 5, 4, 1, "random", seed=12, permute_seed=3), 2)
    if not masked:
        m.dirichlet[:] = 0
    L = oracle_mod.Level(m, power_its=30, lam=lam)
    b_u = L.A(np.where(L.mask_u != 0, 0.0, inputs.field_normal(L.maps.uniq_gid, 3))) + 0.1
    b_u[L.mask_u != 0] = 0.0
    x0_u = None if zero_guess else np.where(L.mask_u != 0, 0.0, inputs.field_normal(L.maps.uniq_gid, 4))
    ox = L.smooth(b_u, x0_u, order)[L.maps.l2u]
    outs = {}
    for env in ("1", "0"):
        monkeypatch.setenv("SEM_COARSE", env)
        with binding.Sem(m.E, m.N, m.vert, m.gid, m.dirichlet if masked else None) as sem:
            sem.geom(with_mass=lam != 0.0)
            sem.set_lambda(lam)
            for dt, tol in ((torch_cuda.float64, 1e-11), (torch_cuda.float32, TOL32)):
                db = to_dev(torch_cuda, b_u[L.maps.l2u], dt)
                dx = torch_cuda.full_like(db, float("nan")) if zero_guess else to_dev(torch_cuda, x0_u[L.maps.l2u], dt)
                sem.cheby(db, dx, order, L.lmin, L.lmax, zero_guess)
                torch_cuda.cuda.synchronize()
                got = dx.cpu().numpy()
                assert relerr(got, ox) <= tol, (env, dt)
                outs[(env, dt)] = got
                if env == "1":                                  # every copy of a unique node holds the same bits
                    first = L.maps.seg_idx[L.maps.seg_off[:-1]]
                    assert np.array_equal(got, got[first][L.maps.l2u])
    assert relerr(outs[("1", torch_cuda.float64)], outs[("0", torch_cuda.float64)]) <= 1e-12


# --------------------------------------------------------------------------- NEXT-4: sharded solver and overlapped apply
def _thread_shards(torch_cuda, sharded, m, world, masked=True, lam_mass=False):
    bnd = sharded.partition_bounds(m.E, world)
    gath = sharded.local_gathers(m.N, [m.gid[bnd[r]:bnd[r + 1]] for r in range(world)],
                                 [m.dirichlet[bnd[r]:bnd[r + 1]] if masked else None for r in range(world)])
    tw = sharded.ThreadWorld(world, timeout=120.0)
    shards = []
    for r in range(world):
        sl = slice(bnd[r], bnd[r + 1])
        s = sharded.ShardedSem(sharded.ThreadComm(tw, r, *gath), bnd[r + 1] - bnd[r], m.N, m.vert[sl], m.gid[sl],
                               m.dirichlet[sl] if masked else None)
        shards.append(s.geom(with_mass=lam_mass))
    return bnd, tw, shards


@pytest.mark.parametrize("world,lam,permute", [(2, 0.0, None), (3, 1.5, 2), (4, 0.0, 2), (3, 0.0, None)])
def test_sharded_pcg_and_overlapped_apply(torch_cuda, binding, oracle_mod, monkeypatch, world, lam, permute):
    """sem_ax_gs_sharded and sem_pcg_sharded with every rank's library call on its own host thread of ONE GPU (buffers
    handed over by device copies between host barriers; no kernel waits on another).  The elements of each rank are
    ordered interface-first, so the exchange starts after the interface chunk (sem_shard_set_interface).  Checked:
    the apply against the oracle and the single-context call (bit-identical off the interface); the solve against the
    oracle's PCG on the whole mesh -- same iteration count, residual history, solution -- and every rank reports the
    same iteration count and residual."""
    from paper_2110_01716_b200 import sharded
    m = (inputs.box_mesh(6, 5, 4, 7, "random", seed=8, permute_seed=permute) if permute is not None
         else inputs.box_mesh(4, 3, 3 * world, 7, "random", seed=8))          # slabs of 3 element layers per rank
    if world == 3 and permute is None:
        monkeypatch.setenv("SEM_CHUNK_GROUPS", "2")     # the interior part is itself cut into several chunks
    om = oracle_mod.Maps(m.gid)
    oG, _, _ = oracle_mod.geom_trilinear(m.vert, m.N)
    mask_u = oracle_mod.mask_unique(m.dirichlet, om)
    xs = np.where(mask_u != 0, 0.0, inputs.field_normal(om.uniq_gid, 5))
    b_u = oracle_mod.apply_Ag(oG, m.N, om, mask_u, xs, lam)
    ores = oracle_mod.pcg(oG, m.N, om, mask_u, b_u, tol=1e-9, maxit=400, lam=lam)
    u = inputs.field_uniform(m.gid, 12).reshape(m.E, -1)
    u_u = np.zeros(om.U)
    u_u[om.l2u] = u.ravel()
    with binding.Sem(m.E, m.N, m.vert, m.gid, m.dirichlet) as one:
        one.geom(with_mass=lam != 0.0)
        du = to_dev(torch_cuda, u.ravel())
        w1 = torch_cuda.empty_like(du)
        one.ax_gs(du, w1, lam)
        w1 = w1.cpu().numpy().reshape(m.E, -1)
    ow = oracle_mod.apply_Ag(oG, m.N, om, np.zeros_like(mask_u), u_u, lam)   # u is continuous: A_g on unique nodes
    ow = np.where(mask_u != 0, 0.0, ow)[om.l2u].reshape(m.E, -1)
    assert relerr(w1, ow) <= TOL64
    bnd, tw, shards = _thread_shards(torch_cuda, sharded, m, world, lam_mass=lam != 0.0)
    try:
        assert all(0 < s.n_iface <= s.E for s in shards)
        if permute is None:                              # lexicographic order: slabs, the interface is one or two layers
            for s in shards:
                e0, ic = s.sem.chunks()
                assert s.n_iface < s.E and ic == 1 and len(e0) >= 3 and s.n_iface <= e0[1] < s.E
                if world == 3:
                    assert len(e0) > 3
        us = [to_dev(torch_cuda, s.to_local(u[bnd[r]:bnd[r + 1]]).ravel()) for r, s in enumerate(shards)]
        ws = [torch_cuda.full_like(v, float("nan")) for v in us]
        for s in shards:
            s.sem.set_lambda(lam)
        sharded.run_ranks(world, lambda r: shards[r].ax_gs(us[r], ws[r], lam), tw)
        torch_cuda.cuda.synchronize()
        for r, s in enumerate(shards):
            got = s.from_local(ws[r].cpu().numpy().reshape(s.E, -1))
            ref = w1[bnd[r]:bnd[r + 1]]
            assert np.max(np.abs(got - ref)) <= TOL64 * np.max(np.abs(w1))
            maps = s.sem.maps()
            shared_u = np.zeros(maps["uniq_gid"].size, bool)
            for q in s.uniq.values():
                shared_u[q.cpu().numpy()] = True
            shared = s.from_local(shared_u[maps["l2u"]].reshape(s.E, -1))
            few = s.from_local(maps["mult"][maps["l2u"]].reshape(s.E, -1)) <= 2   # a + b has one rounding in any order;
            assert np.array_equal(got[~shared & few], ref[~shared & few])          # 3+ copies: the interface-first
            assert (~shared & few).sum() > 0.3 * got.size                          # element order changes the sum order
        # the solve
        b_l = b_u[om.l2u].reshape(m.E, -1)
        bs = [to_dev(torch_cuda, s.to_local(b_l[bnd[r]:bnd[r + 1]]).ravel()) for r, s in enumerate(shards)]
        xs_d = [torch_cuda.zeros_like(v) for v in bs]
        res = sharded.run_ranks(world, lambda r: shards[r].pcg(bs[r], xs_d[r], 1e-9, 400), tw)
        torch_cuda.cuda.synchronize()
        assert all(rr == res[0] for rr in res)                       # same bits on every rank
        assert res[0][0] == ores["iters"] and res[0][1] <= 1e-9
        x_or = ores["x"][om.l2u].reshape(m.E, -1)
        for r, s in enumerate(shards):
            got = s.from_local(xs_d[r].cpu().numpy().reshape(s.E, -1))
            assert np.max(np.abs(got - x_or[bnd[r]:bnd[r + 1]])) <= 1e-8 * np.max(np.abs(x_or))
            hist = s.sem.pcg_history(res[0][0] + 1)
            big = ores["hist"] >= 1e-5
            assert np.max(np.abs(hist[big] - ores["hist"][big]) / ores["hist"][big]) <= 1e-6
        # fixed iteration count ending between two polls of the flag, zero right-hand side
        xs2 = [torch_cuda.zeros_like(v) for v in bs]
        res2 = sharded.run_ranks(world, lambda r: shards[r].pcg(bs[r], xs2[r], 1e-30, 11), tw)
        assert all(rr[0] == 11 for rr in res2)
        assert abs(res2[0][1] - ores["hist"][11]) <= 1e-6 * ores["hist"][11]
        zs = [torch_cuda.zeros_like(v) for v in bs]
        res3 = sharded.run_ranks(world, lambda r: shards[r].pcg(zs[r], xs2[r].zero_(), 1e-8, 10), tw)
        assert all(rr == (0, 0.0) for rr in res3)
    finally:
        for s in shards:
            s.close()


def test_sharded_hooks_nccl_world1(torch_cuda, binding, oracle_mod):
    """The NCCL transport of sharded.DistComm in a one-rank process group on the GPU: the all-reduce hook works in place
    on the library's device scalars (a raw address wrapped as a tensor), there are no peers, and sem_pcg_sharded takes
    the iterations of sem_pcg on the same context."""
    import torch.distributed as dist

    from paper_2110_01716_b200 import sharded
    os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
    os.environ.setdefault("MASTER_PORT", "29547")
    own = not dist.is_initialized()
    if own:
        dist.init_process_group("nccl", rank=0, world_size=1, device_id=torch_cuda.device("cuda", 0))
    try:
        m = inputs.box_mesh(4, 3, 3, 7, "random", seed=4, permute_seed=1)
        om = oracle_mod.Maps(m.gid)
        oG, _, _ = oracle_mod.geom_trilinear(m.vert, m.N)
        mask_u = oracle_mod.mask_unique(m.dirichlet, om)
        b_u = oracle_mod.apply_Ag(oG, m.N, om, mask_u, np.where(mask_u != 0, 0.0, inputs.field_normal(om.uniq_gid, 2)))
        comm = sharded.DistComm()
        t = torch_cuda.arange(4, device="cuda", dtype=torch_cuda.float64)
        v = sharded.device_view(t.data_ptr() + 8, 2)
        v += 10.0
        assert t.tolist() == [0.0, 11.0, 12.0, 3.0]
        sh = sharded.ShardedSem(comm, m.E, m.N, m.vert, m.gid, m.dirichlet).geom()
        try:
            assert sh.plan == {} and sh.n_iface == 0
            b = to_dev(torch_cuda, b_u[om.l2u])
            x = torch_cuda.zeros_like(b)
            it, rel = sh.pcg(b, x, 1e-9, 300)
            x1 = torch_cuda.zeros_like(b)
            it1, rel1 = sh.sem.pcg(b, x1, 1e-9, 300)
            assert it == it1 and abs(rel - rel1) <= 1e-6 * rel1
            assert relerr(x.cpu().numpy(), x1.cpu().numpy()) <= 1e-9
        finally:
            sh.close()
    finally:
        if own:
            dist.destroy_process_group()


@pytest.mark.parametrize("N,nf", [(3, 2), (7, 3), (4, 4), (1, 2), (7, 4)])
def test_gs_many_node_interleaved(torch_cuda, binding, oracle_mod, N, nf):
    """sem_gs_many with field_stride = SEM_INTERLEAVED (fields stored [nL][nf]; 16-byte vector accesses when nf values fill
    whole 16-byte words): every field bit-identical to the oracle's gather-scatter (same ascending-index sums), FP32
    1e-6; 1 or 5 fields are refused."""
    m = inputs.box_mesh(4, 4, 3, N, permute_seed=6)
    om = oracle_mod.Maps(m.gid)
    rng = np.random.default_rng(300 + N)
    w = rng.standard_normal((nf, m.nL))
    ow = np.stack([oracle_mod.gs(w[f].copy(), om) for f in range(nf)])
    with binding.Sem(m.E, m.N, m.vert, m.gid) as sem:
        dw = to_dev(torch_cuda, np.ascontiguousarray(w.T))
        sem.gs_many(dw, interleaved=True)
        assert np.array_equal(dw.cpu().numpy().T, ow)
        d32 = to_dev(torch_cuda, np.ascontiguousarray(w.T.astype(np.float32)))
        sem.gs_many(d32, interleaved=True)
        assert relerr(d32.cpu().numpy().T, ow) <= 1e-6
        for bad in (1, 5):
            with pytest.raises(binding.SemError):
                sem._check(sem._L.sem_gs_many(sem._h, dw.data_ptr(), bad, binding.SEM_INTERLEAVED, binding.SEM_F64,
                                              binding.SEM_OP_ADD))


@pytest.mark.parametrize("lam", [0.0, 2.5])
def test_ax_recomputed_G_tensor_core_kernel(torch_cuda, binding, oracle_mod, lam):
    """a9 at p = 8, FP64: ax_dmma_rg (the factors recomputed in registers from the 8 vertices, contractions on the tensor
    cores) with several elements per persistent warp (both u / vertex buffers and their barrier phases wrap) and a ragged
    last round; against the oracle (1e-12), the stored-G operator and ax_simple's recomputation; Helmholtz term included."""
    m = inputs.box_mesh(14, 13, 13, 7, "random", seed=9, permute_seed=1)          # 2366 elements on <= 1184 warps
    oG, _, rc = oracle_mod.geom_trilinear(m.vert, m.N)
    assert rc == 0
    u = inputs.field_uniform(m.gid, 4)
    ow = oracle_mod.ax(oG, u, m.N, lam)
    du = to_dev(torch_cuda, u.ravel())
    got = {}
    for mode, variant in ((binding.SEM_G_RECOMPUTE, 0), (binding.SEM_G_RECOMPUTE, 1), (binding.SEM_G_STORED, 0)):
        with binding.Sem(m.E, m.N, m.vert, m.gid) as sem:
            sem.geom(mode=mode, with_mass=lam != 0.0)
            sem.set_variant(variant)
            dw = torch_cuda.full_like(du, float("nan"))
            sem.ax(du, dw, lam)
            got[(mode, variant)] = dw.cpu().numpy().reshape(ow.shape)
            if mode == binding.SEM_G_RECOMPUTE and variant == 0:                  # run to run: bit-identical
                dw2 = torch_cuda.full_like(du, float("nan"))
                sem.ax(du, dw2, lam)
                assert torch_cuda.equal(dw, dw2)
    for k, w in got.items():
        assert relerr(w, ow) <= TOL64, k


@pytest.mark.parametrize("N,dtype", [(1, "f64"), (2, "f32"), (3, "f64"), (4, "f64"), (4, "f32"), (5, "f64"), (6, "f64"),
                                     (6, "f32"), (7, "f32"), (8, "f64"), (9, "f64"), (9, "f32"), (10, "f64"), (11, "f64"),
                                     (11, "f32"), (7, "f64v2")])
def test_ax_recomputed_G_streaming_kernel(torch_cuda, binding, oracle_mod, N, dtype):
    """a9 at the other orders: ax_stream<..., RG> (no G ring; the factors recomputed per node from the vertices) with more
    element groups than resident CTAs (the u buffers wrap, ragged last group), Helmholtz term included, against the
    oracle -- FP64 1e-12, FP32 1e-5 -- and against ax_simple's recomputation."""
    n = {1: 30, 2: 24, 3: 22, 4: 18, 5: 16, 6: 15, 7: 14, 8: 13, 9: 12, 10: 11, 11: 11}[N]
    m = inputs.box_mesh(n, n, n + 1, N, "random", seed=20 + N, permute_seed=N)
    variant = 2 if dtype == "f64v2" else 0                      # p = 8 FP64: variant 2 selects the streaming kernel
    f64 = dtype != "f32"
    tdt, tol = (torch_cuda.float64, TOL64) if f64 else (torch_cuda.float32, TOL32)
    lam = 1.5
    oG, _, rc = oracle_mod.geom_trilinear(m.vert, m.N)
    assert rc == 0
    u = inputs.field_uniform(m.gid, 6)
    ow = oracle_mod.ax(oG, u, m.N, lam)
    du = to_dev(torch_cuda, u.ravel(), tdt)
    with binding.Sem(m.E, m.N, m.vert, m.gid) as sem:
        sem.geom(mode=binding.SEM_G_RECOMPUTE, with_mass=True)
        outs = []
        for v in (variant, 1):
            sem.set_variant(v)
            dw = torch_cuda.full_like(du, float("nan"))
            sem.ax(du, dw, lam)
            outs.append(dw.cpu().numpy().reshape(ow.shape))
            assert relerr(outs[-1], ow) <= tol, v
        assert relerr(outs[0], outs[1].astype(np.float64)) <= 10 * tol


@pytest.mark.parametrize("N,inner", [(7, "0"), (5, "0"), (7, "1")])
def test_recomputed_G_through_chunks_and_inner_context(torch_cuda, binding, oracle_mod, monkeypatch, N, inner):
    """SEM_G_RECOMPUTE on the paths large meshes take: the chunked operator / gather-scatter (element ranges offset into
    the vertex array) and the renumbered inner context of sem_pcg, both forced on a small scrambled mesh.  Ax+gs equals the
    oracle and is bit-identical to the un-chunked recomputed result; the PCG loop takes the oracle's iteration count."""
    m = inputs.box_mesh(6, 5, 4, N, "random", seed=4, permute_seed=9)
    om = oracle_mod.Maps(m.gid)
    oG, _, _ = oracle_mod.geom_trilinear(m.vert, m.N)
    mask_u = oracle_mod.mask_unique(m.dirichlet, om)
    u = inputs.field_uniform(m.gid, 5)
    ow = _ax_gs_oracle(oracle_mod, m, u, True)
    xs = np.where(mask_u != 0, 0.0, inputs.field_normal(om.uniq_gid, 7))
    b_u = oracle_mod.apply_Ag(oG, m.N, om, mask_u, xs)
    ores = oracle_mod.pcg(oG, m.N, om, mask_u, b_u, tol=1e-9, maxit=300)
    monkeypatch.setenv("SEM_INNER", inner)
    outs = []
    for chunk in (None, "3"):
        if chunk is None:
            monkeypatch.delenv("SEM_CHUNK_GROUPS", raising=False)
        else:
            monkeypatch.setenv("SEM_CHUNK_GROUPS", chunk)
        with binding.Sem(m.E, m.N, m.vert, m.gid, m.dirichlet) as sem:
            sem.geom(mode=binding.SEM_G_RECOMPUTE)
            du = to_dev(torch_cuda, u.ravel())
            dw = torch_cuda.full_like(du, float("nan"))
            sem.ax_gs(du, dw)
            outs.append(dw.clone())
            assert relerr(dw.cpu().numpy(), ow) <= TOL64
            b = to_dev(torch_cuda, b_u[om.l2u])
            x = torch_cuda.zeros_like(b)
            it, _ = sem.pcg(b, x, 1e-9, 300)
            assert it == ores["iters"] and relerr(x.cpu().numpy(), ores["x"][om.l2u]) <= TOLPCG
    assert torch_cuda.equal(outs[0], outs[1])


@pytest.mark.parametrize("nf,side_stream", [(1, True), (2, True), (3, True), (4, True), (5, True), (8, True), (5, False)])
def test_pcg_many_groups_and_graph_replay(torch_cuda, binding, oracle_mod, nf, side_stream):
    """sem_pcg_many for 1 ... 8 fields (vector kernels in groups of 3 and 2 fields, single leftovers) on a non-default stream,
    where 16 lockstep iterations are one replayed CUDA graph, and on the default stream (eager launches): every field takes
    the iteration count of sem_pcg on it alone and reaches its solution at 1e-9; the fields stop at different iterations
    (different tolerances are emulated by scaling: one field is zero, one is a smooth mode)."""
    m = inputs.box_mesh(5, 4, 3, 7, "random", seed=12)
    lam = 3.0
    om = oracle_mod.Maps(m.gid)
    mask_u = oracle_mod.mask_unique(m.dirichlet, om)
    xyz = oracle_mod.node_xyz(m.vert, m.N).reshape(-1, 3)
    smooth = np.sin(np.pi * xyz[:, 0]) * np.sin(np.pi * xyz[:, 1]) * np.sin(np.pi * xyz[:, 2])
    stream = torch_cuda.cuda.Stream() if side_stream else torch_cuda.cuda.current_stream()
    with torch_cuda.cuda.stream(stream):
        with binding.Sem(m.E, m.N, m.vert, m.gid, m.dirichlet) as sem:
            sem.geom(with_mass=True)
            sem.set_lambda(lam)
            live = to_dev(torch_cuda, (mask_u[om.l2u] == 0).astype(np.float64))
            us = []
            for f in range(nf):
                if f == 1:
                    us.append(torch_cuda.zeros(sem.nL, device="cuda", dtype=torch_cuda.float64))
                elif f == 2:
                    us.append(to_dev(torch_cuda, smooth) * live)
                else:
                    us.append(to_dev(torch_cuda, inputs.field_normal(om.uniq_gid, 80 + f)[om.l2u]) * live)
            b = torch_cuda.zeros(nf, sem.nL, device="cuda", dtype=torch_cuda.float64)
            for f in range(nf):
                sem.ax_gs(us[f].contiguous(), b[f], lam)
            ref = []
            for f in range(nf):
                x1 = torch_cuda.zeros(sem.nL, device="cuda", dtype=torch_cuda.float64)
                it1, rel1 = sem.pcg(b[f].contiguous(), x1, 1e-9, 300)
                ref.append((it1, x1))
            x = torch_cuda.zeros_like(b)
            its, rels = sem.pcg_many(b, x, 1e-9, 300)
            stream.synchronize()
            assert len(set(r[0] for r in ref)) >= (2 if nf > 1 else 1)          # the fields do stop at different iterations
            for f in range(nf):
                assert its[f] == ref[f][0], (f, its, [r[0] for r in ref])
                if ref[f][0]:
                    assert relerr(x[f].cpu().numpy(), ref[f][1].cpu().numpy()) <= TOLPCG, f
            x.zero_()
            its2, _ = sem.pcg_many(b, x, 1e-30, 21)                              # one full batch + 5 iterations of the next
            assert all(i == (0 if f == 1 else 21) for f, i in enumerate(its2))
