"""GPU parity tests added in round 2 (through the C ABI, against the CPU oracle): the stated sizes VERDICT r1 found
missing (config 4's FP32 coarse levels at E = 7200; config 5 at its full 10^6 elements, where G offsets pass 2^31),
the tensor-core operator kernel, and the regression tests of the round-1 advisor findings."""
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
