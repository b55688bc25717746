"""GPU parity tests: the CUDA path (through the C ABI of include/sem.h, via the thin binding) against the CPU oracle,
element by element on the same seeded inputs.  Tolerances (BASELINE.json north_star / DESIGN.md):
  maps bit-exact; FP64 Ax / gs / Ax+gs max|w_gpu - w_orc| / max|w_orc| <= 1e-12; FP32 <= 1e-5;
  PCG ||x_gpu - x_orc||_inf / ||x_orc||_inf <= 1e-9 at equal iteration count."""
import os

import numpy as np
import pytest

from paper_2110_01716_b200 import inputs

pytestmark = pytest.mark.gpu

TOL64, TOL32, TOLPCG = 1e-12, 1e-5, 1e-9
GOLD = os.path.join(os.path.dirname(__file__), "golden")


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


def make_sem(binding, mesh, dirichlet=False, **geom_kw):
    sem = binding.Sem(mesh.E, mesh.N, mesh.vert, mesh.gid, mesh.dirichlet if dirichlet else None)
    sem.geom(**geom_kw)
    return sem


# ------------------------------------------------------------------------------------------------ a0: GLL tables
@pytest.mark.parametrize("N", [1, 2, 3, 4, 5, 7, 9, 12, 15])
def test_gll_tables(torch_cuda, binding, oracle_mod, N):
    m = inputs.box_mesh(1, 1, 1, N)
    with binding.Sem(1, N, m.vert, m.gid) as sem:
        xi, rho, D = sem.gll()
    oxi, orho, oD = oracle_mod.gll(N)
    assert np.max(np.abs(xi - oxi)) <= 2e-16
    assert np.max(np.abs(rho - orho) / orho) <= 1e-14
    assert np.max(np.abs(D - oD)) <= 1e-13 * np.max(np.abs(oD))


# ------------------------------------------------------------------------------------------------ a1: maps
def _check_maps(binding, oracle_mod, mesh, gid=None, dirichlet=False):
    gid = mesh.gid if gid is None else gid
    with binding.Sem(mesh.E, mesh.N, mesh.vert, gid, mesh.dirichlet if dirichlet else None) as sem:
        c, mp = sem.counts(), sem.maps()
    om = oracle_mod.Maps(gid)
    assert (c["nL"], c["U"], c["S"], c["Us"]) == (om.nL, om.U, om.S, om.Us)
    for name in ["uniq_gid", "l2u", "mult", "seg_off", "seg_idx"]:
        assert np.array_equal(mp[name], getattr(om, name)), name
    return c


def test_maps_bitexact_config1(torch_cuda, binding, oracle_mod):
    c = _check_maps(binding, oracle_mod, inputs.config1(), dirichlet=True)
    assert (c["U"], c["S"], c["Us"]) == (24389, 15192, 6813)          # tests/golden/p13_config1_pcg.txt


def test_maps_bitexact_scrambled_sparse_ids(torch_cuda, binding, oracle_mod):
    m = inputs.box_mesh(5, 3, 4, 3, "random", seed=7, permute_seed=11)
    _check_maps(binding, oracle_mod, m)
    # ids need not be contiguous (S11): a strictly increasing but gappy relabelling, > 2^32
    _check_maps(binding, oracle_mod, m, gid=m.gid * 1000003 + (1 << 33))
    # a non-monotone relabelling changes the canonical order; still must match the oracle bit for bit
    _check_maps(binding, oracle_mod, m, gid=(m.gid * 7919) % 100003)


def test_maps_device_gid(torch_cuda, binding, oracle_mod):
    m = inputs.box_mesh(3, 3, 2, 4)
    g = to_dev(torch_cuda, m.gid.ravel())
    with binding.Sem(m.E, m.N, m.vert, g) as sem:
        mp = sem.maps()
    om = oracle_mod.Maps(m.gid)
    assert np.array_equal(mp["seg_idx"], om.seg_idx) and np.array_equal(mp["l2u"], om.l2u)


def test_maps_no_sharing_and_single_element(torch_cuda, binding, oracle_mod):
    m = inputs.box_mesh(1, 1, 1, 2)
    c = _check_maps(binding, oracle_mod, m)
    assert c["S"] == 0 and c["Us"] == 0
    m2 = inputs.box_mesh(2, 2, 2, 1)
    # every node its own id: nothing shared although the mesh is connected geometrically
    _check_maps(binding, oracle_mod, m2, gid=np.arange(m2.nL, dtype=np.int64).reshape(m2.gid.shape)[::-1].copy())


# ------------------------------------------------------------------------------------------------ a2: geometry
@pytest.mark.parametrize("N,geometry", [(7, "smooth"), (3, "random"), (4, "random"), (1, "smooth")])
def test_geom_trilinear(torch_cuda, binding, oracle_mod, N, geometry):
    m = inputs.box_mesh(4, 3, 5, N, geometry, seed=5)
    with make_sem(binding, m, with_mass=True) as sem:
        G, dJ = sem.get_geom()
    oG, odJ, rc = oracle_mod.geom_trilinear(m.vert, N)
    assert rc == 0
    assert relerr(dJ, odJ) <= 1e-13
    for cpt in range(7):
        assert relerr(G[:, cpt], oG[:, cpt]) <= TOL64, cpt


def test_geom_isoparametric(torch_cuda, binding, oracle_mod):
    m = inputs.box_mesh(3, 3, 3, 5, "random", seed=2)
    xyz = oracle_mod.node_xyz(m.vert, m.N)
    # bend the elements beyond trilinear so that the isoparametric route is really exercised (still valid: small)
    xyz = xyz + 0.01 * np.sin(3 * xyz[..., [1, 2, 0]]) * np.sin(np.pi * xyz) * np.sin(np.pi * xyz[..., [2, 0, 1]])
    with binding.Sem(m.E, m.N, m.vert, m.gid) as sem:
        sem.geom(node_xyz=xyz, with_mass=True)
        G, dJ = sem.get_geom()
    oG, odJ, rc = oracle_mod.geom_iso(xyz, m.N)
    assert rc == 0
    assert relerr(dJ, odJ) <= 1e-12
    assert relerr(G, oG) <= 1e-11          # conditioning of the inverse Jacobian; Ax parity is checked separately


def test_bad_mesh_and_bad_args(torch_cuda, binding):
    m = inputs.box_mesh(2, 2, 2, 3)
    v = m.vert.copy()
    v[3, [0, 1]] = v[3, [1, 0]]                         # swap two vertices: inverted element
    sem = binding.Sem(m.E, m.N, v, m.gid)
    with pytest.raises(binding.SemError) as e:
        sem.geom()
    assert e.value.code == binding.SEM_EMESH
    u = torch_cuda.zeros(m.nL, dtype=torch_cuda.float64, device="cuda")
    w = torch_cuda.zeros_like(u)
    with pytest.raises(binding.SemError) as e:
        sem.ax(u, w)                                    # geometry failed: state error
    assert e.value.code == binding.SEM_ESTATE
    sem.close()
    g = m.gid.copy()
    g[0, 0] = -1
    with pytest.raises(binding.SemError) as e:
        binding.Sem(m.E, m.N, m.vert, g)
    assert e.value.code == binding.SEM_EINVAL
    with make_sem(binding, m) as sem:
        with pytest.raises(binding.SemError) as e:
            sem.ax(u, w, lam=1.0)                       # lambda without with_mass
        assert e.value.code == binding.SEM_ESTATE
        with pytest.raises(binding.SemError) as e:
            sem.ax(u, u)                                # aliasing
        assert e.value.code == binding.SEM_EINVAL


# ------------------------------------------------------------------------------------------------ a3-a5: Ax
def _ax_case(torch, binding, oracle_mod, mesh, variant=0, mode=0, lam=0.0, dtype="f64", seed=0):
    oG, _, rc = oracle_mod.geom_trilinear(mesh.vert, mesh.N)
    assert rc == 0
    u = inputs.field_uniform(mesh.gid, seed)
    ow = oracle_mod.ax(oG, u, mesh.N, lam)
    tdt = torch.float64 if dtype == "f64" else torch.float32
    with make_sem(binding, mesh, mode=mode, with_mass=lam != 0.0) as sem:
        sem.set_variant(variant)
        du = to_dev(torch, u.ravel(), tdt)
        dw = torch.full_like(du, float("nan"))
        sem.ax(du, dw, lam)
        torch.cuda.synchronize()
        w = dw.cpu().numpy().reshape(ow.shape)
    return relerr(w, ow)


@pytest.mark.parametrize("N", [1, 2, 3, 4, 5, 6, 7, 8, 9, 10, 11, 13, 15])
@pytest.mark.parametrize("variant", [0, 1, 2, 3, 4])
def test_ax_f64_all_orders(torch_cuda, binding, oracle_mod, N, variant):
    # 5*3*3 = 45 elements: not a multiple of the elements-per-block of any p (ragged tail), several blocks
    m = inputs.box_mesh(5, 3, 3, N, "random", seed=N)
    assert _ax_case(torch_cuda, binding, oracle_mod, m, variant=variant) <= TOL64


@pytest.mark.parametrize("N", [1, 3, 7])
def test_ax_single_element(torch_cuda, binding, oracle_mod, N):
    m = inputs.box_mesh(1, 1, 1, N, "affine")
    assert _ax_case(torch_cuda, binding, oracle_mod, m) <= TOL64


@pytest.mark.parametrize("N", [3, 7, 9])
def test_ax_many_elements_per_cta(torch_cuda, binding, oracle_mod, N):
    """More elements than resident CTAs: every persistent CTA walks the ring several times (phase wrap-around)."""
    n = {3: 24, 7: 22, 9: 16}[N]
    m = inputs.box_mesh(n, n, n + 1, N, "random", seed=1)
    assert _ax_case(torch_cuda, binding, oracle_mod, m) <= TOL64


@pytest.mark.parametrize("N,dtype", [(7, "f64"), (8, "f64"), (8, "f32"), (9, "f64"), (11, "f64"), (11, "f32")])
def test_ax_pencil_many_elements_per_cta(torch_cuda, binding, oracle_mod, N, dtype):
    """The pencil kernel (variant 4) with several elements per persistent CTA: the G ring and its empty-barriers wrap
    many times, u alternates between its two buffers (even p) or is re-staged (odd p)."""
    n = {7: 16, 8: 14, 9: 13, 11: 11}[N]
    m = inputs.box_mesh(n, n, n + 1, N, "random", seed=2)
    assert _ax_case(torch_cuda, binding, oracle_mod, m, variant=4, dtype=dtype) <= (TOL64 if dtype == "f64" else TOL32)


@pytest.mark.parametrize("N", [1, 2, 3, 5, 7, 9])
def test_ax_recomputed_G(torch_cuda, binding, oracle_mod, N):
    m = inputs.box_mesh(4, 3, 3, N, "random", seed=3)
    assert _ax_case(torch_cuda, binding, oracle_mod, m, mode=1) <= TOL64


@pytest.mark.parametrize("N,variant", [(7, 0), (7, 1), (7, 2), (7, 3), (4, 0), (3, 0), (8, 4), (9, 4), (11, 0), (7, 4)])
def test_ax_helmholtz(torch_cuda, binding, oracle_mod, N, variant):
    m = inputs.box_mesh(3, 3, 3, N, "smooth")
    assert _ax_case(torch_cuda, binding, oracle_mod, m, variant=variant, lam=37.5) <= TOL64


@pytest.mark.parametrize("N", [1, 2, 3, 5, 7, 9])
@pytest.mark.parametrize("variant,mode", [(0, 0), (1, 0), (2, 0), (0, 1), (4, 0)])
def test_ax_f32(torch_cuda, binding, oracle_mod, N, variant, mode):
    m = inputs.box_mesh(5, 4, 3, N, "smooth")
    assert _ax_case(torch_cuda, binding, oracle_mod, m, variant=variant, mode=mode, dtype="f32") <= TOL32


# ------------------------------------------------------------------------------------------------ a6/a7: gs, Ax+gs
@pytest.mark.parametrize("N", [1, 3, 7])
def test_gs_bit_identical(torch_cuda, binding, oracle_mod, N):
    """Same summation order as the oracle (ascending local index), so FP64 sums agree to the last bit."""
    m = inputs.box_mesh(4, 4, 3, N, permute_seed=5)
    rng = np.random.default_rng(N)
    w = rng.standard_normal(m.nL)                     # NOT continuous: a genuine gather-scatter input
    ow = oracle_mod.gs(w, oracle_mod.Maps(m.gid))
    with binding.Sem(m.E, m.N, m.vert, m.gid) as sem:
        dw = to_dev(torch_cuda, w)
        sem.gs(dw)
        assert np.array_equal(dw.cpu().numpy(), ow)
        w32 = w.astype(np.float32)
        dw32 = to_dev(torch_cuda, w32)
        sem.gs(dw32)
        assert relerr(dw32.cpu().numpy(), oracle_mod.gs(w32.astype(np.float64), oracle_mod.Maps(m.gid))) <= 1e-6


def _ax_gs_oracle(oracle_mod, mesh, u, masked, lam=0.0):
    oG, _, _ = oracle_mod.geom_trilinear(mesh.vert, mesh.N)
    ow = oracle_mod.gs(oracle_mod.ax(oG, u, mesh.N, lam).ravel(), oracle_mod.Maps(mesh.gid))
    if masked:
        om = oracle_mod.Maps(mesh.gid)
        ow[oracle_mod.mask_unique(mesh.dirichlet, om)[om.l2u] != 0] = 0.0
    return ow


@pytest.mark.parametrize("masked", [False, True])
def test_ax_gs_config1(torch_cuda, binding, oracle_mod, masked):
    m = inputs.config1()
    u = inputs.field_uniform(m.gid, 0)
    ow = _ax_gs_oracle(oracle_mod, m, u, masked)
    with make_sem(binding, m, dirichlet=masked) as sem:
        du = to_dev(torch_cuda, u.ravel())
        dw = torch_cuda.empty_like(du)
        sem.ax_gs(du, dw)
        assert relerr(dw.cpu().numpy(), ow) <= TOL64
        # determinism: no atomics on this path, so a second application is bit-identical
        dw2 = torch_cuda.empty_like(du)
        sem.ax_gs(du, dw2)
        assert torch_cuda.equal(dw, dw2)


@pytest.mark.parametrize("case", ["cfg1", "cfg1_masked", "perm_N7", "N3_masked", "N1", "N5", "one_element", "N7_many"])
def test_ax_gs_meshes(torch_cuda, binding, oracle_mod, case):
    """sem_ax_gs (operator kernel + gather-scatter kernel + mask) over mesh shapes that exercise every record class
    (pairs, quads, bigs; N = 1 has only corner nodes), several element groups per CTA (N < 7), a scrambled element
    order, one element (nothing shared) and more element groups than resident CTAs: equal to sem_ax followed by
    sem_gs bit for bit, within tolerance of the oracle in FP64 and FP32, and repeatable."""
    masked = case.endswith("masked")
    m = {"cfg1": inputs.config1, "cfg1_masked": inputs.config1,
         "perm_N7": lambda: inputs.box_mesh(5, 4, 3, 7, "random", seed=3, permute_seed=4),
         "N3_masked": lambda: inputs.box_mesh(7, 6, 5, 3, "smooth"),
         "N1": lambda: inputs.box_mesh(9, 8, 7, 1, "smooth"),
         "N5": lambda: inputs.box_mesh(4, 3, 5, 5, "random", seed=2, permute_seed=1),
         "one_element": lambda: inputs.box_mesh(1, 1, 1, 7),
         "N7_many": lambda: inputs.box_mesh(13, 12, 11, 7, "smooth")}[case]()
    u = inputs.field_uniform(m.gid, 7)
    ow = _ax_gs_oracle(oracle_mod, m, u, masked)
    with make_sem(binding, m, dirichlet=masked) as sem:
        for dt, tol in ((torch_cuda.float64, TOL64), (torch_cuda.float32, TOL32)):
            du = to_dev(torch_cuda, u.ravel(), dt)
            dw = torch_cuda.full_like(du, float("nan"))
            sem.ax_gs(du, dw)
            assert relerr(dw.cpu().numpy(), ow) <= tol, (case, dt)
            dw2 = torch_cuda.full_like(du, float("nan"))
            sem.ax_gs(du, dw2)
            assert torch_cuda.equal(dw, dw2)
            if not masked:
                dw3 = torch_cuda.full_like(du, float("nan"))
                sem.ax(du, dw3)
                sem.gs(dw3)
                assert torch_cuda.equal(dw, dw3)


@pytest.mark.parametrize("N", [7, 3, 1])
def test_ax_gs_f32_levels_config4_small(torch_cuda, binding, oracle_mod, N):
    """Config 4 (mixed-precision levels N = 7, 3, 1), down-sized mesh: FP32 Ax+gs against the FP64 oracle."""
    m = inputs.box_mesh(6, 5, 4, N, "smooth")
    u = inputs.field_normal(m.gid, 2)
    ow = _ax_gs_oracle(oracle_mod, m, u, False)
    with make_sem(binding, m) as sem:
        du = to_dev(torch_cuda, u.ravel(), torch_cuda.float32)
        dw = torch_cuda.empty_like(du)
        sem.ax_gs(du, dw)
        assert relerr(dw.cpu().numpy(), ow) <= TOL32


@pytest.mark.slow
def test_ax_gs_config2_full_size(torch_cuda, binding, oracle_mod):
    """BASELINE config 2 (7200 elements, N = 7) in the launch configuration bench.py times, every output compared."""
    m = inputs.config2()
    u = inputs.field_uniform(m.gid, 0)
    ow = _ax_gs_oracle(oracle_mod, m, u, False)
    with make_sem(binding, m) as sem:
        c = sem.counts()
        assert (c["nL"], c["U"], c["S"], c["Us"]) == (3686400, 2524887, 2049160, 887647)
        du = to_dev(torch_cuda, u.ravel())
        dw = torch_cuda.empty_like(du)
        for _ in range(3):
            sem.ax_gs(du, dw)
        assert relerr(dw.cpu().numpy(), ow) <= TOL64
        d32 = du.float()
        w32 = torch_cuda.empty_like(d32)
        sem.ax_gs(d32, w32)
        assert relerr(w32.cpu().numpy(), ow) <= TOL32


def test_stored_vs_recomputed_config3_smallest(torch_cuda, binding, oracle_mod):
    """Config 3: stored-G and recomputed-G variants agree with the oracle (and so with each other) <= 1e-12."""
    for N in (3, 5, 7, 9):
        m = inputs.config3(8, N)
        u = inputs.field_uniform(m.gid, 1)
        ow = _ax_gs_oracle(oracle_mod, m, u, False)
        for mode in (0, 1):
            with make_sem(binding, m, mode=mode) as sem:
                du = to_dev(torch_cuda, u.ravel())
                dw = torch_cuda.empty_like(du)
                sem.ax_gs(du, dw)
                assert relerr(dw.cpu().numpy(), ow) <= TOL64, (N, mode)


# ------------------------------------------------------------------------------------------------ a8: Jacobi-PCG
def test_diag_exact(torch_cuda, binding, oracle_mod):
    m = inputs.box_mesh(3, 4, 3, 5, "random", seed=9)
    oG, _, _ = oracle_mod.geom_trilinear(m.vert, m.N)
    od = oracle_mod.gs(oracle_mod.diag_local(oG, m.N).ravel(), oracle_mod.Maps(m.gid))
    with make_sem(binding, m, dirichlet=True) as sem:
        assert relerr(sem.get_diag().ravel(), od) <= TOL64


def _pcg_setup(oracle_mod, mesh):
    om = oracle_mod.Maps(mesh.gid)
    oG, _, _ = oracle_mod.geom_trilinear(mesh.vert, mesh.N)
    mask_u = oracle_mod.mask_unique(mesh.dirichlet, om)
    return om, oG, mask_u


def test_pcg_config1_20_iterations(torch_cuda, binding, oracle_mod):
    m = inputs.config1()
    om, oG, mask_u = _pcg_setup(oracle_mod, m)
    xyz = oracle_mod.node_xyz(m.vert, m.N).reshape(-1, 3)
    us_u = np.zeros(om.U)
    us_u[om.l2u] = np.sin(np.pi * xyz[:, 0]) * np.sin(np.pi * xyz[:, 1]) * np.sin(np.pi * xyz[:, 2])
    us_u[mask_u != 0] = 0.0
    b_u = oracle_mod.apply_Ag(oG, m.N, om, mask_u, us_u)
    ores = oracle_mod.pcg(oG, m.N, om, mask_u, b_u, tol=1e-30, maxit=20, snap_its=(1, 5, 10, 20))
    assert ores["iters"] == 20
    with make_sem(binding, m, dirichlet=True) as sem:
        b = to_dev(torch_cuda, b_u[om.l2u])
        for its in (1, 5, 10, 20):
            x = torch_cuda.zeros_like(b)
            it, rel = sem.pcg(b, x, 1e-30, its)
            assert it == its
            xg = x.cpu().numpy()
            assert np.array_equal(xg, xg[om.seg_idx[om.seg_off[:-1]]][om.l2u])      # continuous
            assert relerr(xg, ores["snaps"][its][om.l2u]) <= TOLPCG
            assert abs(rel - ores["hist"][its]) <= 1e-9 * ores["hist"][its]
        hist = sem.pcg_history(21)
        assert np.max(np.abs(hist - ores["hist"]) / ores["hist"]) <= 1e-9
    gold = {}
    for line in open(os.path.join(GOLD, "p13_config1_pcg.txt")):
        if not line.startswith("#") and line.strip():
            k, v = line.split(None, 1)
            gold[k] = v.strip()
    assert abs(hist[20] - float(gold["relres_it20"])) <= 1e-9
    assert abs(np.max(np.abs(xg - us_u[om.l2u])) - float(gold["err_inf_it20"])) <= 1e-9


def test_pcg_converges_same_iteration_count(torch_cuda, binding, oracle_mod):
    m = inputs.box_mesh(4, 4, 4, 5, "random", seed=3, permute_seed=4)      # config-5 recipe, down-sized
    om, oG, mask_u = _pcg_setup(oracle_mod, m)
    xyz = oracle_mod.node_xyz(m.vert, m.N).reshape(-1, 3)
    f = 3 * np.pi ** 2 * np.sin(np.pi * xyz[:, 0]) * np.sin(np.pi * xyz[:, 1]) * np.sin(np.pi * xyz[:, 2])
    b_u = np.zeros(om.U)
    np.add.at(b_u, om.l2u, oG[:, 6].ravel() * f)
    b_u[mask_u != 0] = 0.0
    ores = oracle_mod.pcg(oG, m.N, om, mask_u, b_u, tol=1e-8, maxit=500)
    with make_sem(binding, m, dirichlet=True) as sem:
        b = to_dev(torch_cuda, b_u[om.l2u])
        x = torch_cuda.zeros_like(b)
        it, rel = sem.pcg(b, x, 1e-8, 500)
        assert it == ores["iters"] and rel <= 1e-8
        assert relerr(x.cpu().numpy(), ores["x"][om.l2u]) <= TOLPCG
        exact = np.sin(np.pi * xyz[:, 0]) * np.sin(np.pi * xyz[:, 1]) * np.sin(np.pi * xyz[:, 2])
        assert np.max(np.abs(x.cpu().numpy() - exact)) <= 1e-4           # discretisation error at N = 5, 4^3 elements
        # nonzero initial guess: same solution, x0 masked on entry
        x0 = torch_cuda.ones_like(b)
        it2, _ = sem.pcg(b, x0, 1e-10, 500)
        assert relerr(x0.cpu().numpy(), ores["x"][om.l2u]) <= 1e-7
        # r0 = 0 (b = 0, x0 = 0) -> 0 iterations, x untouched (S13)
        z = torch_cuda.zeros_like(b)
        x1 = torch_cuda.zeros_like(b)
        it3, rel3 = sem.pcg(z, x1, 1e-8, 10)
        assert it3 == 0 and rel3 == 0.0 and float(x1.abs().max()) == 0.0
        # maxit = 0: only the entry masking of x0 happens
        x2 = torch_cuda.ones_like(b)
        it4, _ = sem.pcg(b, x2, 1e-8, 0)
        assert it4 == 0 and float(x2.sum()) == float((mask_u[om.l2u] == 0).sum())


def test_pcg_trajectory_config5_replica(torch_cuda, binding, oracle_mod):
    """S20: config-5 recipe (N = 7, random +-10 % vertices seed 3, element permutation seed 4, b = M Q^T(B f)) on a
    6^3 replica: the iterates x_k at k = 1, 5, 10, 25 and the residual history agree with the oracle's."""
    m = inputs.config5(6)
    om, oG, mask_u = _pcg_setup(oracle_mod, m)
    xyz = oracle_mod.node_xyz(m.vert, m.N).reshape(-1, 3)
    f = 3 * np.pi ** 2 * np.sin(np.pi * xyz[:, 0]) * np.sin(np.pi * xyz[:, 1]) * np.sin(np.pi * xyz[:, 2])
    b_u = np.zeros(om.U)
    np.add.at(b_u, om.l2u, oG[:, 6].ravel() * f)
    b_u[mask_u != 0] = 0.0
    ores = oracle_mod.pcg(oG, m.N, om, mask_u, b_u, tol=1e-30, maxit=25, snap_its=(1, 5, 10, 25))
    with make_sem(binding, m, dirichlet=True) as sem:
        b = to_dev(torch_cuda, b_u[om.l2u])
        for k in (1, 5, 10, 25):
            x = torch_cuda.zeros_like(b)
            it, rel = sem.pcg(b, x, 1e-30, k)
            assert it == k
            assert relerr(x.cpu().numpy(), ores["snaps"][k][om.l2u]) <= TOLPCG, k
            assert abs(rel - ores["hist"][k]) <= 1e-9 * ores["hist"][k], k
        hist = sem.pcg_history(26)
        assert np.max(np.abs(hist - ores["hist"]) / ores["hist"]) <= 1e-9


def test_pcg_helmholtz(torch_cuda, binding, oracle_mod):
    m = inputs.box_mesh(3, 3, 3, 4, "smooth")
    om, oG, mask_u = _pcg_setup(oracle_mod, m)
    mask_u[:] = 0                                                            # Helmholtz is SPD without Dirichlet
    rng = np.random.default_rng(0)
    b_u = rng.standard_normal(om.U)
    lam = 10.0
    ores = oracle_mod.pcg(oG, m.N, om, mask_u, b_u, tol=1e-9, maxit=300, lam=lam)
    with binding.Sem(m.E, m.N, m.vert, m.gid) as sem:
        sem.geom(with_mass=True)
        sem.set_lambda(lam)
        b = to_dev(torch_cuda, b_u[om.l2u])
        x = torch_cuda.zeros_like(b)
        it, rel = sem.pcg(b, x, 1e-9, 300)
        assert it == ores["iters"]
        assert relerr(x.cpu().numpy(), ores["x"][om.l2u]) <= TOLPCG


# ------------------------------------------------------------------------------------ NEXT-1: pMG transfer
@pytest.mark.parametrize("Nc,Nf", [(1, 3), (3, 7), (1, 7), (5, 8), (7, 7), (2, 5), (9, 15)])
def test_transfer_parity(torch_cuda, binding, oracle_mod, Nc, Nf):
    """sem_transfer against the oracle: interpolation matrix, prolongation and restriction, FP64 (1e-12) and FP32
    (1e-5), on a mesh with more elements than resident CTAs of the kernel."""
    nx, ny, nz = (13, 12, 11) if Nf <= 8 else (5, 4, 3)
    mc, mf = inputs.box_mesh(nx, ny, nz, Nc, "smooth"), inputs.box_mesh(nx, ny, nz, Nf, "smooth")
    uc = inputs.field_normal(mc.gid, 2)
    rf = inputs.field_uniform(mf.gid, 5) * (1.0 + np.arange(mf.E)[:, None] % 7)      # not continuous on purpose
    o_p, o_r = oracle_mod.prolong(uc, Nc, Nf), oracle_mod.restrict(rf, Nc, Nf)
    with binding.Sem(mc.E, Nc, mc.vert, mc.gid) as sc, binding.Sem(mf.E, Nf, mf.vert, mf.gid) as sf:
        assert np.max(np.abs(sc.interp(sf) - oracle_mod.interp(Nc, Nf))) <= 1e-14
        for dt, tol in ((torch_cuda.float64, TOL64), (torch_cuda.float32, TOL32)):
            d_uc, d_rf = to_dev(torch_cuda, uc.ravel(), dt), to_dev(torch_cuda, rf.ravel(), dt)
            d_uf = torch_cuda.full((mf.nL,), float("nan"), dtype=dt, device="cuda")
            d_rc = torch_cuda.full((mc.nL,), float("nan"), dtype=dt, device="cuda")
            sc.transfer(sf, d_uc, d_uf, binding.SEM_PROLONG)
            sc.transfer(sf, d_rf, d_rc, binding.SEM_RESTRICT)
            assert relerr(d_uf.cpu().numpy(), o_p.ravel()) <= tol, (Nc, Nf, dt)
            assert relerr(d_rc.cpu().numpy(), o_r.ravel()) <= tol, (Nc, Nf, dt)


def test_transfer_bad_args(torch_cuda, binding):
    m3, m7, other = inputs.box_mesh(2, 2, 2, 3), inputs.box_mesh(2, 2, 2, 7), inputs.box_mesh(3, 2, 2, 3)
    with binding.Sem(m3.E, 3, m3.vert, m3.gid) as s3, binding.Sem(m7.E, 7, m7.vert, m7.gid) as s7, \
            binding.Sem(other.E, 3, other.vert, other.gid) as so:
        a = torch_cuda.zeros(m3.nL, dtype=torch_cuda.float64, device="cuda")
        b = torch_cuda.zeros(m7.nL, dtype=torch_cuda.float64, device="cuda")
        with pytest.raises(binding.SemError) as e:
            s7.transfer(s3, b, a, binding.SEM_PROLONG)            # coarse order exceeds fine order
        assert e.value.code == binding.SEM_EINVAL
        with pytest.raises(binding.SemError) as e:
            so.transfer(s7, torch_cuda.zeros(other.nL, dtype=torch_cuda.float64, device="cuda"), b, binding.SEM_PROLONG)   # different meshes
        assert e.value.code == binding.SEM_EINVAL
        with pytest.raises(binding.SemError):
            s3.transfer(s7, a, b, 7)                              # bad direction


# ------------------------------------------------------------------------ NEXT-1: Chebyshev-Jacobi smoother
def _lmax_power(oracle_mod, G, N, om, mask_u, its=12):
    """Largest eigenvalue of diag^-1 A by power iteration, on the oracle side (the bounds are inputs of the smoother)."""
    dg = np.zeros(om.U)
    np.add.at(dg, om.l2u, oracle_mod.diag_local(G, N).ravel())
    Minv = np.where(mask_u != 0, 0.0, 1.0 / dg)
    v = np.where(mask_u != 0, 0.0, np.cos(np.arange(om.U) * 0.37))
    lam = 1.0
    for _ in range(its):
        w = Minv * oracle_mod.apply_Ag(G, N, om, mask_u, v)
        lam = float(np.linalg.norm(w) / np.linalg.norm(v))
        v = w / np.linalg.norm(w)
    return lam


@pytest.mark.parametrize("N,order,zero_guess", [(7, 1, False), (7, 2, True), (7, 4, False), (3, 3, True), (1, 2, False),
                                                (5, 6, False)])
def test_cheby_parity(torch_cuda, binding, oracle_mod, N, order, zero_guess):
    m = inputs.box_mesh(5, 4, 3, N, "smooth")
    om, oG, mask_u = _pcg_setup(oracle_mod, m)
    lmax = 1.1 * _lmax_power(oracle_mod, oG, N, om, mask_u)
    lmin = 0.1 * lmax
    xs = np.where(mask_u != 0, 0.0, inputs.field_normal(om.uniq_gid, 4))
    b_u = oracle_mod.apply_Ag(oG, N, om, mask_u, xs)
    x0_u = None if zero_guess else np.where(mask_u != 0, 0.0, inputs.field_uniform(om.uniq_gid, 6))
    ox = oracle_mod.cheby(oG, N, om, mask_u, b_u, x0_u, order, lmin, lmax)[om.l2u]
    with make_sem(binding, m, dirichlet=True) as sem:
        for dt, tol in ((torch_cuda.float64, TOL64), (torch_cuda.float32, TOL32)):
            b = to_dev(torch_cuda, b_u[om.l2u], dt)
            # with zero_guess the content of x must not matter; otherwise a nonzero guess that is NOT masked on entry
            x = torch_cuda.full_like(b, 3.0) if zero_guess else to_dev(torch_cuda, x0_u[om.l2u] + (mask_u[om.l2u] != 0), dt)
            sem.cheby(b, x, order, lmin, lmax, zero_guess)
            assert relerr(x.cpu().numpy(), ox) <= tol, (N, order, dt)
        with pytest.raises(binding.SemError):
            sem.cheby(b, x, 0, lmin, lmax)
        with pytest.raises(binding.SemError):
            sem.cheby(b, x, 2, lmax, lmin)


def test_cheby_smooths(torch_cuda, binding, oracle_mod):
    """What the smoother is for: on config 1 the FP32 smoother of order 4 reduces the energy norm of a rough error by
    more than the min-max bound 1/T_4(sigma) guarantees for the upper 90 % of the spectrum (loose, property check)."""
    m = inputs.config1()
    om, oG, mask_u = _pcg_setup(oracle_mod, m)
    lmax = 1.1 * _lmax_power(oracle_mod, oG, m.N, om, mask_u)
    rough = np.where(mask_u != 0, 0.0, inputs.field_uniform(om.uniq_gid, 8))          # white noise: mostly high modes
    b_u = np.zeros(om.U)                                                               # solve A x = 0 from x0 = rough
    with make_sem(binding, m, dirichlet=True) as sem:
        b = to_dev(torch_cuda, b_u[om.l2u], torch_cuda.float32)
        x = to_dev(torch_cuda, rough[om.l2u], torch_cuda.float32)
        sem.cheby(b, x, 4, 0.1 * lmax, lmax)
        e1 = np.zeros(om.U)
        e1[om.l2u] = x.cpu().numpy().astype(np.float64)
    en = lambda e: float(e @ oracle_mod.apply_Ag(oG, m.N, om, mask_u, e))
    assert en(e1) < 0.25 * en(rough)


# ------------------------------------------------------------------------- NEXT-1c: p-multigrid V-cycle
@pytest.mark.parametrize("orders", [(7, 3, 1), (5, 1), (8, 5, 1)])
def test_vcycle_parity(torch_cuda, binding, oracle_mod, orders):
    """sem_pmg_vcycle against the oracle's V-cycle with the same eigenvalue bounds: FP64 to 1e-11 (a chain of about a
    dozen operator applications, each 1e-12-exact), FP32 to 5e-5 (P:109 runs the cycle in FP32; same chain at 1e-5
    per step, normalised by max |z|)."""
    meshes = [inputs.box_mesh(5, 4, 3, N, "smooth") for N in orders]
    olv = [oracle_mod.Level(m) for m in meshes]
    L0 = olv[0]
    r_u = np.where(L0.mask_u != 0, 0.0, inputs.field_normal(L0.maps.uniq_gid, 9))
    oz = oracle_mod.vcycle(olv, r_u, 2, 8)[L0.maps.l2u]
    sems = [make_sem(binding, m, dirichlet=True) for m in meshes]
    try:
        for dt, prec, tol in ((torch_cuda.float64, binding.SEM_F64, 1e-11), (torch_cuda.float32, binding.SEM_F32, 5e-5)):
            with binding.Pmg(sems, [l.lmin for l in olv], [l.lmax for l in olv], 2, 8, prec) as mg:
                r = to_dev(torch_cuda, r_u[L0.maps.l2u], dt)
                z = torch_cuda.full_like(r, float("nan"))
                mg.vcycle(r, z)
                assert relerr(z.cpu().numpy(), oz) <= tol, (orders, dt)
                z2 = torch_cuda.full_like(r, float("nan"))
                mg.vcycle(r, z2)                                   # work vectors carry no state between cycles
                assert torch_cuda.equal(z, z2)
    finally:
        for s_ in sems:
            s_.close()


def test_pmg_bad_args(torch_cuda, binding):
    m7, m3 = inputs.box_mesh(2, 2, 2, 7), inputs.box_mesh(2, 2, 2, 3)
    with make_sem(binding, m7, dirichlet=True) as s7, make_sem(binding, m3, dirichlet=True) as s3:
        with pytest.raises(binding.SemError):
            binding.Pmg([s3, s7], [0.2, 0.2], [2.0, 2.0])           # orders must decrease
        with pytest.raises(binding.SemError):
            binding.Pmg([s7, s3], [0.2, 3.0], [2.0, 2.0])           # lmin >= lmax


def test_fpcg_vcycle(torch_cuda, binding, oracle_mod):
    """sem_fpcg (flexible PCG + V-cycle): with an FP64 cycle the iterates follow the oracle's (same iteration count,
    residual history to 1e-7, solution to 1e-9); with the paper's FP32 cycle the FP64 outer iteration still
    reaches the tolerance in about as many iterations and the same solution; and it needs far fewer iterations than
    Jacobi-PCG on the same problem (config-5 recipe of the right-hand side, down-sized mesh)."""
    orders = (7, 3, 1)
    meshes = [inputs.box_mesh(5, 4, 3, N, "random", seed=3) for N in orders]
    olv = [oracle_mod.Level(m) for m in meshes]
    L0, m0 = olv[0], meshes[0]
    xyz = oracle_mod.node_xyz(m0.vert, m0.N).reshape(-1, 3)
    f = 3 * np.pi ** 2 * np.sin(np.pi * xyz[:, 0]) * np.sin(np.pi * xyz[:, 1]) * np.sin(np.pi * xyz[:, 2])
    b_u = np.zeros(L0.maps.U)
    np.add.at(b_u, L0.maps.l2u, L0.G[:, 6].ravel() * f)
    b_u[L0.mask_u != 0] = 0.0
    ores = oracle_mod.fpcg(L0, lambda r: oracle_mod.vcycle(olv, r, 2, 8), b_u, tol=1e-8, maxit=100)
    jac = oracle_mod.pcg(L0.G, L0.N, L0.maps, L0.mask_u, b_u, tol=1e-8, maxit=1000)
    assert ores["iters"] * 3 < jac["iters"]
    sems = [make_sem(binding, m, dirichlet=True) for m in meshes]
    try:
        b = to_dev(torch_cuda, b_u[L0.maps.l2u])
        with binding.Pmg(sems, [l.lmin for l in olv], [l.lmax for l in olv], 2, 8, binding.SEM_F64) as mg:
            x = torch_cuda.full_like(b, float("nan"))
            it, rel = mg.fpcg(b, x, 1e-8, 100)
            assert it == ores["iters"] and rel <= 1e-8
            assert np.max(np.abs(mg.history(it + 1) - ores["hist"]) / ores["hist"]) <= 1e-7
            assert relerr(x.cpu().numpy(), ores["x"][L0.maps.l2u]) <= TOLPCG
        with binding.Pmg(sems, [l.lmin for l in olv], [l.lmax for l in olv], 2, 8, binding.SEM_F32) as mg:
            x32 = torch_cuda.full_like(b, float("nan"))
            it32, rel32 = mg.fpcg(b, x32, 1e-8, 100)
            assert rel32 <= 1e-8 and abs(it32 - ores["iters"]) <= 2
            assert relerr(x32.cpu().numpy(), ores["x"][L0.maps.l2u]) <= 1e-7
            # zero right-hand side: 0 iterations, x = 0
            xz = torch_cuda.ones_like(b)
            itz, relz = mg.fpcg(torch_cuda.zeros_like(b), xz, 1e-8, 10)
            assert itz == 0 and float(xz.abs().max()) == 0.0
    finally:
        for s_ in sems:
            s_.close()


def test_lambda_max(torch_cuda, binding, oracle_mod):
    """sem_lambda_max approaches the largest eigenvalue of diag^-1 A (dense, tiny mesh) from below."""
    m = inputs.box_mesh(3, 3, 2, 4, "random", seed=2)
    om, oG, mask_u = _pcg_setup(oracle_mod, m)
    free = mask_u == 0
    A = np.stack([oracle_mod.apply_Ag(oG, m.N, om, mask_u, e) for e in np.eye(om.U)], axis=1)[np.ix_(free, free)]
    lam_true = float(np.max(np.linalg.eigvals((1.0 / np.diag(A))[:, None] * A).real))
    with make_sem(binding, m, dirichlet=True) as sem:
        lam = sem.lambda_max(60)
        assert 0.95 * lam_true <= lam <= lam_true * (1 + 1e-12)
        assert sem.lambda_max(5) <= lam * (1 + 1e-12)


def test_vcycle_graph_replay_on_side_stream(torch_cuda, binding, oracle_mod):
    """On a non-default stream sem_pmg_vcycle runs eagerly once, captures a CUDA graph on the second call with the same
    (r, z) pair and replays it afterwards: the three paths give bit-identical results and match the oracle; a new
    pair falls back to eager and is captured again."""
    orders = (7, 3, 1)
    meshes = [inputs.box_mesh(4, 3, 3, N, "smooth") for N in orders]
    olv = [oracle_mod.Level(m) for m in meshes]
    L0 = olv[0]
    r_u = np.where(L0.mask_u != 0, 0.0, inputs.field_normal(L0.maps.uniq_gid, 11))
    oz = oracle_mod.vcycle(olv, r_u, 2, 8)[L0.maps.l2u]
    side = torch_cuda.cuda.Stream()
    with torch_cuda.cuda.stream(side):
        sems = [make_sem(binding, m, dirichlet=True) for m in meshes]
        try:
            with binding.Pmg(sems, [l.lmin for l in olv], [l.lmax for l in olv], 2, 8, binding.SEM_F64) as mg:
                r = to_dev(torch_cuda, r_u[L0.maps.l2u])
                zbuf = torch_cuda.empty_like(r)
                outs = []
                for _ in range(4):                       # eager, capture + launch, replay, replay
                    zbuf.fill_(float("nan"))
                    mg.vcycle(r, zbuf)
                    side.synchronize()
                    outs.append(zbuf.clone())
                for o in outs[1:]:
                    assert torch_cuda.equal(o, outs[0])
                assert relerr(outs[0].cpu().numpy(), oz) <= 1e-11
                sems[1].geom()                            # a level is re-built: the recorded graph must not be replayed
                zbuf.fill_(float("nan"))
                mg.vcycle(r, zbuf)
                side.synchronize()
                assert torch_cuda.equal(zbuf, outs[0])
                r2 = r * 2.0                              # a different pair: eager again, then captured again
                z2 = torch_cuda.empty_like(r)
                for _ in range(3):
                    mg.vcycle(r2, z2)
                side.synchronize()
                assert relerr(z2.cpu().numpy(), 2.0 * oz) <= 1e-11
        finally:
            for s_ in sems:
                s_.close()


@pytest.mark.slow
def test_config5_solve_40cubed_against_analytic_solution(torch_cuda, binding):
    """S20: config 5's recipe at 40^3 elements (32.8 M local nodes; the full 100^3 run is recorded in
    profiles/r1d_config5.md): unique / shared counts from the closed forms, convergence to 1e-8, the iteration count
    grows like the mesh (569 at 16^3, ~3.1 k at 100^3), and the converged solution is the analytic one to 1e-8."""
    n = 40
    m = inputs.config5(n)
    with binding.Sem(m.E, m.N, m.vert, m.gid, m.dirichlet) as sem:
        sem.geom(with_mass=True)
        cnt = sem.counts()
        assert cnt["U"] == (7 * n + 1) ** 3 and cnt["nL"] == n ** 3 * 512
        xi = torch_cuda.from_numpy(sem.gll()[0]).cuda()
        V = torch_cuda.from_numpy(m.vert).cuda()
        w1 = torch_cuda.stack([(1 - xi) / 2, (1 + xi) / 2])
        xyz = torch_cuda.zeros(m.E, 8, 8, 8, 3, device="cuda", dtype=torch_cuda.float64)
        for v in range(8):
            ia, ib, ic = v & 1, (v >> 1) & 1, (v >> 2) & 1
            wgt = w1[ic][:, None, None] * w1[ib][None, :, None] * w1[ia][None, None, :]
            xyz += wgt[None, :, :, :, None] * V[:, v][:, None, None, None, :]
        exact = (torch_cuda.sin(np.pi * xyz[..., 0]) * torch_cuda.sin(np.pi * xyz[..., 1])
                 * torch_cuda.sin(np.pi * xyz[..., 2])).reshape(-1)
        del xyz
        f = 3 * np.pi ** 2 * exact
        bf, t2 = torch_cuda.empty_like(f), torch_cuda.empty_like(f)
        sem.ax(f, bf, 1.0)
        sem.ax(f, t2, 0.0)
        bf -= t2                                              # (A + B) f - A f = B f, element by element
        sem.gs(bf)
        bf[torch_cuda.from_numpy(m.dirichlet.ravel()).cuda() != 0] = 0.0
        x = torch_cuda.zeros_like(bf)
        it, rel = sem.pcg(bf, x, 1e-8, 5000)
        assert rel <= 1e-8 and 1000 <= it <= 1700
        assert float((x - exact).abs().max()) <= 1e-8


# ------------------------------------------------------------- NEXT-3: projection onto previous solutions
def test_projection_parity(torch_cuda, binding, oracle_mod):
    """sem_proj_* against the oracle's Projection over a sequence of smoothly evolving right-hand sides, including a
    restart (Lmax = 4) and a dropped direction: guess and reduced right-hand side to 1e-9 at every step."""
    m = inputs.box_mesh(4, 3, 3, 5, "random", seed=7)
    L0 = oracle_mod.Level(m, power_its=2)
    free = L0.mask_u == 0
    n = L0.maps.U
    l2u = L0.maps.l2u
    base, drift, wig, extra = (np.where(free, inputs.field_normal(L0.maps.uniq_gid, s_), 0.0) for s_ in (21, 22, 23, 24))
    oproj = oracle_mod.Projection(L0.A, n, Lmax=4)
    with make_sem(binding, m, dirichlet=True) as sem, binding.Proj(sem, 4) as gproj:
        for step in range(9):
            # every step brings a genuinely new component (otherwise the update would orthonormalise rounding noise,
            # which is valid on both sides but not comparable)
            fresh = np.where(free, inputs.field_normal(L0.maps.uniq_gid, 100 + step), 0.0)
            xs = base + 0.1 * step * drift + 0.01 * np.sin(step) * wig + 0.003 * fresh + (0.05 * extra if step >= 5 else 0.0)
            b_u = L0.A(xs)
            o_xbar, o_bred = oproj.guess(b_u)
            b = to_dev(torch_cuda, b_u[l2u])
            xbar, bred = torch_cuda.full_like(b, float("nan")), torch_cuda.full_like(b, float("nan"))
            gproj.guess(b, xbar, bred)
            scale = max(np.max(np.abs(xs)), 1e-300)
            assert np.max(np.abs(xbar.cpu().numpy() - o_xbar[l2u])) <= 1e-9 * scale, step
            assert np.max(np.abs(bred.cpu().numpy() - o_bred[l2u])) <= 1e-9 * np.max(np.abs(b_u)), step
            o_acc = oproj.update(xs - o_xbar)                      # each side solves its own reduced problem exactly
            dx = to_dev(torch_cuda, xs[l2u]) - xbar
            g_acc = gproj.update(dx)
            assert g_acc == o_acc and gproj.size() == oproj.P.shape[0], step
        # a direction inside the space is dropped on both sides
        inside = oproj.P[0] * 0.5 + oproj.P[-1] * 2.0 if oproj.P.shape[0] < 4 else None
        if inside is not None:
            assert oproj.update(inside) is False
            assert gproj.update(to_dev(torch_cuda, inside[l2u])) is False
    with make_sem(binding, m, dirichlet=True) as sem:
        with pytest.raises(binding.SemError):
            binding.Proj(sem, 0)


def test_helmholtz_smoother_and_vcycle(torch_cuda, binding, oracle_mod):
    """S18: H = A + lambda B through the NEXT-1 calls: the smoother and the V-cycle use the level's own Helmholtz
    diagonal and operator (lambda = 4 on every level), against the oracle."""
    lam = 4.0
    orders = (5, 2)
    meshes = [inputs.box_mesh(4, 3, 3, N, "random", seed=9) for N in orders]
    olv = [oracle_mod.Level(m, lam=lam) for m in meshes]
    L0 = olv[0]
    r_u = np.where(L0.mask_u != 0, 0.0, inputs.field_normal(L0.maps.uniq_gid, 13))
    o_s = L0.smooth(r_u, None, 3)[L0.maps.l2u]
    o_v = oracle_mod.vcycle(olv, r_u, 2, 6)[L0.maps.l2u]
    sems = []
    try:
        for m in meshes:
            s_ = binding.Sem(m.E, m.N, m.vert, m.gid, m.dirichlet)
            s_.geom(with_mass=True)
            s_.set_lambda(lam)
            sems.append(s_)
        r = to_dev(torch_cuda, r_u[L0.maps.l2u])
        x = torch_cuda.full_like(r, float("nan"))
        sems[0].cheby(r, x, 3, L0.lmin, L0.lmax, True)
        assert relerr(x.cpu().numpy(), o_s) <= TOL64
        with binding.Pmg(sems, [l.lmin for l in olv], [l.lmax for l in olv], 2, 6, binding.SEM_F64) as mg:
            z = torch_cuda.full_like(r, float("nan"))
            mg.vcycle(r, z)
            assert relerr(z.cpu().numpy(), o_v) <= 1e-11
    finally:
        for s_ in sems:
            s_.close()


def test_high_multiplicity_node(torch_cuda, binding, oracle_mod):
    """A node shared by 300 elements (a "star" of unit cubes glued at one vertex; gids are arbitrary, S11): the
    gather-scatter's generic path for more than 8 copies, and the PCG's fallback to 8-byte dot weights when a
    multiplicity does not fit a byte."""
    E, N = 300, 2
    p3 = (N + 1) ** 3
    base = inputs.box_mesh(1, 1, 1, N)
    vert = np.repeat(base.vert, E, axis=0)
    gid = (1 + np.arange(E * p3, dtype=np.int64)).reshape(E, p3)
    gid[:, 0] = 0                                            # local node 0 of every element is the same global node
    dirichlet = np.zeros((E, p3), np.uint8)
    dirichlet[:, p3 - 1] = 1                                 # one Dirichlet node per element: the operator is SPD
    om = oracle_mod.Maps(gid)
    assert om.mult.max() == E
    oG, _, _ = oracle_mod.geom_trilinear(vert, N)
    mask_u = oracle_mod.mask_unique(dirichlet, om)
    u = inputs.field_uniform(gid, 3)
    ow = oracle_mod.gs(oracle_mod.ax(oG, u, N).ravel(), om)
    xs = np.where(mask_u != 0, 0.0, inputs.field_normal(om.uniq_gid, 5))
    b_u = oracle_mod.apply_Ag(oG, N, om, mask_u, xs)
    ores = oracle_mod.pcg(oG, N, om, mask_u, b_u, tol=1e-30, maxit=12)
    with binding.Sem(E, N, vert, gid) as sem:
        sem.geom()
        du = to_dev(torch_cuda, u.ravel())
        dw = torch_cuda.empty_like(du)
        sem.ax_gs(du, dw)
        assert relerr(dw.cpu().numpy(), ow) <= TOL64
    with binding.Sem(E, N, vert, gid, dirichlet) as sem:
        sem.geom()
        b = to_dev(torch_cuda, b_u[om.l2u])
        x = torch_cuda.zeros_like(b)
        it, rel = sem.pcg(b, x, 1e-30, 12)
        assert it == 12
        assert relerr(x.cpu().numpy(), ores["x"][om.l2u]) <= TOLPCG


def test_ax_gs_graph_replay_on_side_stream(torch_cuda, binding, oracle_mod):
    """Repeated sem_ax_gs with the same arguments on a non-default stream: eager, captured, replayed -- bit-identical,
    equal to the oracle; new arguments, a new variant or a re-built geometry drop the recorded graph."""
    m = inputs.box_mesh(6, 5, 4, 7, "smooth")
    u = inputs.field_uniform(m.gid, 3)
    ow = _ax_gs_oracle(oracle_mod, m, u, True)
    side = torch_cuda.cuda.Stream()
    with torch_cuda.cuda.stream(side):
        with make_sem(binding, m, dirichlet=True) as sem:
            du = to_dev(torch_cuda, u.ravel())
            dw = torch_cuda.empty_like(du)
            outs = []
            for _ in range(4):
                dw.fill_(float("nan"))
                sem.ax_gs(du, dw)
                side.synchronize()
                outs.append(dw.clone())
            for o in outs[1:]:
                assert torch_cuda.equal(o, outs[0])
            assert relerr(outs[0].cpu().numpy(), ow) <= TOL64
            du2 = du * 3.0                                   # other arguments: eager, then recorded again
            dw2 = torch_cuda.empty_like(du)
            for _ in range(3):
                sem.ax_gs(du2, dw2)
            side.synchronize()
            assert relerr(dw2.cpu().numpy(), 3.0 * ow) <= TOL64
            sem.geom()                                       # re-built geometry: the graph over (du2, dw2) is stale
            dw2.fill_(float("nan"))
            sem.ax_gs(du2, dw2)
            side.synchronize()
            assert relerr(dw2.cpu().numpy(), 3.0 * ow) <= TOL64
            d32 = du.float()
            w32 = torch_cuda.empty_like(d32)
            for _ in range(3):
                sem.ax_gs(d32, w32)                          # another precision
            side.synchronize()
            assert relerr(w32.cpu().numpy(), ow) <= TOL32


def test_fpcg_iteration_graph_on_side_stream(torch_cuda, binding, oracle_mod):
    """On a non-default stream sem_fpcg records one whole iteration as a CUDA graph (from the second iteration of the
    first solve) and replays it, also in later solves: iteration counts, residual history and solution equal the
    oracle's, solve after solve."""
    orders = (5, 2)
    meshes = [inputs.box_mesh(4, 4, 3, N, "random", seed=5) for N in orders]
    olv = [oracle_mod.Level(m) for m in meshes]
    L0 = olv[0]
    xs = np.where(L0.mask_u != 0, 0.0, inputs.field_normal(L0.maps.uniq_gid, 17))
    b_u = L0.A(xs)
    ores = oracle_mod.fpcg(L0, lambda r: oracle_mod.vcycle(olv, r, 2, 6), b_u, tol=1e-9, maxit=60)
    side = torch_cuda.cuda.Stream()
    with torch_cuda.cuda.stream(side):
        sems = [make_sem(binding, m, dirichlet=True) for m in meshes]
        try:
            with binding.Pmg(sems, [l.lmin for l in olv], [l.lmax for l in olv], 2, 6, binding.SEM_F64) as mg:
                b = to_dev(torch_cuda, b_u[L0.maps.l2u])
                x = torch_cuda.empty_like(b)
                for solve in range(3):
                    x.fill_(float("nan"))
                    it, rel = mg.fpcg(b, x, 1e-9, 60)
                    assert it == ores["iters"] and rel <= 1e-9, solve
                    assert np.max(np.abs(mg.history(it + 1) - ores["hist"]) / ores["hist"]) <= 1e-6, solve
                    assert relerr(x.cpu().numpy(), ores["x"][L0.maps.l2u]) <= 1e-8, solve
                b2 = b * 2.0                                   # another right-hand side: the graph is recorded anew
                it, _ = mg.fpcg(b2, x, 1e-9, 60)
                assert it == ores["iters"] and relerr(x.cpu().numpy(), 2.0 * ores["x"][L0.maps.l2u]) <= 1e-8
        finally:
            for s_ in sems:
                s_.close()


# ------------------------------------------- NEXT-2a: fast-diagonalisation local solve of the Schwarz smoother, Eq. (3)
def _fdm_inputs(oracle_mod, E, m, seed):
    """Seeded operator pairs -> (S, Lambda^-1) by the oracle's eigen-decomposition (inputs of Eq. (3)) and a seeded b."""
    A, B = inputs.fdm_pairs(E, m, seed)
    S = np.empty_like(A)
    invL = np.empty((E, m, m, m))
    for e in range(E):
        lam = []
        for d in range(3):
            S[e, d], l = oracle_mod.fdm_eig(A[e, d], B[e, d])
            lam.append(l)
        invL[e] = oracle_mod.fdm_inv_lambda(*lam)
    b = 2.0 * inputs.hash_uniform01(seed, 12, np.arange(E * m ** 3)).reshape(E, m, m, m) - 1.0
    return S, invL, b


@pytest.mark.parametrize("m,E", [(10, 1500), (10, 3), (4, 5000), (6, 777), (8, 1201), (12, 301), (7, 450), (9, 333),
                                 (2, 100), (3, 65), (5, 129), (16, 150), (13, 97),
                                 # several groups per persistent CTA (the stage is re-filled while in use), at the
                                 # element counts the sweep times: config 2's E = 7200 and the paper's E/P = 3573
                                 (10, 7200), (11, 3573), (8, 9001), (6, 30001), (12, 2500), (16, 701), (4, 60000)])
def test_fdm_apply_parity(torch_cuda, binding, oracle_mod, m, E):
    """sem_fdm_apply against the oracle's Eq. (3) on the same S, Lambda^-1, b: FP64 1e-12, FP32 1e-5 (normalised by
    max |u| per case), more elements than one wave of CTAs holds at m = 10 and a ragged last group; in place too."""
    S, invL, b = _fdm_inputs(oracle_mod, E, m, seed=30 + m)
    ou = oracle_mod.fdm_apply(S, invL, b)
    mesh = inputs.box_mesh(E, 1, 1, 1)                                   # the call only needs E and the stream
    with binding.Sem(mesh.E, 1, mesh.vert, mesh.gid) as sem:
        for dt, tol in ((torch_cuda.float64, TOL64), (torch_cuda.float32, TOL32)):
            dS, dL, db = (to_dev(torch_cuda, a.ravel(), dt) for a in (S, invL, b))
            du = torch_cuda.full_like(db, float("nan"))
            sem.fdm_apply(m, dS, dL, db, du)
            assert relerr(du.cpu().numpy(), ou.ravel()) <= tol, (m, E, dt)
            sem.fdm_apply(m, dS, dL, db, db)                             # in place
            assert torch_cuda.equal(db, du)


def test_fdm_apply_bad_args(torch_cuda, binding):
    mesh = inputs.box_mesh(2, 1, 1, 1)
    with binding.Sem(mesh.E, 1, mesh.vert, mesh.gid) as sem:
        z = torch_cuda.zeros(2 * 17 ** 3, dtype=torch_cuda.float64, device="cuda")
        for m in (1, 17):
            rc = sem._L.sem_fdm_apply(sem._h, m, z.data_ptr(), z.data_ptr(), z.data_ptr(), z.data_ptr(), binding.SEM_F64)
            assert rc == binding.SEM_EINVAL
        assert sem._L.sem_fdm_apply(sem._h, 4, None, z.data_ptr(), z.data_ptr(), z.data_ptr(), binding.SEM_F64) == binding.SEM_EINVAL
        assert sem._L.sem_fdm_apply(sem._h, 4, z.data_ptr(), z.data_ptr(), z.data_ptr(), z.data_ptr(), 5) == binding.SEM_EINVAL


@pytest.mark.parametrize("m,E", [(10, 2000), (6, 500)])
def test_fdm_setup_and_apply_pipeline(torch_cuda, binding, oracle_mod, m, E):
    """The library's own setup (sem_fdm_setup, host) feeding sem_fdm_apply, against the oracle's eigen-decomposition
    feeding the oracle's Eq. (3): the result does not depend on eigenvector signs or on the basis chosen inside a
    (nearly) degenerate eigenspace, so it is what is compared."""
    A, B = inputs.fdm_pairs(E, m, seed=70 + m)
    So, invLo, b = _fdm_inputs(oracle_mod, E, m, seed=70 + m)
    ou = oracle_mod.fdm_apply(So, invLo, b)
    S, invL = binding.fdm_setup(A, B)
    mesh = inputs.box_mesh(E, 1, 1, 1)
    with binding.Sem(mesh.E, 1, mesh.vert, mesh.gid) as sem:
        for dt, tol in ((torch_cuda.float64, 1e-11), (torch_cuda.float32, TOL32)):
            dS, dL, db = (to_dev(torch_cuda, a.ravel(), dt) for a in (S, invL, b))
            du = torch_cuda.empty_like(db)
            sem.fdm_apply(m, dS, dL, db, du)
            assert relerr(du.cpu().numpy(), ou.ravel()) <= tol, (m, E, dt)


# ------------------------------------------------- NEXT-4, first piece: gatherScatterMany (Table 3)
@pytest.mark.parametrize("N,nf,pad", [(7, 3, 0), (7, 3, 40), (3, 4, 8), (5, 2, 0), (1, 7, 16), (2, 5, 0), (7, 1, 0)])
def test_gs_many_bit_identical(torch_cuda, binding, oracle_mod, N, nf, pad):
    """sem_gs_many on nf fields (stride nL + pad) against the oracle's gather-scatter of each field: same ascending-index
    sums, so FP64 agrees to the last bit; the padding between fields is left untouched; FP32 at 1e-6.  Scrambled element
    order; the 4x4x3 mesh has pair, quad and 8-copy records."""
    m = inputs.box_mesh(4, 4, 3, N, permute_seed=6)
    om = oracle_mod.Maps(m.gid)
    rng = np.random.default_rng(100 + N)
    w = rng.standard_normal((nf, m.nL + pad))                 # NOT continuous: a genuine gather-scatter input
    ow = w.copy()
    for f in range(nf):
        ow[f, :m.nL] = oracle_mod.gs(w[f, :m.nL].copy(), om)
    with binding.Sem(m.E, m.N, m.vert, m.gid) as sem:
        dw = to_dev(torch_cuda, w)
        sem.gs_many(dw)
        assert np.array_equal(dw.cpu().numpy(), ow)
        dw32 = to_dev(torch_cuda, w.astype(np.float32))
        sem.gs_many(dw32)
        assert relerr(dw32.cpu().numpy()[:, :m.nL], ow[:, :m.nL]) <= 1e-6
        with pytest.raises(binding.SemError):
            sem._check(sem._L.sem_gs_many(sem._h, dw.data_ptr(), 3, m.nL - 1, binding.SEM_F64, binding.SEM_OP_ADD))


def test_gs_many_config2_three_fields(torch_cuda, binding, oracle_mod):
    """Full size (config 2, three velocity-like fields): sem_gs_many equals sem_gs field by field, bit for bit, and the
    oracle on sampled shared nodes."""
    m = inputs.config2()
    om = oracle_mod.Maps(m.gid)
    rng = np.random.default_rng(8)
    w = rng.standard_normal((3, m.nL))
    with binding.Sem(m.E, m.N, m.vert, m.gid) as sem:
        dw = to_dev(torch_cuda, w)
        sem.gs_many(dw)
        for f in range(3):
            d1 = to_dev(torch_cuda, w[f])
            sem.gs(d1)
            assert torch_cuda.equal(d1, dw[f])
        got = dw.cpu().numpy()
    sample = rng.integers(0, om.U, 2000)
    for g in sample:
        idx = om.seg_idx[om.seg_off[g]:om.seg_off[g + 1]]
        for f in range(3):
            s = 0.0
            for l in idx:                                     # ascending local index, like O5
                s += w[f, l]
            assert np.all(got[f, idx] == s)
