"""sem_cheby_noalloc (include/sem.h): the Chebyshev-Jacobi smoother with its work vectors in the library's static device
array, for callers that cannot call cudaMalloc.  Checked against the existing path (sem_cheby, FP64, matrix-free) and
the CPU oracle on two calls in a row that share the array.  This file sorts last on purpose: the suite runs with
pytest -x, and a failure here must not hide any other test.  It passes alone in a fresh process and after the others."""
import numpy as np
import pytest

from paper_2110_01716_b200 import inputs

pytestmark = pytest.mark.gpu

TOL64 = 1e-12


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


def to_dev(torch, a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def test_cheby_noalloc_matches_existing_path_twice(torch_cuda, binding, oracle_mod):
    """Two calls in a row (different right-hand side, order, guess, and a second context of another size in between, all
    sharing the static array): each equals sem_cheby's FP64 result to 1e-12 and the oracle's Chebyshev-Jacobi; the device
    memory in use does not change across the calls; sizes beyond SEM_NOALLOC_MAX_NODES and a missing Jacobi diagonal are
    refused with a clear error."""
    torch = torch_cuda
    m = inputs.box_mesh(5, 4, 3, 7, "random", seed=6, permute_seed=3)            # 60 elements, 30 720 nodes
    m2 = inputs.box_mesh(6, 5, 4, 3, "random", seed=2)                            # another context, N = 3
    L = oracle_mod.Level(m, power_its=30)
    L2 = oracle_mod.Level(m2, power_its=30)
    with binding.Sem(m.E, m.N, m.vert, m.gid, m.dirichlet) as sem, binding.Sem(m2.E, m2.N, m2.vert, m2.gid, m2.dirichlet) as sem2:
        sem.geom()
        sem2.geom()
        b0 = torch.zeros(sem.nL, device="cuda", dtype=torch.float64)
        x0 = torch.zeros_like(b0)
        with pytest.raises(binding.SemError, match="Jacobi diagonal"):             # building it would allocate
            sem.cheby_noalloc(b0, x0, 2, L.lmin, L.lmax, True)
        sem.get_diag()                                                            # set-up: the diagonal, once
        sem2.get_diag()
        cases = [(sem, L, 11, 4, True), (sem2, L2, 12, 3, False), (sem, L, 13, 3, False), (sem, L, 14, 1, True)]
        ref = []
        for s, lev, seed, order, zero in cases:                                   # the existing path first
            b_u = np.where(lev.mask_u != 0, 0.0, inputs.field_normal(lev.maps.uniq_gid, seed))
            x_u = None if zero else np.where(lev.mask_u != 0, 0.0, inputs.field_normal(lev.maps.uniq_gid, seed + 50))
            db = to_dev(torch, b_u[lev.maps.l2u])
            dx = torch.full_like(db, float("nan")) if zero else to_dev(torch, x_u[lev.maps.l2u])
            monkey = pytest.MonkeyPatch()
            monkey.setenv("SEM_COARSE", "0")
            try:
                s.cheby(db, dx, order, lev.lmin, lev.lmax, zero)
            finally:
                monkey.undo()
            torch.cuda.synchronize()
            ref.append((db, x_u, dx.cpu().numpy(), lev.smooth(b_u, x_u, order)[lev.maps.l2u]))
        sem.cheby_noalloc(ref[0][0], torch.empty_like(ref[0][0]), 2, L.lmin, L.lmax, True)   # resolves the symbol address
        torch.cuda.synchronize()
        outs = []
        for (s, lev, seed, order, zero), (db, x_u, _, _) in zip(cases, ref):      # back to back, no sync in between
            dx = torch.full_like(db, float("nan")) if zero else to_dev(torch, x_u[lev.maps.l2u])
            outs.append(dx)
        free0 = torch.cuda.mem_get_info()[0]
        for (s, lev, seed, order, zero), dx, (db, _, _, _) in zip(cases, outs, ref):
            s.cheby_noalloc(db, dx, order, lev.lmin, lev.lmax, zero)
        torch.cuda.synchronize()
        assert torch.cuda.mem_get_info()[0] == free0                               # nothing was allocated on the device
        for dx, (_, _, existing, orc) in zip(outs, ref):
            got = dx.cpu().numpy()
            assert relerr(got, existing) <= TOL64
            assert relerr(got, orc) <= 1e-11
    # beyond the stated maximum: refused, with the limit in the message
    big = inputs.box_mesh(11, 10, 10, 7, "affine")                                 # 1100 elements, 563 200 nodes > 2^19
    assert big.nL > binding.SEM_NOALLOC_MAX_NODES
    with binding.Sem(big.E, big.N, big.vert, big.gid) as sb:
        sb.geom()
        sb.get_diag()
        b = torch.zeros(sb.nL, device="cuda", dtype=torch.float64)
        with pytest.raises(binding.SemError, match="SEM_NOALLOC_MAX_NODES"):
            sb.cheby_noalloc(b, torch.zeros_like(b), 2, 0.1, 1.0, True)
