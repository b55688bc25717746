"""Pins for the CPU oracle: everything here is fixed by the paper's definitions and by
mathematics, and is computed WITHOUT the oracle's own formulas (closed forms, numpy.polynomial, dense Kronecker /
weak-form brute force, dense Cholesky), so that a dropped term, wrong sign/index or transposed operand fails."""
import os

import numpy as np
import numpy.polynomial.legendre as npleg
import numpy.polynomial.polynomial as nppoly
import pytest

from paper_2110_01716_b200 import inputs

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def read_golden(name):
    out = {}
    for line in open(os.path.join(GOLD, name)):
        if line.startswith("#") or not line.strip():
            continue
        k, v = line.split(None, 1)
        out[k] = v.strip()
    return out


# ---------- independent 1-D data (numpy.polynomial, Lagrange polynomials differentiated explicitly) -------------
def ref_gll(N):
    PN = npleg.Legendre.basis(N)
    xi = np.concatenate([[-1.0], np.sort(PN.deriv().roots().real), [1.0]])
    rho = 2.0 / (N * (N + 1) * PN(xi) ** 2)
    return xi, rho


def ref_D(xi):
    p = xi.size
    D = np.zeros((p, p))
    for l in range(p):
        others = np.delete(xi, l)
        c = nppoly.polyfromroots(others) / np.prod(xi[l] - others)   # h_l as monomial coefficients
        D[:, l] = nppoly.polyval(xi, nppoly.polyder(c))              # dh_l/dr at xi_i
    return D


def ref_trilinear(vert_e, r, s, t):
    """x(r,s,t) for one element; r,s,t arrays of equal shape -> [...,3]."""
    X = 0.0
    for v in range(8):
        a, b, c = v & 1, (v >> 1) & 1, (v >> 2) & 1
        phi = (1 + (2 * a - 1) * r) * (1 + (2 * b - 1) * s) * (1 + (2 * c - 1) * t) / 8.0
        X = X + phi[..., None] * vert_e[v]
    return X


def dense_element_matrix(vert_e, N):
    """Weak-form brute force: A_mn = sum_q rho_q detJ_q grad(phi_m)(x_q) . grad(phi_n)(x_q) with PHYSICAL gradients,
    phi the 3-D Lagrange basis; the O(N^6) formation of P:75 / P:107.  Also returns the diagonal mass."""
    xi, rho = ref_gll(N)
    D1 = ref_D(xi)
    p = N + 1
    I = np.eye(p)
    Dref = [np.kron(I, np.kron(I, D1)), np.kron(I, np.kron(D1, I)), np.kron(D1, np.kron(I, I))]  # d/dr, d/ds, d/dt
    T, S, R = np.meshgrid(xi, xi, xi, indexing="ij")            # node (k,j,i): t=xi_k, s=xi_j, r=xi_i
    X = ref_trilinear(vert_e, R.ravel(), S.ravel(), T.ravel())  # [p^3,3]
    W = (rho[:, None, None] * rho[None, :, None] * rho[None, None, :]).ravel()
    J = np.stack([np.stack([Dref[b] @ X[:, a] for b in range(3)], axis=-1) for a in range(3)], axis=1)  # [q,a,b]
    det = np.linalg.det(J)
    Rinv = np.linalg.inv(J)                                      # [q,b,a] = dr_b/dx_a
    A = np.zeros((p ** 3, p ** 3))
    for a in range(3):
        Ga = sum(Rinv[:, b, a][:, None] * Dref[b] for b in range(3))   # d phi_n / d x_a at q
        A += Ga.T @ ((W * det)[:, None] * Ga)
    return A, W * det


def assemble_dense(mesh):
    gids, inv = np.unique(mesh.gid.ravel(), return_inverse=True)
    inv = inv.reshape(mesh.gid.shape)
    U = gids.size
    A = np.zeros((U, U))
    B = np.zeros(U)
    for e in range(mesh.E):
        Ae, Be = dense_element_matrix(mesh.vert[e], mesh.N)
        A[np.ix_(inv[e], inv[e])] += Ae
        np.add.at(B, inv[e], Be)
    return A, B, inv


def tiny_mesh(N=3):
    m = inputs.box_mesh(2, 2, 2, N, "affine")
    # perturb the single interior vertex (it is vertex 7 of element 0, 6 of element 1, ... ) consistently
    target = np.array([0.5, 0.5, 0.5])
    sel = np.all(np.isclose(m.vert, target), axis=-1)
    m.vert[sel] = target + np.array([0.07, -0.05, 0.04])
    return m


# ---------------------------------------------- P1, P2 -----------------------------------------------------------
def test_P1_closed_forms(oracle_mod):
    xi, rho, D = oracle_mod.gll(1)
    assert np.allclose(xi, [-1, 1], atol=0) and np.allclose(rho, [1, 1], atol=1e-15)
    assert np.allclose(D, [[-0.5, 0.5], [-0.5, 0.5]], atol=1e-15)
    xi, rho, D = oracle_mod.gll(2)
    assert np.allclose(xi, [-1, 0, 1], atol=1e-16) and np.allclose(rho, [1 / 3, 4 / 3, 1 / 3], atol=1e-15)
    assert np.allclose(D, [[-1.5, 2, -0.5], [-0.5, 0, 0.5], [0.5, -2, 1.5]], atol=1e-14)
    xi, rho, _ = oracle_mod.gll(3)
    assert np.allclose(xi, [-1, -1 / np.sqrt(5), 1 / np.sqrt(5), 1], atol=1e-15)
    assert np.allclose(rho, [1 / 6, 5 / 6, 5 / 6, 1 / 6], atol=1e-15)
    xi, rho, _ = oracle_mod.gll(4)
    assert np.allclose(xi, [-1, -np.sqrt(3 / 7), 0, np.sqrt(3 / 7), 1], atol=1e-15)
    assert np.allclose(rho, [1 / 10, 49 / 90, 32 / 45, 49 / 90, 1 / 10], atol=1e-15)
    xi, rho, D = oracle_mod.gll(7)   # standard Lobatto tables
    assert np.allclose(xi[4:], [0.2092992179024789, 0.5917001814331423, 0.8717401485096066, 1.0], atol=1e-15)
    assert np.allclose(rho[4:], [0.4124587946587038, 0.3411226924835044, 0.2107042271435061, 1 / 28], atol=1e-15)
    assert D[0, 0] == pytest.approx(-14.0, abs=1e-13) and D[0, 7] == pytest.approx(0.5, abs=1e-13)
    assert D[7, 7] == pytest.approx(14.0, abs=1e-13)


@pytest.mark.parametrize("N", [1, 2, 3, 4, 5, 6, 7, 8, 9, 11, 15])
def test_P2_exactness_and_independent_tables(oracle_mod, N):
    xi, rho, D = oracle_mod.gll(N)
    rxi, rrho = ref_gll(N)
    assert np.allclose(xi, rxi, atol=2e-14) and np.allclose(rho, rrho, rtol=1e-12)
    assert np.allclose(D, ref_D(rxi), atol=1e-10 * N * N)
    assert np.all(np.diff(xi) > 0) and np.allclose(xi, -xi[::-1], atol=0)
    assert abs(rho.sum() - 2.0) < 1e-14
    assert np.abs(D.sum(axis=1)).max() < 1e-12 * N * N             # D annihilates constants
    for m in range(1, N + 1):                                      # D xi^m = m xi^(m-1) exactly for m <= N
        assert np.allclose(D @ xi ** m, m * xi ** (m - 1), atol=1e-11 * N)
    for m in range(0, 2 * N):                                      # quadrature exact to degree 2N-1
        exact = 0.0 if m % 2 else 2.0 / (m + 1)
        assert abs(rho @ xi ** m - exact) < 1e-14
    # antisymmetry D[i,l] = -D[N-i,N-l] (centro-skew-symmetric): catches a transposed / flipped operand
    assert np.allclose(D, -D[::-1, ::-1], atol=1e-12 * N * N)


# ---------------------------------------------- P3..P8, P11 ------------------------------------------------------
@pytest.fixture(scope="module")
def cfg1(oracle_mod):
    m = inputs.config1()
    xyz = oracle_mod.node_xyz(m.vert, m.N)
    G, dJ, rc = oracle_mod.geom_iso(xyz, m.N)
    assert rc == 0
    maps = oracle_mod.Maps(m.gid)
    return m, xyz, G, dJ, maps


def test_O2_nodes_match_independent_trilinear(oracle_mod, cfg1):
    m, xyz, *_ = cfg1
    xi, _ = ref_gll(m.N)
    T, S, R = np.meshgrid(xi, xi, xi, indexing="ij")
    for e in (0, 21, 63):
        assert np.allclose(xyz[e], ref_trilinear(m.vert[e], R.ravel(), S.ravel(), T.ravel()), atol=1e-15)


def test_P3_constants_annihilated(oracle_mod, cfg1):
    m, xyz, G, *_ = cfg1
    w = oracle_mod.ax(G, np.ones((m.E, m.p ** 3)), m.N)
    scale = np.abs(oracle_mod.ax(G, xyz[..., 0].copy(), m.N)).max()
    assert np.abs(w).max() < 1e-13 * scale


def test_P4_symmetric_positive_semidefinite(oracle_mod, cfg1):
    m, xyz, G, dJ, maps = cfg1
    u = inputs.field_uniform(m.gid, 11)
    v = inputs.field_uniform(m.gid, 12)
    Au, Av = oracle_mod.ax(G, u, m.N), oracle_mod.ax(G, v, m.N)
    assert abs((v * Au).sum() - (u * Av).sum()) < 1e-13 * abs((u * Au).sum())
    assert (u * Au).sum() > 0 and (v * Av).sum() > 0
    # the same through gs: (QQ^T A u) weighted by 1/mult is the assembled product
    wts = 1.0 / maps.mult[maps.l2u].reshape(u.shape)
    gAu, gAv = oracle_mod.gs(Au, maps), oracle_mod.gs(Av, maps)
    assert abs((wts * v * gAu).sum() - (wts * u * gAv).sum()) < 1e-13 * abs((wts * u * gAu).sum())


def test_P5_volume_and_P13_detJ(oracle_mod, cfg1):
    m, xyz, G, dJ, maps = cfg1
    assert abs(G[:, 6].sum() - 1.0) < 1e-13                       # sum of B = volume of [0,1]^3
    gold = read_golden("p13_config1_pcg.txt")
    assert dJ.min() == pytest.approx(float(gold["detJ_min"]), rel=1e-10)
    assert dJ.max() == pytest.approx(float(gold["detJ_max"]), rel=1e-10)
    for cfg in (inputs.config3(3, 2), inputs.config3(2, 5)):
        Gc, dJc, rc = oracle_mod.geom_trilinear(cfg.vert, cfg.N)
        assert rc == 0 and abs(Gc[:, 6].sum() - 1.0) < 1e-13


def test_P6_linear_field_energy(oracle_mod, cfg1):
    m, xyz, G, *_ = cfg1
    for d in range(3):
        u = xyz[..., d].copy()
        assert abs((u * oracle_mod.ax(G, u, m.N)).sum() - 1.0) < 1e-12     # |grad x|^2 integrated over the unit box
    u, v = xyz[..., 0].copy(), xyz[..., 1].copy()
    assert abs((v * oracle_mod.ax(G, u, m.N)).sum()) < 1e-12               # grad x . grad y = 0


@pytest.mark.parametrize("N", [2, 3, 7])
def test_P7_affine_kronecker(oracle_mod, N):
    h = np.array([0.5, 0.25, 0.125])                                       # anisotropic box element
    m = inputs.box_mesh(2, 4, 8, N, "affine")
    xi, rho = ref_gll(N)
    D1 = ref_D(xi)
    M, K = np.diag(rho), D1.T @ np.diag(rho) @ D1
    # A_L = (hy hz / (2 hx)) M(x)M(x)K + ... with index order (k,j,i): kron(t, kron(s, r))
    AL = (h[1] * h[2] / (2 * h[0])) * np.kron(M, np.kron(M, K)) + (h[0] * h[2] / (2 * h[1])) * np.kron(M, np.kron(K, M)) \
        + (h[0] * h[1] / (2 * h[2])) * np.kron(K, np.kron(M, M))
    G, dJ, rc = oracle_mod.geom_iso(oracle_mod.node_xyz(m.vert, N), N)
    assert rc == 0
    W = (rho[:, None, None] * rho[None, :, None] * rho[None, None, :]).ravel()
    assert np.allclose(G[5, 0], W * h[1] * h[2] / (2 * h[0]), rtol=1e-12)
    assert np.allclose(G[5, 3], W * h[0] * h[2] / (2 * h[1]), rtol=1e-12)
    assert np.allclose(G[5, 5], W * h[0] * h[1] / (2 * h[2]), rtol=1e-12)
    assert np.abs(G[:, [1, 2, 4]]).max() < 1e-15
    u = inputs.field_uniform(m.gid, 5)
    w = oracle_mod.ax(G, u, N)
    assert np.allclose(w[5], AL @ u[5], atol=1e-13 * np.abs(w).max())
    lam = 0.7                                                              # Helmholtz term (S18)
    wl = oracle_mod.ax(G, u, N, lam)
    assert np.allclose(wl[5], AL @ u[5] + lam * W * np.prod(h) / 8 * u[5], atol=1e-13 * np.abs(wl).max())


def test_P8_trilinear_equals_isoparametric(oracle_mod):
    for m in (inputs.config1(), inputs.config3(3, 4), inputs.config3(2, 9), inputs.config3(3, 1)):
        Gi, dJi, rc1 = oracle_mod.geom_iso(oracle_mod.node_xyz(m.vert, m.N), m.N)
        Gt, dJt, rc2 = oracle_mod.geom_trilinear(m.vert, m.N)
        assert rc1 == 0 and rc2 == 0
        assert np.abs(Gi - Gt).max() < 1e-12 * np.abs(Gi).max()
        assert np.abs(dJi - dJt).max() < 1e-12 * np.abs(dJi).max()


def test_negative_jacobian_flagged(oracle_mod):
    m = inputs.box_mesh(1, 1, 1, 3, "affine")
    m.vert[0, [0, 1]] = m.vert[0, [1, 0]]                                  # swap two vertices: inverted element
    _, _, rc = oracle_mod.geom_trilinear(m.vert, 3)
    assert rc == -2


def test_P11_sin_product_energy(oracle_mod, cfg1):
    m, xyz, G, *_ = cfg1
    u = np.sin(np.pi * xyz[..., 0]) * np.sin(np.pi * xyz[..., 1]) * np.sin(np.pi * xyz[..., 2])
    assert (u * oracle_mod.ax(G, u, m.N)).sum() == pytest.approx(3 * np.pi ** 2 / 8, rel=1e-10)


# ---------------------------------------------- O5/O6 maps and gs ------------------------------------------------
def test_O6_maps_bruteforce(oracle_mod):
    rng = np.random.default_rng(3)
    gid = rng.integers(0, 40, size=300).astype(np.int64) * 1000003        # non-contiguous ids, many duplicates
    mp = oracle_mod.Maps(gid)
    uniq = sorted(set(gid.tolist()))
    assert mp.U == len(uniq) and mp.uniq_gid.tolist() == uniq
    assert mp.l2u.tolist() == [uniq.index(g) for g in gid.tolist()]
    assert mp.mult.tolist() == [gid.tolist().count(g) for g in uniq]
    assert mp.seg_off.tolist() == [0] + np.cumsum(mp.mult).tolist()
    expect_idx = [l for g in uniq for l in range(gid.size) if gid[l] == g]   # (l2u, l) ascending
    assert mp.seg_idx.tolist() == expect_idx
    w = rng.standard_normal(300)
    out = oracle_mod.gs(w, mp)
    for l in range(300):
        assert out[l] == pytest.approx(sum(w[q] for q in range(300) if gid[q] == gid[l]), abs=1e-13)
    with pytest.raises(ValueError):
        oracle_mod.Maps(np.array([3, -1, 2], np.int64))


def test_config1_counts(oracle_mod, cfg1):
    m, *_, maps = cfg1
    gold = read_golden("p13_config1_pcg.txt")
    assert (maps.U, maps.S, maps.Us) == (int(gold["U"]), int(gold["S"]), int(gold["Us"]))
    assert maps.U == m.unique_nodes == 29 ** 3
    hist = {int(k): int(v) for k, v in (t.split(":") for t in gold["mult_hist"].split())}
    bc = np.bincount(maps.mult)
    assert {k: int(bc[k]) for k in np.nonzero(bc)[0]} == hist


# ---------------------------------------------- P9, P10, P14: dense brute force ----------------------------------
@pytest.fixture(scope="module")
def tiny(oracle_mod):
    m = tiny_mesh(3)
    Adense, Bdense, inv = assemble_dense(m)
    G, dJ, rc = oracle_mod.geom_iso(oracle_mod.node_xyz(m.vert, m.N), m.N)
    assert rc == 0 and dJ.min() > 0
    maps = oracle_mod.Maps(m.gid)
    assert np.array_equal(maps.l2u.reshape(inv.shape), inv)
    return m, Adense, Bdense, G, maps


def test_P9_dense_assembly_matches_matrix_free(oracle_mod, tiny):
    m, Adense, Bdense, G, maps = tiny
    U = maps.U
    assert U == 343
    nomask = np.zeros(U, np.uint8)
    Amf = np.stack([oracle_mod.apply_Ag(G, m.N, maps, nomask, np.eye(U)[g]) for g in range(U)], axis=1)
    assert np.abs(Amf - Adense).max() < 1e-13 * np.abs(Adense).max()
    assert np.abs(Adense - Adense.T).max() < 1e-14 * np.abs(Adense).max()
    ev = np.linalg.eigvalsh(0.5 * (Adense + Adense.T))
    assert abs(ev[0]) < 1e-12 * ev[-1] and ev[1] > 1e-6 * ev[-1]          # exactly one zero eigenvalue
    Bo = np.zeros(U)
    np.add.at(Bo, maps.l2u, G[:, 6].ravel())
    assert np.allclose(Bo, Bdense, rtol=1e-12)
    lam = 2.5                                                              # Helmholtz: A + lam B
    y = oracle_mod.apply_Ag(G, m.N, maps, nomask, np.arange(U) / U, lam)
    assert np.allclose(y, (Adense + lam * np.diag(Bdense)) @ (np.arange(U) / U), atol=1e-13 * np.abs(y).max())


def test_P10_exact_diagonal(oracle_mod, tiny):
    m, Adense, Bdense, G, maps = tiny
    dl = oracle_mod.diag_local(G, m.N)
    dg = np.zeros(maps.U)
    np.add.at(dg, maps.l2u, dl.ravel())
    assert np.abs(dg - np.diag(Adense)).max() < 1e-13 * np.diag(Adense).max()
    dl2 = oracle_mod.diag_local(G, m.N, 1.5)
    dg2 = np.zeros(maps.U)
    np.add.at(dg2, maps.l2u, dl2.ravel())
    assert np.allclose(dg2, np.diag(Adense) + 1.5 * Bdense, rtol=1e-12)


def test_P14_pcg_vs_dense_solve_and_krylov_optimality(oracle_mod, tiny):
    m, Adense, Bdense, G, maps = tiny
    mask = oracle_mod.mask_unique(m.dirichlet, maps)
    free = np.nonzero(mask == 0)[0]
    assert free.size == 125
    rng = np.random.default_rng(7)
    b = np.zeros(maps.U)
    b[free] = rng.standard_normal(free.size)
    Aff = Adense[np.ix_(free, free)]
    L = np.linalg.cholesky(Aff)
    xs = np.zeros(maps.U)
    xs[free] = np.linalg.solve(L.T, np.linalg.solve(L, b[free]))
    res = oracle_mod.pcg(G, m.N, maps, mask, b, tol=1e-13, maxit=500)
    assert res["relres"] <= 1e-13 and res["iters"] <= 125 + 20
    assert np.abs(res["x"] - xs).max() < 1e-10 * np.abs(xs).max()
    assert np.all(res["x"][mask == 1] == 0)
    # x_k minimises the A-norm error over span{M^-1 b, (M^-1 A) M^-1 b, ...}: dense least squares in the A-norm
    Minv = 1.0 / np.diag(Aff)
    for k in (1, 2, 3):
        xk = oracle_mod.pcg(G, m.N, maps, mask, b, tol=1e-30, maxit=k)
        assert xk["iters"] == k
        V = [Minv * b[free]]
        for _ in range(k - 1):
            V.append(Minv * (Aff @ V[-1]))
        V = np.stack(V, axis=1)
        c = np.linalg.solve(V.T @ Aff @ V, V.T @ b[free])
        assert np.abs(xk["x"][free] - V @ c).max() < 1e-9 * np.abs(V @ c).max()
    # relres is the recurrence residual relative to ||r0|| and the history is consistent with the returned value
    r1 = b[free] - Aff @ oracle_mod.pcg(G, m.N, maps, mask, b, tol=1e-30, maxit=5)["x"][free]
    h5 = oracle_mod.pcg(G, m.N, maps, mask, b, tol=1e-30, maxit=5)
    assert h5["hist"][5] == pytest.approx(np.linalg.norm(r1) / np.linalg.norm(b[free]), rel=1e-9)
    # non-zero initial guess converges to the same solution; b = 0 returns x0 (masked) with 0 iterations
    x0 = np.zeros(maps.U)
    x0[free] = rng.standard_normal(free.size)
    res2 = oracle_mod.pcg(G, m.N, maps, mask, b, x0_u=x0, tol=1e-13, maxit=500)
    assert np.abs(res2["x"] - xs).max() < 1e-9 * np.abs(xs).max()
    res3 = oracle_mod.pcg(G, m.N, maps, mask, np.zeros(maps.U), tol=1e-8, maxit=10)
    assert res3["iters"] == 0 and np.all(res3["x"] == 0)


def test_P14_element_permutation_invariance(oracle_mod):
    a = inputs.box_mesh(3, 3, 3, 4, "random", seed=5)
    b = inputs.box_mesh(3, 3, 3, 4, "random", seed=5, permute_seed=9)
    assert not np.array_equal(a.perm, b.perm) and sorted(b.perm.tolist()) == list(range(27))
    out = []
    for m in (a, b):
        G, _, rc = oracle_mod.geom_trilinear(m.vert, m.N)
        maps = oracle_mod.Maps(m.gid)
        u = inputs.field_uniform(m.gid, 0)
        w = oracle_mod.gs(oracle_mod.ax(G, u, m.N), maps)
        wu = np.zeros(maps.U)
        wu[maps.l2u] = w.ravel()
        out.append((maps.uniq_gid, wu))
    assert np.array_equal(out[0][0], out[1][0])
    assert np.abs(out[0][1] - out[1][1]).max() < 1e-13 * np.abs(out[0][1]).max()


# ---------------------------------------------- P12: spectral convergence ----------------------------------------
def test_P12_spectral_convergence(oracle_mod):
    gold = {int(k): float(v) for k, v in read_golden("p12_spectral_convergence.txt").items()}
    errs = {}
    for N in range(2, 9):
        m = inputs.box_mesh(2, 2, 2, N, "affine")
        xyz = oracle_mod.node_xyz(m.vert, N)
        G, _, _ = oracle_mod.geom_iso(xyz, N)
        maps = oracle_mod.Maps(m.gid)
        mask = oracle_mod.mask_unique(m.dirichlet, maps)
        sp = np.sin(np.pi * xyz[..., 0]) * np.sin(np.pi * xyz[..., 1]) * np.sin(np.pi * xyz[..., 2])
        b = np.zeros(maps.U)
        np.add.at(b, maps.l2u, (G[:, 6] * 3 * np.pi ** 2 * sp).ravel())    # Q^T (B f)
        b[mask == 1] = 0
        res = oracle_mod.pcg(G, N, maps, mask, b, tol=1e-14, maxit=2000)
        ue = np.zeros(maps.U)
        ue[maps.l2u] = sp.ravel()
        errs[N] = np.abs(res["x"] - ue).max()
        # Rayleigh quotient of the interpolated eigenfunction approaches 3 pi^2 from below
        um = np.where(mask == 1, 0.0, ue)
        rq = um @ oracle_mod.apply_Ag(G, N, maps, mask, um) / (um ** 2 @ np.bincount(maps.l2u, G[:, 6].ravel()))
        assert rq < 3 * np.pi ** 2 + 1e-9 and abs(rq - 3 * np.pi ** 2) < 0.2 * 30.0 ** (2 - N) + 1e-9
    for N in range(3, 9):
        assert errs[N] < errs[N - 1] / 10.0                                # exponential decay in N
    for N, e in errs.items():
        assert e == pytest.approx(gold[N], rel=0.06)                       # survey cross-check (2 printed digits)


# ---------------------------------------------- P13: config-1 PCG history ----------------------------------------
def test_P13_config1_pcg_history(oracle_mod, cfg1):
    m, xyz, G, dJ, maps = cfg1
    gold = read_golden("p13_config1_pcg.txt")
    mask = oracle_mod.mask_unique(m.dirichlet, maps)
    sp = np.sin(np.pi * xyz[..., 0]) * np.sin(np.pi * xyz[..., 1]) * np.sin(np.pi * xyz[..., 2])
    xu = np.zeros(maps.U)
    xu[maps.l2u] = sp.ravel()
    xu[mask == 1] = 0
    b = oracle_mod.apply_Ag(G, m.N, maps, mask, xu)
    assert np.linalg.norm(b) == pytest.approx(float(gold["norm_b"]), rel=1e-11)
    dg = np.bincount(maps.l2u, oracle_mod.diag_local(G, m.N).ravel())
    assert dg.min() == pytest.approx(float(gold["diag_min"]), rel=1e-11)    # over all unique nodes (corner of the box)
    assert dg.max() == pytest.approx(float(gold["diag_max"]), rel=1e-11)
    z = np.where(mask == 1, 0.0, b / dg)
    alpha1 = (b @ z) / (z @ oracle_mod.apply_Ag(G, m.N, maps, mask, z))
    assert alpha1 == pytest.approx(float(gold["alpha1"]), rel=1e-9)
    res = oracle_mod.pcg(G, m.N, maps, mask, b, tol=1e-30, maxit=20, snap_its=(1, 20))
    assert res["iters"] == 20
    for it in (1, 5, 10, 15, 20):
        assert res["hist"][it] == pytest.approx(float(gold[f"relres_it{it}"]), rel=2e-10)
    assert np.abs(res["snaps"][20] - xu).max() == pytest.approx(float(gold["err_inf_it20"]), rel=1e-9)
    assert np.allclose(res["snaps"][1], alpha1 * z, rtol=1e-12, atol=1e-16)
    full = oracle_mod.pcg(G, m.N, maps, mask, b, tol=1e-14, maxit=400)
    assert abs(full["iters"] - int(gold["iters_to_1e-14"])) <= 2
    assert np.abs(full["x"] - xu).max() < 1e-11                           # converges to the masked sin-product itself


def test_inputs_fields_are_continuous_and_seeded():
    m = inputs.config1()
    u = inputs.field_uniform(m.gid, 0)
    assert u.min() >= -1 and u.max() <= 1 and abs(u.mean()) < 0.02
    _, first = np.unique(m.gid.ravel(), return_index=True)
    _, inv = np.unique(m.gid.ravel(), return_inverse=True)
    assert np.array_equal(u.ravel()[first][inv], u.ravel())              # equal on all copies of a shared node
    assert np.array_equal(u, inputs.field_uniform(m.gid, 0)) and not np.array_equal(u, inputs.field_uniform(m.gid, 1))
    g = inputs.field_normal(m.gid, 2)
    assert abs(g.mean()) < 0.02 and abs(g.std() - 1) < 0.02
    r = inputs.config3(4, 3)
    h = 0.25
    V0 = inputs.vertex_grid(4, 4, 4)
    V1 = inputs.deform_random(V0, 0.1, 1)
    assert np.abs(V1 - V0).max() <= 0.1 * h and np.abs(V1 - V0)[1:-1, 1:-1, 1:-1].min() > 0
    assert np.array_equal(V1[0], V0[0]) and np.array_equal(V1[:, :, -1], V0[:, :, -1])
    assert r.dirichlet.sum() > 0 and r.gid.max() == r.unique_nodes - 1


# ---------------------------------------------------------------------------------- NEXT-1: pMG transfer operators
# P:103 "u_f = (J x J x J) u_c, where J is the 1D polynomial interpolation operator from the coarse GLL points to the
# fine GLL points".  Pins: polynomial reproduction (the defining property of interpolation), partition of unity,
# identity at equal orders, nesting of levels, the paper's level schedules, exact 3-D reproduction, and adjointness of
# the restriction.
@pytest.mark.parametrize("Nc,Nf", [(1, 3), (3, 7), (1, 7), (5, 8), (4, 6), (1, 8), (7, 7), (2, 5)])
def test_T1_interp_reproduces_polynomials(oracle_mod, Nc, Nf):
    J = oracle_mod.interp(Nc, Nf)
    xc, _, _ = oracle_mod.gll(Nc)
    xf, _, _ = oracle_mod.gll(Nf)
    assert J.shape == (Nf + 1, Nc + 1)
    for m in range(Nc + 1):                                   # degree <= Nc is reproduced exactly
        assert np.max(np.abs(J @ xc ** m - xf ** m)) <= 1e-13
    assert np.max(np.abs(J.sum(axis=1) - 1.0)) <= 1e-14       # partition of unity
    assert np.max(np.abs(J[0] - np.eye(Nc + 1)[0])) <= 1e-15 and np.max(np.abs(J[-1] - np.eye(Nc + 1)[-1])) <= 1e-15
    if Nc == Nf:
        assert np.max(np.abs(J - np.eye(Nc + 1))) <= 1e-14


def test_T1_interp_closed_form_N1():
    """N_c = 1: the two cardinal functions are (1 -+ x)/2, so J = [(1 - xi_f)/2, (1 + xi_f)/2] (closed form)."""
    import oracle
    xf, _, _ = oracle.gll(7)
    J = oracle.interp(1, 7)
    assert np.max(np.abs(J - np.stack([(1 - xf) / 2, (1 + xf) / 2], axis=1))) <= 1e-15


def test_T2_levels_nest(oracle_mod):
    """Interpolating 1 -> 3 -> 7 equals interpolating 1 -> 7 (config 4's schedule), likewise the paper's 1-5-8."""
    for a, b, c in ((1, 3, 7), (1, 5, 8), (1, 4, 6)):
        assert np.max(np.abs(oracle_mod.interp(b, c) @ oracle_mod.interp(a, b) - oracle_mod.interp(a, c))) <= 1e-13


def test_T3_prolong_reproduces_3d_polynomial_and_is_kron(oracle_mod):
    Nc, Nf, E = 3, 7, 3
    xc, _, _ = oracle_mod.gll(Nc)
    xf, _, _ = oracle_mod.gll(Nf)
    f = lambda r, s, t: 1.0 + r - 2 * s * t + r ** 3 * s ** 2 - 0.5 * t ** 3 * r * s ** 3        # degree <= 3 per variable
    uc = np.stack([f(xc[None, None, :], xc[None, :, None], xc[:, None, None]) * (e + 1) for e in range(E)])
    uf = oracle_mod.prolong(uc.reshape(E, -1), Nc, Nf).reshape(E, Nf + 1, Nf + 1, Nf + 1)
    for e in range(E):
        assert np.max(np.abs(uf[e] - f(xf[None, None, :], xf[None, :, None], xf[:, None, None]) * (e + 1))) <= 1e-13
    # dense Kronecker product, no shared code: index (k, j, i) with i fastest <-> J (x) J (x) J
    J = oracle_mod.interp(Nc, Nf)
    K = np.kron(J, np.kron(J, J))
    rng = np.random.default_rng(0)
    v = rng.standard_normal((2, (Nc + 1) ** 3))
    assert np.max(np.abs(oracle_mod.prolong(v, Nc, Nf) - v @ K.T)) <= 1e-13
    r = rng.standard_normal((2, (Nf + 1) ** 3))
    assert np.max(np.abs(oracle_mod.restrict(r, Nc, Nf) - r @ K)) <= 1e-13


@pytest.mark.parametrize("Nc,Nf", [(1, 3), (3, 7), (5, 8)])
def test_T4_restriction_is_the_adjoint(oracle_mod, Nc, Nf):
    rng = np.random.default_rng(Nc * 10 + Nf)
    uc = rng.standard_normal((4, (Nc + 1) ** 3))
    rf = rng.standard_normal((4, (Nf + 1) ** 3))
    lhs = np.sum(oracle_mod.prolong(uc, Nc, Nf) * rf)
    rhs = np.sum(uc * oracle_mod.restrict(rf, Nc, Nf))
    assert abs(lhs - rhs) <= 1e-12 * abs(lhs)
    # a transposed operand or swapped index order would break this: restrict(prolong(u)) = (J^T J)^{x3} u
    J = oracle_mod.interp(Nc, Nf)
    M = J.T @ J
    assert np.max(np.abs(oracle_mod.restrict(oracle_mod.prolong(uc, Nc, Nf), Nc, Nf) - uc @ np.kron(M, np.kron(M, M)).T)) <= 1e-12


# ------------------------------------------------------------------------- NEXT-1: Chebyshev-Jacobi smoother
def _dense_masked_operator(oracle_mod, m):
    om = oracle_mod.Maps(m.gid)
    G, _, _ = oracle_mod.geom_trilinear(m.vert, m.N)
    mask_u = oracle_mod.mask_unique(m.dirichlet, om)
    A = np.stack([oracle_mod.apply_Ag(G, m.N, om, mask_u, e) for e in np.eye(om.U)], axis=1)
    return om, G, mask_u, A


def test_C1_chebyshev_error_polynomial(oracle_mod):
    """The smoother's error propagation is the scaled Chebyshev polynomial T_k((theta - t)/delta) / T_k(sigma) of
    M^-1 A (the definition of the method, Saad Alg. 12.1): checked against the dense matrix of a tiny mesh, built from
    numpy's Chebyshev class -- no code shared with the oracle's three-term recurrence."""
    m = inputs.box_mesh(2, 2, 2, 3, "random", seed=5)
    om, G, mask_u, A = _dense_masked_operator(oracle_mod, m)
    free = mask_u == 0
    Af = A[np.ix_(free, free)]
    Dinv = 1.0 / np.diag(Af)
    lam_all = np.linalg.eigvals(Dinv[:, None] * Af).real
    lmax, lmin = 1.1 * lam_all.max(), 0.1 * lam_all.max()
    theta, delta = (lmax + lmin) / 2, (lmax - lmin) / 2
    rng = np.random.default_rng(1)
    xs = np.zeros(om.U); xs[free] = rng.standard_normal(free.sum())
    b = oracle_mod.apply_Ag(G, m.N, om, mask_u, xs)
    x0 = np.zeros(om.U); x0[free] = rng.standard_normal(free.sum())
    B = np.eye(free.sum()) - 0.0                                   # error e_k = p_k(M^-1 A) e_0
    MA = Dinv[:, None] * Af
    for order in (1, 2, 3, 5):
        xk = oracle_mod.cheby(G, m.N, om, mask_u, b, x0, order, lmin, lmax)
        Tk = np.polynomial.chebyshev.Chebyshev.basis(order)
        # evaluate p_k(MA) through the eigen-decomposition of the (similar to symmetric) matrix
        w, V = np.linalg.eig(MA)
        pk = (V * (Tk((theta - w.real) / delta) / Tk(theta / delta))) @ np.linalg.inv(V)
        e_expected = (pk @ (x0 - xs)[free]).real
        assert np.max(np.abs((xk - xs)[free] - e_expected)) <= 1e-10 * np.max(np.abs(e_expected)), order
        assert np.all(xk[~free] == 0.0)
    # order 1 is damped Jacobi with weight 1/theta (closed form)
    x1 = oracle_mod.cheby(G, m.N, om, mask_u, b, x0, 1, lmin, lmax)
    r0 = np.zeros(om.U); r0[free] = Dinv * (b - oracle_mod.apply_Ag(G, m.N, om, mask_u, x0))[free]
    assert np.max(np.abs(x1 - (x0 + r0 / theta))) <= 1e-14


def test_C2_chebyshev_damps_the_upper_spectrum(oracle_mod):
    """On a down-sized smooth mesh with bounds [lmax/10, 1.1 lmax]: in the basis of the generalised eigenvectors
    A v = t M v (A- and M-orthogonal), every error component with t inside the bounds is damped by at least
    1/T_k(sigma) -- the min-max property that makes it a smoother -- and no component below them is amplified."""
    import scipy.linalg
    m = inputs.box_mesh(3, 3, 3, 3, "smooth")
    om, G, mask_u, A = _dense_masked_operator(oracle_mod, m)
    free = mask_u == 0
    Af = A[np.ix_(free, free)]
    Af = 0.5 * (Af + Af.T)
    t, V = scipy.linalg.eigh(Af, np.diag(np.diag(Af)))           # V^T M V = I
    lmax, lmin = 1.1 * t.max(), 0.11 * t.max()
    sigma = (lmax + lmin) / (lmax - lmin)
    rng = np.random.default_rng(3)
    xs = np.zeros(om.U); xs[free] = rng.standard_normal(free.sum())
    b = oracle_mod.apply_Ag(G, m.N, om, mask_u, xs)
    c0 = V.T @ (np.diag(Af) * (0.0 - xs[free]))                  # coefficients of e_0 = x_0 - x* in the basis V
    inside = t >= lmin
    assert inside.sum() > 10 and (~inside).sum() > 3
    for order in (1, 2, 4, 8):
        e = (oracle_mod.cheby(G, m.N, om, mask_u, b, None, order, lmin, lmax) - xs)[free]
        ck = V.T @ (np.diag(Af) * e)
        bound = 1.0 / np.polynomial.chebyshev.Chebyshev.basis(order)(sigma)
        assert np.all(np.abs(ck[inside]) <= bound * np.abs(c0[inside]) * (1 + 1e-9) + 1e-13), order
        assert np.all(np.abs(ck[~inside]) <= np.abs(c0[~inside]) * (1 + 1e-9) + 1e-13), order


# --------------------------------------------------------------------- NEXT-1c: p-multigrid V-cycle
@pytest.fixture(scope="module")
def pmg_levels(oracle_mod):
    return [oracle_mod.Level(inputs.box_mesh(3, 3, 2, N, "smooth")) for N in (5, 3, 1)]


def _dense_of(fn, n):
    return np.stack([fn(e) for e in np.eye(n)], axis=1)


def test_V1_vcycle_is_a_symmetric_contraction(oracle_mod, pmg_levels):
    """With equal pre- and post-smoothing from a zero guess the V-cycle is a fixed symmetric linear operator M^-1
    (every ingredient is linear and restriction is the adjoint of prolongation), M^-1 A has a positive spectrum, and
    the iteration x <- x + M^-1 (b - A x) contracts: rho(I - M^-1 A) < 1, far below the Jacobi smoother's own rate."""
    L0 = pmg_levels[0]
    free = L0.mask_u == 0
    n = L0.maps.U
    Minv = _dense_of(lambda r: oracle_mod.vcycle(pmg_levels, np.where(free, r, 0.0), 2, 8), n)[np.ix_(free, free)]
    A = _dense_of(L0.A, n)[np.ix_(free, free)]
    assert np.max(np.abs(Minv - Minv.T)) <= 1e-10 * np.max(np.abs(Minv))
    ev = np.linalg.eigvals(Minv @ A).real
    assert ev.min() > 0.0
    rho = np.max(np.abs(1.0 - ev))
    assert rho < 0.6
    # the smoother alone (same work on the fine level, no coarse correction) is much worse on the smooth modes
    S = _dense_of(lambda r: L0.smooth(np.where(free, r, 0.0), None, 4), n)[np.ix_(free, free)]
    assert np.max(np.abs(1.0 - np.linalg.eigvals(S @ A).real)) > 0.9


def test_V2_coarse_correction_helps_coarse_space_errors(oracle_mod, pmg_levels):
    """Two levels: for an error that lies in the coarse space (a prolonged coarse function) the cycle -- whose coarse
    problem is solved well (60 Chebyshev steps) -- leaves a much smaller energy-norm error than the same smoothing
    work without the coarse correction.  (It cannot remove it: the re-discretised coarse operator is stiffer than the
    Galerkin one, eig(A_c^-1 P^T A P) in [0.28, 1] on this mesh, so the correction under-shoots.)"""
    L0, L1 = pmg_levels[0], pmg_levels[1]
    rng = np.random.default_rng(2)
    e_c = np.where(L1.mask_u != 0, 0.0, rng.standard_normal(L1.maps.U))
    x_f = np.zeros(L0.maps.U)
    x_f[L0.maps.l2u] = oracle_mod.prolong(e_c[L1.maps.l2u].reshape(-1, (L1.N + 1) ** 3), L1.N, L0.N).ravel()
    x_f[L0.mask_u != 0] = 0.0
    r = L0.A(x_f)
    en = lambda e: float(e @ L0.A(e))
    z_v = oracle_mod.vcycle(pmg_levels[:2], r, 2, 60)
    z_s = L0.smooth(r, None, 4)
    assert en(z_v - x_f) < 0.4 * en(z_s - x_f) and en(z_v - x_f) < en(x_f)


def test_V3_fpcg_with_vcycle_converges_fast_to_the_dense_solution(oracle_mod, pmg_levels):
    """Flexible CG preconditioned by the V-cycle reaches the dense direct solution, in far fewer iterations than
    Jacobi-PCG (the reason the paper uses pMG); with the identity-free Jacobi preconditioner the same
    routine reproduces orc_pcg's iterates (Polak-Ribiere = Fletcher-Reeves when the preconditioner is fixed and SPD)."""
    L0 = pmg_levels[0]
    free = L0.mask_u == 0
    rng = np.random.default_rng(4)
    xs = np.where(free, rng.standard_normal(L0.maps.U), 0.0)
    b = L0.A(xs)
    A = _dense_of(L0.A, L0.maps.U)[np.ix_(free, free)]
    x_dense = np.zeros(L0.maps.U)
    x_dense[free] = np.linalg.solve(A, b[free])
    res = oracle_mod.fpcg(L0, lambda r: oracle_mod.vcycle(pmg_levels, r, 2, 8), b, tol=1e-10, maxit=60)
    assert res["hist"][-1] <= 1e-10 and np.max(np.abs(res["x"] - x_dense)) <= 1e-8 * np.max(np.abs(x_dense))
    jac = oracle_mod.pcg(L0.G, L0.N, L0.maps, L0.mask_u, b, tol=1e-10, maxit=500)
    assert res["iters"] * 3 < jac["iters"]
    fj = oracle_mod.fpcg(L0, lambda r: L0.Minv * r, b, tol=1e-10, maxit=500)
    assert fj["iters"] == jac["iters"]
    assert np.max(np.abs(fj["hist"] - jac["hist"])) <= 1e-6 * 1.0


# ------------------------------------------------------------- NEXT-3: projection onto previous solutions
def test_J1_projection_is_the_A_orthogonal_best_fit(oracle_mod, pmg_levels):
    """The basis stays A-orthonormal, the guess is the A-norm best approximation of the solution in span(P) (checked
    against a dense A-weighted least squares), the reduced right-hand side is b - A xbar, a repeated right-hand side is
    solved by the guess alone, and the space restarts at L_max."""
    L0 = pmg_levels[1]                                     # the N = 3 level: small enough for dense algebra
    free = L0.mask_u == 0
    n = L0.maps.U
    A = _dense_of(L0.A, n)
    rng = np.random.default_rng(5)
    base = np.where(free, rng.standard_normal(n), 0.0)
    drift = np.where(free, rng.standard_normal(n), 0.0)
    wig = np.where(free, rng.standard_normal(n), 0.0)
    proj = oracle_mod.Projection(L0.A, n, Lmax=4)
    res_norms = []
    for m in range(7):
        xs = base + 0.1 * m * drift + 0.01 * np.sin(m) * wig          # a smoothly evolving solution: 3-dimensional span
        b = L0.A(xs)
        xbar, bred = proj.guess(b)
        assert np.max(np.abs(bred - (b - L0.A(xbar)))) <= 1e-10 * np.max(np.abs(b))
        P = proj.P
        if P.shape[0]:
            assert np.max(np.abs(P @ A @ P.T - np.eye(P.shape[0]))) <= 1e-9
            c = np.linalg.solve(P @ A @ P.T, P @ A @ xs)               # A-orthogonal projection of xs on span(P)
            assert np.max(np.abs(xbar - c @ P)) <= 1e-9 * np.max(np.abs(xs))
        res_norms.append(np.linalg.norm(bred) / np.linalg.norm(b))
        proj.update(xs - xbar)                                         # the reduced problem solved exactly
        assert proj.P.shape[0] <= 4
    assert res_norms[0] == 1.0 and res_norms[1] < 0.5 and max(res_norms[3:5]) < 1e-8     # span exhausted after 3
    xbar, bred = proj.guess(b)                                          # the last right-hand side again
    assert np.linalg.norm(bred) <= 1e-8 * np.linalg.norm(b)
    # a direction already in the space is dropped (on a space that is not about to restart)
    p2 = oracle_mod.Projection(L0.A, n, Lmax=30)
    assert p2.update(base) and p2.update(drift)
    assert p2.update(1e-3 * p2.P[0] + 2.0 * p2.P[1]) is False and p2.P.shape[0] == 2


# --------------------------------------- NEXT-2a: fast-diagonalisation local solve of the Schwarz smoother, Eq. (3)
def _spd(rng, m, shift):
    M = rng.standard_normal((m, m))
    return M @ M.T + shift * np.eye(m)


def test_F1_fdm_is_the_inverse_of_the_separable_operator(oracle_mod):
    """Eq. (3) with S_d, lam_d from A_d s = lam B_d s (S^T B S = I) is the exact inverse of the dense
    Bz x By x Ax + Bz x Ay x Bx + Az x By x Bx (x fastest), built here with numpy.kron and solved with a dense LU:
    different dense SPD pairs per direction, so a transposed S, a swapped direction or a wrong Lambda index fails."""
    rng = np.random.default_rng(21)
    m, E = 4, 3
    S = np.empty((E, 3, m, m))
    invL = np.empty((E, m, m, m))
    K = []
    for e in range(E):
        A = [_spd(rng, m, 0.5) for _ in range(3)]
        B = [_spd(rng, m, 2.0) for _ in range(3)]
        lam = []
        for d in range(3):
            S[e, d], l = oracle_mod.fdm_eig(A[d], B[d])
            lam.append(l)
            assert np.max(np.abs(S[e, d].T @ B[d] @ S[e, d] - np.eye(m))) <= 1e-12
            assert np.max(np.abs(S[e, d].T @ A[d] @ S[e, d] - np.diag(l))) <= 1e-11
        invL[e] = oracle_mod.fdm_inv_lambda(*lam)
        K.append(np.kron(B[2], np.kron(B[1], A[0])) + np.kron(B[2], np.kron(A[1], B[0]))
                 + np.kron(A[2], np.kron(B[1], B[0])))
    b = rng.standard_normal((E, m, m, m))
    u = oracle_mod.fdm_apply(S, invL, b)
    for e in range(E):
        ref = np.linalg.solve(K[e], b[e].ravel())
        assert np.max(np.abs(u[e].ravel() - ref)) <= 1e-10 * np.max(np.abs(ref))


def test_F2_fdm_solves_the_7_point_laplacian_with_the_closed_form_spectrum(oracle_mod):
    """Textbook special case: A_d = tridiag(-1, 2, -1), B_d = I on m_x x m_y x m_z interior points.  The eigenvalues are
    2 - 2 cos(q pi / (m+1)) (closed form) and Eq. (3) solves the 7-point finite-difference Poisson problem, checked by
    applying the stencil to the result with plain array shifts.  Unequal sizes are emulated by padding to a cube with
    decoupled identity rows, which also pins that the three directions are not interchanged."""
    m = 6
    T = 2.0 * np.eye(m) - np.eye(m, k=1) - np.eye(m, k=-1)
    Sx, lx = oracle_mod.fdm_eig(T, np.eye(m))
    assert np.max(np.abs(lx - (2.0 - 2.0 * np.cos(np.arange(1, m + 1) * np.pi / (m + 1))))) <= 1e-13
    # anisotropic: x uses T, y uses 4 T, z uses 9 T (grid spacings 1, 1/2, 1/3)
    Sy, ly = oracle_mod.fdm_eig(4.0 * T, np.eye(m))
    Sz, lz = oracle_mod.fdm_eig(9.0 * T, np.eye(m))
    S = np.stack([Sx, Sy, Sz])[None]
    invL = oracle_mod.fdm_inv_lambda(lx, ly, lz)[None]
    rng = np.random.default_rng(22)
    b = rng.standard_normal((1, m, m, m))
    u = oracle_mod.fdm_apply(S, invL, b)[0]
    up = np.pad(u, 1)                                                        # homogeneous Dirichlet halo
    c = up[1:-1, 1:-1, 1:-1]
    lap = (1.0 * (2 * c - up[1:-1, 1:-1, :-2] - up[1:-1, 1:-1, 2:])          # i = x, fastest
           + 4.0 * (2 * c - up[1:-1, :-2, 1:-1] - up[1:-1, 2:, 1:-1])        # j = y
           + 9.0 * (2 * c - up[:-2, 1:-1, 1:-1] - up[2:, 1:-1, 1:-1]))       # k = z
    assert np.max(np.abs(lap - b[0])) <= 1e-11 * np.max(np.abs(b))


def test_F3_fdm_is_symmetric_positive_definite_on_the_synthetic_pairs(oracle_mod):
    """On the seeded operator pairs of inputs.fdm_pairs (the parity and bench inputs): c.F(b) = b.F(c), b.F(b) > 0,
    and F inverts the dense separable operator (m = 5, E = 4)."""
    m, E = 5, 4
    A, B = inputs.fdm_pairs(E, m, seed=6)
    assert np.all(A == np.transpose(A, (0, 1, 3, 2))) and np.all(np.linalg.eigvalsh(A) > 0) and np.all(np.linalg.eigvalsh(B) > 0)
    S = np.empty_like(A)
    invL = np.empty((E, m, m, m))
    for e in range(E):
        lam = []
        for d in range(3):
            S[e, d], l = oracle_mod.fdm_eig(A[e, d], B[e, d])
            lam.append(l)
        invL[e] = oracle_mod.fdm_inv_lambda(*lam)
    rng = np.random.default_rng(23)
    b, c = rng.standard_normal((2, E, m, m, m))
    Fb, Fc = oracle_mod.fdm_apply(S, invL, b), oracle_mod.fdm_apply(S, invL, c)
    for e in range(E):
        assert abs(np.vdot(c[e], Fb[e]) - np.vdot(b[e], Fc[e])) <= 1e-12 * abs(np.vdot(c[e], Fb[e])) + 1e-14
        assert np.vdot(b[e], Fb[e]) > 0
        K = (np.kron(B[e, 2], np.kron(B[e, 1], A[e, 0])) + np.kron(B[e, 2], np.kron(A[e, 1], B[e, 0]))
             + np.kron(A[e, 2], np.kron(B[e, 1], B[e, 0])))
        assert np.max(np.abs(K @ Fb[e].ravel() - b[e].ravel())) <= 1e-10 * np.max(np.abs(b[e]))


# ---------------------------------------- NEXT-2b: overlapping additive Schwarz smoother (reading S29)
def _rectilinear(nx, ny, nz, N, stretch):
    """An affine box mesh whose grid lines are moved by x -> x^stretch per coordinate: elements stay rectangular
    boxes but neighbouring elements have different lengths."""
    m = inputs.box_mesh(nx, ny, nz, N, "affine")
    m.vert = m.vert ** np.asarray(stretch)[None, None, :]
    return m


def _window_ids(mesh, ex, ey, ez):
    """Unique-grid (positional gid) ids of the (N+3)^3 tensor window around element (ex, ey, ez): -1 outside the mesh."""
    N = mesh.N
    NX, NY, NZ = mesh.nx * N + 1, mesh.ny * N + 1, mesh.nz * N + 1
    ids = -np.ones((N + 3, N + 3, N + 3), dtype=np.int64)
    for c in range(N + 3):
        for b in range(N + 3):
            for a in range(N + 3):
                x, y, z = ex * N - 1 + a, ey * N - 1 + b, ez * N - 1 + c
                if 0 <= x < NX and 0 <= y < NY and 0 <= z < NZ:
                    ids[c, b, a] = x + NX * (y + NY * z)
    return ids


@pytest.mark.parametrize("stretch", [(1.0, 1.0, 1.0), (1.6, 0.7, 1.3)])
def test_W1_local_operator_is_the_assembled_operator_on_the_window(oracle_mod, stretch):
    """On a rectilinear mesh the assembled operator is a sum of Kronecker products of the 1-D assembled matrices, so its
    restriction to the tensor window of (N+3)^3 nodes around an element IS Bz x By x Ax + ... with the 1-D matrices
    restricted to the window: the separable local operator of the Schwarz block (reading S29: three assembled 1-D segments,
    retained rows and columns) must equal rows/columns of the dense assembled operator, which is pinned by P9 and shares
    no code with it.  A wrong neighbour length, a wrong corner block of the neighbour's 1-D matrix, a swapped Kronecker
    order or a transposed direction fails.  Interior element (all 6 neighbours) and, with the Dirichlet mask, a corner
    element (3 boundary faces: decoupled ghost and face rows)."""
    N = 3
    m = _rectilinear(3, 3, 3, N, stretch)
    for masked, (ex, ey, ez) in ((False, (1, 1, 1)), (True, (0, 2, 0)), (False, (2, 0, 1))):
        maps = oracle_mod.Maps(m.gid)
        mask_u = oracle_mod.mask_unique(m.dirichlet, maps) if masked else np.zeros(maps.U, np.uint8)
        sw = oracle_mod.Schwarz(m, maps, mask_u)
        G, _, rc = oracle_mod.geom_trilinear(m.vert, N)
        assert rc == 0
        Ad = np.stack([oracle_mod.apply_Ag(G, N, maps, mask_u, e) for e in np.eye(maps.U)], axis=1)
        e = ex + 3 * (ey + 3 * ez)
        (Ax, Ay, Az), (Bx, By, Bz) = sw.A1[e], sw.B1[e]
        K = np.kron(Bz, np.kron(By, Ax)) + np.kron(Bz, np.kron(Ay, Bx)) + np.kron(Az, np.kron(By, Bx))
        ids = _window_ids(m, ex, ey, ez).ravel()
        live = ids >= 0
        u_of = np.searchsorted(maps.uniq_gid, np.maximum(ids, 0))
        live &= mask_u[u_of] == 0                               # Dirichlet nodes are decoupled unit rows in the block
        Aw = Ad[np.ix_(u_of[live], u_of[live])]
        assert np.max(np.abs(K[np.ix_(live, live)] - Aw)) <= 1e-13 * np.max(np.abs(Aw)), (stretch, masked)
        dead = ~live                                            # positions without a node: decoupled from the live ones
        assert not dead.any() or np.max(np.abs(K[np.ix_(live, dead)])) == 0.0
        # the block's node map: every filled position points at the window's node; face layers only
        R = sw.R[e].ravel()
        assert np.array_equal(R[R >= 0], u_of[R >= 0])
        nfaces = int((sw.nbr[e] >= 0).sum())
        assert int((R >= 0).sum()) == (N + 1) ** 3 + nfaces * (N + 1) ** 2


def test_W2_schwarz_is_symmetric_positive_and_better_conditioned_than_jacobi(oracle_mod):
    """sum_e R_e^T A~_e^-1 R_e is symmetric positive definite on the free nodes (every A~_e^-1 is, and the blocks cover
    every node) and so is S = W^1/2 M W^1/2; S A has a real positive spectrum, and on a deformed mesh its condition number is far below that
    of diag^-1 A (why the paper uses it as the pMG smoother).  The weights are 1 / (positions per node):
    their reciprocals add up to the number of filled block positions, p^3 + (#face neighbours) p^2 per element."""
    m = inputs.box_mesh(3, 3, 2, 4, "smooth", amp=0.03)
    L = oracle_mod.Level(m)
    sw = oracle_mod.Schwarz(m, L.maps, L.mask_u)
    free = L.mask_u == 0
    n = L.maps.U
    p = m.N + 1

    def unweighted(r):
        u = oracle_mod.fdm_apply(sw.S, sw.invL, sw.extended_rhs(r))
        z = np.zeros(n)
        np.add.at(z, sw.R[sw.back], u[sw.back])
        return z
    M = _dense_of(unweighted, n)[np.ix_(free, free)]
    assert np.max(np.abs(M - M.T)) <= 1e-12 * np.max(np.abs(M))
    assert np.linalg.eigvalsh(0.5 * (M + M.T)).min() > 0.0
    A = _dense_of(L.A, n)[np.ix_(free, free)]
    S = _dense_of(lambda r: sw.apply(np.where(free, r, 0.0)), n)[np.ix_(free, free)]
    assert np.max(np.abs(S - S.T)) <= 1e-12 * np.max(np.abs(S))
    Wh = np.sqrt(sw.W[free])
    assert np.max(np.abs(S - Wh[:, None] * M * Wh[None, :])) <= 1e-12 * np.max(np.abs(S))
    Lc = np.linalg.cholesky(A)
    ev = np.linalg.eigvalsh(Lc.T @ S @ Lc)                    # = spectrum of S A (similar), real because S, A are SPD
    assert ev.min() > 0.0
    evj = np.linalg.eigvals(np.diag(L.Minv[free]) @ A).real
    assert ev.max() / ev.min() < 0.5 * evj.max() / evj.min()
    assert round(float(np.sum(1.0 / sw.W))) == sum(p ** 3 + int((sw.nbr[e] >= 0).sum()) * p * p for e in range(m.E))
    # masked nodes come out zero; RAS: own nodes only, weights 1 / multiplicity
    z = sw.apply(np.where(free, np.cos(np.arange(n)), 0.0))
    assert np.all(z[~free] == 0.0)
    ras = oracle_mod.Schwarz(m, L.maps, L.mask_u, restricted=True)
    assert np.max(np.abs(ras.W * L.maps.mult - 1.0)) == 0.0


def test_W3_one_affine_element_is_solved_exactly(oracle_mod):
    """One affine element with homogeneous Dirichlet faces: no neighbour, the block is the element, the separable operator
    is the element's own (P7), so S is the exact inverse on the interior nodes: S A x = x.  (A wrong boundary row, weight
    or eigen-index order fails.)  Also with a different length per direction."""
    for scale in ((1.0, 1.0, 1.0), (0.5, 2.0, 1.25)):
        m = inputs.box_mesh(1, 1, 1, 5, "affine")
        m.vert = m.vert * np.asarray(scale)[None, None, :]
        L = oracle_mod.Level(m, power_its=2)
        sw = oracle_mod.Schwarz(m, L.maps, L.mask_u)
        free = L.mask_u == 0
        x = np.where(free, np.sin(1.0 + np.arange(L.maps.U) ** 2), 0.0)
        assert np.max(np.abs(sw.apply(L.A(x)) - x)) <= 1e-11 * np.max(np.abs(x)), scale


def test_W4_chebyshev_with_a_general_preconditioner_reduces_to_chebyshev_jacobi(oracle_mod, pmg_levels):
    """cheby_pc (numpy, any preconditioner) with P = diag^-1 reproduces the C++ oracle's Chebyshev-Jacobi smoother, which
    C1 pins against the exact error polynomial."""
    L0 = pmg_levels[0]
    b = L0.A(np.where(L0.mask_u != 0, 0.0, np.cos(np.arange(L0.maps.U) * 0.37)))
    x0 = np.where(L0.mask_u != 0, 0.0, np.sin(np.arange(L0.maps.U) * 0.11))
    for order, guess in ((1, None), (3, None), (4, x0)):
        ref = L0.smooth(b, guess, order)
        got = oracle_mod.cheby_pc(L0.A, lambda r: L0.Minv * r, b, guess, order, L0.lmin, L0.lmax)
        assert np.max(np.abs(got - ref)) <= 1e-12 * np.max(np.abs(ref)), order


def test_W5_schwarz_smoothing_beats_jacobi_smoothing_in_the_vcycle(oracle_mod):
    """The same V-cycle and flexible PCG with Chebyshev-Schwarz smoothing on the levels that can carry it needs fewer
    iterations than with Chebyshev-Jacobi smoothing ("we switched from Chebyshev-Jacobi to Chebyshev-Schwarz") and
    reaches the same (dense direct) solution."""
    meshes = [inputs.box_mesh(3, 3, 2, N, "smooth") for N in (5, 3, 1)]
    lj = [oracle_mod.Level(m) for m in meshes]
    ls = [oracle_mod.Level(m) for m in meshes]
    for L, m in zip(ls[:-1], meshes[:-1]):
        L.use_schwarz(m)
    L0 = lj[0]
    free = L0.mask_u == 0
    rng = np.random.default_rng(4)
    xs = np.where(free, rng.standard_normal(L0.maps.U), 0.0)
    b = L0.A(xs)
    rj = oracle_mod.fpcg(lj[0], lambda r: oracle_mod.vcycle(lj, r, 2, 8), b, tol=1e-10, maxit=60)
    rs = oracle_mod.fpcg(ls[0], lambda r: oracle_mod.vcycle(ls, r, 2, 8), b, tol=1e-10, maxit=60)
    assert rs["hist"][-1] <= 1e-10 and rs["iters"] < rj["iters"]
    assert np.max(np.abs(rs["x"] - xs)) <= 1e-8 * np.max(np.abs(xs))


def test_W6_results_do_not_depend_on_the_elements_local_orientation(oracle_mod):
    """Rotating every element's local (r, s, t) frame by a seeded proper rotation of the cube (inputs.reorient: the same
    nodes and global ids, neighbours now meet with arbitrary relative orientation, as in an unstructured mesh) changes
    every local array but no unique-node result: the assembled operator, the Jacobi diagonal, the PCG iterates and both
    Schwarz variants.  A face link that assumes aligned neighbours, a wrong factor order or a transposed D fails."""
    m0 = inputs.box_mesh(3, 3, 2, 4, "random", seed=5)
    m1 = inputs.reorient(m0, 7)
    assert not np.array_equal(m0.gid, m1.gid)
    o0, o1 = oracle_mod.Maps(m0.gid), oracle_mod.Maps(m1.gid)
    assert np.array_equal(o0.uniq_gid, o1.uniq_gid) and np.array_equal(o0.mult, o1.mult)
    G0, dJ0, rc0 = oracle_mod.geom_trilinear(m0.vert, m0.N)
    G1, dJ1, rc1 = oracle_mod.geom_trilinear(m1.vert, m1.N)
    assert rc0 == 0 and rc1 == 0 and dJ1.min() > 0.0
    k0, k1 = oracle_mod.mask_unique(m0.dirichlet, o0), oracle_mod.mask_unique(m1.dirichlet, o1)
    assert np.array_equal(k0, k1)
    x = np.where(k0 != 0, 0.0, inputs.field_normal(o0.uniq_gid, 3))
    y0, y1 = oracle_mod.apply_Ag(G0, m0.N, o0, k0, x, 2.0), oracle_mod.apply_Ag(G1, m1.N, o1, k1, x, 2.0)
    assert np.max(np.abs(y0 - y1)) <= 1e-13 * np.max(np.abs(y0))
    d0, d1 = np.zeros(o0.U), np.zeros(o1.U)
    np.add.at(d0, o0.l2u, oracle_mod.diag_local(G0, m0.N).ravel())
    np.add.at(d1, o1.l2u, oracle_mod.diag_local(G1, m1.N).ravel())
    assert np.max(np.abs(d0 - d1)) <= 1e-13 * np.max(np.abs(d0))
    r0 = oracle_mod.pcg(G0, m0.N, o0, k0, y0, tol=1e-10, maxit=300, lam=2.0)
    r1 = oracle_mod.pcg(G1, m1.N, o1, k1, y1, tol=1e-10, maxit=300, lam=2.0)
    assert r0["iters"] == r1["iters"] and np.max(np.abs(r0["x"] - r1["x"])) <= 1e-9 * np.max(np.abs(r0["x"]))
    for restricted in (False, True):
        s0 = oracle_mod.Schwarz(m0, o0, k0, restricted)
        s1 = oracle_mod.Schwarz(m1, o1, k1, restricted)
        z0, z1 = s0.apply(x), s1.apply(x)
        assert np.max(np.abs(z0 - z1)) <= 1e-12 * np.max(np.abs(z0)), restricted
