"""ORACLE — TEST INFRASTRUCTURE ONLY (see oracle/sem_oracle.cpp header).

ctypes/numpy wrapper around the plain CPU C++ oracle of the spectral-element Poisson/Helmholtz hot path of
arXiv 2110.01716.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  It imports nothing from paper_2110_01716_b200 and shares no code with the CUDA path.

Array conventions: p = N+1, local node l = ((e*p + k)*p + j)*p + i (i fastest), vertex v = a+2b+4c,
G[E][7][p^3] = (rr, rs, rt, ss, st, tt, B).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "sem_oracle.cpp")
_SO = os.path.join(_HERE, "liboracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with g++ -O3 -fopenmp (no other tuning).  Returns the .so path."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        cmd = ["g++", "-O3", "-std=c++17", "-fopenmp", "-fPIC", "-shared", "-ffp-contract=off", _SRC, "-o", _SO]
        subprocess.run(cmd, check=True)
    return _SO


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.orc_count_unique.restype = C.c_int64
    return _lib


def _p(a):
    return a.ctypes.data_as(C.c_void_p) if a is not None else None


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def num_threads() -> int:
    return int(lib().orc_num_threads())


def gll(N: int):
    """O1: (xi[p], rho[p], D[p,p]) — D[i,l] = dh_l/dr at xi_i."""
    p = N + 1
    xi, rho, D = np.empty(p), np.empty(p), np.empty((p, p))
    rc = lib().orc_gll(C.c_int(N), _p(xi), _p(rho), _p(D))
    if rc:
        raise ValueError(f"orc_gll rc={rc}")
    return xi, rho, D


def node_xyz(vert: np.ndarray, N: int) -> np.ndarray:
    """O2: trilinear images of the GLL points.  vert[E,8,3] -> xyz[E,p^3,3]."""
    vert = _f64(vert)
    E = vert.shape[0]
    out = np.empty((E, (N + 1) ** 3, 3))
    rc = lib().orc_node_xyz(C.c_int64(E), C.c_int(N), _p(vert), _p(out))
    assert rc == 0
    return out


def geom_iso(xyz: np.ndarray, N: int):
    """O3 (isoparametric): xyz[E,p^3,3] -> (G[E,7,p^3], detJ[E,p^3], rc) ; rc=-2 if some detJ <= 0."""
    xyz = _f64(xyz)
    E = xyz.shape[0]
    p3 = (N + 1) ** 3
    G, dJ = np.empty((E, 7, p3)), np.empty((E, p3))
    rc = lib().orc_geom_iso(C.c_int64(E), C.c_int(N), _p(xyz), _p(G), _p(dJ))
    return G, dJ, rc


def geom_trilinear(vert: np.ndarray, N: int):
    """O3 (trilinear-analytic): vert[E,8,3] -> (G[E,7,p^3], detJ[E,p^3], rc)."""
    vert = _f64(vert)
    E = vert.shape[0]
    p3 = (N + 1) ** 3
    G, dJ = np.empty((E, 7, p3)), np.empty((E, p3))
    rc = lib().orc_geom_trilinear(C.c_int64(E), C.c_int(N), _p(vert), _p(G), _p(dJ))
    return G, dJ, rc


def ax(G: np.ndarray, u: np.ndarray, N: int, lam: float = 0.0) -> np.ndarray:
    """O4: local w = D^T G D u (+ lam B u); no gather-scatter."""
    G, u = _f64(G), _f64(u)
    E = G.shape[0]
    w = np.empty_like(u)
    rc = lib().orc_ax(C.c_int64(E), C.c_int(N), _p(G), _p(u), _p(w), C.c_double(lam))
    assert rc == 0
    return w


class Maps:
    """O6 canonical maps."""

    def __init__(self, gid: np.ndarray):
        gid = np.ascontiguousarray(gid, dtype=np.int64).ravel()
        nL = gid.size
        U = int(lib().orc_count_unique(C.c_int64(nL), _p(gid)))
        self.nL, self.U = nL, U
        self.uniq_gid = np.empty(U, np.int64)
        self.l2u = np.empty(nL, np.int32)
        self.mult = np.empty(U, np.int32)
        self.seg_off = np.empty(U + 1, np.int64)
        self.seg_idx = np.empty(nL, np.int32)
        rc = lib().orc_maps(C.c_int64(nL), _p(gid), C.c_int64(U), _p(self.uniq_gid), _p(self.l2u), _p(self.mult),
                            _p(self.seg_off), _p(self.seg_idx))
        if rc:
            raise ValueError("orc_maps: negative gid or inconsistent U")
        self.S = int(self.mult[self.mult > 1].sum())
        self.Us = int((self.mult > 1).sum())


def gs(w: np.ndarray, maps: Maps) -> np.ndarray:
    """O5: QQ^T, op=add.  Returns a new array."""
    out = _f64(w).copy()
    rc = lib().orc_gs(C.c_int64(maps.nL), C.c_int64(maps.U), _p(maps.l2u), _p(out))
    assert rc == 0
    return out


def diag_local(G: np.ndarray, N: int, lam: float = 0.0) -> np.ndarray:
    """O7: exact diagonal of the local operator, [E,p^3] (assemble with gs())."""
    G = _f64(G)
    E = G.shape[0]
    d = np.empty((E, (N + 1) ** 3))
    rc = lib().orc_diag_local(C.c_int64(E), C.c_int(N), _p(G), _p(d), C.c_double(lam))
    assert rc == 0
    return d


def mask_unique(dirichlet_local, maps: Maps) -> np.ndarray:
    """S14: a unique node is masked if any of its local copies is flagged."""
    m = np.zeros(maps.U, np.uint8)
    if dirichlet_local is not None:
        np.maximum.at(m, maps.l2u, np.ascontiguousarray(dirichlet_local, np.uint8).ravel())
    return m


def apply_Ag(G, N, maps: Maps, mask_u, x_u, lam: float = 0.0) -> np.ndarray:
    """O8: y = M Q^T A_L Q M x in unique storage."""
    G, x_u = _f64(G), _f64(x_u)
    y = np.empty(maps.U)
    mask_u = np.ascontiguousarray(mask_u, np.uint8)
    lib().orc_apply_Ag(C.c_int64(G.shape[0]), C.c_int(N), _p(G), C.c_double(lam), C.c_int64(maps.nL),
                       C.c_int64(maps.U), _p(maps.l2u), _p(mask_u), _p(x_u), _p(y))
    return y


def pcg(G, N, maps: Maps, mask_u, b_u, x0_u=None, tol=1e-8, maxit=100, lam=0.0, snap_its=()):
    """O8 Jacobi-PCG in unique storage.  Returns dict(x, iters, relres, hist, snaps{it: x})."""
    G, b_u = _f64(G), _f64(b_u)
    x = np.zeros(maps.U) if x0_u is None else _f64(x0_u).copy()
    mask_u = np.ascontiguousarray(mask_u, np.uint8)
    hist = np.full(maxit + 1, np.nan)
    relres = C.c_double(0.0)
    snap_its = np.ascontiguousarray(sorted(int(s) for s in snap_its), dtype=np.int32)
    ns = snap_its.size
    xs = np.empty((max(ns, 1), maps.U))
    it = lib().orc_pcg(C.c_int64(G.shape[0]), C.c_int(N), _p(G), C.c_double(lam), C.c_int64(maps.nL), C.c_int64(maps.U),
                       _p(maps.l2u), _p(mask_u), _p(b_u), _p(x), C.c_double(tol), C.c_int(maxit), C.byref(relres),
                       _p(hist), C.c_int(ns), _p(snap_its), _p(xs))
    return dict(x=x, iters=int(it), relres=float(relres.value), hist=hist[: it + 1],
                snaps={int(s): xs[n] for n, s in enumerate(snap_its) if s <= it})


# ---- NEXT-1: p-multigrid transfer operators --------------------------------------------------------------
def interp(Nc: int, Nf: int) -> np.ndarray:
    """J[i, j] = coarse (order Nc) Lagrange cardinal function j at fine (order Nf) GLL point i."""
    J = np.empty((Nf + 1, Nc + 1))
    assert lib().orc_interp(C.c_int(Nc), C.c_int(Nf), _p(J)) == 0
    return J


def prolong(uc: np.ndarray, Nc: int, Nf: int) -> np.ndarray:
    """u_f = (J x J x J) u_c per element; uc [E, (Nc+1)^3] -> [E, (Nf+1)^3]."""
    uc = _f64(uc).reshape(-1, (Nc + 1) ** 3)
    uf = np.empty((uc.shape[0], (Nf + 1) ** 3))
    assert lib().orc_prolong(C.c_int64(uc.shape[0]), C.c_int(Nc), C.c_int(Nf), _p(uc), _p(uf)) == 0
    return uf


def restrict(rf: np.ndarray, Nc: int, Nf: int) -> np.ndarray:
    """r_c = (J^T x J^T x J^T) r_f per element; rf [E, (Nf+1)^3] -> [E, (Nc+1)^3]."""
    rf = _f64(rf).reshape(-1, (Nf + 1) ** 3)
    rc = np.empty((rf.shape[0], (Nc + 1) ** 3))
    assert lib().orc_restrict(C.c_int64(rf.shape[0]), C.c_int(Nc), C.c_int(Nf), _p(rf), _p(rc)) == 0
    return rc


def cheby(G, N, maps: Maps, mask_u, b_u, x0_u, order: int, lmin: float, lmax: float, lam=0.0) -> np.ndarray:
    """Chebyshev-accelerated point-Jacobi smoother (reading S23), `order` steps, unique storage; returns x."""
    G, b_u = _f64(G), _f64(b_u)
    x = np.zeros(maps.U) if x0_u is None else _f64(x0_u).copy()
    mask_u = np.ascontiguousarray(mask_u, np.uint8)
    rc = lib().orc_cheby(C.c_int64(G.shape[0]), C.c_int(N), _p(G), C.c_double(lam), C.c_int64(maps.nL), C.c_int64(maps.U),
                         _p(maps.l2u), _p(mask_u), _p(b_u), _p(x), C.c_int(order), C.c_double(lmin), C.c_double(lmax))
    assert rc == 0
    return x


def cheby_pc(A, P, b_u, x0_u, order: int, lmin: float, lmax: float) -> np.ndarray:
    """The Chebyshev semi-iteration of S23 (Saad, Alg. 12.1) with a general preconditioner application P in place of
    diag^-1 (NEXT-2b: P = the Schwarz operator), written out in numpy:
        theta = (lmax+lmin)/2, delta = (lmax-lmin)/2, sigma = theta/delta, rho_0 = 1/sigma
        r = P(b - A x);  d = r/theta
        k = 1 .. order-1:  x += d;  r -= P(A d);  rho_k = 1/(2 sigma - rho_{k-1});  d = rho_k rho_{k-1} d + (2 rho_k/delta) r
        x += d"""
    theta, delta = 0.5 * (lmax + lmin), 0.5 * (lmax - lmin)
    sigma = theta / delta
    rho = 1.0 / sigma
    x = np.zeros_like(np.asarray(b_u, dtype=np.float64)) if x0_u is None else np.array(x0_u, dtype=np.float64)
    r = P(b_u - A(x)) if x0_u is not None else P(np.asarray(b_u, dtype=np.float64))
    d = r / theta
    for _ in range(1, order):
        x = x + d
        r = r - P(A(d))
        rho1 = 1.0 / (2.0 * sigma - rho)
        d = rho1 * rho * d + (2.0 * rho1 / delta) * r
        rho = rho1
    return x + d


# ---- NEXT-1c: p-multigrid V-cycle preconditioner -------------------------------------------
class Level:
    """One p-multigrid level: its own discretisation of order N on the same elements (S17)."""

    def __init__(self, mesh, lmin_frac: float = 0.1, lmax_safety: float = 1.1, power_its: int = 60, lam: float = 0.0):
        self.N = mesh.N
        self.lam = lam                                  # Helmholtz shift (S18): H = A + lam B on every level
        self.maps = Maps(mesh.gid)
        self.G, _, rc = geom_trilinear(mesh.vert, mesh.N)
        assert rc == 0
        self.mask_u = mask_unique(mesh.dirichlet, self.maps)
        dg = np.zeros(self.maps.U)
        np.add.at(dg, self.maps.l2u, diag_local(self.G, self.N, lam).ravel())
        self.Minv = np.where(self.mask_u != 0, 0.0, 1.0 / dg)
        # eigenvalue bounds of diag^-1 A for the smoother (S23): power iteration x safety, lmin = fraction of lmax
        # (a rough start vector: an under-estimate of lmax would make the smoother amplify the modes above it)
        v = np.where(self.mask_u != 0, 0.0, np.cos(np.arange(self.maps.U) ** 2 * 1.7))
        lam = 1.0
        for _ in range(power_its):
            w = self.Minv * self.A(v)
            lam = float(np.linalg.norm(w) / np.linalg.norm(v))
            v = w / np.linalg.norm(w)
        self.lmax = lmax_safety * lam
        self.lmin = lmin_frac * self.lmax

    def A(self, x_u):
        return apply_Ag(self.G, self.N, self.maps, self.mask_u, x_u, self.lam)

    def smooth(self, b_u, x0_u, order):
        if getattr(self, "schwarz", None) is not None:
            return cheby_pc(self.A, self.schwarz.apply, b_u, x0_u, order, self.slmin, self.slmax)
        return cheby(self.G, self.N, self.maps, self.mask_u, b_u, x0_u, order, self.lmin, self.lmax, self.lam)

    def use_schwarz(self, mesh, restricted: bool = False, lmin_frac: float = 0.1, lmax_safety: float = 1.1,
                    power_its: int = 60):
        """Switch this level's smoother to Chebyshev-accelerated Schwarz (NEXT-2b): bounds of S A by
        power iteration x safety, lmin a fraction of lmax, as for Chebyshev-Jacobi (S23)."""
        self.schwarz = Schwarz(mesh, self.maps, self.mask_u, restricted)
        v = np.where(self.mask_u != 0, 0.0, np.cos(np.arange(self.maps.U) ** 2 * 1.7))
        lam = 1.0
        for _ in range(power_its):
            w = self.schwarz.apply(self.A(v))
            lam = float(np.linalg.norm(w) / np.linalg.norm(v))
            v = w / np.linalg.norm(w)
        self.slmax = lmax_safety * lam
        self.slmin = lmin_frac * self.slmax
        return self


def vcycle(levels, r_u, smooth_order: int, coarse_order: int, lvl: int = 0):
    """z = M^-1 r, one V-cycle (reading S25 in DESIGN.md; the paper gives the ingredients, not the cycle):
        coarsest level:  z = Chebyshev-Jacobi(A, r, coarse_order steps, zero guess)       (stands in for the AMG solve)
        otherwise:       z   = smooth(A, r, zero guess)
                         res = r - A z
                         r_c = M_c Q_c^T J^T (W res)     W = 1/multiplicity on the local copies (un-assembly)
                         z  += J e_c,  e_c = vcycle(r_c)
                         z   = smooth(A, r, guess z)
    Unique storage on every level; J = element-wise (J x J x J) between the two levels' local layouts."""
    L = levels[lvl]
    if lvl == len(levels) - 1:
        return L.smooth(r_u, None, coarse_order)
    C_ = levels[lvl + 1]
    z = L.smooth(r_u, None, smooth_order)
    res = r_u - L.A(z)
    res[L.mask_u != 0] = 0.0
    res_L = (res / L.maps.mult)[L.maps.l2u]                         # each copy carries 1/mult of the functional
    rc_L = restrict(res_L.reshape(-1, (L.N + 1) ** 3), C_.N, L.N).ravel()
    r_c = np.zeros(C_.maps.U)
    np.add.at(r_c, C_.maps.l2u, rc_L)                               # Q_c^T
    r_c[C_.mask_u != 0] = 0.0
    e_c = vcycle(levels, r_c, smooth_order, coarse_order, lvl + 1)
    e_L = prolong(e_c[C_.maps.l2u].reshape(-1, (C_.N + 1) ** 3), C_.N, L.N).ravel()
    e_u = np.zeros(L.maps.U)
    e_u[L.maps.l2u] = e_L                                           # continuous: every copy holds the same value
    e_u[L.mask_u != 0] = 0.0
    return L.smooth(r_u, z + e_u, smooth_order)


def fpcg(level: "Level", precond, b_u, tol=1e-8, maxit=100):
    """Flexible preconditioned CG (the preconditioner may change from iteration to iteration or be inexact, e.g. an FP32
    V-cycle; reading S26): the PCG recurrence of O8 with the Polak-Ribiere beta
        beta = r_new . (z_new - z_old) / (r_old . z_old).
    x0 = 0; returns dict(x, iters, hist) with hist[k] = ||r_k|| / ||r_0||."""
    A = level.A
    x = np.zeros_like(b_u)
    r = np.where(level.mask_u != 0, 0.0, b_u)
    r0 = float(np.linalg.norm(r))
    hist = [1.0 if r0 > 0 else 0.0]
    if r0 == 0.0:
        return dict(x=x, iters=0, hist=np.array(hist))
    z = precond(r)
    p = z.copy()
    rz = float(r @ z)
    it = 0
    while it < maxit:
        q = A(p)
        pq = float(p @ q)
        if not pq > 0.0:
            break
        alpha = rz / pq
        x += alpha * p
        r = r - alpha * q
        it += 1
        hist.append(float(np.linalg.norm(r)) / r0)
        if hist[-1] <= tol:
            break
        z_new = precond(r)
        beta = float(r @ (z_new - z)) / rz
        rz = float(r @ z_new)
        z = z_new
        p = z + beta * p
    return dict(x=x, iters=it, hist=np.array(hist))


# ---- NEXT-3: projection onto previous solutions ----------------------------------------------------------
class Projection:
    """P:111 "For any n x L subspace of R^n with A-orthonormal basis P_L = [p_1 ... p_L], the best-fit approximation to
    the solution of A p^m = b^m is pbar = P_L P_L^T b^m ... The residual for the reduced problem A dp = b^m - A pbar has
    a significantly smaller norm ... We augment the space P_{L+1} = [P_L dp] after orthonormalizing dp against P_L with
    one round of classical Gram-Schmidt ... L_max = 30 before restarting".  Unique storage, plain Euclidean dots.
    Reading S27: A p_i is stored beside p_i, so the reduced right-hand side is b - sum alpha_i (A p_i); the
    norm of the orthogonalised dp comes from the same reduction (dp^T A dp - sum beta_i^2); a restart empties the space
    and the new direction becomes its first vector; a direction whose orthogonalised A-norm^2 is <= 1e-12 of its
    A-norm^2 is dropped (after one round of classical Gram-Schmidt that remainder is rounding noise)."""

    def __init__(self, A, n: int, Lmax: int = 30):
        self.A, self.n, self.Lmax = A, n, Lmax
        self.P = np.zeros((0, n))
        self.AP = np.zeros((0, n))

    def guess(self, b):
        alpha = self.P @ b
        return alpha @ self.P, b - alpha @ self.AP

    def update(self, dx):
        w = self.A(dx)
        if self.P.shape[0] >= self.Lmax:
            self.P, self.AP = np.zeros((0, self.n)), np.zeros((0, self.n))
        beta = self.P @ w                                  # p_i^T A dx
        gamma = float(dx @ w)
        nrm2 = gamma - float(beta @ beta)
        if not (gamma > 0.0) or nrm2 <= 1e-12 * gamma:
            return False
        s = 1.0 / np.sqrt(nrm2)
        self.P = np.vstack([self.P, (dx - beta @ self.P) * s])
        self.AP = np.vstack([self.AP, (w - beta @ self.AP) * s])
        return True


# ---- NEXT-2a: fast-diagonalisation local solve of the Schwarz smoother, Eq. (3) -------------------------
def fdm_eig(A: np.ndarray, B: np.ndarray):
    """One direction of one element: the generalised symmetric eigenproblem A s = lambda B s of the 1-D operator pair
    (stiffness A, mass B; both m x m, symmetric, B positive definite), normalised S^T B S = I so that S^T A S = diag(lam)
    (fast diagonalisation, Deville et al. 2002 as cited at P:103).  Library routine as a step: scipy.linalg.eigh.
    Returns (S[m, m] with eigenvectors in columns, lam[m] ascending)."""
    import scipy.linalg
    lam, S = scipy.linalg.eigh(np.asarray(A, dtype=np.float64), np.asarray(B, dtype=np.float64))
    return S, lam


def fdm_inv_lambda(lam_x, lam_y, lam_z) -> np.ndarray:
    """Lambda^-1 of Eq. (3) as an [m][m][m] array indexed [c][b][a] (z, y, x eigen-index; x fastest): the separable
    operator Bz x By x Ax + Bz x Ay x Bx + Az x By x Bx is diagonalised by Sz x Sy x Sx to lam_x[a] + lam_y[b] + lam_z[c]
    ("Lambda is a diagonal matrix with only 1,000 nonzeros" at m = 10)."""
    lx, ly, lz = (np.asarray(v, dtype=np.float64) for v in (lam_x, lam_y, lam_z))
    return 1.0 / (lz[:, None, None] + ly[None, :, None] + lx[None, None, :])


def fdm_apply(S: np.ndarray, inv_lambda: np.ndarray, b: np.ndarray) -> np.ndarray:
    """Eq. (3), for every element e:  u^e = (S_z x S_y x S_x) Lambda^-1 (S_z^T x S_y^T x S_x^T) b^e.
    S[E][3][m][m] (direction x, y, z; S_d[row][col], eigenvectors in columns), inv_lambda[E][m][m][m], b[E][m][m][m]
    stored [k][j][i] with i (x) fastest, like every local field.  FP64; the three 1-D contractions are written out one
    by one in the order of the formula (transposes first, then the diagonal, then the forward matrices)."""
    S = np.asarray(S, dtype=np.float64)
    b = np.asarray(b, dtype=np.float64)
    u = np.empty_like(b)
    for e in range(b.shape[0]):
        Sx, Sy, Sz = S[e, 0], S[e, 1], S[e, 2]
        t = np.einsum("ia,kji->kja", Sx, b[e])           # S_x^T along i
        t = np.einsum("jb,kja->kba", Sy, t)              # S_y^T along j
        t = np.einsum("kc,kba->cba", Sz, t)              # S_z^T along k
        t = t * inv_lambda[e]
        t = np.einsum("kc,cba->kba", Sz, t)              # S_z
        t = np.einsum("jb,kba->kja", Sy, t)              # S_y
        u[e] = np.einsum("ia,kja->kji", Sx, t)           # S_x
    return u


# ---- NEXT-2b: overlapping additive Schwarz smoother around Eq. (3) (reading S29 in DESIGN.md) ---------------
# P:103 "The Schwarz smoothers are implemented by solving local Poisson problems on domains extended into adjacent elements
# by one layer.  Thus, for an 8 x 8 x 8 brick (N = 7), one solves a 10 x 10 x 10 local problem"; "We exchange
# face data only to get the domain extensions -- meaning 6 exchanges per element instead of 26 ... a restricted additive
# Schwarz (RAS) variant, that does not require communication after the local solve".  The paper cites Lottes & Fischer
# (2005) for the construction and prints none of it; what is written out below is reading S29:
#   * extended block of element e: m = N + 3 points per direction; index 1..N+1 = the element's own nodes, index 0 and
#     m-1 = the face neighbour's node ONE LAYER IN from the shared face; only the 6 face layers are filled ("face data
#     only"), the edge and corner positions of the block hold no node (right-hand side 0, nothing scattered back);
#   * local operator  A~ = Bz x By x Ax + Bz x Ay x Bx + Az x By x Bx  from 1-D stiffness/mass pairs on the extended
#     line [left neighbour | element | right neighbour]: the 1-D spectral-element matrices (2/L) D^T diag(rho) D and
#     (L/2) diag(rho) of the three segments assembled, and the rows/columns of the m retained nodes kept (all other
#     nodes of the neighbours held at zero).  L = mean length of the element's 4 edges in that local direction;
#   * where there is no neighbour the ghost point is decoupled (unit row, zero right-hand side); on a Dirichlet face the
#     face node is decoupled as well;
#   * z = W^1/2 sum_e R_e^T A~_e^-1 R_e (W^1/2 r) with W = 1 / (number of block positions that map to the node), then the
#     Dirichlet mask: the weighting is split over both sides so that S stays symmetric positive definite (S A then has a
#     real positive spectrum, which the Chebyshev acceleration and the CG outer iteration assume); RAS: only the
#     element's own nodes are scattered back, z = W sum_e R^_e^T A~_e^-1 R_e r with W = 1 / multiplicity (not symmetric).
def schwarz_lengths(vert: np.ndarray) -> np.ndarray:
    """L[e][d], d = r, s, t: mean length of the 4 edges of the trilinear element that run in local direction d
    (vertex v = a + 2b + 4c: the edges of direction d join v and v + 2^d for the 4 vertices v whose bit d is 0)."""
    v = _f64(vert).reshape(-1, 8, 3)
    L = np.empty((v.shape[0], 3))
    for d in range(3):
        starts = [q for q in range(8) if not (q >> d) & 1]
        L[:, d] = np.mean([np.linalg.norm(v[:, q + (1 << d)] - v[:, q], axis=1) for q in starts], axis=0)
    return L


def schwarz_ops_1d(N: int, Lm: float, Ll, Lr, dirichlet_l: bool, dirichlet_r: bool):
    """(A, B), each m x m with m = N + 3, of one element's extended line (reading S29).  Lm = the element's length,
    Ll / Lr = the left / right neighbour's length in the direction normal to the shared face (None: no neighbour, then
    dirichlet_l / dirichlet_r says whether that end face is a Dirichlet face)."""
    _, rho, D = gll(N)
    Kh = D.T @ np.diag(rho) @ D                           # reference 1-D stiffness on [-1, 1]
    m = N + 3
    A = np.zeros((m, m))
    B = np.zeros(m)
    A[1:N + 2, 1:N + 2] += (2.0 / Lm) * Kh                # the element itself: block positions 1 .. N+1
    B[1:N + 2] += (Lm / 2.0) * rho
    if Ll is not None:                                    # left neighbour: its last two nodes (one-in, shared face)
        A[0:2, 0:2] += (2.0 / Ll) * Kh[N - 1:N + 1, N - 1:N + 1]
        B[0:2] += (Ll / 2.0) * rho[N - 1:N + 1]
    else:
        A[0, 0], B[0] = 1.0, 1.0                          # no ghost point: decoupled unit row
        if dirichlet_l:
            A[1, :] = 0.0
            A[:, 1] = 0.0
            A[1, 1], B[1] = 1.0, 1.0
    if Lr is not None:                                    # right neighbour: its first two nodes (shared face, one-in)
        A[m - 2:m, m - 2:m] += (2.0 / Lr) * Kh[0:2, 0:2]
        B[m - 2:m] += (Lr / 2.0) * rho[0:2]
    else:
        A[m - 1, m - 1], B[m - 1] = 1.0, 1.0
        if dirichlet_r:
            A[m - 2, :] = 0.0
            A[:, m - 2] = 0.0
            A[m - 2, m - 2], B[m - 2] = 1.0, 1.0
    return A, np.diag(B)


class Schwarz:
    """The additive Schwarz smoother z = S r of one level (unique-node storage), reading S29.
    R[e][c][b][a] = unique node behind position (a, b, c) of element e's extended block, -1 where there is none."""

    def __init__(self, mesh, maps: Maps, mask_u: np.ndarray, restricted: bool = False):
        N, p, E = mesh.N, mesh.N + 1, mesh.vert.shape[0]
        assert N >= 2, "a face needs an interior node to identify the face neighbour"
        m, p3 = N + 3, p ** 3
        self.N, self.m, self.maps, self.mask_u, self.restricted = N, m, maps, np.asarray(mask_u), restricted
        gid = np.ascontiguousarray(mesh.gid, dtype=np.int64).reshape(E, p, p, p)            # [e][k][j][i]
        l2u = maps.l2u.reshape(E, p, p, p)
        L = schwarz_lengths(mesh.vert)
        order = np.argsort(gid.reshape(E, p3), axis=1, kind="stable")                       # per element: gid -> local index
        sorted_gid = np.take_along_axis(gid.reshape(E, p3), order, axis=1)
        R = -np.ones((E, m, m, m), dtype=np.int64)
        R[:, 1:p + 1, 1:p + 1, 1:p + 1] = l2u
        self.nbr = -np.ones((E, 6), dtype=np.int64)
        Lnb = [[None] * 6 for _ in range(E)]
        dirf = np.zeros((E, 6), dtype=bool)
        c0 = p // 2                                                                           # a face-interior node
        for e in range(E):
            for f in range(6):
                axis, side = f // 2, f % 2                                                    # axis 0/1/2 = i/j/k; side 0: index 0, 1: index N
                sl = [slice(None)] * 3                                                        # [k][j][i] slices of my face
                sl[2 - axis] = 0 if side == 0 else N
                fg = gid[e][tuple(sl)]                                                        # [p][p] gids of my face nodes
                ctr = l2u[e][tuple(sl)][c0, c0]
                copies = maps.seg_idx[maps.seg_off[ctr]:maps.seg_off[ctr + 1]] // p3
                others = [int(x) for x in copies if x != e]
                if len(others) != 1:                                                          # domain boundary
                    dirf[e, f] = self.mask_u[ctr] != 0
                    continue
                n = others[0]
                self.nbr[e, f] = n
                pos = np.searchsorted(sorted_gid[n], fg.ravel())
                assert np.array_equal(sorted_gid[n][pos], fg.ravel()), "face nodes not found in the neighbour"
                ln = order[n][pos]                                                            # neighbour's local indices of my face nodes
                ci, cj, ck = ln % p, (ln // p) % p, ln // (p * p)
                coords = [ci, cj, ck]
                naxis = [a for a in range(3) if np.all(coords[a] == coords[a][0]) and coords[a][0] in (0, N)]
                assert len(naxis) == 1
                na = naxis[0]
                coords[na] = np.where(coords[na] == 0, 1, N - 1)                              # one layer in
                one_in = l2u[n].ravel()[coords[0] + p * (coords[1] + p * coords[2])].reshape(fg.shape)
                Lnb[e][f] = L[n, na]
                gl = [slice(1, p + 1)] * 3                                                    # my ghost layer in the block
                gl[2 - axis] = 0 if side == 0 else m - 1
                R[e][tuple(gl)] = one_in
        self.R = R
        # 1-D operator pairs, their eigen-decompositions (Eq. (3)) per element and direction
        self.A1 = np.empty((E, 3, m, m))
        self.B1 = np.empty((E, 3, m, m))
        self.S = np.empty((E, 3, m, m))
        self.invL = np.empty((E, m, m, m))
        for e in range(E):
            lam = []
            for d in range(3):
                self.A1[e, d], self.B1[e, d] = schwarz_ops_1d(N, L[e, d], Lnb[e][2 * d], Lnb[e][2 * d + 1],
                                                              bool(dirf[e, 2 * d]), bool(dirf[e, 2 * d + 1]))
                self.S[e, d], l = fdm_eig(self.A1[e, d], self.B1[e, d])
                lam.append(l)
            tot = lam[2][:, None, None] + lam[1][None, :, None] + lam[0][None, None, :]
            self.invL[e] = np.where(tot > 1e-12 * tot.max(), 1.0 / np.where(tot > 0, tot, 1.0), 0.0)   # all-Neumann block
        own = np.zeros((m, m, m), dtype=bool)
        own[1:p + 1, 1:p + 1, 1:p + 1] = True
        self.back = (R >= 0) & (own[None] if restricted else True)                            # positions scattered back
        cnt = np.zeros(maps.U)
        np.add.at(cnt, R[self.back], 1.0)
        self.W = 1.0 / cnt

    def extended_rhs(self, r_u):
        return np.where(self.R >= 0, np.asarray(r_u)[np.maximum(self.R, 0)], 0.0)

    def apply(self, r_u):
        pre = np.ones(self.maps.U) if self.restricted else np.sqrt(self.W)
        post = self.W if self.restricted else np.sqrt(self.W)
        u = fdm_apply(self.S, self.invL, self.extended_rhs(pre * np.asarray(r_u)))
        z = np.zeros(self.maps.U)
        np.add.at(z, self.R[self.back], u[self.back])
        z *= post
        z[self.mask_u != 0] = 0.0
        return z
