"""Seeded synthetic input generators shared by the oracle-side tests and the CUDA-side tests / bench.

This module holds NONE of the method's arithmetic (no GLL points, no geometric factors, no operator): it only
lays out box meshes of hexahedral elements, moves their vertices, numbers their nodes and draws random fields.
It imports neither `oracle` nor the CUDA binding.  Recipes follow BASELINE.json configs / SURVEY §8(c) S5-S9:

* elements e = ex + nx*(ey + ny*ez) on [0,1]^3; vertex v = a + 2b + 4c of element (ex,ey,ez) is grid vertex
  (ex+a, ey+b, ez+c)                                                              (S4)
* global node ids are positional: gid = (ex*N+i) + NX*((ey*N+j) + NY*(ez*N+k)), NX = nx*N+1, NY = ny*N+1   (S9)
* "smooth" geometry: every component of every vertex moves by amp*sin(2 pi x)sin(2 pi y)sin(2 pi z)        (S6)
* "random" geometry: interior vertices move by U[-frac*h_d, +frac*h_d] per component, boundary fixed       (S7)
* fields are drawn per UNIQUE node by a counter-based 64-bit mixer keyed on (seed, gid), so they are
  continuous across elements and independent of element order                                             (S8)
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np

_M64 = np.uint64(0xFFFFFFFFFFFFFFFF)


def _mix64(x: np.ndarray) -> np.ndarray:
    """splitmix64 finaliser on a uint64 array (wrap-around arithmetic)."""
    with np.errstate(over="ignore"):
        z = x + np.uint64(0x9E3779B97F4A7C15)
        z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
        z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
        return z ^ (z >> np.uint64(31))


def hash_uniform01(seed: int, stream: int, counter: np.ndarray) -> np.ndarray:
    """Uniform in [0,1) from (seed, stream, counter); counter is any integer array."""
    c = np.asarray(counter).astype(np.uint64)
    with np.errstate(over="ignore"):
        key = _mix64(np.uint64(seed) * np.uint64(0xD1342543DE82EF95) + np.uint64(stream) * np.uint64(0xA0761D6478BD642F)
                     + np.uint64(1))
        h = _mix64(_mix64(c ^ key) + key)
    return (h >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


def field_uniform(gid: np.ndarray, seed: int) -> np.ndarray:
    """u ~ U[-1,1] per unique node, scattered to local copies (same shape as gid)."""
    return 2.0 * hash_uniform01(seed, 0, gid) - 1.0


def field_normal(gid: np.ndarray, seed: int) -> np.ndarray:
    """u ~ N(0,1) per unique node (Box-Muller on two hashed uniforms)."""
    u1 = 1.0 - hash_uniform01(seed, 1, gid)          # (0,1]
    u2 = hash_uniform01(seed, 2, gid)
    return np.sqrt(-2.0 * np.log(u1)) * np.cos(2.0 * np.pi * u2)


@dataclass
class BoxMesh:
    nx: int
    ny: int
    nz: int
    N: int
    vert: np.ndarray        # [E,8,3] float64
    gid: np.ndarray         # [E,p^3] int64
    dirichlet: np.ndarray   # [E,p^3] uint8, 1 on the boundary of [0,1]^3
    perm: np.ndarray        # [E] element e of this mesh is lexicographic element perm[e]
    name: str = ""

    @property
    def E(self) -> int:
        return self.vert.shape[0]

    @property
    def p(self) -> int:
        return self.N + 1

    @property
    def nL(self) -> int:
        return self.E * self.p ** 3

    @property
    def unique_nodes(self) -> int:
        return (self.nx * self.N + 1) * (self.ny * self.N + 1) * (self.nz * self.N + 1)

    @property
    def dofs(self) -> int:
        """The paper's n = E N^3."""
        return self.E * self.N ** 3


def vertex_grid(nx: int, ny: int, nz: int) -> np.ndarray:
    """Undeformed vertex coordinates, V[nz+1, ny+1, nx+1, 3]."""
    x = np.arange(nx + 1, dtype=np.float64) / nx
    y = np.arange(ny + 1, dtype=np.float64) / ny
    z = np.arange(nz + 1, dtype=np.float64) / nz
    Z, Y, X = np.meshgrid(z, y, x, indexing="ij")
    return np.stack([X, Y, Z], axis=-1)


def deform_smooth(V: np.ndarray, amp: float) -> np.ndarray:
    d = amp * np.sin(2 * np.pi * V[..., 0]) * np.sin(2 * np.pi * V[..., 1]) * np.sin(2 * np.pi * V[..., 2])
    # force exactly zero displacement on the boundary (sin(2 pi) is 1e-16, not 0)
    d[0, :, :] = d[-1, :, :] = 0.0
    d[:, 0, :] = d[:, -1, :] = 0.0
    d[:, :, 0] = d[:, :, -1] = 0.0
    return V + d[..., None]


def deform_random(V: np.ndarray, frac: float, seed: int) -> np.ndarray:
    nz1, ny1, nx1, _ = V.shape
    vid = np.arange(nz1 * ny1 * nx1, dtype=np.int64).reshape(nz1, ny1, nx1)
    h = np.array([1.0 / (nx1 - 1), 1.0 / (ny1 - 1), 1.0 / (nz1 - 1)])
    out = V.copy()
    interior = np.zeros((nz1, ny1, nx1), bool)
    interior[1:-1, 1:-1, 1:-1] = True
    for d in range(3):
        delta = (2.0 * hash_uniform01(seed, 10 + d, vid) - 1.0) * frac * h[d]
        out[..., d] += np.where(interior, delta, 0.0)
    return out


def box_mesh(nx: int, ny: int, nz: int, N: int, geometry: str = "affine", amp: float = 0.05, frac: float = 0.1,
             seed: int = 0, permute_seed: int | None = None, name: str = "") -> BoxMesh:
    """Build a box mesh of nx*ny*nz hexahedra of order N on [0,1]^3 (see module docstring)."""
    V = vertex_grid(nx, ny, nz)
    if geometry == "smooth":
        V = deform_smooth(V, amp)
    elif geometry == "random":
        V = deform_random(V, frac, seed)
    elif geometry != "affine":
        raise ValueError(geometry)
    E = nx * ny * nz
    e = np.arange(E, dtype=np.int64)
    if permute_seed is not None:
        # seeded permutation of the element list only (S9): sort elements by a hashed key
        e = np.argsort(hash_uniform01(permute_seed, 20, e), kind="stable").astype(np.int64)
    ex, ey, ez = e % nx, (e // nx) % ny, e // (nx * ny)
    vert = np.empty((E, 8, 3))
    for v in range(8):
        a, b, c = v & 1, (v >> 1) & 1, (v >> 2) & 1
        vert[:, v, :] = V[ez + c, ey + b, ex + a, :]
    p = N + 1
    NX, NY, NZ = nx * N + 1, ny * N + 1, nz * N + 1
    i = np.arange(p, dtype=np.int64)
    gx = (ex[:, None] * N + i[None, :])                      # [E,p]
    gy = (ey[:, None] * N + i[None, :])
    gz = (ez[:, None] * N + i[None, :])
    gid = gx[:, None, None, :] + NX * (gy[:, None, :, None] + NY * gz[:, :, None, None])   # [E,k,j,i]
    bx = (gx == 0) | (gx == NX - 1)
    by = (gy == 0) | (gy == NY - 1)
    bz = (gz == 0) | (gz == NZ - 1)
    dirichlet = (bx[:, None, None, :] | by[:, None, :, None] | bz[:, :, None, None]).astype(np.uint8)
    return BoxMesh(nx, ny, nz, N, vert, np.ascontiguousarray(gid.reshape(E, p ** 3)),
                   np.ascontiguousarray(dirichlet.reshape(E, p ** 3)), e, name)


# ---- the BASELINE.json configs ---------------------------------------------------------------------------------
def config1() -> BoxMesh:
    """Tiny oracle-check: 4x4x4 elements, N=7, smooth deformation amp 0.05."""
    return box_mesh(4, 4, 4, 7, "smooth", amp=0.05, name="cfg1_4x4x4_N7_smooth")


def config2() -> BoxMesh:
    """Per-GPU paper scale: 20x20x18 = 7200 elements, N=7 (n = E N^3 = 2 469 600)."""
    return box_mesh(20, 20, 18, 7, "smooth", amp=0.05, name="cfg2_20x20x18_N7_smooth")


def config3(n: int, N: int) -> BoxMesh:
    """Bandwidth sweep: n^3 elements, random +-10% vertex perturbation, seed 1."""
    return box_mesh(n, n, n, N, "random", frac=0.1, seed=1, name=f"cfg3_{n}^3_N{N}_random")


def config4(N: int) -> BoxMesh:
    """Mixed-precision levels: 20x20x18, N in {7,3,1}, smooth deformation."""
    return box_mesh(20, 20, 18, N, "smooth", amp=0.05, name=f"cfg4_20x20x18_N{N}_smooth")


def config5(n: int = 100) -> BoxMesh:
    """Full solve: n^3 elements (100^3 at full size), N=7, random perturbation seed 3, element permutation seed 4."""
    return box_mesh(n, n, n, 7, "random", frac=0.1, seed=3, permute_seed=4, name=f"cfg5_{n}^3_N7_random_perm")


def fdm_pairs(E: int, m: int, seed: int):
    """Seeded stand-in for the 1-D operator pairs (A_d, B_d), d = x, y, z, of the Schwarz smoother's extended local
    problems (the paper does not give their construction, reading S28 in DESIGN.md): on a 1-D grid of m
    interior points clustered towards the ends like GLL points (x_q = -cos(pi q / (m+1)), homogeneous Dirichlet at
    q = 0 and q = m+1), scaled by a seeded element length h_d in [0.5, 1.5], A = the linear finite-element stiffness
    matrix (tridiagonal, SPD) and B = the lumped mass matrix (diagonal, positive).  Returns A[E][3][m][m], B[E][3][m][m]
    (FP64).  Mesh-like data only: the eigen-decomposition and Eq. (3) are the method's, not this module's."""
    cnt = np.arange(E * 3, dtype=np.uint64)
    h = (0.5 + hash_uniform01(seed, 11, cnt)).reshape(E, 3)
    x = -np.cos(np.pi * np.arange(m + 2) / (m + 1))                 # [m+2] reference grid on [-1, 1]
    dx = np.diff(x)                                                 # [m+1]
    A = np.zeros((E, 3, m, m))
    B = np.zeros((E, 3, m, m))
    q = np.arange(m)
    for e in range(E):
        for d in range(3):
            s = 0.5 * h[e, d] * dx                                  # physical cell sizes
            A[e, d, q, q] = 1.0 / s[:-1] + 1.0 / s[1:]
            A[e, d, q[:-1], q[1:]] = A[e, d, q[1:], q[:-1]] = -1.0 / s[1:-1]
            B[e, d, q, q] = 0.5 * (s[:-1] + s[1:])
    return A, B


# ---- re-oriented elements: the same mesh with every element's local frame rotated (unstructured-mesh orientations) -------
def _proper_rotations():
    """The 24 signed permutations (pi, s) of the reference cube with determinant +1: old coordinate a = s[a] * new
    coordinate pi[a]."""
    import itertools
    out = []
    for pi in itertools.permutations(range(3)):
        par = 1
        for a in range(3):
            for b in range(a + 1, 3):
                if pi[a] > pi[b]:
                    par = -par
        for s in itertools.product((1, -1), repeat=3):
            if par * s[0] * s[1] * s[2] == 1:
                out.append((pi, s))
    return out


def reorient(mesh: BoxMesh, seed: int) -> BoxMesh:
    """The same elements, nodes and global ids, but every element's local (r, s, t) frame replaced by one of the 24
    proper rotations of the reference cube, chosen by a hash of (seed, element): local node (i0', i1', i2') of the new
    element is old local node i_a = i'_{pi[a]} (s[a] = +1) or N - i'_{pi[a]} (s[a] = -1), vertices alike.  Neighbouring
    elements then meet with arbitrary relative orientation, as in an unstructured hexahedral mesh; the Jacobian
    determinant stays positive.  Mesh layout only: no method arithmetic."""
    N, p, E = mesh.N, mesh.N + 1, mesh.E
    rots = _proper_rotations()
    pick = (hash_uniform01(seed, 30, np.arange(E)) * len(rots)).astype(np.int64) % len(rots)
    gid = mesh.gid.reshape(E, p, p, p).copy()
    dirf = mesh.dirichlet.reshape(E, p, p, p).copy()
    vert = mesh.vert.copy()
    idx = np.arange(p)
    for e in range(E):
        pi, s = rots[int(pick[e])]
        # new index tuple n = (n0, n1, n2) = (i', j', k'); old index o_a = n[pi[a]] or N - n[pi[a]]
        n = np.meshgrid(idx, idx, idx, indexing="ij")            # n[0] = i', n[1] = j', n[2] = k'  (arrays [i'][j'][k'])
        o = [n[pi[a]] if s[a] > 0 else N - n[pi[a]] for a in range(3)]
        g_old, d_old = mesh.gid.reshape(E, p, p, p)[e], mesh.dirichlet.reshape(E, p, p, p)[e]
        g_new = g_old[o[2], o[1], o[0]]                          # arrays are stored [k][j][i]; result indexed [i'][j'][k']
        d_new = d_old[o[2], o[1], o[0]]
        gid[e] = np.transpose(g_new, (2, 1, 0))
        dirf[e] = np.transpose(d_new, (2, 1, 0))
        for v in range(8):
            nb = [(v >> a) & 1 for a in range(3)]
            ob = [nb[pi[a]] if s[a] > 0 else 1 - nb[pi[a]] for a in range(3)]
            vert[e, v] = mesh.vert[e, ob[0] + 2 * ob[1] + 4 * ob[2]]
    return BoxMesh(mesh.nx, mesh.ny, mesh.nz, N, vert, np.ascontiguousarray(gid.reshape(E, p ** 3)),
                   np.ascontiguousarray(dirf.reshape(E, p ** 3)), mesh.perm, mesh.name + "_reoriented")
