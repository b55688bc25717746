"""CPU-side checks of the boundary: libsem.so builds, loads and exports every symbol include/sem.h declares, the
Python binding names them all, and compute calls fail loudly (no CPU fallback) when there is no CUDA device."""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "sem.h")


def header_symbols():
    txt = open(HEADER).read()
    txt = re.sub(r"/\*.*?\*/", "", txt, flags=re.S)
    return sorted(set(re.findall(r"SEM_API\s+[\w\s\*]+?\b(sem_\w+)\s*\(", txt)))


@pytest.fixture(scope="module")
def built_lib():
    from paper_2110_01716_b200 import build
    return build.build()


def test_header_declares_north_star_calls():
    syms = header_symbols()
    for name in ["sem_mesh_setup", "sem_geom", "sem_ax", "sem_gs", "sem_pcg", "sem_ax_gs"]:
        assert name in syms


def test_library_exports_every_declared_symbol(built_lib):
    L = C.CDLL(built_lib)
    for name in header_symbols():
        assert hasattr(L, name), f"{name} declared in include/sem.h but not exported by libsem.so"


def test_binding_covers_header(built_lib):
    from paper_2110_01716_b200 import binding
    assert sorted(binding.SYMBOLS) == header_symbols()
    binding.lib()   # sets restype/argtypes for every symbol without raising


def test_no_cpu_fallback(built_lib):
    """Without a GPU the library must refuse to compute (SEM_ECUDA), and bad arguments are SEM_EINVAL."""
    import torch
    from paper_2110_01716_b200 import binding, inputs
    L = binding.lib()
    h = C.c_void_p()
    m = inputs.box_mesh(1, 1, 1, 2)
    vert = np.ascontiguousarray(m.vert)
    gid = np.ascontiguousarray(m.gid)
    assert L.sem_mesh_setup(C.byref(h), 0, 2, vert.ctypes.data, gid.ctypes.data, None, None) == binding.SEM_EINVAL
    assert L.sem_mesh_setup(C.byref(h), 1, 0, vert.ctypes.data, gid.ctypes.data, None, None) == binding.SEM_EINVAL
    assert L.sem_mesh_setup(C.byref(h), 1, 16, vert.ctypes.data, gid.ctypes.data, None, None) == binding.SEM_EINVAL
    assert L.sem_mesh_setup(C.byref(h), 1, 2, None, gid.ctypes.data, None, None) == binding.SEM_EINVAL
    if not torch.cuda.is_available():
        rc = L.sem_mesh_setup(C.byref(h), 1, 2, vert.ctypes.data, gid.ctypes.data, None, None)
        assert rc == binding.SEM_ECUDA
        assert b"no CUDA device" in L.sem_last_error(h)
        L.sem_ctx_destroy(h)
        with pytest.raises(binding.SemError):
            binding.Sem(1, 2, vert, gid)


# ------------------------------------------------------------------ NEXT-2a setup: sem_fdm_setup is host logic (no GPU)
def test_fdm_setup_host_matches_the_oracle_eigen_decomposition(built_lib):
    """sem_fdm_setup (Cholesky + cyclic Jacobi in the library) against the oracle's scipy.linalg.eigh on the seeded
    operator pairs: eigenvalues, B-orthonormality, diagonalisation, Lambda^-1, and -- since eigenvectors are unique only
    up to sign and up to rotations inside (nearly) degenerate eigenspaces -- the result of Eq. (3) computed by the oracle
    from the library's (S, Lambda^-1) against the oracle's own."""
    import numpy as np
    import oracle
    from paper_2110_01716_b200 import binding, inputs
    for m, E in ((10, 12), (4, 7), (7, 5), (16, 3), (2, 4)):
        A, B = inputs.fdm_pairs(E, m, seed=50 + m)
        S, invL = binding.fdm_setup(A, B)
        So, invLo = np.empty_like(A), np.empty((E, m, m, m))
        for e in range(E):
            lam = []
            for d in range(3):
                So[e, d], l = oracle.fdm_eig(A[e, d], B[e, d])
                lam.append(l)
                D = S[e, d].T @ A[e, d] @ S[e, d]
                assert np.max(np.abs(np.diag(D) - l)) <= 1e-12 * l[-1]
                assert np.max(np.abs(D - np.diag(np.diag(D)))) <= 1e-11 * l[-1]
                assert np.max(np.abs(S[e, d].T @ B[e, d] @ S[e, d] - np.eye(m))) <= 1e-12
            invLo[e] = oracle.fdm_inv_lambda(*lam)
        assert np.max(np.abs(invL / invLo - 1.0)) <= 1e-12
        b = 2.0 * inputs.hash_uniform01(9, 12, np.arange(E * m ** 3)).reshape(E, m, m, m) - 1.0
        u_lib, u_orc = oracle.fdm_apply(S, invL, b), oracle.fdm_apply(So, invLo, b)
        assert np.max(np.abs(u_lib - u_orc)) <= 1e-11 * np.max(np.abs(u_orc))


def test_fdm_setup_dense_spd_pairs(built_lib):
    """The seeded pairs above have a DIAGONAL mass matrix and a tridiagonal stiffness matrix; here both are dense SPD
    (random orthogonal basis, seeded spectrum), m = 2 ... 16, so the Cholesky factor's off-diagonal code and the
    congruence transform are exercised: S^T B S = I, S^T A S = diag(lambda) ascending, lambda equal to scipy's generalised
    eigenvalues, and Eq. (3) with the library's (S, Lambda^-1) inverts the dense Kronecker-sum operator."""
    import numpy as np
    import scipy.linalg
    import oracle
    from paper_2110_01716_b200 import binding, inputs

    def spd(m, seed, lo, hi):
        Q, _ = np.linalg.qr(2.0 * inputs.hash_uniform01(seed, 3, np.arange(m * m)).reshape(m, m) - 1.0)
        ev = lo + (hi - lo) * inputs.hash_uniform01(seed, 4, np.arange(m))
        return (Q * ev) @ Q.T

    for m in range(2, 17):
        E = 3
        A = np.empty((E, 3, m, m))
        B = np.empty((E, 3, m, m))
        for e in range(E):
            for d in range(3):
                A[e, d] = spd(m, 1000 * m + 10 * e + d, 0.5, 40.0)
                B[e, d] = spd(m, 7000 * m + 10 * e + d, 0.2, 3.0)
        S, invL = binding.fdm_setup(A, B)
        for e in range(E):
            lam = []
            for d in range(3):
                ref = scipy.linalg.eigh(A[e, d], B[e, d], eigvals_only=True)
                D = S[e, d].T @ A[e, d] @ S[e, d]
                assert np.max(np.abs(S[e, d].T @ B[e, d] @ S[e, d] - np.eye(m))) <= 1e-12, (m, e, d)
                assert np.max(np.abs(D - np.diag(np.diag(D)))) <= 1e-11 * ref[-1], (m, e, d)
                assert np.max(np.abs(np.diag(D) - ref)) <= 1e-11 * ref[-1], (m, e, d)
                lam.append(np.diag(D))
            assert np.max(np.abs(invL[e] * oracle.fdm_inv_lambda(*[np.asarray(l) for l in lam])[...] ** -1 - 1.0)) <= 1e-11
        if m <= 6:                                           # Eq. (3) inverts the dense separable operator (kron order z,y,x)
            e = 0
            Ax, Ay, Az = A[e]
            Bx, By, Bz = B[e]
            K = np.kron(Bz, np.kron(By, Ax)) + np.kron(Bz, np.kron(Ay, Bx)) + np.kron(Az, np.kron(By, Bx))
            b = 2.0 * inputs.hash_uniform01(3, 5, np.arange(m ** 3)) - 1.0
            u = oracle.fdm_apply(S[e:e + 1], invL[e:e + 1], b.reshape(1, m, m, m)).ravel()
            assert np.max(np.abs(K @ u - b)) <= 1e-9 * np.max(np.abs(b)), m


def test_fdm_setup_bad_args(built_lib):
    import numpy as np
    from paper_2110_01716_b200 import binding
    A = np.tile(np.eye(3), (1, 3, 1, 1))
    with pytest.raises(binding.SemError):
        binding.fdm_setup(A, -A)                                # mass matrix not positive definite
    with pytest.raises(binding.SemError):
        binding.fdm_setup(np.tile(np.eye(17), (1, 3, 1, 1)), np.tile(np.eye(17), (1, 3, 1, 1)))    # m > 16
