"""Thin ctypes binding over the C-ABI library libsem.so (include/sem.h).  Argument marshalling only: every step of the
hot path runs in the CUDA kernels of the library.  torch is used for device memory and the stream handle.

There is no CPU fallback: if libsem.so is missing the import of this module's `lib()` raises, and every compute call
needs a CUDA device.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libsem.so")

SEM_F64, SEM_F32 = 0, 1
SEM_OP_ADD = 0
SEM_G_STORED, SEM_G_RECOMPUTE = 0, 1
SEM_PROLONG, SEM_RESTRICT = 0, 1
SEM_INTERLEAVED = 1
SEM_NOALLOC_MAX_NODES = 1 << 19
SEM_SCHWARZ_ASM, SEM_SCHWARZ_RAS = 0, 1
SEM_SMOOTH_CHEBY_JACOBI, SEM_SMOOTH_CHEBY_SCHWARZ, SEM_SMOOTH_CHEBY_RAS = 0, 1, 2
SEM_OK, SEM_EINVAL, SEM_EMESH, SEM_ECUDA, SEM_ENOMEM, SEM_ESTATE = 0, -1, -2, -3, -4, -5
_ERRNAME = {-1: "SEM_EINVAL", -2: "SEM_EMESH", -3: "SEM_ECUDA", -4: "SEM_ENOMEM", -5: "SEM_ESTATE"}

# every symbol include/sem.h declares: name -> (restype, argtypes)
_vp, _i64, _i32, _dbl = C.c_void_p, C.c_int64, C.c_int, C.c_double
SYMBOLS = {
    "sem_mesh_setup": (_i32, [C.POINTER(_vp), _i64, _i32, _vp, _vp, _vp, _vp]),
    "sem_geom": (_i32, [_vp, _vp, _i32, _i32]),
    "sem_ax": (_i32, [_vp, _vp, _vp, _i32, _dbl]),
    "sem_gs": (_i32, [_vp, _vp, _i32, _i32]),
    "sem_ax_gs": (_i32, [_vp, _vp, _vp, _i32, _dbl]),
    "sem_gs_many": (_i32, [_vp, _vp, _i32, _i64, _i32, _i32]),
    "sem_pcg": (_i32, [_vp, _vp, _vp, _dbl, _i32, C.POINTER(_i32), C.POINTER(_dbl)]),
    "sem_iface_pack": (_i32, [_vp, _vp, _i64, _vp, _vp, _i32]),
    "sem_iface_add": (_i32, [_vp, _vp, _i64, _vp, _vp, _i32]),
    "sem_ax_gs_many": (_i32, [_vp, _vp, _vp, _i32, _i64, _i32, _dbl]),
    "sem_pcg_many": (_i32, [_vp, _vp, _vp, _i32, _i64, _dbl, _i32, C.POINTER(_i32), C.POINTER(_dbl)]),
    "sem_set_lambda": (_i32, [_vp, _dbl]),
    "sem_get_pcg_history": (_i32, [_vp, _vp, _i32]),
    "sem_get_counts": (_i32, [_vp, C.POINTER(_i64), C.POINTER(_i64), C.POINTER(_i64), C.POINTER(_i64)]),
    "sem_get_maps": (_i32, [_vp, _vp, _vp, _vp, _vp, _vp]),
    "sem_get_gll": (_i32, [_vp, _vp, _vp, _vp]),
    "sem_get_geom": (_i32, [_vp, _vp, _vp]),
    "sem_get_diag": (_i32, [_vp, _vp]),
    "sem_set_variant": (_i32, [_vp, _i32]),
    "sem_transfer": (_i32, [_vp, _vp, _vp, _vp, _i32, _i32]),
    "sem_get_interp": (_i32, [_vp, _vp, _vp]),
    "sem_cheby": (_i32, [_vp, _vp, _vp, _i32, _dbl, _dbl, _i32, _i32]),
    "sem_lambda_max": (_i32, [_vp, _i32, C.POINTER(_dbl)]),
    "sem_cheby_noalloc": (_i32, [_vp, _vp, _vp, _i32, _dbl, _dbl, _i32]),
    "sem_pmg_create": (_i32, [C.POINTER(_vp), _i32, C.POINTER(_vp), C.POINTER(_dbl), C.POINTER(_dbl), _i32, _i32, _i32]),
    "sem_pmg_vcycle": (_i32, [_vp, _vp, _vp]),
    "sem_pmg_destroy": (None, [_vp]),
    "sem_proj_create": (_i32, [C.POINTER(_vp), _vp, _i32]),
    "sem_proj_guess": (_i32, [_vp, _vp, _vp, _vp]),
    "sem_proj_update": (_i32, [_vp, _vp, C.POINTER(_i32)]),
    "sem_proj_size": (_i32, [_vp, C.POINTER(_i32)]),
    "sem_proj_destroy": (None, [_vp]),
    "sem_fpcg": (_i32, [_vp, _vp, _vp, _dbl, _i32, C.POINTER(_i32), C.POINTER(_dbl)]),
    "sem_pmg_get_history": (_i32, [_vp, _vp, _i32]),
    "sem_fdm_apply": (_i32, [_vp, _i32, _vp, _vp, _vp, _vp, _i32]),
    "sem_fdm_setup": (_i32, [_i64, _i32, _vp, _vp, _vp, _vp]),
    "sem_measure_peak": (_i32, [_i32, _vp, C.POINTER(_dbl)]),
    "sem_schwarz_setup": (_i32, [_vp]),
    "sem_schwarz": (_i32, [_vp, _vp, _vp, _i32, _i32]),
    "sem_get_schwarz": (_i32, [_vp, _vp, _vp, _vp, _vp, _i32]),
    "sem_cheby_schwarz": (_i32, [_vp, _vp, _vp, _i32, _dbl, _dbl, _i32, _i32, _i32]),
    "sem_lambda_max_schwarz": (_i32, [_vp, _i32, _i32, C.POINTER(_dbl)]),
    "sem_pmg_set_smoother": (_i32, [_vp, _i32, C.POINTER(_dbl), C.POINTER(_dbl)]),
    "sem_shard_set_interface": (_i32, [_vp, _i64]),
    "sem_get_chunks": (_i32, [_vp, _vp, _i32, C.POINTER(_i32), C.POINTER(_i32)]),
    "sem_ax_gs_sharded": (_i32, [_vp, _vp, _vp, _i32, _dbl, _vp]),
    "sem_pcg_sharded": (_i32, [_vp, _vp, _vp, _dbl, _i32, _vp, C.POINTER(_i32), C.POINTER(_dbl)]),
    "sem_last_error": (C.c_char_p, [_vp]),
    "sem_ctx_destroy": (None, [_vp]),
}

_lib = None

# sem_shard_hooks (include/sem.h): the transport of a sharded solve, called back from inside the library
_GS_HOOK = C.CFUNCTYPE(_i32, _vp, _vp, _i32)
_AR_HOOK = C.CFUNCTYPE(_i32, _vp, _vp, _i32)


class _ShardHooksStruct(C.Structure):
    _fields_ = [("gs_begin", _GS_HOOK), ("gs_end", _GS_HOOK), ("allreduce", _AR_HOOK), ("user", _vp)]


class ShardHooks:
    """Wraps three Python callables as a sem_shard_hooks struct.  gs_begin(w_ptr, prec), gs_end(w_ptr, prec) and
    allreduce(scalars_ptr, n) get raw DEVICE addresses (int).  An exception inside a hook makes the library call fail;
    it is kept in `.error` and re-raised by the binding."""

    def __init__(self, gs_begin, gs_end, allreduce):
        self.error = None

        def guard(fn):
            def call(_user, ptr, k):
                try:
                    fn(int(ptr or 0), int(k))
                    return 0
                except BaseException as exc:          # must not propagate into the C caller
                    self.error = exc
                    return 1
            return call

        self._keep = (_GS_HOOK(guard(gs_begin)), _GS_HOOK(guard(gs_end)), _AR_HOOK(guard(allreduce)))
        self.struct = _ShardHooksStruct(self._keep[0], self._keep[1], self._keep[2], None)

    def ref(self):
        return C.cast(C.byref(self.struct), _vp)


def fdm_setup(A: np.ndarray, B: np.ndarray):
    """sem_fdm_setup (host): A, B [E][3][m][m] float64 -> (S[E][3][m][m], inv_lambda[E][m][m][m]) for sem_fdm_apply."""
    A = np.ascontiguousarray(A, dtype=np.float64)
    B = np.ascontiguousarray(B, dtype=np.float64)
    assert A.ndim == 4 and A.shape == B.shape and A.shape[1] == 3 and A.shape[2] == A.shape[3]
    E, m = A.shape[0], A.shape[2]
    S = np.empty_like(A)
    inv_lambda = np.empty((E, m, m, m))
    rc = lib().sem_fdm_setup(E, m, _np_ptr(A), _np_ptr(B), _np_ptr(S), _np_ptr(inv_lambda))
    if rc != SEM_OK:
        raise SemError(rc, "sem_fdm_setup: bad arguments or a mass matrix that is not positive definite")
    return S, inv_lambda


def measure_peak(kind: int) -> float:
    """sem_measure_peak on torch's current stream: TFLOP/s of kind 0 = FP64 FMA, 1 = FP32 FMA, 2 = FP64 DMMA m8n8k4."""
    import torch
    out = _dbl(0.0)
    rc = lib().sem_measure_peak(kind, C.c_void_p(torch.cuda.current_stream().cuda_stream), C.byref(out))
    if rc != SEM_OK:
        raise SemError(rc, "sem_measure_peak")
    return float(out.value)


class SemError(RuntimeError):
    def __init__(self, code: int, text: str):
        super().__init__(f"{_ERRNAME.get(code, code)}: {text}")
        self.code = code


def lib() -> C.CDLL:
    """Load libsem.so (fails loudly if it has not been built: python -m paper_2110_01716_b200.build)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise FileNotFoundError(f"{LIB_PATH} not built; run `python -m paper_2110_01716_b200.build` "
                                    "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        for name, (res, args) in SYMBOLS.items():
            f = getattr(L, name)
            f.restype, f.argtypes = res, args
        _lib = L
    return _lib


def _np_ptr(a):
    return a.ctypes.data_as(C.c_void_p) if a is not None else None


class Sem:
    """One mesh/discretisation context (sem_mesh_setup ... sem_ctx_destroy).  Method names follow the C ABI."""

    def __init__(self, E: int, N: int, vertex_xyz: np.ndarray, gid, dirichlet: np.ndarray | None = None, stream=None):
        import torch

        if not torch.cuda.is_available():
            raise SemError(SEM_ECUDA, "no CUDA device (libsem has no CPU fallback)")
        self._L = lib()
        self.E, self.N, self.p = int(E), int(N), int(N) + 1
        self.nL = self.E * self.p ** 3
        vert = np.ascontiguousarray(vertex_xyz, dtype=np.float64).reshape(E, 8, 3)
        if isinstance(gid, torch.Tensor):
            assert gid.dtype == torch.int64 and gid.is_contiguous() and gid.numel() == self.nL
            self._gid_keep = gid
            gid_ptr = C.c_void_p(gid.data_ptr())
        else:
            g = np.ascontiguousarray(gid, dtype=np.int64).reshape(-1)
            assert g.size == self.nL
            self._gid_keep = g
            gid_ptr = _np_ptr(g)
        d = None
        if dirichlet is not None:
            d = np.ascontiguousarray(dirichlet, dtype=np.uint8).reshape(-1)
            assert d.size == self.nL
        self._stream = stream if stream is not None else torch.cuda.current_stream()
        self._h = C.c_void_p()
        rc = self._L.sem_mesh_setup(C.byref(self._h), E, N, _np_ptr(vert), gid_ptr, _np_ptr(d),
                                    C.c_void_p(self._stream.cuda_stream))
        self._check(rc)

    # ---- plumbing ----
    def _check(self, rc: int):
        if rc != SEM_OK:
            text = self._L.sem_last_error(self._h) if self._h else b""
            raise SemError(rc, (text or b"").decode())

    def close(self):
        if getattr(self, "_h", None):
            self._L.sem_ctx_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    @staticmethod
    def _prec(t) -> int:
        import torch

        if t.dtype == torch.float64:
            return SEM_F64
        if t.dtype == torch.float32:
            return SEM_F32
        raise TypeError(f"unsupported dtype {t.dtype}")

    def _vec(self, t):
        assert t.is_cuda and t.is_contiguous() and t.numel() == self.nL, "need a contiguous CUDA tensor of nL values"
        return C.c_void_p(t.data_ptr())

    # ---- the C ABI ----
    def geom(self, node_xyz: np.ndarray | None = None, mode: int = SEM_G_STORED, with_mass: bool = False):
        x = None if node_xyz is None else np.ascontiguousarray(node_xyz, dtype=np.float64)
        self._check(self._L.sem_geom(self._h, _np_ptr(x), mode, int(with_mass)))
        self.with_mass = bool(with_mass)
        return self

    def ax(self, u, w, lam: float = 0.0):
        self._check(self._L.sem_ax(self._h, self._vec(u), self._vec(w), self._prec(u), lam))
        return w

    def gs(self, w):
        self._check(self._L.sem_gs(self._h, self._vec(w), self._prec(w), SEM_OP_ADD))
        return w

    def gs_many(self, w, interleaved: bool = False):
        """sem_gs_many in place on a contiguous CUDA tensor: [nfields][stride >= nL], or -- interleaved=True -- the
        node-interleaved layout [nL][nfields] (field_stride = SEM_INTERLEAVED, 2 to 4 fields)."""
        assert w.is_cuda and w.is_contiguous() and w.dim() == 2
        if interleaved:
            assert w.shape[0] == self.nL
            nf, stride = w.shape[1], SEM_INTERLEAVED
        else:
            assert w.shape[1] >= self.nL
            nf, stride = w.shape[0], w.shape[1]
        self._check(self._L.sem_gs_many(self._h, C.c_void_p(w.data_ptr()), nf, stride, self._prec(w), SEM_OP_ADD))
        return w

    def _fields(self, t):
        assert t.is_cuda and t.is_contiguous() and t.dim() == 2 and t.shape[1] >= self.nL, \
            "need a contiguous [nfields][stride >= nL] CUDA tensor"
        return C.c_void_p(t.data_ptr()), int(t.shape[0]), int(t.shape[1])

    def ax_gs_many(self, u, w, lam: float = 0.0):
        """sem_ax_gs_many on contiguous [nfields][stride] CUDA tensors."""
        pu, nf, st = self._fields(u)
        pw, nfw, stw = self._fields(w)
        assert (nf, st) == (nfw, stw) and u.dtype == w.dtype
        self._check(self._L.sem_ax_gs_many(self._h, pu, pw, nf, st, self._prec(u), lam))
        return w

    def pcg_many(self, b, x, tol: float, maxit: int):
        """sem_pcg_many on contiguous [nfields][stride] FP64 CUDA tensors: (iters[nf], relres[nf])."""
        pb, nf, st = self._fields(b)
        px, nfx, stx = self._fields(x)
        assert (nf, st) == (nfx, stx)
        it = (C.c_int * nf)()
        rel = (C.c_double * nf)()
        self._check(self._L.sem_pcg_many(self._h, pb, px, nf, st, tol, maxit, it, rel))
        return list(it), list(rel)

    def _vec_or_ptr(self, w, prec):
        """A field as a CUDA tensor, or as a raw device address (int) with its precision given (hook callbacks)."""
        if isinstance(w, int):
            assert prec in (SEM_F64, SEM_F32)
            return C.c_void_p(w), prec
        return self._vec(w), self._prec(w)

    def iface_pack(self, uniq, w, buf, prec=None):
        """sem_iface_pack: buf[q] = w[first copy of unique node uniq[q]] (uniq: int32 CUDA tensor)."""
        pw, pr = self._vec_or_ptr(w, prec)
        self._check(self._L.sem_iface_pack(self._h, C.c_void_p(uniq.data_ptr()), int(uniq.numel()), pw,
                                           C.c_void_p(buf.data_ptr()), pr))
        return buf

    def iface_add(self, uniq, buf, w, prec=None):
        """sem_iface_add: every copy of unique node uniq[q] += buf[q] (Dirichlet nodes stay zero)."""
        pw, pr = self._vec_or_ptr(w, prec)
        self._check(self._L.sem_iface_add(self._h, C.c_void_p(uniq.data_ptr()), int(uniq.numel()),
                                          C.c_void_p(buf.data_ptr()), pw, pr))
        return w

    def shard_set_interface(self, n_iface_elems: int):
        """sem_shard_set_interface: elements [0, n) are the only ones touching nodes shared with other ranks."""
        self._check(self._L.sem_shard_set_interface(self._h, int(n_iface_elems)))
        return self

    def chunks(self):
        """sem_get_chunks: (element bounds of the chunks, number of leading chunks that precede gs_begin)."""
        n, ic = C.c_int(0), C.c_int(0)
        self._check(self._L.sem_get_chunks(self._h, None, 0, C.byref(n), C.byref(ic)))
        e0 = np.zeros(n.value + 1, dtype=np.int64)
        self._check(self._L.sem_get_chunks(self._h, _np_ptr(e0), e0.size, None, None))
        return e0, ic.value

    def _check_hooks(self, rc: int, hooks: "ShardHooks"):
        if hooks.error is not None:
            exc, hooks.error = hooks.error, None
            raise exc
        self._check(rc)

    def ax_gs_sharded(self, u, w, hooks: "ShardHooks", lam: float = 0.0):
        assert u.dtype == w.dtype
        self._check_hooks(self._L.sem_ax_gs_sharded(self._h, self._vec(u), self._vec(w), self._prec(u), lam, hooks.ref()),
                          hooks)
        return w

    def pcg_sharded(self, b, x, tol: float, maxit: int, hooks: "ShardHooks"):
        """sem_pcg_sharded on this rank's part; returns (iters, relres), the same on every rank."""
        import torch

        assert b.dtype == torch.float64 and x.dtype == torch.float64
        it, rel = C.c_int(0), C.c_double(0.0)
        self._check_hooks(self._L.sem_pcg_sharded(self._h, self._vec(b), self._vec(x), tol, maxit, hooks.ref(),
                                                  C.byref(it), C.byref(rel)), hooks)
        return it.value, rel.value

    def ax_gs(self, u, w, lam: float = 0.0):
        assert u.dtype == w.dtype
        self._check(self._L.sem_ax_gs(self._h, self._vec(u), self._vec(w), self._prec(u), lam))
        return w

    def pcg(self, b, x, tol: float, maxit: int):
        """Returns (iters, relres); x is updated in place."""
        import torch

        assert b.dtype == torch.float64 and x.dtype == torch.float64
        it, rel = C.c_int(0), C.c_double(0.0)
        self._check(self._L.sem_pcg(self._h, self._vec(b), self._vec(x), tol, maxit, C.byref(it), C.byref(rel)))
        return it.value, rel.value

    def set_lambda(self, lam: float):
        self._check(self._L.sem_set_lambda(self._h, lam))

    def transfer(self, fine: "Sem", vin, vout, direction: int):
        """sem_transfer with self as the COARSE context: SEM_PROLONG coarse -> fine, SEM_RESTRICT fine -> coarse."""
        n_in, n_out = (fine.nL, self.nL) if direction == SEM_RESTRICT else (self.nL, fine.nL)
        for t, n in ((vin, n_in), (vout, n_out)):
            assert t.is_cuda and t.is_contiguous() and t.numel() == n and t.dtype == vin.dtype, \
                "need contiguous CUDA tensors of the coarse / fine local sizes"
        rc = self._L.sem_transfer(self._h, fine._h, C.c_void_p(vin.data_ptr()), C.c_void_p(vout.data_ptr()),
                                  self._prec(vin), direction)
        if rc != SEM_OK:
            raise SemError(rc, self._L.sem_last_error(fine._h).decode())
        return vout

    def fdm_apply(self, m: int, S, inv_lambda, b, u):
        """sem_fdm_apply (Eq. (3)): S[E][3][m][m], inv_lambda[E][m^3], b, u [E][m^3]; u may be b."""
        m3 = m * m * m
        for t, n in ((S, self.E * 3 * m * m), (inv_lambda, self.E * m3), (b, self.E * m3), (u, self.E * m3)):
            assert t.is_cuda and t.is_contiguous() and t.numel() == n and t.dtype == b.dtype, \
                "need contiguous CUDA tensors of one dtype with E*3*m*m / E*m^3 values"
        self._check(self._L.sem_fdm_apply(self._h, m, C.c_void_p(S.data_ptr()), C.c_void_p(inv_lambda.data_ptr()),
                                          C.c_void_p(b.data_ptr()), C.c_void_p(u.data_ptr()), self._prec(b)))
        return u

    def interp(self, fine: "Sem") -> np.ndarray:
        J = np.empty((fine.N + 1, self.N + 1))
        rc = self._L.sem_get_interp(self._h, fine._h, _np_ptr(J))
        if rc != SEM_OK:
            raise SemError(rc, self._L.sem_last_error(fine._h).decode())
        return J

    def cheby(self, b, x, order: int, lmin: float, lmax: float, zero_guess: bool = False):
        self._check(self._L.sem_cheby(self._h, self._vec(b), self._vec(x), order, lmin, lmax, int(zero_guess),
                                      self._prec(x)))
        return x

    def cheby_noalloc(self, b, x, order: int, lmin: float, lmax: float, zero_guess: bool = False):
        """sem_cheby_noalloc: FP64, nL <= SEM_NOALLOC_MAX_NODES, work vectors in the library's static device array."""
        import torch

        assert b.dtype == torch.float64 and x.dtype == torch.float64
        self._check(self._L.sem_cheby_noalloc(self._h, self._vec(b), self._vec(x), order, lmin, lmax, int(zero_guess)))
        return x

    def lambda_max(self, iters: int = 30) -> float:
        lam = C.c_double(0.0)
        self._check(self._L.sem_lambda_max(self._h, iters, C.byref(lam)))
        return lam.value

    def set_variant(self, v: int):
        self._check(self._L.sem_set_variant(self._h, v))

    # ---- NEXT-2b: overlapping Schwarz smoother ----
    def schwarz_setup(self):
        self._check(self._L.sem_schwarz_setup(self._h))
        return self

    def schwarz(self, r, z, kind: int = SEM_SCHWARZ_ASM):
        self._check(self._L.sem_schwarz(self._h, self._vec(r), self._vec(z), self._prec(r), kind))
        return z

    def get_schwarz(self, kind: int = SEM_SCHWARZ_ASM):
        """(nbr[E][6], A[E][3][m][m], B[E][3][m][m], W[E][p^3]) of the Schwarz smoother (parity accessor)."""
        m = self.p + 2
        nbr = np.empty((self.E, 6), np.int32)
        A, B = np.empty((self.E, 3, m, m)), np.empty((self.E, 3, m, m))
        W = np.empty((self.E, self.p ** 3))
        self._check(self._L.sem_get_schwarz(self._h, _np_ptr(nbr), _np_ptr(A), _np_ptr(B), _np_ptr(W), kind))
        return nbr, A, B, W

    def cheby_schwarz(self, b, x, order: int, lmin: float, lmax: float, zero_guess: bool = False,
                      kind: int = SEM_SCHWARZ_ASM):
        self._check(self._L.sem_cheby_schwarz(self._h, self._vec(b), self._vec(x), order, lmin, lmax, int(zero_guess),
                                              self._prec(x), kind))
        return x

    def lambda_max_schwarz(self, kind: int = SEM_SCHWARZ_ASM, iters: int = 30) -> float:
        lam = C.c_double(0.0)
        self._check(self._L.sem_lambda_max_schwarz(self._h, kind, iters, C.byref(lam)))
        return lam.value

    def pcg_history(self, n: int) -> np.ndarray:
        h = np.full(n, np.nan)
        self._check(self._L.sem_get_pcg_history(self._h, _np_ptr(h), n))
        return h

    def counts(self):
        v = [C.c_int64(0) for _ in range(4)]
        self._check(self._L.sem_get_counts(self._h, *[C.byref(x) for x in v]))
        return dict(nL=v[0].value, U=v[1].value, S=v[2].value, Us=v[3].value)

    def maps(self):
        c = self.counts()
        out = dict(l2u=np.empty(c["nL"], np.int32), mult=np.empty(c["U"], np.int32),
                   seg_off=np.empty(c["U"] + 1, np.int64), seg_idx=np.empty(c["nL"], np.int32),
                   uniq_gid=np.empty(c["U"], np.int64))
        self._check(self._L.sem_get_maps(self._h, _np_ptr(out["l2u"]), _np_ptr(out["mult"]), _np_ptr(out["seg_off"]),
                                         _np_ptr(out["seg_idx"]), _np_ptr(out["uniq_gid"])))
        return out

    def gll(self):
        p = self.p
        xi, rho, D = np.empty(p), np.empty(p), np.empty((p, p))
        self._check(self._L.sem_get_gll(self._h, _np_ptr(xi), _np_ptr(rho), _np_ptr(D)))
        return xi, rho, D

    def get_geom(self):
        nc = 7 if getattr(self, "with_mass", False) else 6
        G = np.empty((self.E, nc, self.p ** 3))
        dJ = np.empty((self.E, self.p ** 3))
        self._check(self._L.sem_get_geom(self._h, _np_ptr(G), _np_ptr(dJ)))
        return G, dJ

    def get_diag(self) -> np.ndarray:
        d = np.empty((self.E, self.p ** 3))
        self._check(self._L.sem_get_diag(self._h, _np_ptr(d)))
        return d


class Pmg:
    """p-multigrid V-cycle preconditioner over Sem contexts, finest first (sem_pmg_create ... sem_pmg_destroy)."""

    def __init__(self, levels, lmin, lmax, smooth_order: int = 2, coarse_order: int = 8, prec: int = SEM_F32):
        self._L = lib()
        self.levels = list(levels)                     # keep the contexts alive
        n = len(self.levels)
        h = C.c_void_p()
        arr = (C.c_void_p * n)(*[lv._h for lv in self.levels])
        lo, hi = (C.c_double * n)(*lmin), (C.c_double * n)(*lmax)
        rc = self._L.sem_pmg_create(C.byref(h), n, arr, lo, hi, smooth_order, coarse_order, prec)
        if rc != SEM_OK:
            raise SemError(rc, "; ".join(self._L.sem_last_error(lv._h).decode() for lv in self.levels))
        self._h = h

    def set_smoother(self, smoother: int, lmin=None, lmax=None):
        n = len(self.levels)
        lo = (C.c_double * n)(*lmin) if lmin is not None else None
        hi = (C.c_double * n)(*lmax) if lmax is not None else None
        rc = self._L.sem_pmg_set_smoother(self._h, smoother, lo, hi)
        if rc != SEM_OK:
            raise SemError(rc, "; ".join(self._L.sem_last_error(lv._h).decode() for lv in self.levels))
        return self

    def vcycle(self, r, z):
        rc = self._L.sem_pmg_vcycle(self._h, C.c_void_p(r.data_ptr()), C.c_void_p(z.data_ptr()))
        if rc != SEM_OK:
            raise SemError(rc, "; ".join(self._L.sem_last_error(lv._h).decode() for lv in self.levels))
        return z

    def fpcg(self, b, x, tol: float, maxit: int):
        it, rel = C.c_int(0), C.c_double(0.0)
        rc = self._L.sem_fpcg(self._h, C.c_void_p(b.data_ptr()), C.c_void_p(x.data_ptr()), tol, maxit, C.byref(it),
                              C.byref(rel))
        if rc != SEM_OK:
            raise SemError(rc, "; ".join(self._L.sem_last_error(lv._h).decode() for lv in self.levels))
        return it.value, rel.value

    def history(self, n: int) -> np.ndarray:
        h = np.full(n, np.nan)
        self._L.sem_pmg_get_history(self._h, _np_ptr(h), n)
        return h

    def close(self):
        if getattr(self, "_h", None):
            self._L.sem_pmg_destroy(self._h)
            self._h = None

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()


class Proj:
    """Projection onto previous solutions (sem_proj_create ... sem_proj_destroy) on one Sem context."""

    def __init__(self, sem: Sem, Lmax: int = 30):
        self._L, self.sem = lib(), sem
        h = C.c_void_p()
        rc = self._L.sem_proj_create(C.byref(h), sem._h, Lmax)
        if rc != SEM_OK:
            raise SemError(rc, self._L.sem_last_error(sem._h).decode())
        self._h = h

    def _chk(self, rc):
        if rc != SEM_OK:
            raise SemError(rc, self._L.sem_last_error(self.sem._h).decode())

    def guess(self, b, xbar, b_reduced):
        self._chk(self._L.sem_proj_guess(self._h, self.sem._vec(b), self.sem._vec(xbar), self.sem._vec(b_reduced)))
        return xbar, b_reduced

    def update(self, dx) -> bool:
        acc = C.c_int(0)
        self._chk(self._L.sem_proj_update(self._h, self.sem._vec(dx), C.byref(acc)))
        return bool(acc.value)

    def size(self) -> int:
        n = C.c_int(0)
        self._L.sem_proj_size(self._h, C.byref(n))
        return n.value

    def close(self):
        if getattr(self, "_h", None):
            self._L.sem_proj_destroy(self._h)
            self._h = None

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()
