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
