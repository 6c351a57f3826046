"""CPU-only checks of the boundary: libexx.so builds/loads and exports every symbol include/exx.h declares,
argument validation that needs no GPU, and the workload recipe.  No compute calls here."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from paper_1111_0716_b200 import binding as B
from paper_1111_0716_b200 import build as build_mod
from paper_1111_0716_b200 import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def L():
    build_mod.build()
    return B.lib()


def test_header_symbols_are_exported(L):
    hdr = open(os.path.join(ROOT, "include", "exx.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(exx_[a-z0-9_]+)\s*\(", hdr))
    assert declared == set(B.SYMBOLS), declared ^ set(B.SYMBOLS)
    for s in declared:
        assert hasattr(L, s), s
    assert L.exx_version() >= 100


def test_strerror_and_class_names(L):
    for code in range(0, -11, -1):
        assert L.exx_strerror(code)
    assert L.exx_strerror(-99) == b"unknown error"
    names = [L.exx_kernel_class_name(k) for k in range(13)]
    assert all(names) and L.exx_kernel_class_name(13) is None and L.exx_kernel_class_name(-1) is None


def test_create_rejects_bad_arguments_before_touching_the_gpu(L):
    h = C.c_void_p()
    lat = np.ascontiguousarray(W.cubic(10.0).reshape(9))
    k = np.zeros(3)
    w = np.ones(1)
    kp = B.KernelParams(0, 0.0, 1.0)

    def create(grid=(16, 16, 16), lattice=lat, ecut=6.0, kparams=kp, nk=1, nb=2):
        g = (C.c_int * 3)(*grid)
        return L.exx_create(C.byref(h), g, B._dp(lattice), nk, B._dp(k), B._dp(w), ecut, C.byref(kparams), nb, None)

    assert create(grid=(16, 16, 14)) == -2          # 14 = 2*7
    assert create(grid=(16, 1, 16)) == -2
    assert create(grid=(2048, 16, 16)) == -2
    assert create(lattice=np.zeros(9)) == -3
    assert create(ecut=0.0) == -4
    assert create(ecut=float("nan")) == -4
    assert create(kparams=B.KernelParams(2, 0.0, 1.0)) == -5
    assert create(kparams=B.KernelParams(1, 0.0, 1.0)) == -5
    assert create(kparams=B.KernelParams(0, 0.0, float("inf"))) == -5
    assert create(nk=0) == -9
    assert create(nb=0) == -9
    assert L.exx_create(None, None, None, 1, None, None, 1.0, None, 1, None) == -1
    assert not h.value                                # *out untouched on error
    assert L.exx_destroy(None) == -1
    n = C.c_int(7)
    assert L.exx_npw(None, 0, C.byref(n)) == -1 and n.value == 7


def test_build_refuses_code_changing_flags_for_the_stamped_library():
    """libexx.so carries the hash of the standard flags, so build() without out= accepts only ptxas verbosity as an extra."""
    for extra in (["-Xptxas=-O0"], ["-Xptxas", "-O0"], ["-DEXX_DEFAULT_TILE=16"], ["-Xptxas", "-v", "-G"]):
        with pytest.raises(ValueError):
            build_mod.build(extra=extra)
    assert build_mod.build(extra=["-Xptxas", "-v"]) == build_mod.LIB      # up to date: returns without compiling


def test_workload_recipe():
    w = W.make("C4b")
    assert w.nk == 8 and w.nbands == 160 and w.nocc == 160 and w.pair_evals == 1638400
    assert W.make("C2").pair_evals == 27648 and W.make("C5").pair_evals == 65536 and W.make("C4a").pair_evals == 25600
    c = W.make("C1").coefficients([739])
    assert c.shape == (8 * 739,) and c.dtype == np.complex128
    assert np.allclose((np.abs(c.reshape(8, 739)) ** 2).sum(1), 1.0)
    assert np.array_equal(c, W.make("C1").coefficients([739]))      # seeded, reproducible
