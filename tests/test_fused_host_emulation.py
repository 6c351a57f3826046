"""Host-logic test (no GPU): the fused passes' per-thread phases (csrc/exx_fused_phases.h) and the in-register DFT
codelets (csrc/exx_dft.h) are __host__ __device__ code; csrc/exx_host_emu.cpp runs them on the CPU thread by thread and
tile by tile in the order exx_fused.cu launches them.  Compared here with numpy.fft (a library routine, independent of
the product): this checks the index maps of the two-step transforms, the shared-memory layouts, the permuted kernel
table and the accumulation — everything about the kernels except the device-side barriers and memory system.
"""
import ctypes as C
import os
import subprocess

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
SRC = os.path.join(ROOT, "paper_1111_0716_b200", "csrc", "exx_host_emu.cpp")
dp = C.POINTER(C.c_double)


@pytest.fixture(scope="module")
def emu(tmp_path_factory):
    so = str(tmp_path_factory.mktemp("emu") / "libexx_emu.so")
    subprocess.check_call(["g++", "-O2", "-std=c++17", "-fPIC", "-shared", "-ffp-contract=off", "-o", so, SRC])
    L = C.CDLL(so)
    L.exx_emu_dft.argtypes = [C.c_int, C.c_int, dp]
    L.exx_emu_pair.argtypes = [C.c_int, dp, dp, dp, C.c_double, dp, dp]
    L.exx_emu_pair_energy.argtypes = [C.c_int, dp, dp, dp, dp, dp]
    up = C.POINTER(C.c_uint32)
    L.exx_emu_dual.argtypes = [C.c_int, C.c_int, C.c_int, dp, dp, dp, dp, dp, up, up, C.c_uint32, dp, dp]
    return L


def _p(a):
    return a.ctypes.data_as(dp)


@pytest.mark.parametrize("R", [2, 3, 4, 5, 6, 8, 9, 10, 12, 16])
@pytest.mark.parametrize("sign", [-1, 1])
def test_codelets_against_numpy(emu, R, sign):
    rng = np.random.default_rng(100 * R + sign)
    x = rng.standard_normal(R) + 1j * rng.standard_normal(R)
    v = x.copy()
    assert emu.exx_emu_dft(R, sign, _p(v)) == 0
    want = np.fft.fft(x) if sign < 0 else np.fft.ifft(x) * R
    assert np.linalg.norm(v - want) <= 1e-15 * R * np.linalg.norm(want)
    # delta -> constant, constant -> delta (exact)
    d = np.zeros(R, dtype=np.complex128)
    d[0] = 1.0
    emu.exx_emu_dft(R, sign, _p(d))
    assert np.array_equal(d, np.ones(R))


@pytest.mark.parametrize("R1", [2, 4, 5, 6, 8, 9, 10, 12, 16])
def test_three_passes_equal_definition(emu, R1):
    """acc += -w f u_m IFFT[K' FFT[conj(u_m) u_n]] (unnormalised transforms), one pair, whole box."""
    N = 8 * R1
    rng = np.random.default_rng(R1)
    shp = (N, N, N)
    un = rng.standard_normal(shp) + 1j * rng.standard_normal(shp)
    um = rng.standard_normal(shp) + 1j * rng.standard_normal(shp)
    K = rng.random(shp)  # any real table: an asymmetric one catches transposed / mirrored frequency indices
    acc0 = rng.standard_normal(shp) + 1j * rng.standard_normal(shp)
    acc, work = acc0.copy(), np.zeros(shp, dtype=np.complex128)
    wf = 0.7
    assert emu.exx_emu_pair(R1, _p(un), _p(um), _p(K), wf, _p(acc), _p(work)) == 0
    want = -wf * um * np.fft.ifftn(K * np.fft.fftn(np.conj(um) * un)) * N ** 3
    assert np.linalg.norm(acc - acc0 - want) <= 1e-14 * np.linalg.norm(want)


@pytest.mark.parametrize("R1", [2, 4, 5, 6, 8, 9, 10, 12, 16])
def test_energy_route_equals_definition(emu, R1):
    """sum_g K(g) |FFT[conj(u_m) u_n](g)|^2 for one pair (passes A, forward B, p2_x8_energy) against numpy.fft."""
    N = 8 * R1
    rng = np.random.default_rng(1000 + R1)
    shp = (N, N, N)
    un = rng.standard_normal(shp) + 1j * rng.standard_normal(shp)
    um = rng.standard_normal(shp) + 1j * rng.standard_normal(shp)
    K = rng.random(shp)  # asymmetric real table: a mirrored or transposed frequency index changes the sum
    work = np.zeros(shp, dtype=np.complex128)
    e = np.zeros(1)
    assert emu.exx_emu_pair_energy(R1, _p(un), _p(um), _p(K), _p(work), _p(e)) == 0
    want = float((K * np.abs(np.fft.fftn(np.conj(um) * un)) ** 2).sum())
    assert abs(e[0] - want) <= 1e-13 * want


def test_single_plane_wave_pair(emu):
    """u_n = e^{i g_n.r}, u_m = e^{i g_m.r}: the pair density is one plane wave, so the result is K'(g_n-g_m) Ng u_n."""
    R1 = 6
    N = 8 * R1
    j = np.arange(N)
    def pw(g):
        return np.exp(2j * np.pi * (g[0] * j[:, None, None] + g[1] * j[None, :, None] + g[2] * j[None, None, :]) / N)
    gn, gm = (3, -2, 5), (1, 4, -7)
    K = np.random.default_rng(5).random((N, N, N))
    acc, work = np.zeros((N, N, N), dtype=np.complex128), np.zeros((N, N, N), dtype=np.complex128)
    un, um = pw(gn), pw(gm)
    assert emu.exx_emu_pair(R1, _p(un), _p(um), _p(K), 1.0, _p(acc), _p(work)) == 0
    d = [(a - b) % N for a, b in zip(gn, gm)]
    want = -K[d[0], d[1], d[2]] * N ** 3 * un
    assert np.abs(acc - want).max() <= 1e-12 * N ** 3


@pytest.mark.parametrize("R1", [2, 4, 5, 6, 8, 9, 10, 12])
def test_plain_transforms_through_the_passes(emu, R1):
    """S1/S7 use the fused passes as plain 3-D transforms: forward natural -> F layout, inverse F layout -> natural."""
    N = 8 * R1
    emu.exx_emu_fft.argtypes = [C.c_int, C.c_int, dp, dp, C.POINTER(C.c_int64)]
    rng = np.random.default_rng(40 + R1)
    x = rng.standard_normal((N, N, N)) + 1j * rng.standard_normal((N, N, N))
    fidx = np.empty(N ** 3, dtype=np.int64)
    out = np.zeros(N ** 3, dtype=np.complex128)
    assert emu.exx_emu_fft(R1, -1, _p(x.copy()), _p(out), fidx.ctypes.data_as(C.POINTER(C.c_int64))) == 0
    assert np.array_equal(np.sort(fidx), np.arange(N ** 3))      # findex is a permutation of the box
    want = np.fft.fftn(x).reshape(-1)
    assert np.linalg.norm(out[fidx] - want) <= 1e-14 * np.linalg.norm(want)
    # inverse: scatter natural-order coefficients through findex, transform back
    y = rng.standard_normal((N, N, N)) + 1j * rng.standard_normal((N, N, N))
    f = np.zeros(N ** 3, dtype=np.complex128)
    f[fidx] = y.reshape(-1)
    back = np.zeros(N ** 3, dtype=np.complex128)
    assert emu.exx_emu_fft(R1, +1, _p(f), _p(back), None) == 0
    want = np.fft.ifftn(y).reshape(-1) * N ** 3
    assert np.linalg.norm(back - want) <= 1e-14 * np.linalg.norm(want)


@pytest.mark.parametrize("R1,ta,tb", [(2, 5, 3), (4, 6, 4), (5, 3, 3), (6, 5, 2), (9, 5, 2), (10, 3, 2)])
def test_dual_sweep_equals_definition(emu, R1, ta, tb):
    """The dual sweep of pass C (pair symmetry) on a ragged ta x tb batch with holes: rows get
    acc_a -= sum_j coef_b[j] u_b[j] v_ij, columns get acc_b -= sum_i coef_a[i] u_a[i] conj(v_ij), v_ij = IFFT[K FFT[conj(u_b[j]) u_a[i]]],
    against numpy.fft.  Masks as the host builds them: a pair may be skipped altogether, feed one side only, or both."""
    N = 8 * R1
    rng = np.random.default_rng(7000 + R1)
    shp = (N, N, N)
    ua = rng.standard_normal((ta,) + shp) + 1j * rng.standard_normal((ta,) + shp)
    ub = rng.standard_normal((tb,) + shp) + 1j * rng.standard_normal((tb,) + shp)
    K = rng.random(shp)
    coef_a, coef_b = rng.random(ta) + 0.1, rng.random(tb) + 0.1
    coef_b[tb - 1] = 0.0                                   # an empty b-band: no side a for that column
    coef_a[1] = 0.0                                        # an empty a-band: no side b for that row
    ev = np.zeros(ta, dtype=np.uint32)
    bside = np.zeros(ta, dtype=np.uint32)
    amask = 0
    for j in range(tb):
        if coef_b[j] != 0.0:
            amask |= 1 << j
    for i in range(ta):
        for j in range(tb):
            if (i, j) == (2, 0):
                continue                                   # a pair that is not evaluated at all
            sa, sb = coef_b[j] != 0.0, coef_a[i] != 0.0 and (i, j) != (0, 1)   # (0, 1): a "diagonal" pair, side a only
            if sa or sb:
                ev[i] |= 1 << j
            if sb:
                bside[i] |= 1 << j
    acc_a0 = rng.standard_normal((ta,) + shp) + 1j * rng.standard_normal((ta,) + shp)
    acc_b0 = rng.standard_normal((tb,) + shp) + 1j * rng.standard_normal((tb,) + shp)
    acc_a, acc_b = acc_a0.copy(), acc_b0.copy()
    up = C.POINTER(C.c_uint32)
    rc = emu.exx_emu_dual(R1, ta, tb, _p(ua), _p(ub), _p(K), _p(coef_a), _p(coef_b), ev.ctypes.data_as(up), bside.ctypes.data_as(up),
                          amask, _p(acc_a), _p(acc_b))
    if rc == -2:
        pytest.skip("no dual kernel for this grid (FusedCfg<R1>::RG = 0: two single sweeps)")
    assert rc == 0
    want_a, want_b = np.zeros_like(acc_a), np.zeros_like(acc_b)
    for i in range(ta):
        for j in range(tb):
            if not (ev[i] >> j) & 1:
                continue
            v = np.fft.ifftn(K * np.fft.fftn(np.conj(ub[j]) * ua[i])) * N ** 3
            if (amask >> j) & 1:
                want_a[i] -= coef_b[j] * ub[j] * v
            if (bside[i] >> j) & 1:
                want_b[j] -= coef_a[i] * ua[i] * np.conj(v)
    assert np.linalg.norm(acc_a - acc_a0 - want_a) <= 1e-14 * np.linalg.norm(want_a)
    assert np.linalg.norm(acc_b - acc_b0 - want_b) <= 1e-14 * np.linalg.norm(want_b)
