"""Pins for the oracle's building blocks (CPU only): its FFT, its sphere<->box index maps, its Coulomb kernel.

Each check compares the oracle with something OTHER than itself: the O(N^2) definition, closed forms (delta, shift
theorem, Parseval), brute-force enumeration, textbook limits.  See DESIGN.md section 3 (pins).
"""
import math

import numpy as np
import pytest

from oracle import exx_ref as R
from paper_1111_0716_b200 import workloads as W

LENGTHS = [1, 2, 3, 4, 5, 6, 7, 9, 12, 16, 27, 48, 64, 96, 128]


def _rand(n, seed):
    rng = np.random.default_rng(seed)
    return rng.standard_normal(n) + 1j * rng.standard_normal(n)


@pytest.mark.parametrize("n", LENGTHS)
@pytest.mark.parametrize("sign", [-1, +1])
def test_fft1d_equals_naive_dft(n, sign):
    x = _rand(n, n)
    a, b = R.fft1d(x, sign), R.dft1d(x, sign)
    assert np.linalg.norm(a - b) <= 1e-14 * max(1.0, np.linalg.norm(b)) * math.log2(n + 1)


@pytest.mark.parametrize("n", [16, 48, 64, 96, 128])
def test_fft1d_closed_forms(n):
    # delta at j0  ->  exp(-/+ 2 pi i k j0 / n): fixes the sign convention and the index direction
    j0 = 5
    d = np.zeros(n, complex)
    d[j0] = 1.0
    k = np.arange(n)
    for sign in (-1, +1):
        want = np.exp(sign * 2j * np.pi * k * j0 / n)
        assert np.abs(R.fft1d(d, sign) - want).max() < 1e-14
        assert np.abs(R.dft1d(d, sign) - want).max() < 1e-14
    # constant -> n * delta_0
    c = R.fft1d(np.ones(n, complex), -1)
    assert abs(c[0] - n) < 1e-12 and np.abs(c[1:]).max() < 1e-12
    # Parseval and inverse(forward) = n * identity
    x = _rand(n, 100 + n)
    X = R.fft1d(x, -1)
    assert abs(np.vdot(X, X).real - n * np.vdot(x, x).real) < 1e-11 * n
    assert np.abs(R.fft1d(X, +1) - n * x).max() < 1e-12 * n


def test_fft3d_axes_layout_and_library():
    # non-cubic box: a plane wave exp(+i 2 pi (g.j/N)) must transform to Ng * delta at the folded index of g
    N = (4, 6, 3)
    g = (1, -2, 1)
    j = np.meshgrid(*[np.arange(n) for n in N], indexing="ij")
    box = np.exp(2j * np.pi * sum(g[i] * j[i] / N[i] for i in range(3)))
    F = R.fft3d(box, -1)
    want = np.zeros(N, complex)
    want[g[0] % N[0], g[1] % N[1], g[2] % N[2]] = np.prod(N)
    assert np.abs(F - want).max() < 1e-12
    # brute-force triple sum from the definition on random data
    x = _rand(np.prod(N), 7).reshape(N)
    Wm = [np.exp(-2j * np.pi * np.outer(np.arange(n), np.arange(n)) / n) for n in N]
    brute = np.einsum("ai,bj,ck,ijk->abc", Wm[0], Wm[1], Wm[2], x)
    assert np.abs(R.fft3d(x, -1) - brute).max() < 1e-12
    # and an independent library
    big = _rand(12 * 8 * 18, 3).reshape(12, 8, 18)
    assert np.abs(R.fft3d(big, -1) - np.fft.fftn(big)).max() < 1e-11
    assert np.abs(R.fft3d(big, +1) - np.fft.ifftn(big) * big.size).max() < 1e-11


# ----------------------------------------------------------------------------------------------------------------
def _brute_sphere(grid, lattice, kf, ecut):
    """Enumerate the whole box with numpy and test the inequality; returns (indices ascending, relative margin)."""
    B = 2 * np.pi * np.linalg.inv(np.asarray(lattice)).T
    fr = [np.where(2 * np.arange(n) < n, np.arange(n), np.arange(n) - n) for n in grid]
    g = np.stack(np.meshgrid(*fr, indexing="ij"), -1).astype(float) + np.asarray(kf)
    G = g @ B
    e = 0.5 * (G ** 2).sum(-1)
    return np.flatnonzero((e < ecut).ravel()), np.abs(e - ecut).min() / ecut


def _ctx(w):
    return R.RefExx(w.grid, w.lattice, w.kfrac, w.kweight, w.ecut, w.kernel_kind, w.mu, w.scale, w.nbands)


@pytest.mark.parametrize("name", ["C1", "C2", "C3"])
def test_index_map_brute_force(name):
    w = W.make(name)
    o = _ctx(w)
    for k in range(w.nk):
        want, margin = _brute_sphere(w.grid, w.lattice, w.kfrac[k], w.ecut)
        assert margin > 1e-9  # no vector close enough to the cutoff for rounding to decide (reading A11)
        m = o.index_map(k)
        assert m.dtype == np.int32
        assert np.array_equal(m, want)
        assert np.all(np.diff(m) > 0)


def test_index_map_noncubic_kpoint_brute_force():
    lat = W.rhombohedral(7.3, 71.0)
    kf = np.array([[0.1, -0.3, 0.25], [0.5, 0.0, 0.0]])
    o = R.RefExx((12, 18, 16), lat, kf, [0.5, 0.5], 9.0, nbands=2)
    for k in range(2):
        want, margin = _brute_sphere((12, 18, 16), lat, kf[k], 9.0)
        assert margin > 1e-9
        assert np.array_equal(o.index_map(k), want)


def test_index_map_counts_and_checksums():
    # counts and checksums tabulated in SURVEY.md section 8(a)/(c)-PINS (survey probe, numpy)
    expect = {"C1": ([739], 1402128), "C2": ([1580, 1632, 1632, 1632, 1632, 1632, 1632, 1580], 77343110),
              "C3": ([15895], 2015122368), "C4a": ([15465], None), "C5": ([40651], None)}
    for name, (npw, chk) in expect.items():
        w = W.make(name)
        o = _ctx(w)
        assert o.npw == npw
        if chk is not None:
            assert int(o.index_map(0).astype(np.int64).sum()) == chk
        # sphere-volume estimate Omega (2 Ecut)^{3/2} / (6 pi^2): lattice-point discrepancy ~ surface/volume
        est = o.omega * (2 * w.ecut) ** 1.5 / (6 * np.pi ** 2)
        assert abs(o.npw[0] - est) / est < (0.06 if est < 5000 else 0.01)
        # inversion symmetry at Gamma: g in sphere <=> -g in sphere
        if np.all(w.kfrac[0] == 0):
            m = o.index_map(0).astype(np.int64)
            N = w.grid
            j1, j2, j3 = m // (N[1] * N[2]), (m // N[2]) % N[1], m % N[2]
            inv = (((-j1) % N[0]) * N[1] + ((-j2) % N[1])) * N[2] + ((-j3) % N[2])
            assert np.array_equal(np.sort(inv), m)
        o.close()


def test_psi_offsets_and_mp_mesh():
    w = W.make("C2")
    o = _ctx(w)
    assert o.offsets[0] == 0 and o.offsets[-1] == w.nbands * sum(o.npw)
    assert np.allclose(w.kfrac[0], [-0.25, -0.25, -0.25]) and np.allclose(w.kfrac[1], [-0.25, -0.25, 0.25])
    assert np.allclose(w.kfrac[-1], [0.25, 0.25, 0.25]) and abs(w.kweight.sum() - 1) < 1e-15
    # rhombohedral cell: |a_i| = a, a_i.a_j = a^2 cos(alpha), volume a^3 sqrt(1 - 3c^2 + 2c^3)
    A = w.lattice
    c = math.cos(math.radians(58.0))
    assert np.allclose(A @ A.T, 9.55 ** 2 * (np.full((3, 3), c) + (1 - c) * np.eye(3)), atol=1e-12)
    assert abs(o.omega - 9.55 ** 3 * math.sqrt(1 - 3 * c * c + 2 * c ** 3)) < 1e-10
    assert abs(o.omega - 587.624) < 1e-3
    # reciprocal rows: a_i . b_j = 2 pi delta_ij
    assert np.allclose(A @ o.recip().T, 2 * np.pi * np.eye(3), atol=1e-13)


# ----------------------------------------------------------------------------------------------------------------
def test_kernel_bare_closed_form_cubic():
    a = 10.0
    o = R.RefExx((16,) * 3, W.cubic(a), np.zeros((1, 3)), [1.0], 6.0, kind=0, nbands=1)
    K = o.kernel_table(0, 0)
    assert K[0, 0, 0] == 0.0                                   # bare: q+G = 0 term := 0 (reading A6)
    # cubic: G = (2 pi / a) g  =>  4 pi / G^2 = a^2 / (pi |g|^2)
    assert abs(K[1, 0, 0] - a * a / np.pi) < 1e-12
    assert abs(K[0, 15, 0] - a * a / np.pi) < 1e-12             # index 15 is g = -1
    assert abs(K[2, 14, 3] - a * a / (np.pi * (4 + 4 + 9))) < 1e-12
    assert abs(K[8, 0, 0] - a * a / (np.pi * 64)) < 1e-12       # Nyquist index N/2 <-> g = -N/2
    assert np.all(K >= 0)


def test_kernel_hse_limits_and_bounds():
    mu = 0.106
    a = 20.0
    o = R.RefExx((64,) * 3, W.cubic(a), np.zeros((1, 3)), [1.0], 12.0, kind=1, mu=mu, nbands=1)
    ob = R.RefExx((64,) * 3, W.cubic(a), np.zeros((1, 3)), [1.0], 12.0, kind=0, nbands=1)
    K, Kb = o.kernel_table(0, 0), ob.kernel_table(0, 0)
    assert abs(K[0, 0, 0] - np.pi / mu ** 2) < 1e-12 * np.pi / mu ** 2   # finite limit kept (reading A6)
    mask = np.ones(K.shape, bool)
    mask[0, 0, 0] = False
    assert np.all(K[mask] > 0) and np.all(K[mask] <= Kb[mask])      # equal only once exp(-x) < 2^-53
    assert np.all(K[:3, :3, :3][mask[:3, :3, :3]] < Kb[:3, :3, :3][mask[:3, :3, :3]])
    # against the formula in extended precision
    g2 = ((2 * np.pi / a) ** 2) * np.array([1.0, 2.0, 3.0, 1024 * 3.0], dtype=np.longdouble)
    want = 4 * np.pi / g2 * (1 - np.exp(-g2 / (4 * np.longdouble(mu) ** 2)))
    got = np.array([K[1, 0, 0], K[1, 1, 0], K[1, 1, 1], K[32, 32, 32]])
    assert np.abs(got - want.astype(float)).max() / want.max() < 1e-15
    # Q -> infinity: bare; Q -> 0 (huge cell): (pi/mu^2)(1 - x/2), x = Q^2 / 4 mu^2
    assert abs(K[32, 32, 32] / Kb[32, 32, 32] - 1) < 1e-12
    big = R.RefExx((4,) * 3, W.cubic(1.0e5), np.zeros((1, 3)), [1.0], 1e-6, kind=1, mu=mu, nbands=1)
    Kbig = big.kernel_table(0, 0)
    x = (2 * np.pi / 1.0e5) ** 2 / (4 * mu * mu)
    assert abs(Kbig[1, 0, 0] / (np.pi / mu ** 2) - (1 - x / 2)) < 1e-12


def test_kernel_kpoint_shift_and_scale():
    w = W.make("C2")
    o = R.RefExx(w.grid, w.lattice, w.kfrac, w.kweight, w.ecut, 0, 0.0, 0.25, w.nbands)
    B = 2 * np.pi * np.linalg.inv(w.lattice).T
    K = o.kernel_table(7, 0)                     # kappa_7 - kappa_0 = (1/2, 1/2, 1/2)
    for idx, g in (((0, 0, 0), (0, 0, 0)), ((47, 1, 24), (-1, 1, -24)), ((3, 40, 2), (3, -8, 2))):
        Q = (np.array(g) + 0.5) @ B
        assert abs(K[idx] - 0.25 * 4 * np.pi / (Q @ Q)) < 1e-13 * K[idx]
    K00 = o.kernel_table(3, 3)
    assert K00[0, 0, 0] == 0.0 and np.all(K > 0)
    # K_{kq}(g) = K_{qk}(-g) off the Nyquist planes
    Kqk = o.kernel_table(0, 7)
    assert abs(K[3, 40, 2] - Kqk[45, 8, 46]) < 1e-15 * K[3, 40, 2]


def test_create_errors():
    lat = W.cubic(5.0)
    k, wt = np.zeros((1, 3)), [1.0]
    with pytest.raises(R.ExxRefError):
        R.RefExx((8, 8, 8), np.zeros((3, 3)), k, wt, 5.0)
    with pytest.raises(R.ExxRefError):
        R.RefExx((8, 8, 8), lat, k, wt, -1.0)
    with pytest.raises(R.ExxRefError):
        R.RefExx((8, 8, 8), lat, k, wt, 5.0, kind=3)
    with pytest.raises(R.ExxRefError):
        R.RefExx((8, 8, 8), lat, k, wt, 5.0, kind=1, mu=0.0)
    o = R.RefExx((8, 8, 8), lat, k, wt, 5.0, nbands=2)
    psi = W.custom("t", 1, (8, 8, 8), lat, k, wt, 5.0, 2, [1, 1]).coefficients(o.npw)
    with pytest.raises(R.ExxRefError):
        o.apply(psi, [1.0, -0.5])
    with pytest.raises(R.ExxRefError):
        o.apply(psi, [1.0, float("nan")])
