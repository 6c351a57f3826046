"""Pins for the oracle's V_x application and E_x (CPU only).

Nothing here compares the oracle with a re-typing of its own formula: the checks are the closed form for
single-plane-wave bands (BASELINE.json north_star), operator identities (Hermiticity, gauge covariance, unitary
covariance), two independent evaluation routes (E1 vs E2; FFT vs explicit cyclic convolution), a supercell that must
reproduce k-point sampling, and the Hartree energy of a single orbital.  See DESIGN.md section 3.
"""
import numpy as np
import pytest

from oracle import exx_ref as R
from paper_1111_0716_b200 import workloads as W


def _ctx(w):
    return R.RefExx(w.grid, w.lattice, w.kfrac, w.kweight, w.ecut, w.kernel_kind, w.mu, w.scale, w.nbands)


def _small(seed=5, grid=(12, 12, 12), nb=5, occ=(1.0, 1.0, 0.5, 0.25, 0.0), kind=0, mu=0.0, kpts=False, ecut=4.0, scale=1.0):
    lat = W.rhombohedral(6.0, 63.0)
    if kpts:
        kf = np.array([[0.0, 0.0, 0.0], [0.5, 0.0, 0.0], [0.25, -0.25, 0.125]])
        kw = np.array([0.5, 0.25, 0.25])
    else:
        kf, kw = np.zeros((1, 3)), np.ones(1)
    w = W.custom("small", seed, grid, lat, kf, kw, ecut, nb, occ, kind, mu, scale)
    o = _ctx(w)
    return w, o, w.coefficients(o.npw)


def _plane_wave_bands(o, ik_list, g_list):
    """psi holding one plane wave per band: band n of k-point ik has c = delta_{g, g_n}.  Bands not listed stay 0."""
    N = o.grid
    psi = np.zeros(o.ncoef, complex)
    for (ik, n), g in zip(ik_list, g_list):
        lin = ((g[0] % N[0]) * N[1] + (g[1] % N[1])) * N[2] + (g[2] % N[2])
        m = o.index_map(ik)
        pos = np.searchsorted(m, lin)
        assert m[pos] == lin, "plane wave outside the sphere"
        o.band(psi, ik, n)[pos] = 1.0
    return psi


def test_closed_form_single_plane_waves_gamma():
    # BASELINE.json north_star: E_x = -(1/2)(1/Omega) sum f_n f_m 4 pi / |G_n - G_m|^2, zero terms skipped.
    gs = [(0, 0, 0), (1, 0, 0), (0, 2, 0), (-1, 1, 3), (2, -2, 1)]
    f = np.array([1.0, 1.0, 0.5, 1.0, 0.25])
    o = R.RefExx((16,) * 3, W.cubic(10.0), np.zeros((1, 3)), [1.0], 6.0, nbands=5)
    psi = _plane_wave_bands(o, [(0, n) for n in range(5)], gs)
    out = o.apply(psi, f)
    B = 2 * np.pi * np.linalg.inv(W.cubic(10.0)).T
    lam = np.zeros(5)
    for i, a in enumerate(gs):
        for j, b in enumerate(gs):
            d = (np.array(a) - np.array(b)) @ B
            if d @ d > 0:
                lam[i] -= f[j] * 4 * np.pi / (d @ d) / o.omega
    ecf = 0.5 * float(f @ lam)
    e1, per_band = o.energy(psi, f, out)
    e2 = o.energy_e2(psi, f)
    assert abs(ecf - (-0.04836886372955853)) < 1e-15          # value recorded in SURVEY.md section 8(c)-PINS
    assert abs(e1 - ecf) < 1e-15 and abs(e2 - ecf) < 1e-15
    # plane waves are eigenvectors: V_x c_n = lambda_n c_n with lambda_n = -(1/Omega) sum_m f_m K(G_n - G_m)
    for n in range(5):
        assert np.abs(o.band(out, 0, n) - lam[n] * o.band(psi, 0, n)).max() < 1e-16
        assert abs(per_band[n] - 0.5 * f[n] * lam[n]) < 1e-16


def test_closed_form_plane_waves_with_kpoints_and_hse():
    # bands at different k: E_x = -(1/2 Omega) sum w_k w_q f f K(|k_n + G_n - k_m - G_m|), K = HSE, scale 0.25
    lat = W.rhombohedral(8.0, 60.0)
    kf = np.array([[0.0, 0.0, 0.0], [0.25, 0.25, -0.25]])
    kw = np.array([0.75, 0.25])
    mu = 0.3
    o = R.RefExx((12, 12, 12), lat, kf, kw, 5.0, kind=1, mu=mu, scale=0.25, nbands=2)
    bands = [(0, 0), (0, 1), (1, 0), (1, 1)]
    gs = [(0, 0, 0), (1, -1, 0), (0, 1, 1), (-1, 0, 0)]
    occ = np.array([1.0, 0.5, 1.0, 0.3])
    psi = _plane_wave_bands(o, bands, gs)
    out = o.apply(psi, occ)
    B = 2 * np.pi * np.linalg.inv(lat).T
    ecf = 0.0
    for i, (ki, ni) in enumerate(bands):
        for j, (kj, nj) in enumerate(bands):
            t = kf[ki] + np.array(gs[i]) - kf[kj] - np.array(gs[j])
            q2 = (t @ B) @ (t @ B)
            K = 0.25 * (np.pi / mu ** 2 if not t.any() else 4 * np.pi / q2 * (1 - np.exp(-q2 / (4 * mu * mu))))
            ecf += -0.5 / o.omega * kw[ki] * kw[kj] * occ[i] * occ[j] * K
    e1, _ = o.energy(psi, occ, out)
    assert abs(e1 - ecf) < 2e-15 * abs(ecf) + 1e-17
    assert abs(o.energy_e2(psi, occ) - ecf) < 2e-15 * abs(ecf) + 1e-17


@pytest.mark.parametrize("kpts", [False, True])
@pytest.mark.parametrize("kind", [0, 1])
def test_hermiticity_sign_and_two_energy_routes(kpts, kind):
    w, o, psi = _small(kpts=kpts, kind=kind, mu=0.25)
    out = o.apply(psi, w.occ)
    for k in range(w.nk):
        c = np.array([o.band(psi, k, n) for n in range(w.nbands)])
        v = np.array([o.band(out, k, n) for n in range(w.nbands)])
        M = c.conj() @ v.T                                # M_ij = <c_i | V_x c_j>
        assert np.abs(M - M.conj().T).max() < 1e-15 * max(1.0, np.abs(M).max())
        assert np.all(np.linalg.eigvalsh(0.5 * (M + M.conj().T)) < 1e-14)   # V_x is negative semi-definite
    e1, per_band = o.energy(psi, w.occ, out)
    e2 = o.energy_e2(psi, w.occ)
    assert e1 < 0 and np.all(per_band <= 1e-18)
    assert abs(e1 - e2) < 1e-14 * abs(e1)
    assert abs(per_band.sum() - e1) < 1e-15
    assert np.all(per_band[w.occ == 0] == 0)
    # unoccupied bands (f = 0) still get a V_x row (reading A16)
    assert np.linalg.norm(o.band(out, 0, w.nbands - 1)) > 0


def test_gauge_and_unitary_covariance():
    w, o, psi = _small(occ=(1.0, 1.0, 1.0, 0.5, 0.0), kpts=True)
    out = o.apply(psi, w.occ)
    e1, _ = o.energy(psi, w.occ, out)
    # common global phase
    ph = np.exp(0.7j)
    out2 = o.apply(psi * ph, w.occ)
    assert np.abs(out2 - ph * out).max() < 1e-16
    assert abs(o.energy(psi * ph, w.occ, out2)[0] - e1) < 1e-16
    # independent phases per band: V_x (e^{i t_n} c_n) = e^{i t_n} V_x c_n, E_x unchanged
    psi3, want3 = psi.copy(), out.copy()
    for k in range(w.nk):
        for n in range(w.nbands):
            p = np.exp(1j * (0.3 + k + 2.1 * n))
            o.band(psi3, k, n)[:] *= p
            o.band(want3, k, n)[:] *= p
    out3 = o.apply(psi3, w.occ)
    assert np.abs(out3 - want3).max() < 1e-16
    # unitary mix among the three equally occupied bands (same U at every k): out -> U out, E_x unchanged
    rng = np.random.default_rng(2)
    U, _ = np.linalg.qr(rng.standard_normal((3, 3)) + 1j * rng.standard_normal((3, 3)))
    psi4, want4 = psi.copy(), out.copy()
    for k in range(w.nk):
        c = np.array([o.band(psi, k, n) for n in range(3)])
        v = np.array([o.band(out, k, n) for n in range(3)])
        for n in range(3):
            o.band(psi4, k, n)[:] = U[n] @ c
            o.band(want4, k, n)[:] = U[n] @ v
    out4 = o.apply(psi4, w.occ)
    assert np.abs(out4 - want4).max() < 1e-15
    assert abs(o.energy(psi4, w.occ, out4)[0] - e1) < 1e-15


def test_fft_path_equals_no_fft_path_on_C1():
    # C1 is aliased by construction (needs 21 grid points, has 16): the no-FFT route must be cyclic to agree.
    w = W.make("C1")
    o = _ctx(w)
    psi = w.coefficients(o.npw)
    a, b = o.apply(psi, w.occ), o.apply_direct(psi, w.occ)
    for n in range(w.nbands):
        assert np.linalg.norm(o.band(a, 0, n) - o.band(b, 0, n)) < 1e-13 * np.linalg.norm(o.band(b, 0, n))


def test_fft_path_equals_no_fft_path_kpoints_noncubic():
    lat = W.rhombohedral(5.0, 66.0)
    kf = np.array([[0.0, 0.0, 0.0], [0.5, 0.25, -0.25]])
    w = W.custom("k", 9, (6, 8, 9), lat, kf, [0.6, 0.4], 3.5, 3, [1.0, 0.5, 0.0], kernel_kind=1, mu=0.4)
    o = _ctx(w)
    psi = w.coefficients(o.npw)
    a, b = o.apply(psi, w.occ), o.apply_direct(psi, w.occ)
    assert np.linalg.norm(a - b) < 1e-13 * np.linalg.norm(b)


def test_apply_rows_equals_apply_and_to_real():
    w, o, psi = _small(kpts=True)
    full = o.apply(psi, w.occ)
    rows = [(2, 4), (0, 0), (1, 3)]
    got = o.apply_rows(psi, w.occ, rows)
    for (k, n), r in zip(rows, got):
        assert np.abs(r - o.band(full, k, n)).max() < 1e-16
    # u_nk(r_j) against the explicit plane-wave sum at a few grid points
    m = o.index_map(1)
    N = o.grid
    c = o.band(psi, 1, 2)
    u = o.to_real(1, c)
    j1, j2, j3 = m // (N[1] * N[2]), (m // N[2]) % N[1], m % N[2]
    for j in ((0, 0, 0), (1, 2, 3), (11, 5, 7)):
        want = (c * np.exp(2j * np.pi * (j1 * j[0] / N[0] + j2 * j[1] / N[1] + j3 * j[2] / N[2]))).sum()
        assert abs(u[j] - want) < 1e-13


def test_single_orbital_exchange_is_minus_hartree():
    # one occupied band: E_x = -E_H[|u|^2], E_H = (1/2 Omega) sum_g K(g) |n~(g)|^2, n~ = FFT(|u|^2)/Ng  (numpy FFT)
    w, o, psi = _small(nb=2, occ=(1.0, 0.0), grid=(16, 16, 16), ecut=3.0)
    u = o.to_real(0, o.band(psi, 0, 0))
    nt = np.fft.fftn(np.abs(u) ** 2) / u.size
    eh = 0.5 / o.omega * (o.kernel_table(0, 0) * np.abs(nt) ** 2).sum()
    out = o.apply(psi, w.occ)
    assert abs(o.energy(psi, w.occ, out)[0] + eh) < 1e-15


def test_supercell_reproduces_kpoint_sampling():
    # 2x1x1 supercell at Gamma holding the bands of kappa in {(0,0,0), (1/2,0,0)}, w = 1/2 each:
    # coefficient map g' = (2 g_1 + 2 kappa_1, g_2, g_3); E_x(super) = 2 E_x(prim); V_x rows map one to one.
    lat = W.rhombohedral(6.0, 63.0)
    N = (12, 12, 12)
    kf = np.array([[0.0, 0.0, 0.0], [0.5, 0.0, 0.0]])
    nb, occ = 2, np.array([1.0, 0.5])
    wp = W.custom("prim", 21, N, lat, kf, [0.5, 0.5], 4.0, nb, occ)
    op = _ctx(wp)
    psi = wp.coefficients(op.npw)
    outp = op.apply(psi, wp.occ)
    ep, _ = op.energy(psi, wp.occ, outp)

    lat2 = lat.copy()
    lat2[0] *= 2
    N2 = (24, 12, 12)
    os_ = R.RefExx(N2, lat2, np.zeros((1, 3)), [1.0], 4.0, nbands=2 * nb)
    assert os_.npw[0] == op.npw[0] + op.npw[1]
    ms = os_.index_map(0)
    psis = np.zeros(os_.ncoef, complex)
    pos_of = {}
    for k in range(2):
        m = op.index_map(k).astype(np.int64)
        j1, j2, j3 = m // (N[1] * N[2]), (m // N[2]) % N[1], m % N[2]
        g1 = np.where(2 * j1 < N[0], j1, j1 - N[0])
        g1s = 2 * g1 + int(round(2 * kf[k, 0]))
        lin = ((g1s % N2[0]) * N2[1] + j2) * N2[2] + j3
        pos = np.searchsorted(ms, lin)
        assert np.array_equal(ms[pos], lin)
        pos_of[k] = pos
        for n in range(nb):
            os_.band(psis, 0, k * nb + n)[pos] = op.band(psi, k, n)
    occs = np.tile(occ, 2)
    outs = os_.apply(psis, occs)
    es, _ = os_.energy(psis, occs, outs)
    assert abs(es - 2 * ep) < 1e-14 * abs(es)
    for k in range(2):
        for n in range(nb):
            assert np.abs(os_.band(outs, 0, k * nb + n)[pos_of[k]] - op.band(outp, k, n)).max() < 1e-15


def test_C1_whole_config_value_and_independent_library():
    # Whole-config cross-check with an independent FFT library (numpy/pocketfft), same definition (D).
    w = W.make("C1")
    o = _ctx(w)
    psi = w.coefficients(o.npw)
    out = o.apply(psi, w.occ)
    e1, _ = o.energy(psi, w.occ, out)
    m = o.index_map(0)
    K = o.kernel_table(0, 0) / o.omega
    u = []
    for n in range(w.nbands):
        box = np.zeros(w.ng, complex)
        box[m] = o.band(psi, 0, n)
        u.append(np.fft.ifftn(box.reshape(w.grid)) * w.ng)
    for n in (0, 7):
        acc = np.zeros(w.grid, complex)
        for mm in range(w.nbands):
            acc -= u[mm] * np.fft.ifftn(K * np.fft.fftn(np.conj(u[mm]) * u[n]))
        want = (np.fft.fftn(acc) / w.ng).ravel()[m]
        assert np.linalg.norm(o.band(out, 0, n) - want) < 1e-13 * np.linalg.norm(want)
    # value recorded by the survey probe (numpy.fft, not a paper value)
    assert abs(e1 - (-0.0623251812923801)) < 1e-14
    assert abs(np.linalg.norm(o.band(out, 0, 0)) - 0.01853725795907376) < 1e-15


def test_subspace_matrix_pins():
    """exx_ref_subspace against an independent library contraction (numpy.einsum), Hermiticity with all bands occupied, and
    the trace identity E_x = 1/2 sum_k w_k sum_n f_n Re M_nn."""
    w, o, psi = _small(occ=(1.0, 1.0, 1.0, 1.0, 1.0), kpts=True)
    out = o.apply(psi, w.occ)
    e, _ = o.energy(psi, w.occ, out)
    tr = 0.0
    for k in range(w.nk):
        c = np.array([o.band(psi, k, n) for n in range(w.nbands)])
        v = np.array([o.band(out, k, n) for n in range(w.nbands)])
        M = o.subspace(k, psi, out)
        assert M.shape == (w.nbands, w.nbands)
        assert np.abs(M - np.einsum("ig,jg->ij", c.conj(), v)).max() < 1e-16 * w.nbands * 10
        assert np.abs(M - M.conj().T).max() < 1e-15 * np.abs(M).max()
        tr += 0.5 * w.kweight[k] * float((w.occ[k * w.nbands:(k + 1) * w.nbands] * np.diagonal(M).real).sum())
    assert abs(tr - e) < 1e-15
    # a transposed operand or a missing conjugate would fail this: M computed from (psi, out) is not M from (out, psi)^T
    M01 = o.subspace(0, psi, out)
    assert np.abs(o.subspace(0, out, psi) - M01.conj().T).max() < 1e-16


# ---------------------------------------------------------------------------------------------------------------
# exx_ref_apply_to: the operator of (psi, occ) applied to other vectors phi
def test_apply_to_closed_form_plane_wave_eigenvalues():
    """Occupied orbitals = plane waves g_m (weights f_m), trial vectors = plane waves g_i (some among the occupied, some not):
    conj(u_m) t_i is one plane wave, so V_x t_i = lambda_i t_i with lambda_i = -(1/Omega) sum_m f_m K(|G_i - G_m|) (bare kernel, the
    Q = 0 term dropped; HSE keeps pi/mu^2) -- evaluated here from the lattice, no oracle code."""
    gm = [(0, 0, 0), (1, 0, 0), (0, 2, 0), (-1, 1, 3), (2, -2, 1)]
    gi = [(1, 0, 0), (0, 0, 1), (-2, 1, 0), (2, -2, 1), (1, 1, 1)]
    f = np.array([1.0, 1.0, 0.5, 0.0, 0.25])
    lat = W.rhombohedral(9.0, 70.0)
    Bm = 2 * np.pi * np.linalg.inv(lat).T
    for kind, mu in ((0, 0.0), (1, 0.3)):
        o = R.RefExx((16,) * 3, lat, np.zeros((1, 3)), [1.0], 6.0, kind, mu, 1.0, nbands=5)
        psi = _plane_wave_bands(o, [(0, n) for n in range(5)], gm)
        phi = _plane_wave_bands(o, [(0, n) for n in range(5)], gi)
        phi *= np.exp(0.3j) * 1.7            # any amplitude
        out = o.apply_to(psi, f, phi)
        for i, a in enumerate(gi):
            lam = 0.0
            for j, b in enumerate(gm):
                d = (np.array(a) - np.array(b)) @ Bm
                q2 = float(d @ d)
                if q2 > 0:
                    kq = 4 * np.pi / q2 * (1.0 if kind == 0 else -np.expm1(-q2 / (4 * mu * mu)))
                else:
                    kq = 0.0 if kind == 0 else np.pi / mu ** 2
                lam -= f[j] * kq / o.omega
            assert np.linalg.norm(o.band(out, 0, i) - lam * o.band(phi, 0, i)) <= 1e-13 * abs(lam) * np.linalg.norm(o.band(phi, 0, i))


@pytest.mark.parametrize("kpts", [False, True])
def test_apply_to_reduces_to_apply_and_operator_identities(kpts):
    w, o, psi = _small(kpts=kpts, kind=1 if kpts else 0, mu=0.25)
    occ = w.occ
    # phi = psi: the pinned function
    assert np.linalg.norm(o.apply_to(psi, occ, psi) - o.apply(psi, occ)) <= 1e-14 * np.linalg.norm(o.apply(psi, occ))
    rng = np.random.default_rng(77)
    phi = rng.standard_normal(o.ncoef) + 1j * rng.standard_normal(o.ncoef)
    chi = rng.standard_normal(o.ncoef) + 1j * rng.standard_normal(o.ncoef)
    vphi, vchi = o.apply_to(psi, occ, phi), o.apply_to(psi, occ, chi)
    # linear in phi (complex coefficients)
    a, b = 0.7 - 0.2j, -1.3 + 0.5j
    assert np.linalg.norm(o.apply_to(psi, occ, a * phi + b * chi) - (a * vphi + b * vchi)) <= 1e-13 * np.linalg.norm(vphi)
    # Hermitian and negative semi-definite within every k-point, for arbitrary vectors
    for k in range(o.nk):
        P = np.array([o.band(phi, k, i) for i in range(o.nbands)] + [o.band(chi, k, i) for i in range(o.nbands)])
        V = np.array([o.band(vphi, k, i) for i in range(o.nbands)] + [o.band(vchi, k, i) for i in range(o.nbands)])
        M = P.conj() @ V.T
        assert np.abs(M - M.conj().T).max() <= 1e-13 * np.abs(M).max()
        assert np.linalg.eigvalsh(0.5 * (M + M.conj().T)).max() <= 1e-13 * np.abs(M).max()
    # the operator does not depend on the phase of the orbitals that define it
    assert np.linalg.norm(o.apply_to(psi * np.exp(1.1j), occ, phi) - vphi) <= 1e-13 * np.linalg.norm(vphi)


def test_apply_to_block_of_trial_vectors():
    """Fewer (or more) trial vectors per k-point than orbitals: each vector's result is independent of the block it travels in,
    and the plane-wave eigenvalue holds for a block of two."""
    w, o, psi = _small(kpts=True)
    rng = np.random.default_rng(78)
    tot = int(sum(o.npw))
    full = rng.standard_normal(o.ncoef) + 1j * rng.standard_normal(o.ncoef)
    vfull = o.apply_to(psi, w.occ, full)
    for nphi in (1, 2, o.nbands + 2):
        blk = np.concatenate([np.concatenate([o.band(full, k, i % o.nbands) for i in range(nphi)]) for k in range(o.nk)])
        vblk = o.apply_to(psi, w.occ, blk)
        assert vblk.size == nphi * tot
        pos = 0
        for k in range(o.nk):
            for i in range(nphi):
                got = vblk[pos:pos + o.npw[k]]
                pos += o.npw[k]
                assert np.linalg.norm(got - o.band(vfull, k, i % o.nbands)) <= 1e-14 * np.linalg.norm(got)
    gm = [(0, 0, 0), (1, 0, 0), (0, 2, 0)]
    f = np.array([1.0, 0.5, 0.25])
    o2 = R.RefExx((16,) * 3, W.cubic(9.0), np.zeros((1, 3)), [1.0], 6.0, nbands=3)
    psi2 = _plane_wave_bands(o2, [(0, n) for n in range(3)], gm)
    m = o2.index_map(0)
    blk = np.zeros(2 * o2.npw[0], complex)
    gi = [(0, 0, 1), (1, 0, 0)]
    for i, gv in enumerate(gi):
        blk[i * o2.npw[0] + np.searchsorted(m, ((gv[0] % 16) * 16 + (gv[1] % 16)) * 16 + (gv[2] % 16))] = 1.0
    out = o2.apply_to(psi2, f, blk)
    Bm = 2 * np.pi / 9.0
    for i, gv in enumerate(gi):
        lam = -sum(fj * 4 * np.pi / (Bm ** 2 * float((np.array(gv) - np.array(b)) @ (np.array(gv) - np.array(b)))) / o2.omega
                   for fj, b in zip(f, gm) if tuple(b) != tuple(gv))
        assert np.linalg.norm(out[i * o2.npw[0]:(i + 1) * o2.npw[0]] - lam * blk[i * o2.npw[0]:(i + 1) * o2.npw[0]]) <= 1e-13 * abs(lam)


def test_stored_oracle_results_equal_the_survey_probe():
    """tests/golden/exx_C{1,2,3}.json were written by make_golden.py from oracle/ alone.  SURVEY.md section 8(c)-PINS records the same
    three configurations evaluated independently during the survey (numpy.fft, a different program): E_x, the norm of the first
    output row and the checksum of the first index map.  A regenerated golden file that drifts from them fails here, without a GPU."""
    import json
    import os
    gold_dir = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
    survey = {"C1": (-0.0623251812923801, 0.01853725795907376, 1402128),
              "C2": (-0.244336120072931, 0.028385606397239974, 77343110),
              "C3": (-1.4051059069325562, 0.04419327891533337, 2015122368)}
    for name, (ex, norm0, map0) in survey.items():
        gold = json.load(open(os.path.join(gold_dir, "exx_%s.json" % name)))
        assert gold["rows"][0] == [0, 0]
        assert abs(gold["E_x_E1"] - ex) <= 1e-13 * abs(ex), name
        assert abs(gold["E_x_E2"] - ex) <= 1e-13 * abs(ex), name
        assert abs(gold["row_norm"][0] - norm0) <= 1e-13 * norm0, name
        assert gold["map0_sum"] == map0, name
