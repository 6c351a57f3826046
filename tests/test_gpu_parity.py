"""GPU parity tests (-m gpu): the CUDA library, called through its C ABI, against the oracle on the same seeded inputs.

Bars (BASELINE.json north_star): index maps bit-exact; V_x psi_n within 1e-10 relative L2 per band; E_x within 1e-11
relative; fp64.  Building blocks (scatter/gather, FFT, kernel table) are held to tighter, arithmetic-derived bars.
"""
import json
import os

import numpy as np
import pytest

import sys

from oracle import exx_ref as R
from paper_1111_0716_b200 import workloads as W

pytestmark = pytest.mark.gpu

GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
sys.path.insert(0, GOLD)
from probe import probe_vector  # noqa: E402  (seeded probe vectors of the stored per-band functional)
TOL_VX = 1e-10
TOL_EX = 1e-11


@pytest.fixture(scope="module")
def B():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1111_0716_b200 import binding
    binding.lib()  # fails loudly if libexx.so is missing
    return binding


def _pair(B, w):
    o = R.RefExx(w.grid, w.lattice, w.kfrac, w.kweight, w.ecut, w.kernel_kind, w.mu, w.scale, w.nbands)
    g = B.Exx.from_workload(w)
    return o, g


def _rel(a, b):
    return float(np.linalg.norm(a - b) / np.linalg.norm(b))


SMALL = {
    "kpts_frac_occ": dict(grid=(12, 12, 12), lat=("rh", 6.0, 63.0), kf=[[0, 0, 0], [0.5, 0, 0], [0.25, -0.25, 0.125]],
                          kw=[0.5, 0.25, 0.25], ecut=4.0, nb=5, occ=[1, 1, 0.5, 0.25, 0], kind=0, mu=0.0),
    "noncubic_hse": dict(grid=(12, 18, 16), lat=("rh", 7.3, 71.0), kf=[[0.1, -0.3, 0.25], [0.5, 0, 0]], kw=[0.5, 0.5],
                         ecut=5.0, nb=4, occ=[1, 0.7, 0, 0.2], kind=1, mu=0.3),
    "tiny_aliased": dict(grid=(8, 6, 9), lat=("sc", 5.0), kf=[[0, 0, 0]], kw=[1.0], ecut=3.5, nb=3, occ=[1, 1, 1], kind=0, mu=0.0),
    "pow2_rect": dict(grid=(32, 16, 8), lat=("rh", 6.5, 75.0), kf=[[0, 0, 0], [0, 0.5, 0.5]], kw=[0.3, 0.7], ecut=2.5, nb=3,
                      occ=[1, 0.5, 0], kind=1, mu=0.106),
    "one_band": dict(grid=(24, 24, 24), lat=("sc", 9.0), kf=[[0, 0, 0]], kw=[1.0], ecut=5.0, nb=1, occ=[1.0], kind=0, mu=0.0),
    "mixed_27": dict(grid=(27, 24, 36), lat=("rh", 10.0, 80.0), kf=[[0.25, 0.25, 0.25]], kw=[1.0], ecut=4.0, nb=3, occ=[1, 1, 0.5],
                     kind=0, mu=0.0),
}


def _small(name):
    s = SMALL[name]
    lat = W.cubic(s["lat"][1]) if s["lat"][0] == "sc" else W.rhombohedral(s["lat"][1], s["lat"][2])
    return W.custom(name, 77 + len(name), s["grid"], lat, s["kf"], s["kw"], s["ecut"], s["nb"], s["occ"], s["kind"], s["mu"])


# ---------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("name", ["C1", "C2", "C3", "C4a", "C4b", "C5"])
def test_index_maps_bit_exact(B, name):
    w = W.make(name)
    if name in ("C4b", "C5"):  # keep device memory modest: the maps do not depend on the band count
        w.nbands, w.occ_per_k = 2, np.ones(2)
    o, g = _pair(B, w)
    assert g.npw == o.npw and g.offsets == o.offsets
    for k in range(w.nk):
        a, b = g.index_map(k), o.index_map(k)
        assert a.dtype == np.int32 and np.array_equal(a, b)
    g.close()


@pytest.mark.parametrize("name", list(SMALL))
def test_index_maps_and_kernel_tables_small(B, name):
    w = _small(name)
    o, g = _pair(B, w)
    assert g.npw == o.npw
    for k in range(w.nk):
        assert np.array_equal(g.index_map(k), o.index_map(k))
        for q in range(w.nk):
            want = o.kernel_table(k, q) / (o.omega * float(w.ng) ** 2)
            got = g.kernel_table(k, q)
            assert np.abs(got - want).max() <= 4e-16 * np.abs(want).max()
            assert np.array_equal(got == 0, want == 0)
    g.close()


def test_scatter_gather_round_trip_bit_exact(B):
    import torch
    w = W.make("C2")
    w.nbands, w.occ_per_k = 3, np.ones(3)
    o, g = _pair(B, w)
    psi = w.coefficients(o.npw)
    for k in (0, 5):
        coef = np.array([o.band(psi, k, n) for n in range(3)]).reshape(-1)
        cd = torch.from_numpy(coef).cuda()
        box = torch.full((3 * w.ng,), 7.0 + 1j, dtype=torch.complex128, device="cuda")
        g.scatter(k, cd, 3, box)
        hb = box.cpu().numpy().reshape(3, w.ng)
        m = o.index_map(k)
        want = np.zeros((3, w.ng), complex)
        want[:, m] = coef.reshape(3, -1)
        assert np.array_equal(hb.view(np.float64), want.view(np.float64))       # bit identical, zero elsewhere
        back = torch.empty_like(cd)
        g.gather(k, box, 3, back)
        assert np.array_equal(back.cpu().numpy().view(np.float64), coef.view(np.float64))
    g.close()


@pytest.mark.parametrize("grid,nbatch", [((16, 16, 16), 5), ((48, 48, 48), 2), ((12, 18, 16), 3), ((27, 24, 36), 1), ((8, 6, 9), 4),
                                         ((64, 64, 64), 1), ((96, 96, 96), 1), ((128, 128, 128), 1), ((32, 16, 8), 2), ((2, 3, 4), 7),
                                         ((10, 20, 15), 3), ((40, 40, 40), 2), ((25, 6, 5), 2)])
def test_fft3d_against_oracle_fft(B, grid, nbatch):
    import torch
    g = B.Exx(grid, W.cubic(50.0), np.zeros((1, 3)), [1.0], 0.005, nbands=1)  # sphere = {0}: any grid holds it
    rng = np.random.default_rng(sum(grid))
    x = rng.standard_normal((nbatch,) + grid) + 1j * rng.standard_normal((nbatch,) + grid)
    for sign in (-1, +1):
        d = torch.from_numpy(x.reshape(-1).copy()).cuda()
        g.fft3d(d, nbatch, sign)
        got = d.cpu().numpy().reshape((nbatch,) + grid)
        for b in range(nbatch if max(grid) < 64 else 1):
            want = R.fft3d(x[b], sign)
            assert _rel(got[b], want) < 2e-15 * np.log2(np.prod(grid))
    g.close()


# ---------------------------------------------------------------------------------------------------------------
def _check_full(B, w, paths=(0,), tile_m=(0,)):
    """Full element-by-element parity of V_x psi (every band), per-band energies and E_x."""
    o, g = _pair(B, w)
    psi = w.coefficients(o.npw)
    want = o.apply(psi, w.occ)
    e_want, pb_want = o.energy(psi, w.occ, want)
    pd = g.to_device(psi)
    for path in paths:
        for tm in tile_m:
            g.set_option(B.EXX_OPT_PATH, path)
            g.set_option(B.EXX_OPT_TILE_M, tm)
            out = g.apply(pd, w.occ)
            got = out.cpu().numpy()
            for k in range(w.nk):
                for n in range(w.nbands):
                    assert _rel(o.band(got, k, n), o.band(want, k, n)) < TOL_VX, (w.name, path, tm, k, n)
            e, pb = g.energy(pd, w.occ, out)
            assert abs(e - e_want) <= TOL_EX * abs(e_want)
            assert np.abs(pb - pb_want).max() <= TOL_EX * abs(e_want)
            assert abs(pb.sum() - e) <= 1e-14 * abs(e)
            assert e <= 0
            g.set_option(B.EXX_OPT_ENERGY_ROUTE, 1)
            e2, _ = g.energy(pd, w.occ, None)          # library applies V_x itself, then (E1)
            assert abs(e2 - e) <= 1e-15 * abs(e) and g.get_info(B.EXX_INFO_ENERGY_ROUTE) == 1
            assert g.get_info(B.EXX_INFO_PAIRS_ORDERED) == w.pair_evals
            assert g.get_info(B.EXX_INFO_LAUNCHES) > 0
            g.set_option(B.EXX_OPT_ENERGY_ROUTE, 0)
            e3, pb3 = g.energy(pd, w.occ, None)        # pair-density route (E2) where the fused kernels run
            assert g.get_info(B.EXX_INFO_ENERGY_ROUTE) == (2 if g.get_info(B.EXX_INFO_PATH_USED) == 2 else 1)
            assert abs(e3 - e_want) <= TOL_EX * abs(e_want)
            assert np.abs(pb3 - pb_want).max() <= TOL_EX * abs(e_want)
    g.close()
    return o, psi, want


@pytest.mark.parametrize("name", list(SMALL))
def test_apply_small_cases_full_parity(B, name):
    _check_full(B, _small(name), paths=(0, 1), tile_m=(0, 1, 3))


def test_apply_C1_full_parity(B):
    w = W.make("C1")
    o, psi, want = _check_full(B, w, paths=(0, 1), tile_m=(0, 5))
    gold = json.load(open(os.path.join(GOLD, "exx_C1.json")))
    e, _ = o.energy(psi, w.occ, want)
    assert abs(e - gold["E_x_E1"]) < 1e-15


def _check_golden(B, name, live_rows=0, prune=1, symmetry=1, dual=1):
    """Big configs: the GPU applies V_x in full; rows, per-band energies and E_x are compared with stored oracle
    results (tests/golden/make_golden.py) and, for `live_rows` rows, with the oracle run now."""
    import torch
    w = W.make(name)
    if not os.path.exists(os.path.join(GOLD, "exx_%s.json" % name)):
        pytest.skip("golden values for %s not generated (tests/golden/make_golden.py)" % name)
    gold = json.load(open(os.path.join(GOLD, "exx_%s.json" % name)))
    rows_gold = np.load(os.path.join(GOLD, "exx_%s_rows.npz" % name))
    g = B.Exx.from_workload(w)
    assert g.npw == gold["npw"]
    psi = w.coefficients(g.npw)
    assert [psi[0].real, psi[0].imag] == gold["psi_first"]
    pd = g.to_device(psi)
    g.set_option(B.EXX_OPT_PRUNE, prune)
    g.set_option(B.EXX_OPT_SYMMETRY, symmetry)
    g.set_option(B.EXX_OPT_DUAL_SWEEP, dual)
    out = g.apply(pd, w.occ)
    assert g.get_info(B.EXX_INFO_SYMMETRY) == symmetry
    # pair boxes transformed: every ordered pair, or with the symmetry each unordered pair of the nk*nbands occupied bands once
    # unless both are empty (f = 0; C2 has 6 empty bands per k-point, C4's two half-filled bands count as occupied)
    nkb, nempty = w.nk * w.nbands, w.nk * (w.nbands - w.nocc)
    executed = {0: w.pair_evals, 1: nkb * (nkb + 1) // 2 - nempty * (nempty + 1) // 2}[symmetry]
    assert executed == {0: w.pair_evals, 1: {"C2": 17352, "C3": 2080, "C4a": 12880, "C4b": 819840, "C5": 32896}[name]}[symmetry]
    assert g.get_info(B.EXX_INFO_PAIRS_EXECUTED) == executed
    assert g.get_info(B.EXX_INFO_PRUNED) == (1 if (prune and g.get_info(B.EXX_INFO_COMPACT_GRID)) else 0)
    e, pb = g.energy(pd, w.occ, out)
    torch.cuda.synchronize()
    got = out.cpu().numpy()
    for i, (k, n) in enumerate(gold["rows"]):
        want = rows_gold["row%d" % i]
        assert _rel(g.band(got, k, n), want) < TOL_VX, (name, k, n)
        assert abs(pb[k * w.nbands + n] - gold["row_energy"][i]) <= TOL_EX * abs(gold["row_energy"][i]) + 1e-300
    if "E_x_E1" in gold:
        assert abs(e - gold["E_x_E1"]) <= TOL_EX * abs(gold["E_x_E1"])
        assert abs(e - gold["E_x_E2"]) <= TOL_EX * abs(gold["E_x_E2"])
        assert np.abs(pb - np.array(gold["per_band_energy"])).max() <= TOL_EX * abs(gold["E_x_E1"])
        norms = np.array([np.linalg.norm(g.band(got, k, n)) for k in range(w.nk) for n in range(w.nbands)])
        assert np.abs(norms / np.array(gold["per_band_norm"]) - 1).max() < TOL_VX
        if "per_band_probe" in gold:
            # every band's row against the oracle through a third functional, <z_k | V_x c_nk> with a seeded unit probe vector:
            # |<z|got> - <z|want>| <= |got - want| (Cauchy-Schwarz), so the rel-L2 bar of the rows applies to it unchanged
            for k in range(w.nk):
                z = probe_vector(w.seed, k, g.npw[k])
                for n in range(w.nbands):
                    pr = gold["per_band_probe"][k * w.nbands + n]
                    assert abs(np.vdot(z, g.band(got, k, n)) - complex(pr[0], pr[1])) <= TOL_VX * gold["per_band_norm"][k * w.nbands + n], (name, k, n)
    elif "E_x_E2" in gold:
        # rows only plus the oracle's total energy by its second route (E2, forward transforms only: tests/golden/make_golden.py C5:e2)
        assert abs(e - gold["E_x_E2"]) <= TOL_EX * abs(gold["E_x_E2"])
    # properties that hold at any size
    assert e < 0 and abs(pb.sum() - e) <= 1e-13 * abs(e) and np.all(pb <= 0)
    assert g.get_info(B.EXX_INFO_PAIRS_ORDERED) == w.pair_evals
    if live_rows:
        o = R.RefExx(w.grid, w.lattice, w.kfrac, w.kweight, w.ecut, w.kernel_kind, w.mu, w.scale, w.nbands)
        rows = [(w.nk // 2, w.nbands // 3), (0, 1)][:live_rows]
        for (k, n), r in zip(rows, o.apply_rows(psi, w.occ, rows)):
            assert _rel(g.band(got, k, n), r) < TOL_VX, (name, "live", k, n)
    g.close()


def test_apply_C2_parity(B):
    _check_golden(B, "C2", live_rows=1)


def test_apply_C3_parity(B):
    _check_golden(B, "C3", live_rows=1)


def test_apply_C4a_parity(B):
    """The benchmarked configuration against the FULL oracle result: E_x by (E1) and (E2), all 160 per-band energies, norms and
    probe functionals, and 8 complete rows (tile edges 0/31/32/159, interiors 40/95/128, a half-occupied band 158)."""
    gold = json.load(open(os.path.join(GOLD, "exx_C4a.json")))
    assert "E_x_E1" in gold and "E_x_E2" in gold and len(gold["per_band_energy"]) == 160 and len(gold["rows"]) >= 8
    _check_golden(B, "C4a")


def test_apply_C4a_two_sweeps_parity(B):
    """EXX_OPT_DUAL_SWEEP = 0 (two sweeps of the last pass instead of the dual sweep) against the same oracle values."""
    _check_golden(B, "C4a", dual=0)


def test_apply_C5_parity(B):
    _check_golden(B, "C5")


@pytest.mark.skipif(not os.path.exists(os.path.join(GOLD, "exx_C4b.json")), reason="C4b golden rows not generated yet")
def test_apply_C4b_parity(B):
    _check_golden(B, "C4b")


# ---------------------------------------------------------------------------------------------------------------
# compact work grid (EXX_OPT_PRUNE): cells whose box is much larger than 4 gmax + 1
COMPACT = {
    "sc64_gamma": dict(grid=(64, 64, 64), lat=("sc", 10.0), kf=[[0, 0, 0]], kw=[1.0], ecut=12.0, nb=5, occ=[1, 1, 0.5, 0.25, 0],
                       kind=0, mu=0.0, compact=48),
    "rh64_kpts_hse": dict(grid=(64, 64, 64), lat=("rh", 9.0, 62.0), kf=[[0.25, 0.25, 0.25], [-0.25, 0.25, 0.0]], kw=[0.5, 0.5],
                          ecut=9.0, nb=3, occ=[1, 0.6, 0.3], kind=1, mu=0.106, compact=48),
}


FUSED_SIZES = (16, 32, 40, 48, 64, 72, 80, 96, 128)


def _expected_compact(g, w):
    """Smallest supported cubic grid with N >= 4 gmax + 1, if the caller's grid is itself alias-free and larger."""
    gmax = 0
    for k in range(w.nk):
        j = np.stack(np.unravel_index(g.index_map(k), w.grid))
        for ax in range(3):
            f = np.where(2 * j[ax] < w.grid[ax], j[ax], j[ax] - w.grid[ax])
            gmax = max(gmax, int(np.abs(f).max()))
    need = 4 * gmax + 1
    if any(n < need for n in w.grid):
        return 0
    fused = len(set(w.grid)) == 1 and w.grid[0] in FUSED_SIZES
    for n in FUSED_SIZES:
        if n >= need:
            return n if (n ** 3 < w.ng or (not fused and n ** 3 <= 4 * w.ng)) else 0
    return 0


@pytest.mark.parametrize("name", list(COMPACT))
def test_compact_grid_equals_full_grid_and_oracle(B, name):
    s = COMPACT[name]
    lat = W.cubic(s["lat"][1]) if s["lat"][0] == "sc" else W.rhombohedral(s["lat"][1], s["lat"][2])
    w = W.custom(name, 4242, s["grid"], lat, s["kf"], s["kw"], s["ecut"], s["nb"], s["occ"], s["kind"], s["mu"])
    o, g = _pair(B, w)
    compact = _expected_compact(g, w)
    assert compact and compact < 64 and g.get_info(B.EXX_INFO_COMPACT_GRID) == compact
    psi = w.coefficients(o.npw)
    want = o.apply(psi, w.occ)              # the oracle works on the caller's full 64^3 grid
    e_want, _ = o.energy(psi, w.occ, want)
    pd = g.to_device(psi)
    res = {}
    for prune, sym in ((1, 1), (0, 1), (1, 0)):
        g.set_option(B.EXX_OPT_PRUNE, prune)
        g.set_option(B.EXX_OPT_SYMMETRY, sym)
        out = g.apply(pd, w.occ)
        assert g.get_info(B.EXX_INFO_PRUNED) == prune
        assert g.get_info(B.EXX_INFO_SYMMETRY) == sym
        assert (g.get_info(B.EXX_INFO_PAIRS_EXECUTED) < w.pair_evals) == bool(sym)
        assert g.get_info(B.EXX_INFO_WORK_GRID) == (compact if prune else 64)
        assert g.get_info(B.EXX_INFO_PAIRS_ORDERED) == w.pair_evals
        got = out.cpu().numpy()
        for k in range(w.nk):
            for n in range(w.nbands):
                assert _rel(o.band(got, k, n), o.band(want, k, n)) < TOL_VX, (name, prune, k, n)
        e, _ = g.energy(pd, w.occ, out)
        assert abs(e - e_want) <= TOL_EX * abs(e_want)
        res[(prune, sym)] = got
    assert _rel(res[(1, 1)], res[(0, 1)]) < 1e-13
    assert _rel(res[(1, 1)], res[(1, 0)]) < 1e-13
    g.close()


@pytest.mark.parametrize("name", ["C2", "C3"])
def test_pair_symmetry_off_matches_golden(B, name):
    """The default runs use the pair symmetry; this one evaluates every ordered pair (EXX_OPT_SYMMETRY = 0)."""
    _check_golden(B, name, symmetry=0)


NOFUSED = {
    # alias-free caller grids that have no fused kernels of their own: a cubic work grid with up to 4x the points is used instead
    "rect_50_50_64": dict(grid=(50, 50, 64), lat=("sc", 12.0), kf=[[0, 0, 0], [0.25, 0.25, -0.25]], kw=[0.5, 0.5], ecut=20.0, nb=3,
                          occ=[1, 0.5, 0], kind=0, mu=0.0),
    "cubic_54": dict(grid=(54, 54, 54), lat=("sc", 12.0), kf=[[0, 0, 0]], kw=[1.0], ecut=24.5, nb=3, occ=[1, 0.5, 0.25], kind=1, mu=0.106),
}


@pytest.mark.parametrize("name", list(NOFUSED))
def test_cubic_work_grid_for_grids_without_fused_kernels(B, name):
    s = NOFUSED[name]
    lat = W.cubic(s["lat"][1]) if s["lat"][0] == "sc" else W.rhombohedral(s["lat"][1], s["lat"][2])
    w = W.custom(name, 808, s["grid"], lat, s["kf"], s["kw"], s["ecut"], s["nb"], s["occ"], s["kind"], s["mu"])
    o, g = _pair(B, w)
    compact = _expected_compact(g, w)
    assert compact and compact ** 3 >= w.ng and g.get_info(B.EXX_INFO_COMPACT_GRID) == compact   # larger than the caller's box
    psi = w.coefficients(o.npw)
    want = o.apply(psi, w.occ)                 # the oracle works on the caller's grid
    e_want, _ = o.energy(psi, w.occ, want)
    pd = g.to_device(psi)
    res = {}
    for path in (0, 1):                        # auto: fused passes on the cubic grid; 1: generic kernels on the caller's grid
        g.set_option(B.EXX_OPT_PATH, path)
        out = g.apply(pd, w.occ)
        assert g.get_info(B.EXX_INFO_PATH_USED) == (2 if path == 0 else 1)
        assert g.get_info(B.EXX_INFO_PRUNED) == (1 if path == 0 else 0)
        got = out.cpu().numpy()
        for k in range(w.nk):
            for n in range(w.nbands):
                assert _rel(o.band(got, k, n), o.band(want, k, n)) < TOL_VX, (name, path, k, n)
        e, _ = g.energy(pd, w.occ, out)
        assert abs(e - e_want) <= TOL_EX * abs(e_want)
        res[path] = got
    assert _rel(res[0], res[1]) < 1e-13
    g.close()


def test_compact_grid_not_used_when_caller_grid_aliases(B):
    # C1 (16^3, needs 21) is aliased by construction and C3 (needs 61) keeps its 64^3 box: no compact grid
    for name in ("C1", "C3"):
        w = W.make(name)
        w.nbands, w.occ_per_k = 2, np.ones(2)
        g = B.Exx.from_workload(w)
        assert g.get_info(B.EXX_INFO_COMPACT_GRID) == 0
        g.close()
    for name, n in (("C2", 40), ("C4a", 72), ("C5", 96)):
        w = W.make(name)
        w.nbands, w.occ_per_k = 2, np.ones(2)
        g = B.Exx.from_workload(w)
        assert g.get_info(B.EXX_INFO_COMPACT_GRID) == n
        g.close()


@pytest.mark.parametrize("name,prune", [("C2", 1), ("C3", 1), ("C4a", 1), ("C4a", 0)])
def test_apply_is_bitwise_reproducible_at_full_size(B, name, prune):
    """No atomics, fixed summation order, per-thread staging slots: two applies of the same input give identical bits (a race in the
    cp.async staging or in the accumulator updates would show up here) — on the instantiations the BASELINE configs run
    (N = 40, 64, 72 and, with EXX_OPT_PRUNE = 0, 96)."""
    import torch
    w = W.make(name)
    g = B.Exx.from_workload(w)
    g.set_option(B.EXX_OPT_PRUNE, prune)
    pd = g.to_device(w.coefficients(g.npw))
    a = g.apply(pd, w.occ).clone()
    b = g.apply(pd, w.occ)
    assert torch.equal(torch.view_as_real(a), torch.view_as_real(b))
    assert bool(torch.isfinite(torch.view_as_real(a)).all())
    g.close()


def test_apply_C4a_full_grid_parity(B):
    """C4a on the caller's full 96^3 grid (EXX_OPT_PRUNE = 0); test_apply_C4a_parity covers the default (compact 72^3)."""
    _check_golden(B, "C4a", prune=0)


# ---------------------------------------------------------------------------------------------------------------
def test_edge_cases_and_errors(B):
    import torch
    w = _small("kpts_frac_occ")
    o, g = _pair(B, w)
    psi = w.coefficients(o.npw)
    pd = g.to_device(psi)
    # all occupations zero: V_x = 0 exactly, E_x = 0, no pair executed
    out = g.apply(pd, np.zeros(w.nk * w.nbands))
    assert float(out.abs().max()) == 0.0
    assert g.get_info(B.EXX_INFO_PAIRS_EXECUTED) == 0
    assert g.energy(pd, np.zeros(w.nk * w.nbands), out)[0] == 0.0
    # only one occupied band at one k-point: matches the oracle, other k-points still get rows
    occ1 = np.zeros(w.nk * w.nbands)
    occ1[w.nbands + 2] = 0.75
    got = g.apply(pd, occ1).cpu().numpy()
    assert _rel(got, o.apply(psi, occ1)) < TOL_VX
    # errors: aliasing, bad occupations, wrong sizes are refused and leave the output alone
    with pytest.raises(B.ExxError) as ei:
        g.apply(pd, w.occ, pd)
    assert ei.value.code == -10
    bad = w.occ.copy()
    bad[1] = -0.1
    sentinel = torch.full_like(pd, 3.0)
    with pytest.raises(B.ExxError) as ei:
        g.apply(pd, bad, sentinel)
    assert ei.value.code == -6 and float((sentinel - 3.0).abs().max()) == 0.0
    bad[1] = float("inf")
    with pytest.raises(B.ExxError):
        g.energy(pd, bad, out)
    with pytest.raises(B.ExxError):
        g.set_option(99, 1)
    with pytest.raises(B.ExxError):   # sphere does not fit the box
        B.Exx((8, 8, 8), W.cubic(10.0), np.zeros((1, 3)), [1.0], 6.0, nbands=1)
    g.close()


def test_apply_host_matches_device_path(B):
    import torch
    w = W.make("C1")
    o, g = _pair(B, w)
    psi = w.coefficients(o.npw)
    out_d = g.apply(g.to_device(psi), w.occ).cpu().numpy()
    g.set_option(B.EXX_OPT_ENERGY_ROUTE, 1)            # (E1) from V_x psi, as apply_host does
    e_d, _ = g.energy(g.to_device(psi), w.occ, None)
    out_h, e_h = g.apply_host(psi, w.occ)
    assert np.array_equal(out_h.view(np.float64), out_d.view(np.float64)) and e_h == e_d
    pin_in = torch.from_numpy(psi).pin_memory()
    pin_out = torch.empty(g.ncoef, dtype=torch.complex128).pin_memory()
    g.apply_host(pin_in, w.occ, pin_out, want_energy=False)
    assert np.array_equal(pin_out.numpy().view(np.float64), out_d.view(np.float64))
    g.close()


def test_to_real_matches_oracle(B):
    import torch
    w = _small("noncubic_hse")
    o, g = _pair(B, w)
    psi = w.coefficients(o.npw)
    for k in range(w.nk):
        coef = np.array([o.band(psi, k, n) for n in range(w.nbands)]).reshape(-1)
        box = torch.empty(w.nbands * w.ng, dtype=torch.complex128, device="cuda")
        g.to_real(k, torch.from_numpy(coef).cuda(), w.nbands, box)
        hb = box.cpu().numpy().reshape((w.nbands,) + w.grid)
        for n in range(w.nbands):
            assert _rel(hb[n], o.to_real(k, o.band(psi, k, n))) < 1e-14
    g.close()


# ---------------------------------------------------------------------------------------------------------------
# Properties of the GPU result that hold at any size and need no oracle (checked at a full BASELINE size, C3)
def test_gpu_operator_properties_C3(B):
    import torch
    w = W.make("C3")
    g = B.Exx.from_workload(w)
    psi = w.coefficients(g.npw)
    pd = g.to_device(psi)
    out = g.apply(pd, w.occ).clone()
    e, pb = g.energy(pd, w.occ, out)
    npw, nb = g.npw[0], w.nbands
    Cm, Vm = pd.view(nb, npw), out.view(nb, npw)
    # Hermiticity of M_ij = <c_i | V_x c_j> (all 64 bands occupied, so V_x is the full operator on this subspace)
    M = torch.conj(Cm) @ Vm.T
    assert float((M - torch.conj(M.T)).abs().max()) <= 1e-13 * float(M.abs().max())
    # V_x is negative semi-definite on the occupied subspace: all eigenvalues of M <= 0
    ev = torch.linalg.eigvalsh(0.5 * (M + torch.conj(M.T)))
    assert float(ev.max()) <= 1e-14
    assert abs(0.5 * float(torch.diagonal(M).real.sum()) - e) <= 1e-13 * abs(e)
    # covariance under a global phase: c -> e^{i theta} c  =>  V_x c -> e^{i theta} V_x c, E_x unchanged
    ph = complex(np.cos(0.7), np.sin(0.7))
    out2 = g.apply(pd * ph, w.occ)
    assert float((out2 - out * ph).abs().max()) <= 1e-13 * float(out.abs().max())
    e2, _ = g.energy(pd * ph, w.occ, out2)
    assert abs(e2 - e) <= 1e-13 * abs(e)
    # unitary mix of equally occupied bands: c -> U c  =>  out -> U out
    rng = np.random.default_rng(1)
    q, _ = np.linalg.qr(rng.standard_normal((nb, nb)) + 1j * rng.standard_normal((nb, nb)))
    U = torch.from_numpy(q).cuda()
    out3 = g.apply((U @ Cm).reshape(-1).contiguous(), w.occ)
    assert float((out3.view(nb, npw) - U @ Vm).abs().max()) <= 1e-12 * float(out.abs().max())
    g.close()


def test_gpu_closed_form_single_plane_waves(B):
    """Bands that are single plane waves: E_x = -(1/2 Omega) sum_{n,m} f_n f_m 4 pi/|G_n - G_m|^2 (BASELINE north_star closed
    form), evaluated in the test; the GPU (fused path, 48^3) must reproduce it without any oracle in between."""
    import torch
    a, N = 9.0, 48
    w = W.custom("pw48", 1, (N, N, N), W.cubic(a), [[0, 0, 0]], [1.0], 4.0, 5, [1, 1, 0.5, 1, 0.25])
    g = B.Exx.from_workload(w)
    gs = [(0, 0, 0), (1, 0, 0), (0, 2, 0), (-1, 1, 3), (2, -2, 1)]
    m = g.index_map(0)
    psi = np.zeros((5, g.npw[0]), dtype=np.complex128)
    for n, gv in enumerate(gs):
        box = ((gv[0] % N) * N + (gv[1] % N)) * N + (gv[2] % N)
        psi[n, int(np.where(m == box)[0][0])] = 1.0
    f = w.occ
    want = 0.0
    for n in range(5):
        for k in range(5):
            d = np.array(gs[n]) - np.array(gs[k])
            if d.any():
                want -= 0.5 / a ** 3 * f[n] * f[k] * 4 * np.pi / ((2 * np.pi / a) ** 2 * float(d @ d))
    pd = g.to_device(psi.reshape(-1))
    for sym in (1, 0):
        for route in (0, 1):                           # pair-density route (E2) and V_x psi + (E1)
            g.set_option(B.EXX_OPT_SYMMETRY, sym)
            g.set_option(B.EXX_OPT_ENERGY_ROUTE, route)
            e, _ = g.energy(pd, f, None)
            assert g.get_info(B.EXX_INFO_PATH_USED) == 2 and g.get_info(B.EXX_INFO_ENERGY_ROUTE) == 2 - route
            assert abs(e - want) <= 1e-13 * abs(want)
    g.close()


# ---------------------------------------------------------------------------------------------------------------
# S8(f)-1: subspace matrix <c_i | V_x c_j> (exx_subspace, fp64 DMMA ZGEMM)
@pytest.mark.parametrize("name", ["kpts_frac_occ", "noncubic_hse", "one_band"])
def test_subspace_matrix_against_oracle_small(B, name):
    w = _small(name)
    o, g = _pair(B, w)
    psi = w.coefficients(o.npw)
    want_v = o.apply(psi, w.occ)
    pd = g.to_device(psi)
    out = g.apply(pd, w.occ)
    for k in range(w.nk):
        M = g.subspace(k, pd, out).cpu().numpy()
        Mo = o.subspace(k, psi, want_v)
        assert M.shape == (w.nbands, w.nbands)
        assert np.abs(M - Mo).max() <= 1e-12 * max(np.abs(Mo).max(), 1e-300)
    g.close()


def test_subspace_matrix_C3_full_size(B):
    """Full BASELINE size (64 bands, 15 895 plane waves; ragged: 64 = 8 tiles, npw not a multiple of 4): element-wise against
    the oracle's triple loop on the GPU's own V_x psi, plus Hermiticity and the trace identity."""
    w = W.make("C3")
    o, g = _pair(B, w)
    psi = w.coefficients(g.npw)
    pd = g.to_device(psi)
    out = g.apply(pd, w.occ)
    e, _ = g.energy(pd, w.occ, out)
    M = g.subspace(0, pd, out).cpu().numpy()
    Mo = o.subspace(0, psi, out.cpu().numpy())
    assert np.abs(M - Mo).max() <= 1e-13 * np.abs(Mo).max()
    assert np.abs(M - M.conj().T).max() <= 1e-13 * np.abs(M).max()
    assert abs(0.5 * np.diagonal(M).real.sum() - e) <= 1e-13 * abs(e)
    g.close()


def test_subspace_matrix_ragged_band_count(B):
    # 5 and 13 bands: tiles of 8 with a ragged edge in both directions; random (non-V_x) right-hand side
    import torch
    for nb in (5, 13):
        w = W.custom("rag", 9, (12, 12, 12), W.cubic(6.0), [[0, 0, 0], [0.5, 0, 0]], [0.5, 0.5], 4.0, nb, np.ones(nb))
        o, g = _pair(B, w)
        psi = w.coefficients(o.npw)
        rhs = W.custom("rag2", 10, (12, 12, 12), W.cubic(6.0), [[0, 0, 0], [0.5, 0, 0]], [0.5, 0.5], 4.0, nb, np.ones(nb)).coefficients(o.npw)
        for k in range(w.nk):
            M = g.subspace(k, g.to_device(psi), g.to_device(rhs)).cpu().numpy()
            assert np.abs(M - o.subspace(k, psi, rhs)).max() <= 1e-13
        g.close()


# ---------------------------------------------------------------------------------------------------------------
# The job-list driven fused loop nest: ragged band tiles, holes in the occupations, k-points, both symmetry modes, small tiles
@pytest.mark.parametrize("tile", [0, 4, 7])
def test_fused_ragged_tiles_and_occupation_holes(B, tile):
    nb = 19
    occ = np.array([1, 0, 1, 0.5, 0, 0, 1, 1, 0.25, 0, 1, 0, 0, 0, 1, 0.75, 0, 0, 0], dtype=float)
    w = W.custom("ragged48", 2024, (48, 48, 48), W.rhombohedral(7.5, 66.0), [[0.0, 0.0, 0.0], [0.25, -0.25, 0.5]], [0.4, 0.6], 5.0, nb, occ)
    o, g = _pair(B, w)
    psi = w.coefficients(o.npw)
    want = o.apply(psi, w.occ)
    e_want, pb_want = o.energy(psi, w.occ, want)
    pd = g.to_device(psi)
    res = {}
    for sym in (1, 0):
        g.set_option(B.EXX_OPT_SYMMETRY, sym)
        g.set_option(B.EXX_OPT_TILE_N, tile)
        g.set_option(B.EXX_OPT_TILE_M, tile)
        out = g.apply(pd, w.occ)
        assert g.get_info(B.EXX_INFO_PATH_USED) == 2 and g.get_info(B.EXX_INFO_SYMMETRY) == sym
        assert g.get_info(B.EXX_INFO_PAIRS_ORDERED) == w.pair_evals
        got = out.cpu().numpy()
        for k in range(w.nk):
            for n in range(nb):
                assert _rel(o.band(got, k, n), o.band(want, k, n)) < TOL_VX, (sym, tile, k, n)
        e, pb = g.energy(pd, w.occ, out)
        assert abs(e - e_want) <= TOL_EX * abs(e_want)
        assert np.abs(pb - pb_want).max() <= TOL_EX * abs(e_want)
        res[sym] = got
    assert _rel(res[1], res[0]) < 1e-13
    # the same apply twice gives bit-identical results (fixed summation order, no atomics)
    again = g.apply(pd, w.occ).cpu().numpy()
    assert np.array_equal(again.view(np.float64), res[0].view(np.float64))
    g.close()


def test_fused_128_full_grid_against_live_oracle(B):
    """The N = 128 (R1 = 16) instantiation of the fused passes, which the default (compact-grid) runs of C5 never use: a C5-shaped
    cell with 3 bands on the caller's full 128^3 grid (EXX_OPT_PRUNE = 0), both symmetry modes, against the oracle run now."""
    w = W.custom("c5_small", 555, (128, 128, 128), W.cubic(30.0), [[0, 0, 0]], [1.0], 10.0, 3, [1.0, 0.5, 0.0], kernel_kind=1, mu=0.106)
    o, g = _pair(B, w)
    assert g.get_info(B.EXX_INFO_COMPACT_GRID) == 96
    psi = w.coefficients(o.npw)
    want = o.apply(psi, w.occ)
    e_want, _ = o.energy(psi, w.occ, want)
    pd = g.to_device(psi)
    g.set_option(B.EXX_OPT_PRUNE, 0)
    for sym in (1, 0):
        g.set_option(B.EXX_OPT_SYMMETRY, sym)
        out = g.apply(pd, w.occ)
        assert g.get_info(B.EXX_INFO_WORK_GRID) == 128 and g.get_info(B.EXX_INFO_PATH_USED) == 2
        got = out.cpu().numpy()
        for n in range(w.nbands):
            assert _rel(o.band(got, 0, n), o.band(want, 0, n)) < TOL_VX, (sym, n)
        e, _ = g.energy(pd, w.occ, out)
        assert abs(e - e_want) <= TOL_EX * abs(e_want)
    g.close()


FUSED_EVERY = {
    # N: (lattice, kfrac, kweight, ecut, occupations, kernel kind, mu) — one small cell per instantiation of the fused passes that
    # no BASELINE configuration reaches on its own; run on the caller's grid (EXX_OPT_PRUNE = 0)
    32: (("rh", 8.0, 70.0), [[0, 0, 0], [0.5, 0.25, 0]], [0.5, 0.5], 3.0, [1, 0.5, 0, 1], 0, 0.0),        # alias-free: pair symmetry on
    "32a": (("sc", 10.0), [[0, 0, 0]], [1.0], 20.0, [1, 1, 0.5, 0, 1], 1, 0.106),                         # needs 41 > 32: aliased, symmetry off
    40: (("sc", 11.0), [[0.25, 0.25, 0.25]], [1.0], 5.0, [1, 0, 0.5, 1, 1], 0, 0.0),
    80: (("rh", 16.0, 62.0), [[0, 0, 0], [0.25, -0.25, 0.25]], [0.25, 0.75], 4.0, [1, 0.5, 0, 1], 1, 0.2),
}


@pytest.mark.parametrize("key", list(FUSED_EVERY))
def test_fused_every_instantiation_against_live_oracle(B, key):
    lat, kf, kw, ecut, occ, kind, mu = FUSED_EVERY[key]
    n = int(str(key).rstrip("a"))
    lattice = W.cubic(lat[1]) if lat[0] == "sc" else W.rhombohedral(lat[1], lat[2])
    w = W.custom("fused%s" % key, 31 + n, (n, n, n), lattice, kf, kw, ecut, len(occ), occ, kind, mu)
    o, g = _pair(B, w)
    psi = w.coefficients(o.npw)
    want = o.apply(psi, w.occ)
    e_want, _ = o.energy(psi, w.occ, want)
    pd = g.to_device(psi)
    g.set_option(B.EXX_OPT_PRUNE, 0)
    out = g.apply(pd, w.occ)
    assert g.get_info(B.EXX_INFO_WORK_GRID) == n and g.get_info(B.EXX_INFO_PATH_USED) == 2
    assert g.get_info(B.EXX_INFO_SYMMETRY) == (0 if str(key).endswith("a") else 1)
    got = out.cpu().numpy()
    for k in range(w.nk):
        for b in range(w.nbands):
            assert _rel(o.band(got, k, b), o.band(want, k, b)) < TOL_VX, (key, k, b)
    e, _ = g.energy(pd, w.occ, out)
    assert abs(e - e_want) <= TOL_EX * abs(e_want)
    g.close()


# ---------------------------------------------------------------------------------------------------------------
# S8(f)-2: mixed precision (EXX_OPT_PRECISION = 1): fp32 pair transforms, fp64 S1 / S7 / accumulators.  The paper's own bar
# for this mode is 1e-5 relative agreement with fp64; the fp64 bars above do not apply to it.
@pytest.mark.parametrize("name", ["C2", "C3", "C4a"])
def test_mixed_precision_agrees_with_fp64_within_paper_bar(B, name):
    w = W.make(name)
    g = B.Exx.from_workload(w)
    psi = w.coefficients(g.npw)
    pd = g.to_device(psi)
    out64 = g.apply(pd, w.occ).clone()
    e64, _ = g.energy(pd, w.occ, out64)
    assert g.get_info(B.EXX_INFO_PRECISION) == 0
    g.set_option(B.EXX_OPT_PRECISION, 1)
    out32 = g.apply(pd, w.occ)
    assert g.get_info(B.EXX_INFO_PRECISION) == 1 and g.get_info(B.EXX_INFO_PAIRS_ORDERED) == w.pair_evals
    e32, _ = g.energy(pd, w.occ, out32)
    a, b = out32.cpu().numpy(), out64.cpu().numpy()
    worst = max(_rel(g.band(a, k, n), g.band(b, k, n)) for k in range(w.nk) for n in range(w.nbands))
    assert worst < 1e-5, worst
    assert abs(e32 - e64) <= 1e-6 * abs(e64)
    # and it is a different computation, not the fp64 path under another name
    assert worst > 1e-9
    g.set_option(B.EXX_OPT_PRECISION, 0)
    again = g.apply(pd, w.occ)
    assert np.array_equal(again.cpu().numpy().view(np.float64), b.view(np.float64))
    g.close()


def test_mixed_precision_against_oracle_small(B):
    w = W.custom("mixed48", 77, (48, 48, 48), W.rhombohedral(8.0, 64.0), [[0.25, 0.25, 0.25], [-0.25, 0.25, 0.0]], [0.5, 0.5], 6.0, 4,
                 [1.0, 1.0, 0.5, 0.0])
    o, g = _pair(B, w)
    psi = w.coefficients(o.npw)
    want = o.apply(psi, w.occ)
    e_want, _ = o.energy(psi, w.occ, want)
    pd = g.to_device(psi)
    for sym in (1, 0):
        g.set_option(B.EXX_OPT_SYMMETRY, sym)
        g.set_option(B.EXX_OPT_PRECISION, 1)
        out = g.apply(pd, w.occ)
        got = out.cpu().numpy()
        for k in range(w.nk):
            for n in range(w.nbands):
                assert _rel(o.band(got, k, n), o.band(want, k, n)) < 1e-5
        e, _ = g.energy(pd, w.occ, out)
        assert abs(e - e_want) <= 1e-6 * abs(e_want)
    g.close()


def test_mixed_precision_dual_sweep_against_two_sweeps(B):
    """In mixed mode the dual sweep sums the second side's products over the (at most RG) rows of a row group in fp32 before they
    reach the fp64 accumulators, while two sweeps add every product into fp64 directly: the two differ at fp32 rounding level
    (not at 1e-13 like in fp64 mode) and both stay inside the mode's bar against the oracle."""
    w = W.custom("mixed48d", 78, (48, 48, 48), W.rhombohedral(8.0, 64.0), [[0.25, 0.25, 0.25], [-0.25, 0.25, 0.0]], [0.5, 0.5], 6.0, 6,
                 [1.0, 1.0, 0.5, 0.0, 1.0, 0.25])
    o, g = _pair(B, w)
    psi = w.coefficients(o.npw)
    want = o.apply(psi, w.occ)
    pd = g.to_device(psi)
    g.set_option(B.EXX_OPT_PRUNE, 0)          # stay on 48^3, which has a dual kernel
    g.set_option(B.EXX_OPT_PRECISION, 1)
    outs = {}
    for dual in (1, 0):
        g.set_option(B.EXX_OPT_DUAL_SWEEP, dual)
        outs[dual] = g.apply(pd, w.occ).cpu().numpy()
        assert g.get_info(B.EXX_INFO_PRECISION) == 1 and g.get_info(B.EXX_INFO_SYMMETRY) == 1
        assert (g.kernel_times()["fused_pass_r"][1] > 0) == bool(dual)
        for k in range(w.nk):
            for n in range(w.nbands):
                assert _rel(o.band(outs[dual], k, n), o.band(want, k, n)) < 1e-5
    worst = max(_rel(o.band(outs[1], k, n), o.band(outs[0], k, n)) for k in range(w.nk) for n in range(w.nbands))
    assert worst < 2e-6, worst
    g.close()


# ---------------------------------------------------------------------------------------------------------------
# S8(f)-3: stand-alone batched 3-D transform through the fused passes
@pytest.mark.parametrize("n", [16, 32, 40, 48, 64, 72, 80])
def test_fft3d_fused_against_oracle_fft(B, n):
    import torch
    g = B.Exx((n, n, n), W.cubic(10.0), np.zeros((1, 3)), [1.0], 2.0, nbands=1)
    fidx = g.findex()
    assert np.array_equal(np.sort(fidx), np.arange(n ** 3, dtype=np.int32))
    rng = np.random.default_rng(n)
    nbatch = 3
    x = rng.standard_normal((nbatch, n, n, n)) + 1j * rng.standard_normal((nbatch, n, n, n))
    xin = torch.from_numpy(x.reshape(-1).copy()).cuda()
    out = torch.empty_like(xin)
    g.fft3d_fused(xin, nbatch, -1, out)
    assert np.array_equal(xin.cpu().numpy(), x.reshape(-1))            # forward leaves its input alone
    got = out.cpu().numpy().reshape(nbatch, -1)
    for b in range(nbatch if n < 64 else 1):
        want = R.fft3d(x[b], -1).reshape(-1)
        assert _rel(got[b][fidx], want) < 2e-15 * np.log2(n ** 3)
    # inverse of the forward gives back Ng * x
    back = torch.empty_like(xin)
    g.fft3d_fused(out, nbatch, +1, back)
    assert _rel(back.cpu().numpy(), x.reshape(-1) * n ** 3) < 1e-14
    # agrees with the generic natural-order transform of the library too
    ref = xin.clone()
    g.fft3d(ref, nbatch, -1)
    assert _rel(got[:, fidx].reshape(-1), ref.cpu().numpy()) < 1e-14
    g.close()


def test_fft3d_fused_refuses_unsupported_grids(B):
    import torch
    g = B.Exx((12, 18, 16), W.cubic(6.0), np.zeros((1, 3)), [1.0], 2.0, nbands=1)
    a = torch.zeros(g.ng, dtype=torch.complex128, device="cuda")
    with pytest.raises(B.ExxError) as ei:
        g.fft3d_fused(a, 1, -1, torch.empty_like(a))
    assert ei.value.code == -2
    g.close()


@pytest.mark.parametrize("n", [72, 48])
def test_fused_small_batches_dual_and_two_sweeps(B, n):
    """The fused kernels of the benchmarked instantiation (N = 72: R1 = 9, dual sweep with 4 rows per CTA; N = 48: R1 = 6) on a
    problem small enough for the full oracle and for compute-sanitizer (profiles/r2_sanitizer.md): 5 bands cut into 3 x 3 batches
    (a diagonal batch, an off-diagonal one, a ragged last one), an empty band and a half-filled one, pair symmetry with the dual
    sweep and with two sweeps, and no symmetry."""
    w = W.custom("small%d" % n, 7200 + n, (n, n, n), W.cubic(10.0), [[0, 0, 0]], [1.0], 6.0, 5, [1.0, 1.0, 0.5, 0.0, 1.0])
    o, g = _pair(B, w)
    psi = w.coefficients(o.npw)
    want = o.apply(psi, w.occ)
    e_want, pb_want = o.energy(psi, w.occ, want)
    pd = g.to_device(psi)
    g.set_option(B.EXX_OPT_PRUNE, 0)
    g.set_option(B.EXX_OPT_TILE_N, 3)
    g.set_option(B.EXX_OPT_TILE_M, 3)
    outs = []
    import torch
    pad = 4096
    guard = torch.full((g.ncoef + 2 * pad,), float("nan"), dtype=torch.complex128, device="cuda")   # `out` between NaN canaries
    for sym, dual in ((1, 1), (1, 0), (0, 1)):
        g.set_option(B.EXX_OPT_SYMMETRY, sym)
        g.set_option(B.EXX_OPT_DUAL_SWEEP, dual)
        out = g.apply(pd, w.occ, guard[pad:pad + g.ncoef])
        torch.cuda.synchronize()
        assert bool(torch.isnan(guard[:pad].real).all()) and bool(torch.isnan(guard[pad + g.ncoef:].real).all())   # nothing written outside out
        assert not bool(torch.isnan(out.real).any())
        assert g.get_info(B.EXX_INFO_PATH_USED) == 2 and g.get_info(B.EXX_INFO_WORK_GRID) == n and g.get_info(B.EXX_INFO_SYMMETRY) == sym
        assert g.get_info(B.EXX_INFO_PAIRS_ORDERED) == w.pair_evals
        got = out.cpu().numpy()
        for b in range(w.nbands):
            assert _rel(o.band(got, 0, b), o.band(want, 0, b)) < TOL_VX, (n, sym, dual, b)
        e, pb = g.energy(pd, w.occ, out)
        assert abs(e - e_want) <= TOL_EX * abs(e_want) and np.abs(pb - pb_want).max() <= TOL_EX * abs(e_want)
        outs.append(got)
        out2 = g.apply(pd, w.occ)                       # fixed summation order: bit-identical from run to run
        assert np.array_equal(out2.cpu().numpy(), got)
    assert _rel(outs[0], outs[1]) < 1e-13 and _rel(outs[0], outs[2]) < 1e-13
    g.close()


def test_sphere_pruned_transforms_are_bit_identical(B):
    """EXX_OPT_PRUNE_SPHERE (S1 reads / S7 writes only the x rows of the frequency box that can hold sphere coefficients) changes
    no bit of V_x psi or E_x, with k-points (spheres shifted per k: the row mask is the union) and on a compact work grid."""
    for w in (W.custom("prune48", 4811, (48, 48, 48), W.rhombohedral(8.0, 64.0), [[0.25, 0.25, 0.25], [-0.25, 0.25, 0.0]], [0.5, 0.5], 6.0, 4,
                       [1.0, 1.0, 0.5, 0.0]), W.make("C2")):
        o, g = _pair(B, w)
        psi = w.coefficients(o.npw)
        pd = g.to_device(psi)
        res = []
        for val in (1, 0):
            g.set_option(B.EXX_OPT_PRUNE_SPHERE, val)
            assert g.get_option(B.EXX_OPT_PRUNE_SPHERE) == val
            out = g.apply(pd, w.occ)
            res.append((out.cpu().numpy(), g.energy(pd, w.occ, out)[0], g.energy(pd, w.occ, None)[0]))
        assert np.array_equal(res[0][0], res[1][0]) and res[0][1] == res[1][1] and res[0][2] == res[1][2]
        if w.name != "C2":
            want = o.apply(psi, w.occ)
            for k in range(w.nk):
                for n in range(w.nbands):
                    assert _rel(o.band(res[0][0], k, n), o.band(want, k, n)) < TOL_VX
        g.close()


def test_measured_fp64_peak_is_plausible(B):
    """exx_measure_fp64_peak (bench.py's fp64 roofline denominator): a B200 delivers 25-40 TFLOP/s of fp64 FMA depending on its clocks."""
    gf = B.measure_fp64_peak()
    assert 1.0e4 < gf < 6.0e4, gf


def test_fused_degenerate_cases(B):
    """Fused path edge cases: a single band, all occupations zero, one occupied band among empties."""
    import torch
    for nb, occ in ((1, [1.0]), (3, [0.0, 0.0, 0.0]), (5, [0.0, 0.0, 0.7, 0.0, 0.0])):
        w = W.custom("deg48", 31 + nb, (48, 48, 48), W.cubic(8.0), [[0, 0, 0]], [1.0], 5.0, nb, occ)
        o, g = _pair(B, w)
        psi = w.coefficients(o.npw)
        want = o.apply(psi, w.occ)
        pd = g.to_device(psi)
        for sym in (1, 0):
            g.set_option(B.EXX_OPT_SYMMETRY, sym)
            out = g.apply(pd, w.occ)
            assert g.get_info(B.EXX_INFO_PATH_USED) == 2
            assert g.get_info(B.EXX_INFO_PAIRS_ORDERED) == w.pair_evals
            got = out.cpu().numpy()
            if not any(occ):
                assert float(np.abs(got).max()) == 0.0 and g.get_info(B.EXX_INFO_PAIRS_EXECUTED) == 0
                assert g.energy(pd, w.occ, out)[0] == 0.0
            else:
                for n in range(nb):
                    assert _rel(o.band(got, 0, n), o.band(want, 0, n)) < TOL_VX, (nb, sym, n)
                e, _ = g.energy(pd, w.occ, out)
                e_want, _ = o.energy(psi, w.occ, want)
                assert abs(e - e_want) <= TOL_EX * abs(e_want)
        g.close()


# ---------------------------------------------------------------------------------------------------------------
# E_x from psi alone: the pair-density route (E2), EXX_OPT_ENERGY_ROUTE = 0
@pytest.mark.parametrize("tile", [0, 5])
def test_energy_route_ragged_tiles_occupation_holes_kpoints(B, tile):
    """Every combination the batch logic has: k-points with unequal weights, fractional and zero occupations, ragged tiles,
    pair symmetry on and off, against the oracle's (E1) and its independent (E2); bitwise reproducible."""
    nb = 19
    occ = np.array([1, 0, 1, 0.5, 0, 0, 1, 1, 0.25, 0, 1, 0, 0, 0, 1, 0.75, 0, 0, 0], dtype=float)
    w = W.custom("ragged48", 2024, (48, 48, 48), W.rhombohedral(7.5, 66.0), [[0.0, 0.0, 0.0], [0.25, -0.25, 0.5]], [0.4, 0.6], 5.0, nb, occ)
    o, g = _pair(B, w)
    psi = w.coefficients(o.npw)
    e_want, pb_want = o.energy(psi, w.occ, o.apply(psi, w.occ))
    e2_want = o.energy_e2(psi, w.occ)
    assert abs(e2_want - e_want) <= 1e-12 * abs(e_want)
    pd = g.to_device(psi)
    nocc = int((np.asarray(w.occ) != 0).reshape(w.nk, nb).sum(axis=1)[0])
    for sym in (1, 0):
        g.set_option(B.EXX_OPT_SYMMETRY, sym)
        g.set_option(B.EXX_OPT_TILE_N, tile)
        g.set_option(B.EXX_OPT_TILE_M, tile)
        e, pb = g.energy(pd, w.occ, None)
        assert g.get_info(B.EXX_INFO_ENERGY_ROUTE) == 2 and g.get_info(B.EXX_INFO_SYMMETRY) == sym
        # only pairs of two occupied bands are transformed
        assert g.get_info(B.EXX_INFO_PAIRS_ORDERED) == (w.nk * nocc) ** 2
        assert g.get_info(B.EXX_INFO_PAIRS_EXECUTED) == ((w.nk * nocc) * (w.nk * nocc + 1) // 2 if sym else (w.nk * nocc) ** 2)
        assert abs(e - e_want) <= TOL_EX * abs(e_want) and abs(e - e2_want) <= TOL_EX * abs(e_want)
        assert np.abs(pb - pb_want).max() <= TOL_EX * abs(e_want)
        assert np.all(pb[np.asarray(w.occ) == 0] == 0.0) and abs(pb.sum() - e) <= 1e-14 * abs(e)
        e_again, pb_again = g.energy(pd, w.occ, None)
        assert e_again == e and np.array_equal(pb_again, pb)
    assert g.energy(pd, np.zeros(w.nk * nb), None)[0] == 0.0
    g.close()


@pytest.mark.parametrize("name", ["C2", "C3", "C4a", "C4b", "C5"])
def test_energy_route_full_size_against_golden(B, name):
    """At BASELINE's full sizes, in the default launch configuration: E_x and the per-band terms of the pair-density route
    against the stored oracle values (E1 and E2 of tests/golden/make_golden.py)."""
    w = W.make(name)
    gold = json.load(open(os.path.join(GOLD, "exx_%s.json" % name)))
    g = B.Exx.from_workload(w)
    psi = w.coefficients(g.npw)
    pd = g.to_device(psi)
    e, pb = g.energy(pd, w.occ, None)
    assert g.get_info(B.EXX_INFO_ENERGY_ROUTE) == 2 and g.get_info(B.EXX_INFO_PATH_USED) == 2
    nocc = int((np.asarray(w.occ) != 0).sum())
    assert g.get_info(B.EXX_INFO_PAIRS_ORDERED) == nocc * nocc
    assert e < 0 and np.all(pb <= 0) and abs(pb.sum() - e) <= 1e-13 * abs(e)
    for i, (k, n) in enumerate(gold["rows"]):
        assert abs(pb[k * w.nbands + n] - gold["row_energy"][i]) <= TOL_EX * abs(gold["row_energy"][i]) + 1e-300
    if "E_x_E1" in gold:
        assert abs(e - gold["E_x_E1"]) <= TOL_EX * abs(gold["E_x_E1"])
        assert abs(e - gold["E_x_E2"]) <= TOL_EX * abs(gold["E_x_E2"])
        assert np.abs(pb - np.array(gold["per_band_energy"])).max() <= TOL_EX * abs(gold["E_x_E1"])
    e_again, pb_again = g.energy(pd, w.occ, None)       # fixed summation order, no atomics: bit-identical
    assert e_again == e and np.array_equal(pb_again, pb)
    # and against this library's own V_x psi route
    g.set_option(B.EXX_OPT_ENERGY_ROUTE, 1)
    e1, pb1 = g.energy(pd, w.occ, None)
    assert g.get_info(B.EXX_INFO_ENERGY_ROUTE) == 1
    assert abs(e - e1) <= 1e-12 * abs(e1) and np.abs(pb - pb1).max() <= 1e-12 * abs(e1)
    g.close()


def test_energy_route_aliased_grid_generic_fallback_and_mixed_precision(B):
    # C1: fused kernels on an aliased grid (no pair symmetry): (E1) = (E2) holds on any grid (K' real, Parseval)
    w = W.make("C1")
    o, g = _pair(B, w)
    psi = w.coefficients(o.npw)
    e_want, pb_want = o.energy(psi, w.occ, o.apply(psi, w.occ))
    pd = g.to_device(psi)
    e, pb = g.energy(pd, w.occ, None)
    assert g.get_info(B.EXX_INFO_ENERGY_ROUTE) == 2 and g.get_info(B.EXX_INFO_SYMMETRY) == 0
    assert abs(e - e_want) <= TOL_EX * abs(e_want) and np.abs(pb - pb_want).max() <= TOL_EX * abs(e_want)
    # generic kernels asked for: no pair-density route there, the library falls back to V_x psi + (E1)
    g.set_option(B.EXX_OPT_PATH, 1)
    e, _ = g.energy(pd, w.occ, None)
    assert g.get_info(B.EXX_INFO_ENERGY_ROUTE) == 1 and g.get_info(B.EXX_INFO_PATH_USED) == 1
    assert abs(e - e_want) <= TOL_EX * abs(e_want)
    g.close()
    # mixed precision (not under the fp64 bars): fp32 transforms, fp64 sums
    w = W.make("C3")
    g = B.Exx.from_workload(w)
    pd = g.to_device(w.coefficients(g.npw))
    e64, _ = g.energy(pd, w.occ, None)
    g.set_option(B.EXX_OPT_PRECISION, 1)
    e32, _ = g.energy(pd, w.occ, None)
    assert g.get_info(B.EXX_INFO_PRECISION) == 1 and g.get_info(B.EXX_INFO_ENERGY_ROUTE) == 2
    assert 0 < abs(e32 - e64) <= 1e-5 * abs(e64)
    g.close()


# ---------------------------------------------------------------------------------------------------------------
# exx_apply_to: the operator of (psi, occ) applied to other vectors phi (FOCK_ACC on trial wavefunctions)
def _random_phi(w, npw_total, seed):
    rng = np.random.default_rng(seed)
    return rng.standard_normal(npw_total) + 1j * rng.standard_normal(npw_total)


@pytest.mark.parametrize("name", ["kpts_frac_occ", "noncubic_hse", "tiny_aliased", "one_band", "mixed_27"])
def test_apply_to_small_cases_against_oracle(B, name):
    """Fused kernels on the compact grid, generic kernels (EXX_OPT_PATH = 1, pruning off) and shards: V_x[psi, occ] phi per vector
    at the 1e-10 bar against the oracle's exx_ref_apply_to."""
    import torch
    w = _small(name)
    o, g = _pair(B, w)
    psi = w.coefficients(o.npw)
    phi = _random_phi(w, o.ncoef, 31)
    want = o.apply_to(psi, w.occ, phi)
    pd, fd = g.to_device(psi), g.to_device(phi)
    for path, prune, P in ((0, 1, 1), (1, 0, 1), (0, 1, 2), (0, 0, 3)):
        g.set_option(B.EXX_OPT_PATH, path)
        g.set_option(B.EXX_OPT_PRUNE, prune)
        acc = None
        for r in range(P):
            g.set_option(B.EXX_OPT_SHARD_COUNT, P)
            g.set_option(B.EXX_OPT_SHARD_RANK, r)
            part = g.apply_to(pd, w.occ, fd).clone()
            acc = part if acc is None else acc + part
        g.set_option(B.EXX_OPT_SHARD_COUNT, 1)
        g.set_option(B.EXX_OPT_SHARD_RANK, 0)
        assert g.get_info(B.EXX_INFO_SYMMETRY) == 0
        got = acc.cpu().numpy()
        for k in range(w.nk):
            for n in range(w.nbands):
                assert _rel(o.band(got, k, n), o.band(want, k, n)) < TOL_VX, (name, path, prune, P, k, n)
    # phi = psi is exx_apply
    a, b = g.apply(pd, w.occ).clone(), g.apply_to(pd, w.occ, pd)
    assert (a - b).abs().max().item() <= 1e-13 * a.abs().max().item()
    with pytest.raises(B.ExxError):
        g.apply_to(pd, w.occ, fd, fd)      # out may not alias phi
    g.close()


def test_apply_to_fused_kpoints_ragged_tiles(B):
    nb = 11
    occ = np.array([1, 0, 1, 0.5, 0, 0, 1, 1, 0.25, 0, 0.75], dtype=float)
    w = W.custom("to48", 4048, (48, 48, 48), W.rhombohedral(7.5, 66.0), [[0.0, 0.0, 0.0], [0.25, -0.25, 0.5]], [0.4, 0.6], 5.0, nb, occ, 1, 0.2)
    o, g = _pair(B, w)
    psi = w.coefficients(o.npw)
    phi = _random_phi(w, o.ncoef, 32)
    want = o.apply_to(psi, w.occ, phi)
    pd, fd = g.to_device(psi), g.to_device(phi)
    # blocks of 1, 3 and nb + 2 trial vectors per k-point (FOCK_ACC's NSIM blocks), default and small ragged tiles, generic path
    tot = int(sum(o.npw))
    for nphi, tile, path in ((1, 0, 0), (3, 2, 0), (nb + 2, 3, 0), (3, 0, 1)):
        blk = _random_phi(w, nphi * tot, 40 + nphi)
        want_b = o.apply_to(psi, w.occ, blk)
        g.set_option(B.EXX_OPT_TILE_N, tile)
        g.set_option(B.EXX_OPT_TILE_M, tile)
        g.set_option(B.EXX_OPT_PATH, path)
        got_b = g.apply_to(pd, w.occ, g.to_device(blk)).cpu().numpy()
        assert g.get_info(B.EXX_INFO_PAIRS_ORDERED) == w.nk * w.nk * nphi * w.nocc
        pos = 0
        for k in range(w.nk):
            for i in range(nphi):
                sl = slice(pos, pos + o.npw[k])
                pos += o.npw[k]
                assert _rel(got_b[sl], want_b[sl]) < TOL_VX, (nphi, tile, path, k, i)
        # the projected operator <phi_i|V_x phi_j> of the block (exx_subspace_block, DMMA) against numpy on the oracle's vectors
        vd = g.to_device(want_b)
        pos = 0
        for k in range(w.nk):
            P = blk[pos:pos + nphi * o.npw[k]].reshape(nphi, o.npw[k])
            V = want_b[pos:pos + nphi * o.npw[k]].reshape(nphi, o.npw[k])
            pos += nphi * o.npw[k]
            M = g.subspace_block(k, g.to_device(blk), vd).cpu().numpy()
            Mw = P.conj() @ V.T
            assert np.abs(M - Mw).max() <= 1e-13 * np.abs(Mw).max(), (nphi, k)
            assert np.abs(Mw - Mw.conj().T).max() <= 1e-12 * np.abs(Mw).max()
    g.set_option(B.EXX_OPT_PATH, 0)
    # EXX_OPT_KEEP_U: psi unchanged between calls -> S1 of psi skipped, same bits; a changed psi with the option off is picked up
    g.set_option(B.EXX_OPT_TILE_N, 0)
    g.set_option(B.EXX_OPT_TILE_M, 0)
    blk = g.to_device(_random_phi(w, 2 * tot, 50))
    first = g.apply_to(pd, w.occ, blk).clone()
    n_first = g.get_info(B.EXX_INFO_LAUNCHES)
    g.set_option(B.EXX_OPT_KEEP_U, 1)
    kept = g.apply_to(pd, w.occ, blk)
    assert g.get_info(B.EXX_INFO_LAUNCHES) < n_first and bool((kept == first).all())
    e_keep, _ = g.energy(pd, w.occ, None)
    g.set_option(B.EXX_OPT_KEEP_U, 0)
    assert e_keep == g.energy(pd, w.occ, None)[0]
    other = g.apply_to(pd * (0.5 + 0.5j), w.occ, blk)       # |0.5 + 0.5i|^2 = 1/2: the operator is quadratic in the orbitals
    assert (other - 0.5 * first).abs().max().item() <= 1e-13 * first.abs().max().item()
    for tile in (0, 3):
        g.set_option(B.EXX_OPT_TILE_N, tile)
        g.set_option(B.EXX_OPT_TILE_M, tile)
        out = g.apply_to(pd, w.occ, fd)
        assert g.get_info(B.EXX_INFO_PATH_USED) == 2 and g.get_info(B.EXX_INFO_PAIRS_ORDERED) == w.pair_evals
        got = out.cpu().numpy()
        for k in range(w.nk):
            for n in range(nb):
                assert _rel(o.band(got, k, n), o.band(want, k, n)) < TOL_VX, (tile, k, n)
        again = g.apply_to(pd, w.occ, fd).cpu().numpy()
        assert np.array_equal(again.view(np.float64), got.view(np.float64))
    g.close()


def test_apply_to_C3_full_size_properties_and_sampled_rows(B):
    """BASELINE configs[2] at full size (64 bands, 64^3, HSE): trial vectors = random vectors; two of them against the oracle row by
    row (the oracle's apply_to on a problem padded with zero vectors would take minutes, so the rows are obtained from
    exx_ref_apply_rows on an extended orbital set with the trial vector appended at zero occupation), and the operator
    identities that hold at any size: linearity, Hermiticity of <phi_i|V_x phi_j> (exx_subspace), phi = psi equals exx_apply."""
    w = W.make("C3")
    g = B.Exx.from_workload(w)
    psi = w.coefficients(g.npw)
    pd = g.to_device(psi)
    phi = _random_phi(w, g.ncoef, 33)
    fd = g.to_device(phi)
    vphi = g.apply_to(pd, w.occ, fd).clone()
    a = g.apply(pd, w.occ).clone()
    b = g.apply_to(pd, w.occ, pd)
    assert (a - b).abs().max().item() <= 1e-13 * a.abs().max().item()
    lin = g.apply_to(pd, w.occ, 0.5 * fd + (0.25 - 1.0j) * pd)
    assert (lin - (0.5 * vphi + (0.25 - 1.0j) * a)).abs().max().item() <= 1e-13 * vphi.abs().max().item()
    M = g.subspace(0, fd, vphi).cpu().numpy()
    assert np.abs(M - M.conj().T).max() <= 1e-12 * np.abs(M).max()
    assert np.linalg.eigvalsh(0.5 * (M + M.conj().T)).max() <= 1e-12 * np.abs(M).max()
    # sampled rows against the oracle: a context with one more band, the trial vector stored there with f = 0 (reading A16:
    # an empty band still receives V_x, and contributes nothing as m)
    o = R.RefExx(w.grid, w.lattice, w.kfrac, w.kweight, w.ecut, w.kernel_kind, w.mu, w.scale, w.nbands + 1)
    got = vphi.cpu().numpy()
    npw = g.npw[0]
    for i in (0, 41):
        ext = np.concatenate([psi, phi[i * npw:(i + 1) * npw]])
        occ_ext = np.concatenate([w.occ, [0.0]])
        row = o.apply_rows(ext, occ_ext, [(0, w.nbands)])[0]
        assert _rel(got[i * npw:(i + 1) * npw], row) < TOL_VX, i
    g.close()
