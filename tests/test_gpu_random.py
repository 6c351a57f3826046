"""GPU parity on seeded random problems (-m gpu): cell, grid (fused and generic), k-points and weights, cutoff, kernel, band count,
occupations that differ from k-point to k-point, and every option that changes how the work is cut up (pair symmetry, dual sweep, compact grid,
batch tiles, generic kernels, shards).  Each case: V_x psi per band at 1e-10 and E_x / per-band terms at 1e-11 against the oracle,
for the shards' sum, for (E1) from the summed V_x psi and for the pair-density route from psi alone; then exx_apply_to on random trial vectors.
"""
import numpy as np
import pytest

from oracle import exx_ref as R
from paper_1111_0716_b200 import workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1111_0716_b200 import binding
    binding.lib()
    return binding


def _case(seed):
    rng = np.random.default_rng(seed)
    if rng.random() < 0.7:
        n = int(rng.choice([16, 32, 40, 48, 24, 20]))
        grid = (n, n, n)
    else:
        grid = tuple(int(x) for x in rng.choice([8, 9, 10, 12, 15, 16, 18, 20, 24], 3))
    lat = W.rhombohedral(float(rng.uniform(5, 9)), float(rng.uniform(58, 88))) if rng.random() < 0.6 else W.cubic(float(rng.uniform(5, 10)))
    nk = int(rng.choice([1, 1, 2, 3]))
    kf = rng.uniform(-0.5, 0.5, (nk, 3)) if rng.random() < 0.7 else rng.choice([0.0, 0.25, -0.25, 0.5], (nk, 3))
    if nk == 1 and rng.random() < 0.5:
        kf[:] = 0
    kw = rng.uniform(0.2, 1.0, nk)
    kw /= kw.sum()
    nb = int(rng.integers(1, 14))
    ecut = float(rng.uniform(1.5, 6.0))
    kind = int(rng.integers(0, 2))
    mu = float(rng.uniform(0.1, 0.5)) if kind else 0.0
    w = W.custom("rnd%d" % seed, seed, grid, lat, kf, kw, ecut, nb, np.ones(nb), kind, mu, float(rng.choice([1.0, 0.25])))
    occ = rng.choice([0.0, 1.0, 1.0, 0.5, 0.3], nk * nb).astype(np.float64)   # per k-point
    if rng.random() < 0.1:
        occ[:] = 0
    opts = dict(sym=int(rng.integers(0, 2)), prune=int(rng.integers(0, 2)), tn=int(rng.choice([0, 1, 2, 3, 5, 8])),
                tm=int(rng.choice([0, 1, 2, 3, 5, 8])), path=int(rng.choice([0, 0, 0, 1])), P=int(rng.choice([1, 1, 2, 3])))
    opts["dual"] = int(rng.integers(0, 2))   # drawn last: the cases of the earlier options are unchanged
    return w, occ, opts


@pytest.mark.parametrize("block", range(6))
def test_random_problems_against_oracle(B, block):
    ran = 0
    rng_phi = np.random.default_rng(9000 + block)
    for seed in range(20 * block, 20 * block + 20):
        w, occ, opts = _case(seed)
        o = R.RefExx(w.grid, w.lattice, w.kfrac, w.kweight, w.ecut, w.kernel_kind, w.mu, w.scale, w.nbands)
        try:
            g = B.Exx.from_workload(w)
        except B.ExxError as e:          # the random cutoff sphere does not fit the random box
            assert e.code == -2, (seed, e)
            continue
        psi = w.coefficients(o.npw)
        want = o.apply(psi, occ)
        e_want, pb_want = o.energy(psi, occ, want)
        tol_e = 1e-11 * abs(e_want)
        pd = g.to_device(psi)
        g.set_option(B.EXX_OPT_SYMMETRY, opts["sym"])
        g.set_option(B.EXX_OPT_PRUNE, opts["prune"])
        g.set_option(B.EXX_OPT_TILE_N, opts["tn"])
        g.set_option(B.EXX_OPT_TILE_M, opts["tm"])
        g.set_option(B.EXX_OPT_PATH, opts["path"])
        g.set_option(B.EXX_OPT_DUAL_SWEEP, opts["dual"])
        acc, e_parts, pb_parts = None, 0.0, 0.0
        for r in range(opts["P"]):
            g.set_option(B.EXX_OPT_SHARD_COUNT, opts["P"])
            g.set_option(B.EXX_OPT_SHARD_RANK, r)
            part = g.apply(pd, occ).clone()
            acc = part if acc is None else acc + part
            e_r, pb_r = g.energy(pd, occ, None)
            e_parts, pb_parts = e_parts + e_r, pb_parts + pb_r
        g.set_option(B.EXX_OPT_SHARD_COUNT, 1)
        g.set_option(B.EXX_OPT_SHARD_RANK, 0)
        got = acc.cpu().numpy()
        for k in range(w.nk):
            for n in range(w.nbands):
                a, b = o.band(got, k, n), o.band(want, k, n)
                assert np.linalg.norm(a - b) <= 1e-10 * np.linalg.norm(b), (seed, opts, k, n)
        e, pb = g.energy(pd, occ, acc)
        assert abs(e - e_want) <= tol_e and np.abs(pb - pb_want).max() <= tol_e, (seed, opts)
        assert abs(e_parts - e_want) <= tol_e and np.abs(pb_parts - pb_want).max() <= tol_e, (seed, opts)
        # the same operator on random trial vectors (exx_apply_to), same options
        nphi, tot = int(rng_phi.integers(1, w.nbands + 3)), int(sum(o.npw))          # a block of nphi trial vectors per k-point
        phi = rng_phi.standard_normal(nphi * tot) + 1j * rng_phi.standard_normal(nphi * tot)
        want_phi = o.apply_to(psi, occ, phi)
        got_phi = g.apply_to(pd, occ, g.to_device(phi)).cpu().numpy()
        pos = 0
        for k in range(w.nk):
            for n in range(nphi):
                a, b = got_phi[pos:pos + o.npw[k]], want_phi[pos:pos + o.npw[k]]
                pos += o.npw[k]
                assert np.linalg.norm(a - b) <= 1e-10 * np.linalg.norm(b) + 1e-300, (seed, opts, "apply_to", nphi, k, n)
        g.close()
        ran += 1
    assert ran >= 15
