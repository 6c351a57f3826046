"""S8(f)-4 on one GPU (-m gpu): the shards of an apply, run one after the other on the same device, add up to the unsharded
result and to the oracle; every shard executes exactly the pairs exx_shard_plan gives it; the NCCL exchange step runs in a
world of one.  (More than one GPU is never needed here: shards do not wait on one another.)"""
import os
import socket

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


CASES = {
    # fused path, k-points, pair symmetry, occupation holes, ragged band tiles (tile 4 -> several batches per k-pair)
    "fused48_kpts": dict(grid=(48, 48, 48), lat=("rh", 8.0, 64.0), kf=[[0.25, 0.25, 0.25], [-0.25, 0.25, 0.0]], kw=[0.5, 0.5],
                         ecut=6.0, nb=10, occ=[1, 1, 0.5, 0, 1, 1, 0.25, 0, 1, 1], kind=0, mu=0.0, tile=4),
    # compact work grid (64^3 caller grid -> 32^3) with HSE
    "compact64": dict(grid=(64, 64, 64), lat=("sc", 9.0), kf=[[0, 0, 0]], kw=[1.0], ecut=5.0, nb=9, occ=[1, 1, 1, 1, 0.5, 0.5, 0, 1, 1],
                      kind=1, mu=0.106, tile=4),
    # generic path (non-cubic grid): output rows are shared out
    "generic_rect": dict(grid=(12, 18, 16), lat=("rh", 7.3, 71.0), kf=[[0.1, -0.3, 0.25], [0.5, 0, 0]], kw=[0.5, 0.5], ecut=5.0,
                         nb=4, occ=[1, 0.7, 0, 0.2], kind=1, mu=0.3, tile=0),
}


def _make(name):
    s = CASES[name]
    lat = W.cubic(s["lat"][1]) if s["lat"][0] == "sc" else W.rhombohedral(s["lat"][1], s["lat"][2])
    return W.custom(name, 999 + len(name), s["grid"], lat, s["kf"], s["kw"], s["ecut"], s["nb"], s["occ"], s["kind"], s["mu"]), s["tile"]


@pytest.mark.parametrize("name", list(CASES))
@pytest.mark.parametrize("P", [2, 3])
def test_shards_add_up_to_the_full_apply_and_the_oracle(B, name, P):
    w, tile = _make(name)
    o = R.RefExx(w.grid, w.lattice, w.kfrac, w.kweight, w.ecut, w.kernel_kind, w.mu, w.scale, w.nbands)
    g = B.Exx.from_workload(w)
    if tile:
        g.set_option(B.EXX_OPT_TILE_N, tile)
        g.set_option(B.EXX_OPT_TILE_M, tile)
    psi = w.coefficients(o.npw)
    want = o.apply(psi, w.occ)
    e_want, _ = o.energy(psi, w.occ, want)
    pd = g.to_device(psi)
    full = g.apply(pd, w.occ).clone()
    fused = g.get_info(B.EXX_INFO_PATH_USED) == 2
    sym = g.get_info(B.EXX_INFO_SYMMETRY)
    total_exec = g.get_info(B.EXX_INFO_PAIRS_EXECUTED)
    plan = B.shard_plan(w.nk, w.nbands, w.occ, sym, tile, P)[0] if fused else None
    acc = None
    executed = []
    for r in range(P):
        g.set_option(B.EXX_OPT_SHARD_COUNT, P)
        g.set_option(B.EXX_OPT_SHARD_RANK, r)
        part = g.apply(pd, w.occ)
        executed.append(g.get_info(B.EXX_INFO_PAIRS_EXECUTED))
        acc = part.clone() if acc is None else acc + part
    assert sum(executed) == total_exec and all(e < total_exec for e in executed)
    # E_x from psi alone (pair-density route on the fused path, V_x psi + (E1) on the generic one): the shards' partial sums add up
    e_parts, pb_parts = [], []
    for r in range(P):
        g.set_option(B.EXX_OPT_SHARD_RANK, r)
        e_r, pb_r = g.energy(pd, w.occ, None)
        assert g.get_info(B.EXX_INFO_ENERGY_ROUTE) == (2 if fused else 1)
        e_parts.append(e_r)
        pb_parts.append(pb_r)
    assert abs(sum(e_parts) - e_want) <= 1e-11 * abs(e_want)
    assert np.abs(sum(pb_parts) - o.energy(psi, w.occ, want)[1]).max() <= 1e-11 * abs(e_want)
    if fused:
        assert executed == plan.tolist()
    g.set_option(B.EXX_OPT_SHARD_COUNT, 1)
    g.set_option(B.EXX_OPT_SHARD_RANK, 0)
    got, ref = acc.cpu().numpy(), full.cpu().numpy()
    for k in range(w.nk):
        for n in range(w.nbands):
            a, b, c = o.band(got, k, n), o.band(ref, k, n), o.band(want, k, n)
            assert np.linalg.norm(a - b) <= 1e-13 * np.linalg.norm(b)          # shards vs one GPU: summation order only
            assert np.linalg.norm(a - c) <= 1e-10 * np.linalg.norm(c)          # shards vs oracle: the north_star bar
    e, _ = g.energy(pd, w.occ, acc)
    assert abs(e - e_want) <= 1e-11 * abs(e_want)
    g.close()


def test_rank_out_of_range_is_an_error(B):
    w, _ = _make("generic_rect")
    g = B.Exx.from_workload(w)
    pd = g.to_device(w.coefficients(g.npw))
    g.set_option(B.EXX_OPT_SHARD_RANK, 2)
    with pytest.raises(B.ExxError):
        g.apply(pd, w.occ)
    g.set_option(B.EXX_OPT_SHARD_COUNT, 3)
    g.apply(pd, w.occ)
    with pytest.raises(B.ExxError):
        g.set_option(B.EXX_OPT_SHARD_COUNT, 0)
    g.close()


def test_apply_sharded_through_nccl_world_of_one(B):
    """The user-facing call (shard options + all-reduce over NCCL) in a process group of one rank: equals apply."""
    import torch
    import torch.distributed as dist
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    created = not dist.is_initialized()
    if created:
        dist.init_process_group("nccl", init_method="tcp://127.0.0.1:%d" % port, rank=0, world_size=1, device_id=torch.device("cuda:0"))
    try:
        w, tile = _make("fused48_kpts")
        g = B.Exx.from_workload(w)
        pd = g.to_device(w.coefficients(g.npw))
        a = g.apply(pd, w.occ).clone()
        b = g.apply_sharded(pd, w.occ)
        assert torch.equal(a, b)
        assert g.get_option(B.EXX_OPT_SHARD_COUNT) == 1 and g.get_option(B.EXX_OPT_SHARD_RANK) == 0
        # a partial result really goes through the collective: rank 0 of 2 as the only member doubles nothing and sums itself
        c = g.apply_sharded(pd, w.occ, world=2, rank=0)
        d = g.apply_sharded(pd, w.occ, world=2, rank=1)
        assert (c + d - a).abs().max().item() <= 1e-13 * a.abs().max().item()
        # the same for E_x from psi alone: partial sums through the collective
        e, pb = g.energy(pd, w.occ, None)
        e1, pb1 = g.energy_sharded(pd, w.occ)
        assert e1 == e and np.array_equal(pb1, pb)
        (e_a, pb_a), (e_b, pb_b) = g.energy_sharded(pd, w.occ, world=2, rank=0), g.energy_sharded(pd, w.occ, world=2, rank=1)
        assert abs(e_a + e_b - e) <= 1e-13 * abs(e) and np.abs(pb_a + pb_b - pb).max() <= 1e-13 * abs(e)
        assert g.get_option(B.EXX_OPT_SHARD_COUNT) == 1 and g.get_option(B.EXX_OPT_SHARD_RANK) == 0
        g.close()
    finally:
        if created:
            dist.destroy_process_group()


def test_shards_of_C4a_add_up_at_full_size(B):
    """BASELINE configs[3] (C4a, 160 bands, compact 72^3 grid, pair symmetry) cut into 8 shards, run one after the other: every
    shard executes the pairs the plan gives it, the shards' outputs add up to the one-GPU apply to 1e-13 per band, and the rows
    the oracle stored (and their energies) are met at 1e-10 / 1e-11."""
    import json
    import torch
    w = W.make("C4a")
    g = B.Exx.from_workload(w)
    pd = g.to_device(w.coefficients(g.npw))
    full = g.apply(pd, w.occ).clone()
    P = 8
    plan, _ = B.shard_plan(w.nk, w.nbands, w.occ, True, 0, P)
    acc = torch.zeros_like(full)
    part = g.empty_like_psi()
    for r in range(P):
        g.set_option(B.EXX_OPT_SHARD_COUNT, P)
        g.set_option(B.EXX_OPT_SHARD_RANK, r)
        g.apply(pd, w.occ, part)
        assert g.get_info(B.EXX_INFO_PAIRS_EXECUTED) == plan[r]
        acc += part
    g.set_option(B.EXX_OPT_SHARD_COUNT, 1)
    g.set_option(B.EXX_OPT_SHARD_RANK, 0)
    a, f = acc.cpu().numpy(), full.cpu().numpy()
    for n in range(w.nbands):
        assert np.linalg.norm(g.band(a, 0, n) - g.band(f, 0, n)) <= 1e-13 * np.linalg.norm(g.band(f, 0, n))
    # against the stored oracle rows (tests/golden/make_golden.py calls only oracle/): the north_star bars
    gdir = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
    gold = json.load(open(os.path.join(gdir, "exx_C4a.json")))
    rows = np.load(os.path.join(gdir, "exx_C4a_rows.npz"))
    e, pb = g.energy(pd, w.occ, acc)
    for i, (k, n) in enumerate(gold["rows"]):
        want = rows["row%d" % i]
        assert np.linalg.norm(g.band(a, k, n) - want) <= 1e-10 * np.linalg.norm(want)
        assert abs(pb[k * w.nbands + n] - gold["row_energy"][i]) <= 1e-11 * abs(gold["row_energy"][i])
    assert e < 0 and abs(pb.sum() - e) <= 1e-13 * abs(e)
    g.close()
