"""S8(f)-4, host side (no GPU): how the fused path's pair batches are shared out among shards (exx_shard_plan), and the
world-size-2 exchange step (one all-reduce of the sphere coefficients) over gloo."""
import json
import os
import socket
import subprocess
import sys

import numpy as np
import pytest

from paper_1111_0716_b200 import binding as B
from paper_1111_0716_b200 import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _brute(nk, nb, occ, sym):
    """pairs transformed and pass executions, counted pair by pair from the rule in include/exx.h / DESIGN.md 5.4"""
    occ = np.asarray(occ, float).reshape(nk, nb)
    pairs = passes = 0
    for k in range(nk):
        for q in range(nk):
            for a in range(nb):
                for b in range(nb):
                    fa, fb = occ[k, a], occ[q, b]
                    if sym:
                        if (k, a) > (q, b) or (fa == 0 and fb == 0):
                            continue
                        pairs += 1
                        passes += 2 + (fb != 0) + (fa != 0 and (k, a) != (q, b))
                    elif fb != 0:
                        pairs += 1
                        passes += 3
    return pairs, passes


@pytest.mark.parametrize("sym", [True, False])
@pytest.mark.parametrize("nk,nb,tile", [(1, 5, 0), (1, 37, 16), (3, 20, 7), (2, 33, 16), (1, 16, 16), (4, 9, 4)])
def test_plan_covers_every_pair_exactly_once(nk, nb, tile, sym):
    rng = np.random.default_rng(nk * 100 + nb)
    occ = rng.choice([0.0, 0.0, 0.5, 1.0, 1.0], size=nk * nb)
    want = _brute(nk, nb, occ, sym)
    for P in (1, 2, 3, 8, 64):
        pairs, passes = B.shard_plan(nk, nb, occ, sym, tile, P)
        assert pairs.sum() == want[0] and passes.sum() == want[1]
        assert (pairs >= 0).all() and pairs.shape == (P,)


def test_plan_balance_on_the_paper_shaped_workloads():
    # C4a (Gamma, 158 + 2 half occupied bands): 55 batches of <= 256 pairs; C4b: 36 k-pairs x 55/100 batches
    for name, bound in (("C4a", {2: 1.01, 4: 1.01, 8: 1.05}), ("C4b", {2: 1.001, 8: 1.001}), ("C5", {2: 1.01, 8: 1.03})):
        w = W.make(name)
        for P, mx in bound.items():
            _, passes = B.shard_plan(w.nk, w.nbands, w.occ, True, 0, P)
            assert passes.max() <= mx * passes.mean(), (name, P, passes)
    w = W.make("C4a")
    pairs, passes = B.shard_plan(1, 160, w.occ, True, 0, 1)
    assert pairs[0] == 160 * 161 // 2 and passes[0] == 2 * pairs[0] + 160 * 160        # every ordered pair accumulates once


def test_plan_is_deterministic_and_rejects_bad_arguments():
    occ = np.ones(40)
    a = B.shard_plan(2, 20, occ, True, 8, 3)
    b = B.shard_plan(2, 20, occ, True, 8, 3)
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1])
    for bad in (dict(nshards=0), dict(tile=33), dict(tile=-1)):
        kw = dict(symmetry=True, tile=0, nshards=2)
        kw.update(bad)
        with pytest.raises(B.ExxError):
            B.shard_plan(2, 20, occ, **kw)
    with pytest.raises(B.ExxError):
        B.shard_plan(2, 20, -occ, True, 0, 2)


WORKER = r"""
import os, sys, json
sys.path.insert(0, %r)
import numpy as np, torch, torch.distributed as dist
from paper_1111_0716_b200 import binding as B
rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
dist.init_process_group("gloo", rank=rank, world_size=world)
occ = np.r_[np.ones(30), 0.5, 0.0]
pairs, passes = B.shard_plan(1, 32, occ, True, 8, world)
# every rank computes the same plan
got = [None] * world
dist.all_gather_object(got, (pairs.tolist(), passes.tolist()))
same = all(g == got[0] for g in got)
# the exchange step: partial results (here: a stand-in with known sum) added over the ranks, complex128, in place
part = torch.arange(6, dtype=torch.float64).view(3, 2).contiguous()
part = torch.view_as_complex(part) * (rank + 1)
B.all_reduce_sum(part)
print(json.dumps({"rank": rank, "same": same, "pairs": pairs.tolist(), "sum": torch.view_as_real(part).reshape(-1).tolist()}))
dist.destroy_process_group()
"""


def test_exchange_step_gloo_world2(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER % ROOT)
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), WORLD_SIZE="2", LOCAL_RANK=str(r), MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True))
    outs = []
    for p in procs:
        o, e = p.communicate(timeout=180)
        assert p.returncode == 0, e[-2000:]
        outs.append(json.loads(o.strip().splitlines()[-1]))
    assert all(o["same"] for o in outs)
    assert outs[0]["pairs"] == outs[1]["pairs"] and sum(outs[0]["pairs"]) == _brute(1, 32, np.r_[np.ones(30), 0.5, 0.0], True)[0]
    assert all(o["sum"] == [3.0 * v for v in range(6)] for o in outs)      # (1 + 2) x the stand-in, on both ranks
