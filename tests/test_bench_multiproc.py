"""The N > 1 path of bench.py on the CPU (gloo, world_size 2): the path is "replicas only", so the only
multi-rank logic is the rank/world discovery and the max-over-ranks timing reduction; both are exercised here."""
import json
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys, json
sys.path.insert(0, %r)
import torch, torch.distributed as dist
import bench
rank, world, local = bench.dist_setup(2)
dist.init_process_group("gloo", rank=rank, world_size=world)
t = bench.max_over_ranks(10.0 + 5.0 * rank, world, torch.device("cpu"))
dist.barrier()
print(json.dumps({"rank": rank, "world": world, "local": local, "max": t}))
dist.destroy_process_group()
"""


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def test_max_over_ranks_gloo_world2(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER % ROOT)
    port = _free_port()
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), WORLD_SIZE="2", LOCAL_RANK=str(r), MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True))
    outs = []
    for p in procs:
        o, e = p.communicate(timeout=180)
        assert p.returncode == 0, e[-2000:]
        outs.append(json.loads(o.strip().splitlines()[-1]))
    assert sorted(o["rank"] for o in outs) == [0, 1]
    assert all(o["world"] == 2 and o["max"] == 15.0 for o in outs)   # every rank sees the slowest rank's time


def test_reference_arm_runs_on_rank0_only():
    """--impl reference under N > 1: rank 0 prints the line, the other ranks exit 0 without work."""
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0",
                        "--workload", "C1"], env=env, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0 and r.stdout.strip() == ""
    env["RANK"] = "0"
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0",
                        "--workload", "C1"], env=env, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0
    line = json.loads(r.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["unit"] == "pair-evals/s" and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["e2e"]["h2d_bytes_per_step"] == 0


def test_ncu_counters_are_refused_for_another_build(tmp_path, monkeypatch):
    """bench.py prints roofline.traffic / dram_frac / fp64_frac only from an ncu capture of the build it is running: a capture whose
    recorded source hash differs from libexx.so's stamp (or of another work grid) is refused with the reason, never rescaled."""
    sys.path.insert(0, ROOT)
    import bench
    cap = {"source": "test", "srchash": "abc", "work_grid": 72, "units_per_launch": {"fused_pass_a": 1},
           "dram_bytes_per_launch": {"fused_pass_a": 1.0}, "fp64_flops_per_launch": {"fused_pass_a": 1.0}}
    p = tmp_path / "cap.json"
    p.write_text(json.dumps(cap))
    monkeypatch.setattr(bench, "NCU_COUNTERS", str(p))
    monkeypatch.setattr(bench, "lib_source_hash", lambda: "abc")
    got, why = bench.ncu_counters(72 ** 3)
    assert got is not None and got["srchash"] == "abc" and "ncu_counters" in why
    got, why = bench.ncu_counters(96 ** 3)
    assert got is None and "work grid" in why
    monkeypatch.setattr(bench, "lib_source_hash", lambda: "other")
    got, why = bench.ncu_counters(72 ** 3)
    assert got is None and "another build" in why
    monkeypatch.setattr(bench, "NCU_COUNTERS", str(tmp_path / "missing.json"))
    got, why = bench.ncu_counters(72 ** 3)
    assert got is None and "no capture" in why
