#!/usr/bin/env python
"""bench.py — band-pair exchange evaluations per second for one full V_x application (+ E_x) on synthetic
boron-shaped workloads (BASELINE.json metric), one process per GPU.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C4a] [--impl ours|reference]

A step = one pass of the whole hot path (S1..S8 of DESIGN.md: scatter + inverse FFT of every band, all band pairs,
forward FFT + gather, energy reduction) over the workload.  `value` times it with psi already in HBM; `e2e` times the
same call through exx_apply_host with pinned HOST buffers (H2D of psi, D2H of V_x psi and E_x inside the timed region).
N > 1 runs N independent replicas by default (BASELINE.json north_star: one GPU, no sharding): weak
scaling, no collective on the data path; timing is barrier + max over ranks.  `--parallel shard` instead shares the pair
batches of ONE workload out over the N ranks (every rank holds psi, runs its batches, one NCCL all-reduce of
V_x psi per step): strong scaling.
`--impl reference` times the oracle (oracle/, plain CPU code, as it stands) on a bounded sample of the same workload.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_1111_0716_b200 import workloads as W  # noqa: E402

METRIC = "band_pair_exchange_evals_per_s"
UNIT = "pair-evals/s"


def read_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            d = json.load(open(p))
            return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler(threading.Thread):
    """nvidia-smi clocks / throttle reasons sampled during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.rows, self.stop_flag = index, [], False

    def run(self):
        while not self.stop_flag:
            try:
                out = subprocess.run(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q, "--format=csv,noheader,nounits"],
                                     capture_output=True, text=True, timeout=5).stdout.strip()
                if out:
                    self.rows.append([x.strip() for x in out.split(",")])
            except Exception:
                pass
            time.sleep(0.1)

    def summary(self):
        sm = [float(r[0]) for r in self.rows if r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = sorted({names[i] for r in self.rows if len(r) >= 7 for i in range(4) if r[3 + i].lower().startswith("active")})
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None, "reasons": reasons,
                "samples": len(self.rows)}


def dist_setup(n):
    """torchrun sets RANK/WORLD_SIZE/LOCAL_RANK/MASTER_*; single process otherwise."""
    rank, world = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    return rank, world, local


def max_over_ranks(x, world, device):
    if world == 1:
        return x
    import torch
    import torch.distributed as dist
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def run_reference(args, rank, world):
    """The oracle timed on the host cores, rank 0 only; each step = one output row (all (q,m) pairs of band (0,0))."""
    if rank != 0:
        return 0
    from oracle import exx_ref as R
    w = W.make(args.workload)
    o = R.RefExx(w.grid, w.lattice, w.kfrac, w.kweight, w.ecut, w.kernel_kind, w.mu, w.scale, w.nbands)
    psi = w.coefficients(o.npw)
    pairs = w.nk * w.nocc
    for _ in range(args.warmup):
        o.apply_rows(psi, w.occ, [(0, 0)])
    t0 = time.perf_counter()
    for _ in range(args.steps):
        o.apply_rows(psi, w.occ, [(0, 0)])
    dt = (time.perf_counter() - t0) / args.steps
    v = pairs / dt
    sample = "one V_x row (k0, band 0): %d pair evaluations incl. the real-space transforms of the %d bands it needs" % (pairs, pairs + 1)
    line = {"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic", "config": {"workload": w.name, "description": w.description, "sample": sample},
            "cpu_baseline": {"value": v, "unit": UNIT, "cores": R.num_threads(), "kind": "oracle", "sample": sample},
            "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}, "gpu_launches": 0}
    print(json.dumps(line))
    return 0


# algorithmic bytes per work unit of each kernel class, in units of Ng bytes:
# a generic box pass reads and writes one complex128 box (32 Ng); each fused pass moves 32 Ng per pair box (96 Ng for the
# three passes = the B_model of the pair evaluation; the dual sweep of pass C serves both accumulations of a symmetric pair
# and is still booked at 32 Ng per box: work box 16 + one u read 16); pass R is booked at the partial box it reads (16 Ng per unit);
# its read-modify-write of the accumulator (32 Ng per COLUMN, shared by the up to tile_n/RG partial boxes of that column: 4 Ng per
# unit at C4a, 19.9 B/pt measured) is not a per-unit quantity and is left out: a lower bound, used only if pass R ever dominates.
BYTES_PER_UNIT_NG = {"fft_axis_generic": 32, "codensity": 32, "kernel_multiply": 32, "accumulate": 32,
                     "fused_pass_a": 32, "fused_pass_b": 32, "fused_pass_c": 32, "fused_fft_pass": 32, "fused_pass_r": 16,
                     "scatter": 16, "gather": 16}
NCU_COUNTERS = os.path.join(ROOT, "profiles", "ncu_counters_r3.json")


def lib_source_hash():
    """The source hash libexx.so was built from (paper_1111_0716_b200/build.py keeps it beside the library)."""
    try:
        from paper_1111_0716_b200 import build as b
        return open(b.STAMP).read().strip()
    except Exception:
        return None


def ncu_counters(ngw):
    """Per-unit DRAM bytes and fp64 instruction counts of the fused kernels from the committed `ncu --set full` capture
    (profiles/ncu_counters_r3.json), or (None, why) when that capture was taken from other sources or another work grid:
    a stale capture is never printed."""
    try:
        tj = json.load(open(NCU_COUNTERS))
    except Exception as e:  # noqa: BLE001
        return None, "no capture (%s)" % type(e).__name__
    if tj.get("srchash") != lib_source_hash():
        return None, "capture is of another build (source hash differs)"
    if tj.get("work_grid", 0) ** 3 != ngw:
        return None, "capture is of another work grid"
    return tj, "profiles/ncu_counters_r3.json (%s)" % tj.get("source", "")


def run_ours(args, rank, world, local):
    import torch
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)
    from paper_1111_0716_b200 import binding as B
    B.lib()
    w = W.make(args.workload)
    g = B.Exx.from_workload(w)
    if args.path is not None:
        g.set_option(B.EXX_OPT_PATH, args.path)
    if args.precision == "mixed":   # the paper's second mode; NOT the graded fp64 configuration
        g.set_option(B.EXX_OPT_PRECISION, 1)
    psi = w.coefficients(g.npw)
    occ = w.occ
    pd = g.to_device(psi)
    out = g.empty_like_psi()
    pin_in = torch.from_numpy(psi).pin_memory()
    pin_out = torch.empty(g.ncoef, dtype=torch.complex128).pin_memory()
    peak, peak_src = read_peaks()

    shard = args.parallel == "shard"

    def apply_dev():
        if shard:   # this rank's pair batches, then one all-reduce of the sphere coefficients (binding.apply_sharded)
            g.apply_sharded(pd, occ, out, rank=rank, world=world)
        else:
            g.apply(pd, occ, out)

    def step_dev():
        apply_dev()
        return g.energy(pd, occ, out)[0]

    def step_host():
        if not shard:
            return g.apply_host(pin_in, occ, pin_out)[1]
        pd.copy_(pin_in, non_blocking=True)
        apply_dev()
        pin_out.copy_(out, non_blocking=True)
        return g.energy(pd, occ, out)[0]

    def sync_all():
        torch.cuda.synchronize()
        if world > 1:
            torch.distributed.barrier()

    for _ in range(args.warmup):
        ex = step_dev()
    # ---- timed region 1: inputs resident in HBM (events on the stream libexx launches on = torch's current stream)
    g.set_option(B.EXX_OPT_PROFILE, 0)
    sampler = ClockSampler(local)
    sync_all()
    sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(args.steps):
        ex = step_dev()
    e1.record()
    sync_all()
    sampler.stop_flag = True
    ms = max_over_ranks(e0.elapsed_time(e1), world, dev) / args.steps
    launches = g.get_info(B.EXX_INFO_LAUNCHES)
    pairs_ord, pairs_exec = g.get_info(B.EXX_INFO_PAIRS_ORDERED), g.get_info(B.EXX_INFO_PAIRS_EXECUTED)

    # ---- timed region 2: per-kernel-class device time (events around every launch) over the same K steps
    g.set_option(B.EXX_OPT_PROFILE, 1)
    acc = {}
    sync_all()
    p0, p1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    p0.record()
    for _ in range(args.steps):
        apply_dev()
        for name, (t, n, u) in g.kernel_times().items():
            a = acc.setdefault(name, [0.0, 0, 0])
            a[0] += t; a[1] += n; a[2] += u
        g.energy(pd, occ, out)
    p1.record()
    sync_all()
    ms_prof = p0.elapsed_time(p1) / args.steps
    g.set_option(B.EXX_OPT_PROFILE, 0)
    # grid the pair pipeline actually transformed (the compact work grid when EXX_OPT_PRUNE is active):
    # all algorithmic-byte figures below use THAT grid, never the caller's larger box
    nw = g.get_info(B.EXX_INFO_WORK_GRID)
    ngw = nw ** 3 if g.get_info(B.EXX_INFO_PRUNED) else w.ng
    dom = max(acc, key=lambda k: acc[k][0])
    t_dom, n_dom, u_dom = acc[dom]
    bytes_dom = BYTES_PER_UNIT_NG.get(dom, 32) * ngw * u_dom
    achieved = bytes_dom / (t_dom * 1e-3) / 1e9 if t_dom > 0 else 0.0
    # DRAM bytes and fp64 instruction counts per unit from the committed ncu capture of THIS build (refused when the hash differs)
    ncu, ncu_src = ncu_counters(ngw)
    traffic = None
    if ncu and dom in ncu["dram_bytes_per_launch"]:
        traffic = ncu["dram_bytes_per_launch"][dom] / ncu["units_per_launch"][dom] * (u_dom / max(1, n_dom))
    roofline = {"bound": "hbm", "kernel": dom, "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                "traffic": traffic, "traffic_source": ncu_src, "peak_source": peak_src, "avg_launch_us": 1e3 * t_dom / max(1, n_dom),
                "algorithmic_bytes_per_launch": bytes_dom / max(1, n_dom), "share_of_step": t_dom / args.steps / ms_prof,
                "grid_points_transformed": ngw, "model": "32 B per transformed grid point per pair box (SURVEY.md 8(d)); not a DRAM counter",
                "kernel_ms_per_step": {k: v[0] / args.steps for k, v in acc.items() if v[1]}}
    if traffic is not None:
        roofline["dram_frac"] = traffic / (1e-3 * t_dom / max(1, n_dom)) / 1e9 / peak
    # ---- the pipeline figures.  SURVEY.md 8(d) grades  B_model x (pairs executed) / (t x peak)  with B_model = 96 bytes per
    # transformed grid point (three passes x 32) and gives the 64-byte floor (perfect reuse of u) beside it; bytes are counted per
    # EXECUTED pair (a symmetric pair is transformed once), never per ordered pair.  pass_execution_frac counts 32 B/pt for every
    # pass execution of the run (a second pass-C sweep included where the dual sweep is off) and is NOT the graded number.
    fused = [k for k in ("fused_pass_a", "fused_pass_b", "fused_pass_c", "fused_fft_pass") if k in acc]
    pass_units = sum(acc[k][2] for k in fused) / args.steps
    if pass_units == 0:  # generic path: 9 box passes per pair
        pass_units = sum(acc[k][2] for k in ("fft_axis_generic", "codensity", "kernel_multiply", "accumulate") if k in acc) / args.steps
    t_s = ms * 1e-3
    pipeline = {"bytes_per_pass_execution": 32 * ngw, "pass_executions_per_step": pass_units, "pairs_executed": pairs_exec,
                "pairs_ordered": pairs_ord, "symmetry": g.get_info(B.EXX_INFO_SYMMETRY), "unit": "GB/s", "peak": peak,
                "survey_frac": 96.0 * ngw * pairs_exec / t_s / 1e9 / peak, "floor_frac": 64.0 * ngw * pairs_exec / t_s / 1e9 / peak,
                "pass_execution_frac": 32.0 * ngw * pass_units / t_s / 1e9 / peak,
                "us_per_executed_pair": 1e3 * ms / max(1, pairs_exec),
                "us_per_ordered_pair": 1e3 * ms / max(1, pairs_ord), "ms_per_step_profiled": ms_prof,
                "work_grid": [nw] * 3 if ngw != w.ng else list(w.grid)}
    pipeline["achieved"] = pipeline["survey_frac"] * peak
    pipeline["frac"] = pipeline["survey_frac"]
    # fp64 ALU fraction: DFMA/DADD/DMUL executed per unit (hardware counters of the capture) x units / time against the fp64 peak
    # measured now by exx_measure_fp64_peak; dram_frac: the capture's DRAM bytes per unit x units / time against the copy peak
    fp64_peak = B.measure_fp64_peak()
    pipeline["fp64_peak_gflops_measured"] = fp64_peak
    pipeline["counters_source"] = ncu_src
    if ncu:
        flops = dram = 0.0
        for k in acc:
            if k in ncu["units_per_launch"]:
                per_unit = 1.0 / ncu["units_per_launch"][k]
                flops += ncu["fp64_flops_per_launch"][k] * per_unit * acc[k][2] / args.steps
                dram += ncu["dram_bytes_per_launch"][k] * per_unit * acc[k][2] / args.steps
        pipeline["fp64_flops_per_step"] = flops
        pipeline["fp64_frac"] = flops / t_s / 1e9 / fp64_peak
        pipeline["dram_bytes_per_step"] = dram
        pipeline["dram_frac"] = dram / t_s / 1e9 / peak
    else:
        pipeline["fp64_frac"] = pipeline["dram_frac"] = None

    # ---- the same apply on the caller's FULL grid (EXX_OPT_PRUNE = 0): the graded "96^3" pipeline number of BASELINE.md
    full = None
    if ngw != w.ng and not args.no_full_grid and not shard:
        g.set_option(B.EXX_OPT_PRUNE, 0)
        for _ in range(2):
            g.apply(pd, occ, out)
        sync_all()
        f0, f1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        f0.record()
        for _ in range(args.steps):
            g.apply(pd, occ, out)
            ex_f = g.energy(pd, occ, out)[0]
        f1.record()
        sync_all()
        ms_f = max_over_ranks(f0.elapsed_time(f1), world, dev) / args.steps
        pe_f = g.get_info(B.EXX_INFO_PAIRS_EXECUTED)
        full = {"grid": list(w.grid), "ms_per_step": ms_f, "value": world * pairs_ord / (ms_f * 1e-3), "unit": UNIT,
                "us_per_executed_pair": 1e3 * ms_f / max(1, pe_f), "us_per_ordered_pair": 1e3 * ms_f / max(1, pairs_ord),
                "pairs_executed": pe_f, "survey_frac": 96.0 * w.ng * pe_f / (ms_f * 1e-3) / 1e9 / peak,
                "floor_frac": 64.0 * w.ng * pe_f / (ms_f * 1e-3) / 1e9 / peak, "E_x": ex_f}
        assert abs(ex_f - ex) <= (1e-11 if args.precision == "fp64" else 1e-5) * abs(ex)
        g.set_option(B.EXX_OPT_PRUNE, 1)

    # ---- E_x from psi alone by the pair-density route (EXX_OPT_ENERGY_ROUTE = 0): for information, not the headline
    energy_only = None
    if not shard:
        g.energy(pd, occ, None)
        sync_all()
        q0, q1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        q0.record()
        for _ in range(args.steps):
            ex_q = g.energy(pd, occ, None)[0]
        q1.record()
        sync_all()
        ms_q = max_over_ranks(q0.elapsed_time(q1), world, dev) / args.steps
        pq = g.get_info(B.EXX_INFO_PAIRS_ORDERED)
        energy_only = {"route": {1: "E1 from V_x psi", 2: "E2 pair densities"}.get(g.get_info(B.EXX_INFO_ENERGY_ROUTE)), "ms_per_step": ms_q,
                       "pairs_ordered": pq, "pairs_executed": g.get_info(B.EXX_INFO_PAIRS_EXECUTED), "value": world * pq / (ms_q * 1e-3), "unit": UNIT,
                       "gpu_launches": g.get_info(B.EXX_INFO_LAUNCHES), "E_x": ex_q}
        assert abs(ex_q - ex) <= (1e-11 if args.precision == "fp64" else 1e-5) * abs(ex)

    # ---- the operator applied to a block of trial vectors (exx_apply_to; FOCK_ACC's NSIM block): for information
    apply_to = None
    if not shard and args.precision == "fp64":
        nphi = min(8, w.nbands)
        tot = int(sum(g.npw))
        gen = torch.Generator(device="cuda").manual_seed(1234)
        blk = torch.view_as_complex(torch.randn(nphi * tot, 2, dtype=torch.float64, device="cuda", generator=gen))
        blk_out = torch.empty_like(blk)
        g.set_option(B.EXX_OPT_KEEP_U, 1)          # psi does not change between these calls
        g.apply_to(pd, occ, blk, blk_out)
        sync_all()
        a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a0.record()
        for _ in range(args.steps):
            g.apply_to(pd, occ, blk, blk_out)
        a1.record()
        sync_all()
        g.set_option(B.EXX_OPT_KEEP_U, 0)
        ms_a = max_over_ranks(a0.elapsed_time(a1), world, dev) / args.steps
        pa = g.get_info(B.EXX_INFO_PAIRS_EXECUTED)
        apply_to = {"nphi_per_k": nphi, "ms_per_call": ms_a, "pairs_executed": pa, "us_per_pair": 1e3 * ms_a / max(1, pa),
                    "value": world * pa / (ms_a * 1e-3), "unit": UNIT, "gpu_launches": g.get_info(B.EXX_INFO_LAUNCHES), "keep_u": 1}

    # ---- the plain pipeline on the caller's grid: no compact grid, no pair symmetry (every ordered pair through passes A, B, C):
    # the figure to hold against BASELINE.md's "apply <= 0.562 s at 96^3" without either shortcut
    plain = None
    if not shard and not args.no_full_grid and args.precision == "fp64":
        g.set_option(B.EXX_OPT_PRUNE, 0)
        g.set_option(B.EXX_OPT_SYMMETRY, 0)
        g.apply(pd, occ, out)
        sync_all()
        r0, r1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        r0.record()
        for _ in range(max(1, args.steps // 2)):
            g.apply(pd, occ, out)
            ex_p = g.energy(pd, occ, out)[0]
        r1.record()
        sync_all()
        ms_p = max_over_ranks(r0.elapsed_time(r1), world, dev) / max(1, args.steps // 2)
        pe_p = g.get_info(B.EXX_INFO_PAIRS_EXECUTED)
        plain = {"grid": list(w.grid), "pruned": 0, "pair_symmetry": g.get_info(B.EXX_INFO_SYMMETRY), "ms_per_step": ms_p,
                 "pairs_executed": pe_p, "value": world * pe_p / (ms_p * 1e-3), "unit": UNIT, "us_per_pair": 1e3 * ms_p / max(1, pe_p),
                 "survey_frac": 96.0 * w.ng * pe_p / (ms_p * 1e-3) / 1e9 / peak, "E_x": ex_p}
        assert abs(ex_p - ex) <= 1e-11 * abs(ex)
        g.set_option(B.EXX_OPT_PRUNE, 1)
        g.set_option(B.EXX_OPT_SYMMETRY, 1)
        g.apply(pd, occ, out)   # `out` back to the default mode's result for the legs below

    # ---- subspace matrix <psi_i|V_x psi_j> (exx_subspace, fp64 DMMA ZGEMM): 8 nb^2 npw flops per k-point
    subspace = None
    if not shard and args.precision == "fp64":
        m = g.subspace(0, pd, out)
        sync_all()
        s0, s1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        reps = 20
        s0.record()
        for _ in range(reps):
            g.subspace(0, pd, out, m)
        s1.record()
        sync_all()
        ms_s = s0.elapsed_time(s1) / reps
        fl = 8.0 * w.nbands * w.nbands * g.npw[0]
        # yardstick only, never on the product path: the same contraction as a library ZGEMM (torch.matmul -> cuBLAS)
        a_m = pd[g.offsets[0]:g.offsets[0] + w.nbands * g.npw[0]].view(w.nbands, g.npw[0])
        b_m = out[g.offsets[0]:g.offsets[0] + w.nbands * g.npw[0]].view(w.nbands, g.npw[0])
        bt = b_m.t().contiguous()
        ref_m = torch.matmul(a_m.conj(), bt)
        sync_all()
        y0, y1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        y0.record()
        for _ in range(reps):
            torch.matmul(a_m.conj(), bt, out=ref_m)
        y1.record()
        sync_all()
        ms_y = y0.elapsed_time(y1) / reps
        subspace = {"shape": [w.nbands, w.nbands, g.npw[0]], "ms_per_call": ms_s, "gflops": fl / (ms_s * 1e-3) / 1e9,
                    "yardstick_cublas_zgemm": {"ms_per_call": ms_y, "gflops": fl / (ms_y * 1e-3) / 1e9,
                                               "max_abs_diff": float((ref_m - m).abs().max().item()),
                                               "note": "torch.matmul(conj(A), B^T) on the same operands (conj materialised inside the timed call); a yardstick, not on the product path"},
                    "fp64_peak_gflops_measured": fp64_peak, "frac_of_fp64_peak": fl / (ms_s * 1e-3) / 1e9 / fp64_peak,
                    "kernel": "mma.sync.m8n8k4.f64 (DMMA), 32 x 32 tile per warp, register-pipelined fragment loads, split-K with fixed-order reduction",
                    "hermiticity_defect": float((m - m.conj().T).abs().max().item()) if w.nocc == w.nbands else None}

    # ---- timed region 3: end to end through exx_apply_host, pinned host buffers, copies inside the timed region
    for _ in range(min(2, args.warmup)):
        step_host()
    sync_all()
    h0, h1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    h0.record()
    for _ in range(args.steps):
        ex_h = step_host()
    h1.record()
    sync_all()
    ms_e2e = max_over_ranks(h0.elapsed_time(h1), world, dev) / args.steps
    assert ex_h == ex or abs(ex_h - ex) <= (1e-12 if args.precision == "fp64" else 1e-5) * abs(ex)

    # replicas: every rank did the whole workload; shard: the ranks together did it once (pairs_ord is this rank's share)
    job_pairs = w.pair_evals if shard else world * pairs_ord
    value = job_pairs / (ms * 1e-3)
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms, "higher_is_better": True, "scaling": "strong" if shard else "weak", "vs_baseline": None,
            "dtype": "f64" if args.precision == "fp64" else "f32 transforms + f64 accumulation (mixed; outside the fp64 parity contract)",
            "data": "synthetic",
            "config": {"workload": w.name, "description": w.description, "grid": list(w.grid), "nk": w.nk, "nbands": w.nbands,
                       "pairs_per_step": job_pairs if shard else pairs_ord,
                       "parallelism": ("pair batches sharded x%d + all-reduce of V_x psi" if shard else "replicas x%d") % world,
                       "path": {1: "generic", 2: "fused"}.get(g.get_info(B.EXX_INFO_PATH_USED)),
                       "tile_n": g.get_info(B.EXX_INFO_TILE_N), "tile_m": g.get_info(B.EXX_INFO_TILE_M),
                       "pruned": g.get_info(B.EXX_INFO_PRUNED), "pair_symmetry": g.get_info(B.EXX_INFO_SYMMETRY), "work_grid": pipeline["work_grid"],
                       "pairs_executed_per_step": pairs_exec,
                       # whether the dual-sweep kernel RAN in the timed applies (pass R launches > 0), not the option's value: grids
                       # without a dual kernel (40^3, 64^3, 128^3) run two sweeps whatever EXX_OPT_DUAL_SWEEP says
                       "dual_sweep": int(acc.get("fused_pass_r", (0.0, 0, 0))[1] > 0), "dual_sweep_option": g.get_option(B.EXX_OPT_DUAL_SWEEP),
                       "l2": "inputs larger than L2: the real-space cache u_nk(r) is %.2f GB, streamed every step" % (w.nk * w.nbands * ngw * 16 / 1e9)},
            "E_x": ex, "vx_apply_ms": ms, "clocks": sampler.summary(), "roofline": roofline, "pipeline_roofline": pipeline,
            "e2e": {"value": job_pairs / (ms_e2e * 1e-3), "unit": UNIT, "ms_per_step": ms_e2e,
                    "h2d_bytes_per_step": g.ncoef * 16, "d2h_bytes_per_step": g.ncoef * 16 + 8},
            "gpu_launches": launches * args.steps}
    if full is not None:
        line["full_grid"] = full
    if energy_only is not None:
        line["energy_only"] = energy_only
    if apply_to is not None:
        line["apply_to"] = apply_to
    if plain is not None:
        line["plain_pipeline"] = plain
    if subspace is not None:
        line["subspace"] = subspace
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        line["cpu_baseline"] = cpu_baseline(w, psi)
    if rank == 0:
        print(json.dumps(line))
    g.close()
    if world > 1:
        torch.distributed.destroy_process_group()
    return 0


def cpu_baseline(w, psi, nrows=3):
    """The oracle as it stands on the host cores: `nrows` V_x rows (all (q,m) pairs of bands 0.. of k-point 0) of the same
    workload, about 10-15 s of CPU work at C4a."""
    from oracle import exx_ref as R
    o = R.RefExx(w.grid, w.lattice, w.kfrac, w.kweight, w.ecut, w.kernel_kind, w.mu, w.scale, w.nbands)
    nrows = min(nrows, w.nbands)
    pairs = nrows * w.nk * w.nocc
    t0 = time.perf_counter()
    o.apply_rows(psi, w.occ, [(0, n) for n in range(nrows)])
    dt = time.perf_counter() - t0
    return {"value": pairs / dt, "unit": UNIT, "cores": R.num_threads(), "kind": "oracle", "seconds": dt,
            "sample": "%d V_x rows (k0, bands 0..%d): %d pair evaluations incl. the real-space transforms of the bands they need "
                      "(done once)" % (nrows, nrows - 1, pairs)}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="C4a", choices=list(W.ALL))
    ap.add_argument("--path", type=int, default=None, help="EXX_OPT_PATH override: 1 generic, 2 fused")
    ap.add_argument("--precision", default="fp64", choices=["fp64", "mixed"],
                    help="mixed = EXX_OPT_PRECISION 1 (fp32 pair transforms); for information only, the default fp64 run is the benchmark")
    ap.add_argument("--parallel", default="replicas", choices=["replicas", "shard"],
                    help="N > 1: independent replicas (default, weak scaling) or the pair batches of one workload shared out (strong scaling)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-full-grid", action="store_true", help="skip the extra full-grid (EXX_OPT_PRUNE = 0) timing")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    rank, world, local = dist_setup(args.gpus)
    if args.impl == "reference":
        return run_reference(args, rank, world)
    return run_ours(args, rank, world, local)


if __name__ == "__main__":
    sys.exit(main())
