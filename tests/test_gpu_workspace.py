"""Device-memory bookkeeping of libexx on the GPU (-m gpu): what a context allocates and when, and the out-of-memory branches.

A 180 GB device never refuses these allocations by itself, so the library has a test hook: while EXX_TEST_FAIL_ALLOC names a tag
("part": partial boxes of the dual sweep; "acc": accumulator boxes of the full-grid buffers) that allocation reports failure.
"""
import os

import numpy as np
import pytest

from paper_1111_0716_b200 import workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1111_0716_b200 import binding
    binding.lib()
    return binding


@pytest.fixture(autouse=True)
def _no_hook_left_behind():
    os.environ.pop("EXX_TEST_FAIL_ALLOC", None)
    yield
    os.environ.pop("EXX_TEST_FAIL_ALLOC", None)


def _workload():
    # caller's grid 48^3 (R1 = 6, has a dual-sweep kernel); the spheres also fit a compact 32^3 grid, so the 48^3 buffers are only made
    # by the first apply with EXX_OPT_PRUNE = 0
    return W.custom("ws48", 4849, (48, 48, 48), W.cubic(10.0), [[0, 0, 0]], [1.0], 6.0, 6, [1.0, 1.0, 0.5, 0.0, 1.0, 1.0])


def _ctx(B, w):
    g = B.Exx.from_workload(w)
    g.set_option(B.EXX_OPT_PRUNE, 0)
    return g


def test_partial_boxes_are_allocated_by_the_first_dual_sweep_only(B):
    w = _workload()
    g = _ctx(B, w)
    pd = g.to_device(w.coefficients(g.npw))
    box = 16 * 48 ** 3
    g.set_option(B.EXX_OPT_SYMMETRY, 0)
    plain = g.apply(pd, w.occ).cpu().numpy()
    ws_plain = g.get_info(B.EXX_INFO_WORKSPACE_BYTES)
    g.set_option(B.EXX_OPT_SYMMETRY, 1)
    g.set_option(B.EXX_OPT_DUAL_SWEEP, 0)
    two = g.apply(pd, w.occ).cpu().numpy()
    assert g.get_info(B.EXX_INFO_SYMMETRY) == 1
    assert g.get_info(B.EXX_INFO_WORKSPACE_BYTES) == ws_plain          # two sweeps need no partial boxes: none were made
    assert g.kernel_times()["fused_pass_r"][1] == 0
    g.set_option(B.EXX_OPT_DUAL_SWEEP, 1)
    dual = g.apply(pd, w.occ).cpu().numpy()
    extra = g.get_info(B.EXX_INFO_WORKSPACE_BYTES) - ws_plain
    t = g.get_info(B.EXX_INFO_TILE_N)
    assert extra > 0 and extra % box == 0 and extra // box <= t * t     # (row groups) x (columns) boxes, fewer than the pair boxes
    assert g.kernel_times()["fused_pass_r"][1] > 0
    g.apply(pd, w.occ)
    assert g.get_info(B.EXX_INFO_WORKSPACE_BYTES) == ws_plain + extra   # made once
    scale = np.linalg.norm(plain)
    assert np.linalg.norm(two - plain) < 1e-13 * scale and np.linalg.norm(dual - plain) < 1e-13 * scale
    g.close()


def test_refused_partial_boxes_fall_back_to_two_sweeps(B):
    w = _workload()
    g = _ctx(B, w)
    pd = g.to_device(w.coefficients(g.npw))
    g.set_option(B.EXX_OPT_DUAL_SWEEP, 0)
    two = g.apply(pd, w.occ).cpu().numpy()
    ws = g.get_info(B.EXX_INFO_WORKSPACE_BYTES)
    g.set_option(B.EXX_OPT_DUAL_SWEEP, 1)
    os.environ["EXX_TEST_FAIL_ALLOC"] = "part"
    out = g.apply(pd, w.occ).cpu().numpy()                               # not an error: the apply runs two sweeps
    assert g.kernel_times()["fused_pass_r"][1] == 0 and g.get_info(B.EXX_INFO_SYMMETRY) == 1
    assert g.get_info(B.EXX_INFO_WORKSPACE_BYTES) == ws
    assert np.array_equal(out, two)                                      # the very same kernels in the same order
    g.close()


def test_failed_workspace_allocation_leaves_a_clean_context(B):
    w = _workload()
    ref = _ctx(B, w)
    pd = ref.to_device(w.coefficients(ref.npw))
    want = ref.apply(pd, w.occ).cpu().numpy()
    ws_want = ref.get_info(B.EXX_INFO_WORKSPACE_BYTES)
    ref.close()
    g = _ctx(B, w)
    ws0 = g.get_info(B.EXX_INFO_WORKSPACE_BYTES)
    os.environ["EXX_TEST_FAIL_ALLOC"] = "acc"
    for _ in range(2):                                                   # part-way failure (after the u cache and the pair workspace)
        with pytest.raises(B.ExxError) as ei:
            g.apply(pd, w.occ)
        assert ei.value.code == -7
        assert g.get_info(B.EXX_INFO_WORKSPACE_BYTES) == ws0             # everything the attempt took was given back and un-counted
    del os.environ["EXX_TEST_FAIL_ALLOC"]
    got = g.apply(pd, w.occ).cpu().numpy()                               # the retry starts clean
    assert g.get_info(B.EXX_INFO_WORKSPACE_BYTES) == ws_want
    assert np.array_equal(got, want)
    g.close()


def test_calls_from_another_stream_are_refused(B):
    """The library orders its work on the context's creation stream only; the binding refuses a call made under another torch
    stream instead of letting it race, and a context created with an explicit stream lives on that stream's device."""
    import torch
    w = _workload()
    side = torch.cuda.Stream()
    g = B.Exx.from_workload(w, stream=side)
    assert g.device == side.device.index
    with torch.cuda.stream(side):
        pd = g.to_device(w.coefficients(g.npw))
        out = g.apply(pd, w.occ)
    side.synchronize()
    assert bool(torch.isfinite(out.real).all())
    with pytest.raises(RuntimeError, match="creation stream"):
        g.apply(pd, w.occ)                                               # current stream is the default one here
    other = torch.cuda.Stream()
    with torch.cuda.stream(other), pytest.raises(RuntimeError, match="creation stream"):
        g.apply(pd, w.occ)
    g.close()
