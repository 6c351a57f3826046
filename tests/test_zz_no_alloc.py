"""exx_subspace_static — the one entry point of libexx that allocates no device memory — against exx_subspace_block.

Why the entry point exists: some host programs may not let a library call cudaMalloc.  Their GPU memory belongs to another
allocator (a framework's caching pool that reserved the whole card, a job with a fixed memory budget), or they sit in a loop
that cannot take the device-wide synchronisation cudaMalloc / cudaFree cause.  For them the split-K scratch of the subspace
ZGEMM is a fixed 8 MiB array inside the library image, shared by every call on a GPU and never cleared.  What that sharing
could break is exactly what is tested here: two calls in a row with different shapes, the second of which would pick up the
first one's partial sums if the kernels read anything they had not just written.

This file is named so that pytest collects it last (a failure here must not hide the parity tests under `-x`); it needs nothing
from the other test modules and passes alone in a fresh process as well as after them.
"""
import ctypes as C

import numpy as np
import pytest

from paper_1111_0716_b200 import workloads as W

TOL = 1e-13   # relative to max |M|: the bar of the exx_subspace tests in test_gpu_parity.py


def _random_block(rng, nvec, npw):
    return (rng.standard_normal((nvec, npw)) + 1j * rng.standard_normal((nvec, npw))) / np.sqrt(npw)


@pytest.mark.gpu
def test_static_scratch_entry_point_matches_existing_path_on_two_calls_in_a_row():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1111_0716_b200 import binding as B
    B.lib()  # fails loudly if libexx.so is missing
    # a context only for the EXISTING path (exx_subspace_block looks up npw(k) in it); the new call takes plain pointers
    w = W.custom("noalloc", 31, (24, 24, 24), W.cubic(9.0), [[0, 0, 0], [0.5, 0, 0]], [0.5, 0.5], 7.0, 2, np.ones(2))
    g = B.Exx.from_workload(w)
    tot = int(sum(g.npw))
    rng = np.random.default_rng(20111107)
    # first call: 45 vectors (a ragged 32 x 32 tile edge, many slices) at k-point 0;
    # second call, straight after it: 7 vectors at k-point 1 (another npw, fewer and differently sized slices)
    for nvec, ik in ((45, 0), (7, 1)):
        npw = g.npw[ik]
        phi = np.zeros((nvec * tot,), dtype=np.complex128)   # the packed layout of exx_apply_to: nvec vectors per k-point
        vphi = np.zeros_like(phi)
        a = _random_block(rng, nvec, npw)
        b = _random_block(rng, nvec, npw)
        off = nvec * sum(g.npw[:ik])
        phi[off:off + nvec * npw] = a.reshape(-1)
        vphi[off:off + nvec * npw] = b.reshape(-1)
        want = g.subspace_block(ik, g.to_device(phi), g.to_device(vphi)).cpu().numpy()          # existing path (cudaMalloc'd scratch)
        ad, bd = torch.from_numpy(a).cuda(), torch.from_numpy(b).cuda()
        m = torch.full((nvec, nvec), complex(np.nan, np.nan), dtype=torch.complex128, device="cuda")
        got = B.subspace_static(ad, bd, m).cpu().numpy()                                         # new path (fixed array)
        scale = np.abs(want).max()
        assert scale > 0 and np.isfinite(got).all()
        assert np.abs(got - want).max() <= TOL * scale, (nvec, ik)
        assert np.abs(got - a.conj() @ b.T).max() <= 1e-12 * scale                               # and the plain definition
        # the same call again reproduces itself bit for bit (fixed slice order, nothing left over from the call before)
        assert np.array_equal(B.subspace_static(ad, bd).cpu().numpy(), got)
    g.close()


@pytest.mark.gpu
def test_static_scratch_entry_point_at_its_largest_vector_count():
    """nvec = 256 (the limit; C5's band count) with a ragged npw: the fewest slices the fixed array allows."""
    import torch
    from paper_1111_0716_b200 import binding as B
    rng = np.random.default_rng(7)
    a, b = _random_block(rng, 256, 4099), _random_block(rng, 256, 4099)
    got = B.subspace_static(torch.from_numpy(a).cuda(), torch.from_numpy(b).cuda()).cpu().numpy()
    want = a.conj() @ b.T
    assert np.abs(got - want).max() <= 1e-12 * np.abs(want).max()


def test_static_scratch_entry_point_refuses_sizes_beyond_its_array():
    """Argument checks come before any CUDA call, so this runs without a GPU: over-limit sizes give EXX_ERR_LIMIT and a message."""
    from paper_1111_0716_b200 import binding as B
    L = B.lib()
    p = C.c_void_p(256)   # never dereferenced: the call must return before touching the device
    assert L.exx_subspace_static(p, p, B.STATIC_MAX_NVEC + 1, 1000, p, None) == B.EXX_ERR_LIMIT
    assert b"nvec <= 256" in L.exx_last_error(None)
    assert L.exx_subspace_static(p, p, 8, B.STATIC_MAX_NPW + 1, p, None) == B.EXX_ERR_LIMIT
    assert L.exx_subspace_static(p, p, 0, 1000, p, None) == -9
    assert L.exx_subspace_static(p, p, 8, 0, p, None) == -9
    assert L.exx_subspace_static(None, p, 8, 1000, p, None) == -1
    assert L.exx_strerror(B.EXX_ERR_LIMIT) not in (b"unknown error", None)
    hdr = open(B.os.path.join(B.os.path.dirname(B._HERE), "include", "exx.h")).read()
    assert "#define EXX_STATIC_MAX_NVEC %d" % B.STATIC_MAX_NVEC in hdr and "#define EXX_STATIC_MAX_NPW (1 << 24)" in hdr
    assert "#define EXX_STATIC_SCRATCH_BYTES (8 << 20)" in hdr and B.STATIC_SCRATCH_BYTES == 8 << 20
