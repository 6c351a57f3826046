"""Thin Python binding of libexx (include/exx.h): argument marshalling only.

Every step of the path runs in the CUDA library; torch is used for device memory and the stream handle.
There is no CPU fallback: if libexx.so cannot be loaded, every entry point raises.
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("EXX_LIB") or os.path.join(_HERE, "libexx.so")  # EXX_LIB: use another build of the same library

EXX_OPT_PATH, EXX_OPT_TILE_N, EXX_OPT_TILE_M, EXX_OPT_PRUNE, EXX_OPT_PROFILE, EXX_OPT_SYMMETRY = 1, 2, 3, 4, 5, 6
EXX_OPT_PRECISION = 8
EXX_OPT_SHARD_COUNT, EXX_OPT_SHARD_RANK = 9, 10
EXX_OPT_ENERGY_ROUTE = 11
EXX_OPT_KEEP_U = 12
EXX_OPT_DUAL_SWEEP = 13
EXX_OPT_PRUNE_SPHERE = 14
(EXX_INFO_LAUNCHES, EXX_INFO_PAIRS_ORDERED, EXX_INFO_PAIRS_EXECUTED, EXX_INFO_PATH_USED, EXX_INFO_WORKSPACE_BYTES,
 EXX_INFO_NCOEF, EXX_INFO_TILE_N, EXX_INFO_TILE_M, EXX_INFO_PRUNED, EXX_INFO_NUM_KERNEL_CLASSES, EXX_INFO_WORK_GRID,
 EXX_INFO_COMPACT_GRID, EXX_INFO_SYMMETRY) = range(1, 14)
EXX_INFO_PRECISION = 15
EXX_INFO_ENERGY_ROUTE = 16

# every symbol include/exx.h declares (tests/test_abi.py checks the library exports them all)
SYMBOLS = ("exx_create", "exx_destroy", "exx_npw", "exx_index_map", "exx_psi_offset", "exx_set_option", "exx_get_option",
           "exx_get_info", "exx_get_kernel_time", "exx_kernel_class_name", "exx_apply", "exx_energy", "exx_apply_host",
           "exx_scatter", "exx_gather", "exx_fft3d", "exx_to_real", "exx_kernel_table", "exx_strerror", "exx_last_error",
           "exx_version", "exx_subspace", "exx_fft3d_fused", "exx_findex", "exx_shard_plan", "exx_apply_to", "exx_subspace_block", "exx_measure_fp64_peak",
           "exx_subspace_static")


class KernelParams(C.Structure):
    _fields_ = [("kind", C.c_int), ("mu", C.c_double), ("scale", C.c_double)]


class ExxError(RuntimeError):
    def __init__(self, code, detail=""):
        self.code = code
        msg = "libexx error %d: %s" % (code, lib().exx_strerror(code).decode())
        if detail:
            msg += " [" + detail + "]"
        super().__init__(msg)


_lib = None


def lib():
    """Load libexx.so (built in-tree by paper_1111_0716_b200.build).  Raises if it is missing: no fallback."""
    global _lib
    if _lib is None:
        if not os.environ.get("EXX_LIB"):
            # compile (or re-compile after a source change) the CUDA library in-tree; compiling is not a fallback path.  A build
            # error is re-raised even when an older libexx.so is still on disk: only a library whose source stamp matches the
            # sources is ever loaded, so tests and bench.py cannot report numbers for code that was never built.
            from . import build as _build
            try:
                _build.build()
            except Exception as e:  # noqa: BLE001
                raise RuntimeError("libexx.so could not be built from the current sources (%s); refusing to load a stale "
                                   "library (set EXX_LIB to load a specific build); there is no CPU fallback" % e) from e
            if _build.needs_build():
                raise RuntimeError("libexx.so does not match the sources after the build step; there is no CPU fallback")
        if not os.path.exists(LIB_PATH):
            raise RuntimeError("libexx.so not found at %s: build it with `python -m paper_1111_0716_b200.build` "
                               "(there is no CPU fallback)" % LIB_PATH)
        L = C.CDLL(LIB_PATH)
        vp, dp, ip = C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_int)
        i64p = C.POINTER(C.c_int64)
        L.exx_create.argtypes = [C.POINTER(vp), ip, dp, C.c_int, dp, dp, C.c_double, C.POINTER(KernelParams), C.c_int, vp]
        L.exx_destroy.argtypes = [vp]
        L.exx_npw.argtypes = [vp, C.c_int, ip]
        L.exx_index_map.argtypes = [vp, C.c_int, C.POINTER(C.c_int32)]
        L.exx_psi_offset.argtypes = [vp, C.c_int, i64p]
        L.exx_set_option.argtypes = [vp, C.c_int, C.c_int64]
        L.exx_get_option.argtypes = [vp, C.c_int, i64p]
        L.exx_get_info.argtypes = [vp, C.c_int, i64p]
        L.exx_get_kernel_time.argtypes = [vp, C.c_int, dp, i64p, i64p]
        L.exx_kernel_class_name.argtypes = [C.c_int]
        L.exx_kernel_class_name.restype = C.c_char_p
        L.exx_apply.argtypes = [vp, vp, dp, vp]
        L.exx_apply_to.argtypes = [vp, vp, dp, vp, C.c_int, vp]
        L.exx_subspace_block.argtypes = [vp, C.c_int, vp, vp, C.c_int, vp]
        L.exx_energy.argtypes = [vp, vp, dp, vp, dp, dp]
        L.exx_apply_host.argtypes = [vp, vp, dp, vp, dp]
        L.exx_subspace.argtypes = [vp, C.c_int, vp, vp, vp]
        L.exx_fft3d_fused.argtypes = [vp, vp, C.c_int, C.c_int, vp]
        L.exx_findex.argtypes = [vp, C.POINTER(C.c_int32)]
        L.exx_shard_plan.argtypes = [C.c_int, C.c_int, dp, C.c_int, C.c_int, C.c_int, i64p, i64p]
        L.exx_scatter.argtypes = [vp, C.c_int, vp, C.c_int, vp]
        L.exx_gather.argtypes = [vp, C.c_int, vp, C.c_int, vp]
        L.exx_fft3d.argtypes = [vp, vp, C.c_int, C.c_int]
        L.exx_to_real.argtypes = [vp, C.c_int, vp, C.c_int, vp]
        L.exx_kernel_table.argtypes = [vp, C.c_int, C.c_int, dp]
        L.exx_strerror.argtypes = [C.c_int]
        L.exx_strerror.restype = C.c_char_p
        L.exx_last_error.argtypes = [vp]
        L.exx_last_error.restype = C.c_char_p
        L.exx_version.restype = C.c_int
        L.exx_measure_fp64_peak.argtypes = [vp, dp]
        L.exx_subspace_static.argtypes = [vp, vp, C.c_int, C.c_int64, vp, vp]
        _lib = L
    return _lib


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def shard_plan(nk, nbands, occ, symmetry=True, tile=0, nshards=1):
    """exx_shard_plan: (pairs, passes) per shard, two int64 arrays of nshards entries.  Host only: needs no GPU."""
    occ = np.ascontiguousarray(occ, dtype=np.float64).reshape(-1)
    assert occ.size == nk * nbands
    pairs, passes = np.zeros(nshards, dtype=np.int64), np.zeros(nshards, dtype=np.int64)
    i64p = C.POINTER(C.c_int64)
    rc = lib().exx_shard_plan(nk, nbands, _dp(occ), int(bool(symmetry)), int(tile), int(nshards), pairs.ctypes.data_as(i64p),
                              passes.ctypes.data_as(i64p))
    if rc:
        raise ExxError(rc)
    return pairs, passes


def measure_fp64_peak(stream=None):
    """exx_measure_fp64_peak: the device's fp64 vector-pipe peak in GFLOP/s from a DFMA loop (measurement aid for bench.py)."""
    import torch
    g = C.c_double()
    st = stream if stream is not None else torch.cuda.current_stream().cuda_stream
    rc = lib().exx_measure_fp64_peak(C.c_void_p(st), C.cast(C.byref(g), C.POINTER(C.c_double)))
    if rc:
        raise ExxError(rc)
    return g.value


EXX_ERR_LIMIT = -11
STATIC_MAX_NVEC, STATIC_MAX_NPW, STATIC_SCRATCH_BYTES = 256, 1 << 24, 8 << 20


def subspace_static(a_dev, b_dev, m_dev=None, stream=None):
    """exx_subspace_static: M[i, j] = sum_g conj(a[i, g]) b[j, g] for two (nvec, npw) complex128 CUDA tensors, without any device
    allocation inside the library (for processes whose GPU memory belongs to another allocator, or that cannot take cudaMalloc's
    device-wide synchronisation).  Pass m_dev (nvec x nvec complex128) to keep this wrapper from allocating the result either.  The
    scratch is one fixed 8 MiB array per GPU shared by all calls: nvec <= 256, npw <= 2^24 (ExxError code -11 beyond), and calls
    that may overlap on the GPU race — keep them ordered.  Make the first call on a device before any stream capture."""
    import torch
    assert a_dev.is_cuda and b_dev.is_cuda and a_dev.dtype == b_dev.dtype == torch.complex128
    assert a_dev.dim() == 2 and a_dev.shape == b_dev.shape and a_dev.is_contiguous() and b_dev.is_contiguous()
    if a_dev.device.index != torch.cuda.current_device() or b_dev.device != a_dev.device:
        raise RuntimeError("subspace_static works on the current device: make cuda:%d current" % a_dev.device.index)
    nvec, npw = int(a_dev.shape[0]), int(a_dev.shape[1])
    L = lib()
    if (nvec > STATIC_MAX_NVEC or npw > STATIC_MAX_NPW) and m_dev is None:
        # let the library refuse (same error as with a caller-provided m_dev) without allocating a result first
        rc = L.exx_subspace_static(C.c_void_p(a_dev.data_ptr()), C.c_void_p(b_dev.data_ptr()), nvec, npw, C.c_void_p(a_dev.data_ptr()), None)
        raise ExxError(rc, L.exx_last_error(None).decode())
    if m_dev is None:
        m_dev = torch.empty((nvec, nvec), dtype=torch.complex128, device=a_dev.device)
    assert m_dev.is_cuda and m_dev.dtype == torch.complex128 and m_dev.is_contiguous() and m_dev.numel() == nvec * nvec
    st = stream if stream is not None else torch.cuda.current_stream()
    rc = L.exx_subspace_static(C.c_void_p(a_dev.data_ptr()), C.c_void_p(b_dev.data_ptr()), nvec, npw, C.c_void_p(m_dev.data_ptr()),
                               C.c_void_p(st.cuda_stream))
    if rc:
        raise ExxError(rc, L.exx_last_error(None).decode())
    return m_dev


def all_reduce_sum(t, group=None):
    """Sum a complex128 (or real) tensor over the ranks of a torch.distributed group, in place: the one exchange step of the
    sharded path.  NCCL on CUDA tensors; gloo works for the CPU tests."""
    import torch
    import torch.distributed as dist
    dist.all_reduce(torch.view_as_real(t) if t.is_complex() else t, op=dist.ReduceOp.SUM, group=group)
    return t


class Exx:
    """exx_ctx wrapper.  Methods carry the C names without the prefix: apply, energy, apply_host, ..."""

    def __init__(self, grid, lattice, kfrac, kweight, ecut, kind=0, mu=0.0, scale=1.0, nbands=1, stream=None):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("libexx needs a CUDA device (no CPU fallback)")
        self._torch = torch
        L = lib()
        self.grid = tuple(int(g) for g in grid)
        self.ng = self.grid[0] * self.grid[1] * self.grid[2]
        self.nk = len(kweight)
        self.nbands = int(nbands)
        lat = np.ascontiguousarray(lattice, dtype=np.float64).reshape(9)
        kf = np.ascontiguousarray(kfrac, dtype=np.float64).reshape(self.nk * 3)
        kw = np.ascontiguousarray(kweight, dtype=np.float64)
        kp = KernelParams(int(kind), float(mu), float(scale))
        self.stream = stream if stream is not None else torch.cuda.current_stream()
        # libexx enqueues everything on `self.stream`; the context lives on that stream's device (which need not be the current one
        # when the caller hands in a stream), so it is created with that device current
        self.device = self.stream.device.index if getattr(self.stream, "device", None) is not None else torch.cuda.current_device()
        self._h = C.c_void_p()
        g = (C.c_int * 3)(*self.grid)
        with torch.cuda.device(self.device):
            rc = L.exx_create(C.byref(self._h), g, _dp(lat), self.nk, _dp(kf), _dp(kw), float(ecut), C.byref(kp), self.nbands,
                              C.c_void_p(self.stream.cuda_stream))
        if rc:
            raise ExxError(rc, L.exx_last_error(None).decode())
        self.npw = []
        for k in range(self.nk):
            n = C.c_int()
            self._chk(L.exx_npw(self._h, k, C.byref(n)))
            self.npw.append(n.value)
        self.offsets = []
        for k in range(self.nk + 1):
            o = C.c_int64()
            self._chk(L.exx_psi_offset(self._h, k, C.byref(o)))
            self.offsets.append(o.value)
        self.ncoef = self.offsets[-1]

    @classmethod
    def from_workload(cls, w, stream=None):
        return cls(w.grid, w.lattice, w.kfrac, w.kweight, w.ecut, w.kernel_kind, w.mu, w.scale, w.nbands, stream)

    def _chk(self, rc):
        if rc:
            raise ExxError(rc, lib().exx_last_error(self._h).decode())

    def close(self):
        if getattr(self, "_h", None):
            lib().exx_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- queries
    def index_map(self, ik):
        m = np.empty(self.npw[ik], dtype=np.int32)
        self._chk(lib().exx_index_map(self._h, ik, m.ctypes.data_as(C.POINTER(C.c_int32))))
        return m

    def kernel_table(self, ik, iq):
        K = np.empty(self.grid, dtype=np.float64)
        self._chk(lib().exx_kernel_table(self._h, ik, iq, _dp(K)))
        return K

    def set_option(self, opt, value):
        self._chk(lib().exx_set_option(self._h, opt, int(value)))

    def get_option(self, opt):
        v = C.c_int64()
        self._chk(lib().exx_get_option(self._h, opt, C.byref(v)))
        return v.value

    def get_info(self, what):
        v = C.c_int64()
        self._chk(lib().exx_get_info(self._h, what, C.byref(v)))
        return v.value

    def kernel_times(self):
        """{class name: (ms_total, launches, units)} for the last apply (ms needs EXX_OPT_PROFILE = 1)."""
        res = {}
        for k in range(self.get_info(EXX_INFO_NUM_KERNEL_CLASSES)):
            ms, n, u = C.c_double(), C.c_int64(), C.c_int64()
            self._chk(lib().exx_get_kernel_time(self._h, k, C.byref(ms), C.byref(n), C.byref(u)))
            res[lib().exx_kernel_class_name(k).decode()] = (ms.value, n.value, u.value)
        return res

    # ---- device helpers (torch = memory only)
    def _dev(self, t, nelem):
        torch = self._torch
        # the library orders its work on the creation stream only: a call made under another torch stream (or device) would race
        # with the producers/consumers of its tensors, so it is refused rather than silently unordered
        if torch.cuda.current_device() != self.device or t.device.index != self.device:
            raise RuntimeError("this Exx context lives on cuda:%d; call it with that device current and tensors on it" % self.device)
        if torch.cuda.current_stream().cuda_stream != self.stream.cuda_stream:
            raise RuntimeError("call Exx on its creation stream (torch.cuda.stream(ctx.stream)): libexx enqueues on that stream only")
        assert t.is_cuda and t.dtype == torch.complex128 and t.is_contiguous() and t.numel() == nelem, \
            "expected a contiguous complex128 CUDA tensor with %d elements" % nelem
        return C.c_void_p(t.data_ptr())

    def _occ(self, occ):
        occ = np.ascontiguousarray(occ, dtype=np.float64).reshape(-1)
        assert occ.size == self.nk * self.nbands
        return occ

    def empty_like_psi(self):
        return self._torch.empty(self.ncoef, dtype=self._torch.complex128, device="cuda")

    def to_device(self, psi_host):
        return self._torch.from_numpy(np.ascontiguousarray(psi_host, dtype=np.complex128).reshape(-1)).cuda()

    # ---- the calls of include/exx.h
    def apply(self, psi_dev, occ, out_dev=None):
        out_dev = self.empty_like_psi() if out_dev is None else out_dev
        occ = self._occ(occ)
        self._chk(lib().exx_apply(self._h, self._dev(psi_dev, self.ncoef), _dp(occ), self._dev(out_dev, self.ncoef)))
        return out_dev

    def apply_to(self, psi_dev, occ, phi_dev, out_dev=None):
        """out = V_x[psi, occ] phi: the operator defined by the orbitals psi applied to a block of trial vectors phi, nphi per
        k-point packed like psi (nphi = phi.numel() / sum_k npw(k))."""
        occ = self._occ(occ)
        tot = int(sum(self.npw))
        n = int(phi_dev.numel())
        if n % tot or n < tot:
            raise ValueError("phi must hold a whole number of vectors per k-point (%d elements each set)" % tot)
        if out_dev is None:
            out_dev = self._torch.empty_like(phi_dev)
        self._chk(lib().exx_apply_to(self._h, self._dev(psi_dev, self.ncoef), _dp(occ), self._dev(phi_dev, n), n // tot,
                                     self._dev(out_dev, n)))
        return out_dev

    def apply_sharded(self, psi_dev, occ, out_dev=None, group=None, rank=None, world=None):
        """V_x psi with the pair work shared out over the ranks of a torch.distributed group (one process per GPU, every rank
        holding all of psi): this rank's share through exx_apply (EXX_OPT_SHARD_COUNT / _RANK), then ONE all-reduce of the
        sphere coefficients.  Every rank returns the full V_x psi."""
        import torch.distributed as dist
        world = dist.get_world_size(group) if world is None else world
        rank = dist.get_rank(group) if rank is None else rank
        self.set_option(EXX_OPT_SHARD_COUNT, world)
        self.set_option(EXX_OPT_SHARD_RANK, rank)
        try:
            out_dev = self.apply(psi_dev, occ, out_dev)
        finally:
            self.set_option(EXX_OPT_SHARD_RANK, 0)
            self.set_option(EXX_OPT_SHARD_COUNT, 1)
        if world > 1:
            all_reduce_sum(out_dev, group)
        return out_dev

    def energy_sharded(self, psi_dev, occ, group=None, rank=None, world=None):
        """E_x from psi alone with the pair work shared out like apply_sharded: this rank's partial sum through exx_energy
        (EXX_OPT_SHARD_COUNT / _RANK; pair-density route on the fused path), then ONE all-reduce of nk*nbands + 1 doubles
        ("E_x is one scalar all-reduce").  Every rank returns the full (E_x, per-band terms)."""
        import torch.distributed as dist
        world = dist.get_world_size(group) if world is None else world
        rank = dist.get_rank(group) if rank is None else rank
        self.set_option(EXX_OPT_SHARD_COUNT, world)
        self.set_option(EXX_OPT_SHARD_RANK, rank)
        try:
            ex, pb = self.energy(psi_dev, occ, None)
        finally:
            self.set_option(EXX_OPT_SHARD_RANK, 0)
            self.set_option(EXX_OPT_SHARD_COUNT, 1)
        if world > 1:
            t = self._torch.from_numpy(np.concatenate([pb, [ex]])).to(psi_dev.device)
            all_reduce_sum(t, group)
            r = t.cpu().numpy()
            ex, pb = float(r[-1]), r[:-1].copy()
        return ex, pb

    def energy(self, psi_dev, occ, vxpsi_dev=None):
        """(E_x, per-band terms).  Without vxpsi_dev the library works from psi alone (EXX_OPT_ENERGY_ROUTE)."""
        occ = self._occ(occ)
        ex = C.c_double()
        pb = np.empty(self.nk * self.nbands)
        vx = self._dev(vxpsi_dev, self.ncoef) if vxpsi_dev is not None else None
        self._chk(lib().exx_energy(self._h, self._dev(psi_dev, self.ncoef), _dp(occ), vx,
                                   C.cast(C.byref(ex), C.POINTER(C.c_double)), _dp(pb)))
        return ex.value, pb

    def subspace(self, ik, psi_dev, vxpsi_dev, m_dev=None):
        """M[i, j] = <c_i | (V_x c)_j> within k-point ik: (nbands, nbands) complex128 CUDA tensor."""
        if m_dev is None:
            m_dev = self._torch.empty((self.nbands, self.nbands), dtype=self._torch.complex128, device="cuda")
        self._chk(lib().exx_subspace(self._h, ik, self._dev(psi_dev, self.ncoef), self._dev(vxpsi_dev, self.ncoef),
                                     self._dev(m_dev, self.nbands * self.nbands)))
        return m_dev

    def subspace_block(self, ik, phi_dev, vphi_dev, m_dev=None):
        """M[i, j] = <phi_i | vphi_j> within k-point ik for blocks of nphi vectors per k-point (layout of apply_to)."""
        tot = int(sum(self.npw))
        n = int(phi_dev.numel())
        nphi = n // tot
        if m_dev is None:
            m_dev = self._torch.empty((nphi, nphi), dtype=self._torch.complex128, device="cuda")
        self._chk(lib().exx_subspace_block(self._h, ik, self._dev(phi_dev, nphi * tot), self._dev(vphi_dev, nphi * tot), nphi,
                                           self._dev(m_dev, nphi * nphi)))
        return m_dev

    def apply_host(self, psi_host, occ, out_host=None, want_energy=True):
        """psi_host/out_host: complex128 numpy arrays or pinned CPU torch tensors (ncoef elements)."""
        occ = self._occ(occ)
        if out_host is None:
            out_host = np.empty(self.ncoef, dtype=np.complex128)
        ex = C.c_double()
        exp = C.cast(C.byref(ex), C.POINTER(C.c_double)) if want_energy else None
        self._chk(lib().exx_apply_host(self._h, C.c_void_p(_host_ptr(psi_host, self.ncoef)), _dp(occ),
                                       C.c_void_p(_host_ptr(out_host, self.ncoef)), exp))
        return out_host, (ex.value if want_energy else None)

    def scatter(self, ik, coef_dev, nbatch, box_dev):
        self._chk(lib().exx_scatter(self._h, ik, self._dev(coef_dev, nbatch * self.npw[ik]), nbatch, self._dev(box_dev, nbatch * self.ng)))
        return box_dev

    def gather(self, ik, box_dev, nbatch, coef_dev):
        self._chk(lib().exx_gather(self._h, ik, self._dev(box_dev, nbatch * self.ng), nbatch, self._dev(coef_dev, nbatch * self.npw[ik])))
        return coef_dev

    def fft3d(self, box_dev, nbatch, sign):
        self._chk(lib().exx_fft3d(self._h, self._dev(box_dev, nbatch * self.ng), nbatch, sign))
        return box_dev

    def fft3d_fused(self, in_dev, nbatch, sign, out_dev):
        self._chk(lib().exx_fft3d_fused(self._h, self._dev(in_dev, nbatch * self.ng), nbatch, sign, self._dev(out_dev, nbatch * self.ng)))
        return out_dev

    def findex(self):
        f = np.empty(self.ng, dtype=np.int32)
        self._chk(lib().exx_findex(self._h, f.ctypes.data_as(C.POINTER(C.c_int32))))
        return f

    def to_real(self, ik, coef_dev, nbatch, box_dev):
        self._chk(lib().exx_to_real(self._h, ik, self._dev(coef_dev, nbatch * self.npw[ik]), nbatch, self._dev(box_dev, nbatch * self.ng)))
        return box_dev

    def band(self, arr, ik, n):
        o = self.offsets[ik] + n * self.npw[ik]
        return arr.reshape(-1)[o:o + self.npw[ik]]


def _host_ptr(a, nelem):
    if isinstance(a, np.ndarray):
        assert a.dtype == np.complex128 and a.flags["C_CONTIGUOUS"] and a.size == nelem
        return a.ctypes.data
    assert (not a.is_cuda) and a.is_contiguous() and a.numel() == nelem  # torch CPU tensor (pinned or not)
    return a.data_ptr()
