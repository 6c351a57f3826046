"""ctypes binding of the oracle library (oracle/exx_ref.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs may import this.  It imports nothing from paper_1111_0716_b200.

Argument marshalling only; every number is computed by exx_ref.c.
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "exx_ref.c")
_LIB = os.path.join(_HERE, "libexx_ref.so")
_CFLAGS = ["-O2", "-std=c11", "-fopenmp", "-ffp-contract=off", "-fcx-limited-range", "-shared", "-fPIC"]


def build(force=False):
    """Compile oracle/exx_ref.c -> oracle/libexx_ref.so with gcc (rebuilds when the source is newer)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp.%d" % os.getpid()
        subprocess.check_call(["gcc"] + _CFLAGS + ["-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        dp, ip, vp = C.POINTER(C.c_double), C.POINTER(C.c_int), C.c_void_p
        L.exx_ref_create.argtypes = [C.POINTER(vp), ip, dp, C.c_int, dp, dp, C.c_double, C.c_int, C.c_double, C.c_double, C.c_int]
        L.exx_ref_destroy.argtypes = [vp]
        L.exx_ref_npw.argtypes = [vp, C.c_int, ip]
        L.exx_ref_index_map.argtypes = [vp, C.c_int, C.POINTER(C.c_int32)]
        L.exx_ref_psi_offset.argtypes = [vp, C.c_int, C.POINTER(C.c_int64)]
        L.exx_ref_omega.argtypes = [vp]
        L.exx_ref_omega.restype = C.c_double
        L.exx_ref_recip.argtypes = [vp, dp]
        L.exx_ref_kernel_table.argtypes = [vp, C.c_int, C.c_int, dp]
        L.exx_ref_to_real.argtypes = [vp, C.c_int, dp, dp]
        L.exx_ref_apply.argtypes = [vp, dp, dp, dp]
        L.exx_ref_apply_to.argtypes = [vp, dp, dp, dp, C.c_int, dp]
        L.exx_ref_apply_rows.argtypes = [vp, dp, dp, C.c_int, ip, dp]
        L.exx_ref_apply_direct.argtypes = [vp, dp, dp, dp]
        L.exx_ref_energy.argtypes = [vp, dp, dp, dp, dp, dp]
        L.exx_ref_energy_e2.argtypes = [vp, dp, dp, dp]
        L.exx_ref_subspace.argtypes = [vp, C.c_int, dp, dp, dp]
        L.exx_ref_dft1d.argtypes = [C.c_int, C.c_int, dp, dp]
        L.exx_ref_dft1d.restype = None
        L.exx_ref_fft1d.argtypes = [C.c_int, C.c_int, dp, dp]
        L.exx_ref_fft1d.restype = None
        L.exx_ref_fft3d.argtypes = [ip, C.c_int, dp]
        L.exx_ref_fft3d.restype = None
        L.exx_ref_strerror.argtypes = [C.c_int]
        L.exx_ref_strerror.restype = C.c_char_p
        L.exx_ref_num_threads.restype = C.c_int
        _lib = L
    return _lib


class ExxRefError(RuntimeError):
    def __init__(self, code):
        self.code = code
        super().__init__("exx_ref error %d: %s" % (code, lib().exx_ref_strerror(code).decode()))


def _chk(rc):
    if rc != 0:
        raise ExxRefError(rc)


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _c128(a):
    a = np.ascontiguousarray(a, dtype=np.complex128)
    return a


def num_threads():
    return int(lib().exx_ref_num_threads())


def dft1d(x, sign):
    x = _c128(x)
    out = np.empty_like(x)
    lib().exx_ref_dft1d(x.size, sign, _dp(x), _dp(out))
    return out


def fft1d(x, sign):
    x = _c128(x)
    out = np.empty_like(x)
    lib().exx_ref_fft1d(x.size, sign, _dp(x), _dp(out))
    return out


def fft3d(box, sign):
    box = _c128(box).copy()
    n = (C.c_int * 3)(*box.shape)
    lib().exx_ref_fft3d(n, sign, _dp(box))
    return box


class RefExx:
    """Oracle context: same roles as the product's exx_create/apply/energy, on host arrays."""

    def __init__(self, grid, lattice, kfrac, kweight, ecut, kind=0, mu=0.0, scale=1.0, nbands=1):
        self.grid = tuple(int(g) for g in grid)
        self.nk = len(kweight)
        self.nbands = int(nbands)
        lat = np.ascontiguousarray(lattice, dtype=np.float64).reshape(9)
        kf = np.ascontiguousarray(kfrac, dtype=np.float64).reshape(self.nk * 3)
        kw = np.ascontiguousarray(kweight, dtype=np.float64)
        self.kweight = kw.copy()
        self._h = C.c_void_p()
        g = (C.c_int * 3)(*self.grid)
        _chk(lib().exx_ref_create(C.byref(self._h), g, _dp(lat), self.nk, _dp(kf), _dp(kw), float(ecut), int(kind), float(mu),
                                  float(scale), self.nbands))
        self.npw = []
        for k in range(self.nk):
            n = C.c_int()
            _chk(lib().exx_ref_npw(self._h, k, C.byref(n)))
            self.npw.append(n.value)
        self.offsets = [0]
        for k in range(self.nk):
            self.offsets.append(self.offsets[-1] + self.nbands * self.npw[k])
        self.ncoef = self.offsets[-1]
        self.omega = float(lib().exx_ref_omega(self._h))

    def close(self):
        if self._h:
            lib().exx_ref_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def recip(self):
        b = np.empty(9)
        _chk(lib().exx_ref_recip(self._h, _dp(b)))
        return b.reshape(3, 3)

    def index_map(self, ik):
        m = np.empty(self.npw[ik], dtype=np.int32)
        _chk(lib().exx_ref_index_map(self._h, ik, m.ctypes.data_as(C.POINTER(C.c_int32))))
        return m

    def kernel_table(self, ik, iq):
        K = np.empty(self.grid, dtype=np.float64)
        _chk(lib().exx_ref_kernel_table(self._h, ik, iq, _dp(K)))
        return K

    def to_real(self, ik, coef):
        coef = _c128(coef)
        assert coef.size == self.npw[ik]
        box = np.empty(self.grid, dtype=np.complex128)
        _chk(lib().exx_ref_to_real(self._h, ik, _dp(coef), _dp(box)))
        return box

    def _occ(self, occ):
        occ = np.ascontiguousarray(occ, dtype=np.float64).reshape(-1)
        assert occ.size == self.nk * self.nbands
        return occ

    def apply(self, psi, occ):
        psi = _c128(psi).reshape(-1)
        assert psi.size == self.ncoef
        occ = self._occ(occ)
        out = np.empty_like(psi)
        _chk(lib().exx_ref_apply(self._h, _dp(psi), _dp(occ), _dp(out)))
        return out

    def apply_to(self, psi, occ, phi):
        """The operator built from (psi, occ) applied to the vectors phi: nphi vectors per k-point packed like psi
        (nphi = phi.size / sum_k npw(k))."""
        psi, phi = _c128(psi).reshape(-1), _c128(phi).reshape(-1)
        tot = int(sum(self.npw))
        assert psi.size == self.ncoef and phi.size % tot == 0 and phi.size >= tot
        occ = self._occ(occ)
        out = np.empty_like(phi)
        _chk(lib().exx_ref_apply_to(self._h, _dp(psi), _dp(occ), _dp(phi), phi.size // tot, _dp(out)))
        return out

    def apply_rows(self, psi, occ, rows):
        """rows: list of (ik, n).  Returns a list of arrays, one per row, each npw(ik) long."""
        psi = _c128(psi).reshape(-1)
        assert psi.size == self.ncoef
        occ = self._occ(occ)
        rows = [(int(k), int(n)) for k, n in rows]
        r = np.ascontiguousarray(np.array(rows, dtype=np.int32).reshape(-1))
        tot = sum(self.npw[k] for k, _ in rows)
        out = np.empty(tot, dtype=np.complex128)
        _chk(lib().exx_ref_apply_rows(self._h, _dp(psi), _dp(occ), len(rows), r.ctypes.data_as(C.POINTER(C.c_int)), _dp(out)))
        res, pos = [], 0
        for k, _ in rows:
            res.append(out[pos:pos + self.npw[k]])
            pos += self.npw[k]
        return res

    def apply_direct(self, psi, occ):
        psi = _c128(psi).reshape(-1)
        assert psi.size == self.ncoef
        occ = self._occ(occ)
        out = np.empty_like(psi)
        _chk(lib().exx_ref_apply_direct(self._h, _dp(psi), _dp(occ), _dp(out)))
        return out

    def energy(self, psi, occ, vxpsi):
        """(E1).  Returns (E_x, per_band[nk*nb])."""
        psi = _c128(psi).reshape(-1)
        vx = _c128(vxpsi).reshape(-1)
        occ = self._occ(occ)
        ex = C.c_double()
        pb = np.empty(self.nk * self.nbands)
        _chk(lib().exx_ref_energy(self._h, _dp(psi), _dp(occ), _dp(vx), C.cast(C.byref(ex), C.POINTER(C.c_double)), _dp(pb)))
        return ex.value, pb

    def subspace(self, ik, psi, vxpsi):
        """M[i, j] = <c_i | (V_x c)_j> within k-point ik (nb x nb complex)."""
        psi = _c128(psi).reshape(-1)
        vx = _c128(vxpsi).reshape(-1)
        m = np.empty((self.nbands, self.nbands), dtype=np.complex128)
        _chk(lib().exx_ref_subspace(self._h, ik, _dp(psi), _dp(vx), _dp(m)))
        return m

    def energy_e2(self, psi, occ):
        psi = _c128(psi).reshape(-1)
        occ = self._occ(occ)
        ex = C.c_double()
        _chk(lib().exx_ref_energy_e2(self._h, _dp(psi), _dp(occ), C.cast(C.byref(ex), C.POINTER(C.c_double))))
        return ex.value

    def band(self, arr, ik, n):
        """View of band (ik, n) inside a packed psi-layout array."""
        o = self.offsets[ik] + n * self.npw[ik]
        return np.asarray(arr).reshape(-1)[o:o + self.npw[ik]]
