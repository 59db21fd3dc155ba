"""ctypes binding of the fp64 CPU oracle (oracle/qxd_ref.cpp).

TEST INFRASTRUCTURE, NOT PRODUCT CODE: only tests/, ``__graft_entry__.smoke()`` and
``bench.py``'s cpu_baseline / ``--impl reference`` legs may import this module.  It never
imports the CUDA package and the CUDA package never imports it.

Array conventions (numpy, C-contiguous):
  U    complex128 [T,L1,L2,L3,4,3,3]   SU(3) links on the PHYSICAL lattice (row-major a,b)
  A    float64    [T,L1,L2,L3,4]       U(1) field on the physical lattice (or None: QCD only)
  psi  complex128 [T,X1,L2,L3,4,3]     spinor on the EXTENDED lattice (Eq. (1))
  psi_e complex128 [V/2,4,3]           even sites in increasing Lambda order
"""
from __future__ import annotations

import ctypes as C
import numpy as np

from . import build as _build

_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build())
        vp, d, i, l = C.c_void_p, C.c_double, C.c_int, C.c_long
        L.qxd_ref_create.restype = vp
        L.qxd_ref_create.argtypes = [i, i, i, i, i]
        L.qxd_ref_destroy.argtypes = [vp]
        L.qxd_ref_volume.restype = l
        L.qxd_ref_volume.argtypes = [vp]
        L.qxd_ref_gauge_load.argtypes = [vp, vp, vp, d]
        L.qxd_ref_set_quark.argtypes = [vp, d, d]
        L.qxd_ref_set_csw.argtypes = [vp, d, d]
        L.qxd_ref_site_matrix.argtypes = [vp, l, vp]
        L.qxd_ref_clover_build.argtypes = [vp, d, d]
        L.qxd_ref_clover_max_offdiag.restype = d
        L.qxd_ref_clover_max_offdiag.argtypes = [vp]
        L.qxd_ref_clover_max_antiherm.restype = d
        L.qxd_ref_clover_max_antiherm.argtypes = [vp]
        L.qxd_ref_clover_packed.argtypes = [vp, vp, i]
        L.qxd_ref_apply_Dw.argtypes = [vp, vp, vp]
        L.qxd_ref_apply_Dw_sites.argtypes = [vp, vp, l, vp, vp]
        L.qxd_ref_apply_Dhat.argtypes = [vp, vp, vp, i]
        L.qxd_ref_clover_build_range.argtypes = [vp, d, d, l, l]
        L.qxd_ref_apply_Dw_range.argtypes = [vp, vp, vp]
        L.qxd_ref_solve.argtypes = [vp, vp, vp, d, i, vp, vp]
        L.qxd_ref_num_threads.restype = i
        _lib = L
    return _lib


def num_threads() -> int:
    return lib().qxd_ref_num_threads()


def _p(a):
    return a.ctypes.data_as(C.c_void_p)


class RefError(RuntimeError):
    pass


def _chk(rc, what):
    if rc != 0:
        raise RefError(f"{what} failed with status {rc}")


class Ref:
    """One oracle context: geometry + gauge field + quark parameters + clover field."""

    def __init__(self, T, L1, L2, L3, bc):
        self.h = lib().qxd_ref_create(T, L1, L2, L3, bc)
        if not self.h:
            raise RefError("qxd_ref_create: invalid geometry")
        self.cstar = bc & 3
        self.dims = (T, L1, L2, L3)
        self.dims_ext = (T, 2 * L1 if self.cstar else L1, L2, L3)
        self.V = lib().qxd_ref_volume(self.h)

    def __del__(self):
        if getattr(self, "h", None):
            lib().qxd_ref_destroy(self.h)
            self.h = None

    def gauge_load(self, U, A=None, qel=1.0):
        U = np.ascontiguousarray(U, dtype=np.complex128)
        assert U.shape == self.dims + (4, 3, 3), U.shape
        if A is not None:
            A = np.ascontiguousarray(A, dtype=np.float64)
            assert A.shape == self.dims + (4,), A.shape
        _chk(lib().qxd_ref_gauge_load(self.h, _p(U), _p(A) if A is not None else None, qel), "gauge_load")

    def set_quark(self, kappa, q=0.0):
        _chk(lib().qxd_ref_set_quark(self.h, kappa, q), "set_quark")

    def set_csw(self, csw, csw_qed=0.0):
        _chk(lib().qxd_ref_set_csw(self.h, csw, csw_qed), "set_csw")

    def clover_build(self, csw, csw_qed=0.0):
        _chk(lib().qxd_ref_clover_build(self.h, csw, csw_qed), "clover_build")

    def clover_diagnostics(self):
        return (lib().qxd_ref_clover_max_offdiag(self.h), lib().qxd_ref_clover_max_antiherm(self.h))

    def site_matrix(self, site):
        out = np.empty((12, 12), dtype=np.complex128)
        _chk(lib().qxd_ref_site_matrix(self.h, int(site), _p(out)), "site_matrix")
        return out

    def clover_packed(self, inverse=False):
        out = np.empty((self.V, 2, 36), dtype=np.float64)
        _chk(lib().qxd_ref_clover_packed(self.h, _p(out), int(inverse)), "clover_packed")
        return out

    def _spinor(self, psi):
        psi = np.ascontiguousarray(psi, dtype=np.complex128)
        assert psi.size == self.V * 12, psi.shape
        return psi

    def apply_Dw(self, psi):
        psi = self._spinor(psi)
        out = np.empty_like(psi)
        _chk(lib().qxd_ref_apply_Dw(self.h, _p(psi), _p(out)), "apply_Dw")
        return out

    def apply_Dw_sites(self, psi, sites):
        psi = self._spinor(psi)
        sites = np.ascontiguousarray(sites, dtype=np.int64)
        out = np.empty((sites.size, 4, 3), dtype=np.complex128)
        _chk(lib().qxd_ref_apply_Dw_sites(self.h, _p(psi), sites.size, _p(sites), _p(out)), "apply_Dw_sites")
        return out

    def clover_build_range(self, csw, csw_qed, lo, hi):
        """Clover blocks for the natural-order site range [lo, hi) only (bounded-sample timing)."""
        _chk(lib().qxd_ref_clover_build_range(self.h, csw, csw_qed, int(lo), int(hi)), "clover_build_range")
        self._range = (int(lo), int(hi))

    def apply_Dw_range(self, psi, out=None):
        psi = self._spinor(psi)
        lo, hi = self._range
        if out is None:
            out = np.empty((hi - lo, 4, 3), dtype=np.complex128)
        _chk(lib().qxd_ref_apply_Dw_range(self.h, _p(psi), _p(out)), "apply_Dw_range")
        return out

    def apply_Dhat(self, psi_e, dagger=False):
        psi_e = np.ascontiguousarray(psi_e, dtype=np.complex128)
        assert psi_e.size == self.V * 6
        out = np.empty_like(psi_e)
        _chk(lib().qxd_ref_apply_Dhat(self.h, _p(psi_e), _p(out), int(dagger)), "apply_Dhat")
        return out

    def solve(self, eta, tol, maxiter=100000):
        eta = self._spinor(eta)
        psi = np.empty_like(eta)
        it = C.c_int(0)
        res = C.c_double(0.0)
        rc = lib().qxd_ref_solve(self.h, _p(eta), _p(psi), tol, maxiter, C.byref(it), C.byref(res))
        if rc not in (0, -5):
            _chk(rc, "solve")
        return psi, dict(status=rc, iters=it.value, relres=res.value)
