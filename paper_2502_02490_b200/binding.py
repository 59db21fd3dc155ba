"""ctypes binding of include/qxd.h -- same names, argument marshalling only.

Every method of :class:`Qxd` forwards to the C entry point of the same name
(``Qxd.gauge_load`` -> ``qxd_gauge_load`` ...).  Tensors are torch CUDA tensors (or pinned /
pageable host tensors for the ``*_host`` calls); the library borrows their memory.
"""
from __future__ import annotations

import ctypes as C
import os

QXD_F64, QXD_F32, QXD_F16 = 0, 1, 2
QXD_CGNE, QXD_BICGSTAB, QXD_GCR, QXD_DFL_GCR = 0, 1, 2, 3
QXD_RECON_NONE, QXD_RECON_12 = 18, 12
QXD_FS_GAUGE, QXD_FS_HOPLINKS, QXD_FS_CLOVER, QXD_FS_HOPLINKS_STALE, QXD_FS_CLOVER_STALE, QXD_FS_LAZY = 1, 2, 4, 8, 16, 32
QXD_DS_DW, QXD_DS_HOP_AINV, QXD_DS_A_XMHOP, QXD_DS_X_MHOP, QXD_DS_AINV_X_MHOP = 0, 1, 2, 3, 4
QXD_DSF_G5IN, QXD_DSF_G5HOP = 1, 2
QXD_OK, QXD_EINVAL, QXD_ESTATE, QXD_EWORKSPACE, QXD_ECUDA, QXD_ENOCONV = 0, -1, -2, -3, -4, -5

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB = None


class QxdError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__(f"qxd status {status}: {msg}")
        self.status = status


class SolveInfo(C.Structure):
    _fields_ = [("algo", C.c_int), ("sloppy", C.c_int), ("delta", C.c_double), ("maxiter", C.c_int),
                ("iters", C.c_int), ("n_reliable", C.c_int), ("true_res", C.c_double), ("seconds", C.c_double)]


def library_path() -> str:
    return os.path.join(_HERE, "libqxd.so")


# every symbol include/qxd.h declares: name -> (restype, argtypes)
_vp, _i, _d, _l, _sz = C.c_void_p, C.c_int, C.c_double, C.c_long, C.c_size_t
SYMBOLS = {
    "qxd_geometry_create": (_i, [_i, _i, _i, _i, _i, C.POINTER(_vp)]),
    "qxd_geometry_destroy": (_i, [_vp]),
    "qxd_set_tile": (_i, [_vp, _i, _i, _i, _i]),
    "qxd_set_block": (_i, [_vp, _i, _i, _i, _i]),
    "qxd_set_cstar_pairing": (_i, [_vp, _i]),
    "qxd_volume": (_l, [_vp]),
    "qxd_site_index": (_i, [_vp, C.POINTER(_i), C.POINTER(_i), C.POINTER(_i)]),
    "qxd_site_coords": (_i, [_vp, _i, _i, C.POINTER(_i)]),
    "qxd_site_neighbour": (_i, [_vp, _i, _i, _i, _i, C.POINTER(_i)]),
    "qxd_workspace_bytes": (_sz, [_vp, _i, _i]),
    "qxd_workspace_bind": (_i, [_vp, _vp, _sz, _i, _i]),
    "qxd_set_stream": (_i, [_vp, _vp]),
    "qxd_gauge_load": (_i, [_vp, _vp, _vp, _d]),
    "qxd_set_quark": (_i, [_vp, _d, _d]),
    "qxd_clover_build": (_i, [_vp, _d, _d]),
    "qxd_set_lazy_refresh": (_i, [_vp, _i]),
    "qxd_refresh": (_i, [_vp]),
    "qxd_field_status": (_i, [_vp, _vp, _vp]),
    "qxd_set_gauge_reconstruct": (_i, [_vp, _i]),
    "qxd_set_gauge_reconstruct_prec": (_i, [_vp, _i, _i]),
    "qxd_clover_export": (_i, [_vp, _vp, _i]),
    "qxd_clover_stats": (_i, [_vp, _vp]),
    "qxd_apply_Dw": (_i, [_vp, _i, _vp, _vp]),
    "qxd_apply_Dhat_eo": (_i, [_vp, _i, _vp, _vp, _i]),
    "qxd_apply_Dw_host": (_i, [_vp, _i, _vp, _vp]),
    "qxd_solve": (_i, [_vp, _vp, _vp, _d, C.POINTER(SolveInfo)]),
    "qxd_solve_host": (_i, [_vp, _vp, _vp, _d, C.POINTER(SolveInfo)]),
    "qxd_set_gcr": (_i, [_vp, _i, _i, _i]),
    "qxd_apply_sap": (_i, [_vp, _i, _vp, _vp]),
    "qxd_set_deflation": (_i, [_vp, _i, _i, _i, _i]),
    "qxd_set_deflation_chirality": (_i, [_vp, _i]),
    "qxd_set_deflation_refine": (_i, [_vp, _i, _i]),
    "qxd_deflation_setup": (_i, [_vp, _i, _vp]),
    "qxd_deflation_info": (_i, [_vp, C.POINTER(_i), C.POINTER(_i), C.POINTER(_i)]),
    "qxd_deflation_op": (_i, [_vp, _i, _vp, _vp]),
    "qxd_sap_block_of": (_i, [_vp, _i, _i, C.POINTER(_i), C.POINTER(_i)]),
    "qxd_solve_multi": (_i, [_vp, _i, _vp, _vp, _d, C.POINTER(SolveInfo)]),
    "qxd_apply_Dw_multi_packed": (_i, [_vp, _i, _i, _vp, _vp]),
    "qxd_set_rhs_per_thread": (_i, [_vp, _i]),
    "qxd_multi_interleave": (_i, [_vp, _i, _i, _vp, _vp, _i]),
    "qxd_apply_Dw_multi_interleaved": (_i, [_vp, _i, _i, _vp, _vp]),
    "qxd_packed_spinor_bytes": (_sz, [_vp, _i, _i]),
    "qxd_spinor_pack": (_i, [_vp, _i, _vp, _vp]),
    "qxd_spinor_unpack": (_i, [_vp, _i, _vp, _vp]),
    "qxd_apply_Dw_packed": (_i, [_vp, _i, _vp, _vp]),
    "qxd_apply_Dhat_packed": (_i, [_vp, _i, _vp, _vp, _i]),
    "qxd_set_dw_sweep": (_i, [_vp, _i]),
    "qxd_openqxd_index": (_i, [_vp, C.POINTER(_i), _vp, _l, _vp]),
    "qxd_openqxd_reorder": (_i, [_vp, C.POINTER(_i), _i, _i, _vp, _vp]),
    "qxd_openqxd_gauge": (_i, [_vp, C.POINTER(_i), _i, _i, _vp, _vp]),
    "qxd_time_slabs": (_i, [_vp, C.POINTER(_i), C.POINTER(_i)]),
    "qxd_dslash_packed": (_i, [_vp, _i, _i, _i, _i, _vp, _vp, _vp, _i, _i]),
    "qxd_clover_apply_packed": (_i, [_vp, _i, _i, _i, _vp, _vp]),
    "qxd_face_bytes": (_sz, [_vp, _i, _i]),
    "qxd_face_gather": (_i, [_vp, _i, _vp, _i, _i, _i, _i, _vp]),
    "qxd_face_scatter": (_i, [_vp, _i, _vp, _i, _i, _i, _i, _vp]),
    "qxd_halo_zero": (_i, [_vp, _i, _vp, _i, _i, _i, _i]),
    "qxd_blas_norm2_dev": (_i, [_vp, _i, _vp, _vp]),
    "qxd_blas_cg_xr_h": (_i, [_vp] * 9),
    "qxd_blas_cg_p_h": (_i, [_vp] * 6),
    "qxd_noalloc_init": (_i, []),
    "qxd_noalloc_max_reals": (_sz, []),
    "qxd_noalloc_last_error": (C.c_char_p, []),
    "qxd_norm2_noalloc": (_i, [_i, _vp, _sz, _vp, _vp]),
    "qxd_blas_cg_xr": (_i, [_vp, _i, _vp, _vp, _vp, _vp, _vp, _vp, _vp]),
    "qxd_blas_cg_p": (_i, [_vp, _i, _vp, _vp, _vp, _vp]),
    "qxd_blas_copy": (_i, [_vp, _i, _vp, _vp]),
    "qxd_blas_zero": (_i, [_vp, _i, _vp]),
    "qxd_blas_convert": (_i, [_vp, _i, _vp, _i, _vp]),
    "qxd_blas_acc_hi": (_i, [_vp, _i, _vp, _vp]),
    "qxd_blas_sub_norm_dev": (_i, [_vp, _i, _vp, _vp, _vp, _vp]),
    "qxd_blas_axpy": (_i, [_vp, _i, _d, _vp, _vp]),
    "qxd_blas_cdot": (_i, [_vp, _i, _vp, _vp, _vp]),
    "qxd_blas_norm2": (_i, [_vp, _i, _vp, _vp]),
    "qxd_launch_count": (_l, [_vp]),
    "qxd_last_error": (C.c_char_p, [_vp]),
    "qxd_version": (C.c_char_p, []),
}


def load_library():
    """dlopen the in-tree libqxd.so (built by paper_2502_02490_b200/build.py).  Fails loudly if missing."""
    global _LIB
    if _LIB is None:
        path = library_path()
        if not os.path.exists(path):
            raise QxdError(QXD_ESTATE, f"{path} not built: run `python -m paper_2502_02490_b200.build` "
                                       "(or __graft_entry__.build()); there is no CPU fallback")
        lib = C.CDLL(path)
        for name, (res, args) in SYMBOLS.items():
            fn = getattr(lib, name)
            fn.restype = res
            fn.argtypes = args
        _LIB = lib
    return _LIB


def _ptr(t):
    return C.c_void_p(t.data_ptr()) if t is not None else None


def noalloc_max_reals():
    return int(load_library().qxd_noalloc_max_reals())


def norm2_noalloc(x, out, stream=None):
    """out[0] = sum of the squares of the reals of ``x`` (qxd_norm2_noalloc: no context, no workspace, no allocation; the
    partial sums live in a static device array of the library).  x: contiguous CUDA tensor, float64 or float32 (complex
    tensors count their real and imaginary parts); out: CUDA float64 tensor with at least one element, written in stream
    order.  Calls that overlap on the GPU race on the shared scratch (include/qxd.h)."""
    import torch
    lib = load_library()
    if not (x.is_cuda and out.is_cuda and x.is_contiguous() and out.dtype == torch.float64 and out.numel() >= 1):
        raise QxdError(QXD_EINVAL, "norm2_noalloc: x and out must be contiguous CUDA tensors, out float64")
    if x.is_complex():
        x = torch.view_as_real(x)
    if x.dtype == torch.float64:
        prec = QXD_F64
    elif x.dtype == torch.float32:
        prec = QXD_F32
    else:
        raise QxdError(QXD_EINVAL, "norm2_noalloc: float64 or float32 data")
    s = stream if stream is not None else torch.cuda.current_stream(x.device)
    with torch.cuda.device(x.device):
        rc = lib.qxd_norm2_noalloc(prec, _ptr(x), x.numel(), _ptr(out), C.c_void_p(s.cuda_stream))
    if rc != QXD_OK:
        raise QxdError(rc, lib.qxd_noalloc_last_error().decode())
    return out


class Qxd:
    """One solver context (qxd_ctx): geometry, workspace, gauge field, quark, clover term."""

    def __init__(self, T, L1, L2, L3, bc, precisions=(QXD_F64,), nrhs=1, tile=None, block=None, device="cuda:0", pairing=None, gcr=None,
                 deflation=None):
        import torch
        if not torch.cuda.is_available():
            raise QxdError(QXD_ECUDA, "no CUDA device: the qxd hot path has no CPU fallback")
        self.torch = torch
        self.lib = load_library()
        self.device = torch.device(device)
        h = C.c_void_p()
        rc = self.lib.qxd_geometry_create(T, L1, L2, L3, bc, C.byref(h))
        if rc != QXD_OK:
            raise QxdError(rc, "qxd_geometry_create: invalid geometry")
        self.h = h
        self.dims = (T, L1, L2, L3)
        self.cstar = bc & 3
        self.dims_ext = (T, 2 * L1 if self.cstar else L1, L2, L3)
        self.V = self.lib.qxd_volume(self.h)
        if pairing is not None and (self.cstar > 0 or pairing):   # None: library default (paired layout for C* geometries)
            self._chk(self.lib.qxd_set_cstar_pairing(self.h, 1 if pairing else 0))
        if tile is not None:
            self._chk(self.lib.qxd_set_tile(self.h, *tile))
        if block is not None:
            self._chk(self.lib.qxd_set_block(self.h, *block))
        if gcr is not None:                     # (nkv, ncy, nmr): Krylov space and SAP parameters of QXD_GCR (row f3)
            self._chk(self.lib.qxd_set_gcr(self.h, *gcr))
        if deflation is not None:               # (ns, ninv, nkc[, nref]): null vectors, setup smoothing passes, coarse GCR steps, refinement rounds
            d = tuple(deflation) + (0,) * (6 - len(deflation))       # fifth entry: 1 = split the null vectors by chirality; sixth: GCR steps of a refinement solve
            if d[4]:
                self._chk(self.lib.qxd_set_deflation_chirality(self.h, 1))
            self._chk(self.lib.qxd_set_deflation(self.h, *d[:4]))
            if d[5] > 1:
                self.set_deflation_refine(d[3], d[5])
        self.prec_mask = 0
        for p in precisions:
            self.prec_mask |= 1 << p
        self.prec_mask |= 1
        nbytes = self.lib.qxd_workspace_bytes(self.h, self.prec_mask, nrhs)
        with torch.cuda.device(self.device):
            self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
            off = (-self.workspace.data_ptr()) % 256
            self._chk(self.lib.qxd_set_stream(self.h, C.c_void_p(torch.cuda.current_stream().cuda_stream)))
            self._chk(self.lib.qxd_workspace_bind(self.h, C.c_void_p(self.workspace.data_ptr() + off), nbytes, self.prec_mask, nrhs))
        self._keep = []

    # -- plumbing ------------------------------------------------------------------------------
    def _chk(self, rc, allow=()):
        if rc != QXD_OK and rc not in allow:
            raise QxdError(rc, self.lib.qxd_last_error(self.h).decode())
        return rc

    def close(self):
        if getattr(self, "h", None):
            self.torch.cuda.synchronize(self.device)
            self.lib.qxd_geometry_destroy(self.h)
            self.h = None
            self.workspace = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _dev(self, a, dtype=None):
        torch = self.torch
        t = torch.as_tensor(a)
        if dtype is not None and t.dtype != dtype:
            t = t.to(dtype)
        return t.to(self.device).contiguous()

    def set_stream(self, stream=None):
        s = stream if stream is not None else self.torch.cuda.current_stream()
        self._chk(self.lib.qxd_set_stream(self.h, C.c_void_p(s.cuda_stream)))

    def launch_count(self):
        return self.lib.qxd_launch_count(self.h)

    # -- setup ---------------------------------------------------------------------------------
    def gauge_load(self, U_su3, A_u1=None, qel=1.0):
        torch = self.torch
        U = self._dev(U_su3, torch.complex128)
        assert tuple(U.shape) == self.dims + (4, 3, 3), U.shape
        A = None
        if A_u1 is not None:
            A = self._dev(A_u1, torch.float64)
            assert tuple(A.shape) == self.dims + (4,), A.shape
        self._chk(self.lib.qxd_gauge_load(self.h, _ptr(U), _ptr(A), float(qel)))
        torch.cuda.synchronize(self.device)  # inputs may be freed after return

    def set_quark(self, kappa, q=0.0):
        self._chk(self.lib.qxd_set_quark(self.h, float(kappa), float(q)))

    def clover_build(self, csw, csw_qed=0.0):
        self._chk(self.lib.qxd_clover_build(self.h, float(csw), float(csw_qed)))

    def set_lazy_refresh(self, on=True):
        self._chk(self.lib.qxd_set_lazy_refresh(self.h, 1 if on else 0))

    def refresh(self):
        self._chk(self.lib.qxd_refresh(self.h))

    def field_status(self):
        """(status bits QXD_FS_*, hopping-link regenerations, clover regenerations)"""
        st = C.c_int(0)
        cnt = (C.c_long * 2)()
        self._chk(self.lib.qxd_field_status(self.h, C.byref(st), cnt))
        return st.value, cnt[0], cnt[1]

    def multi_interleave(self, plain, interleaved, prec, nrhs, to_interleaved=True):
        self._chk(self.lib.qxd_multi_interleave(self.h, prec, nrhs, _ptr(plain), _ptr(interleaved), int(bool(to_interleaved))))

    def apply_Dw_multi_interleaved(self, pin, pout, prec, nrhs):
        self._chk(self.lib.qxd_apply_Dw_multi_interleaved(self.h, prec, nrhs, _ptr(pin), _ptr(pout)))
        return pout

    def set_dw_sweep(self, tseg):
        self._chk(self.lib.qxd_set_dw_sweep(self.h, int(tseg)))

    def clover_stats(self):
        """(parity passes of the unpivoted block inversion, parity passes redone with the pivoted kernel)"""
        cnt = (C.c_long * 2)()
        self._chk(self.lib.qxd_clover_stats(self.h, cnt))
        return cnt[0], cnt[1]

    def clover_export(self, inverse=False):
        out = self.torch.empty((self.V, 2, 36), dtype=self.torch.float64, device=self.device)
        self._chk(self.lib.qxd_clover_export(self.h, _ptr(out), int(inverse)))
        return out

    # -- natural-order operator applications -----------------------------------------------------
    def apply_Dw(self, psi, prec=QXD_F64, out=None):
        torch = self.torch
        psi = self._dev(psi, torch.complex128)
        assert psi.numel() == self.V * 12
        if out is None:
            out = torch.empty_like(psi)
        self._chk(self.lib.qxd_apply_Dw(self.h, prec, _ptr(psi), _ptr(out)))
        return out

    def apply_Dhat_eo(self, psi_e, prec=QXD_F64, dagger=False):
        torch = self.torch
        psi_e = self._dev(psi_e, torch.complex128)
        assert psi_e.numel() == self.V * 6
        out = torch.empty_like(psi_e)
        self._chk(self.lib.qxd_apply_Dhat_eo(self.h, prec, _ptr(psi_e), _ptr(out), int(dagger)))
        return out

    def apply_Dw_host(self, psi_host, out_host, prec=QXD_F64):
        """psi_host/out_host: CPU complex128 tensors (pinned for best throughput)."""
        assert psi_host.device.type == "cpu" and out_host.device.type == "cpu"
        self._chk(self.lib.qxd_apply_Dw_host(self.h, prec, _ptr(psi_host), _ptr(out_host)))
        return out_host

    # -- solver ------------------------------------------------------------------------------------
    def _info(self, algo, sloppy, delta, maxiter):
        info = SolveInfo()
        info.algo, info.sloppy, info.delta, info.maxiter = algo, sloppy, delta, maxiter
        return info

    @staticmethod
    def _report(rc, info):
        return dict(status=rc, iters=info.iters, n_reliable=info.n_reliable, true_res=info.true_res, seconds=info.seconds)

    def solve(self, eta, tol, algo=QXD_CGNE, sloppy=QXD_F64, delta=0.0, maxiter=0, psi=None):
        torch = self.torch
        eta = self._dev(eta, torch.complex128)
        assert eta.numel() == self.V * 12
        if psi is None:
            psi = torch.empty_like(eta)
        info = self._info(algo, sloppy, delta, maxiter)
        rc = self._chk(self.lib.qxd_solve(self.h, _ptr(eta), _ptr(psi), float(tol), C.byref(info)), allow=(QXD_ENOCONV,))
        return psi, self._report(rc, info)

    def set_deflation_refine(self, nref, steps=1):
        """nref refinement rounds of the deflation space at the next deflation_setup; steps > 1: inverse iteration by that many deflated GCR steps."""
        self._chk(self.lib.qxd_set_deflation_refine(self.h, nref, steps))

    def deflation_setup(self, random_vectors, prec=QXD_F16):
        """random_vectors: ns packed fp32 full-lattice spinors back to back (uint8 tensor on the device)."""
        self._chk(self.lib.qxd_deflation_setup(self.h, prec, _ptr(random_vectors)))

    def deflation_info(self):
        nb, ns, rd = C.c_int(0), C.c_int(0), C.c_int(0)
        self._chk(self.lib.qxd_deflation_info(self.h, C.byref(nb), C.byref(ns), C.byref(rd)))
        return nb.value, ns.value, bool(rd.value)

    def deflation_op(self, op, tin, tout):
        self._chk(self.lib.qxd_deflation_op(self.h, op, _ptr(tin), _ptr(tout)))
        return tout

    def apply_sap(self, pin, pout, prec=QXD_F16):
        """pout = M_sap pin on fp32 packed full-lattice spinors; prec = storage precision of the block operator."""
        self._chk(self.lib.qxd_apply_sap(self.h, prec, _ptr(pin), _ptr(pout)))
        return pout

    def solve_multi(self, eta, tol, sloppy=QXD_F32, delta=0.0, maxiter=0, psi=None):
        """eta: [nrhs, T, X1, L2, L3, 4, 3] complex128 (device).  Returns psi and one report per right-hand side."""
        torch = self.torch
        eta = self._dev(eta, torch.complex128)
        nrhs = eta.numel() // (self.V * 12)
        assert nrhs * self.V * 12 == eta.numel() and nrhs >= 1
        if psi is None:
            psi = torch.empty_like(eta)
        infos = (SolveInfo * nrhs)()
        infos[0].algo, infos[0].sloppy, infos[0].delta, infos[0].maxiter = QXD_CGNE, sloppy, delta, maxiter
        rc = self._chk(self.lib.qxd_solve_multi(self.h, nrhs, _ptr(eta), _ptr(psi), float(tol), infos), allow=(QXD_ENOCONV,))
        return psi, [self._report(rc, infos[k]) for k in range(nrhs)]

    # -- openQxD field orders (row f1) ---------------------------------------------------------------
    def openqxd_index(self, xs, block):
        torch = self.torch
        x = self._dev(xs, torch.int32).reshape(-1, 4)
        out = torch.empty(x.shape[0], dtype=torch.int64, device=self.device)
        self._chk(self.lib.qxd_openqxd_index(self.h, (C.c_int * 4)(*block), _ptr(x), x.shape[0], _ptr(out)))
        return out.cpu().numpy()

    def openqxd_reorder(self, field, reals_per_site, to_openqxd, block):
        torch = self.torch
        f = self._dev(field, torch.float64).reshape(-1)
        assert f.numel() == self.V * reals_per_site, (f.numel(), self.V, reals_per_site)
        out = torch.empty_like(f)
        self._chk(self.lib.qxd_openqxd_reorder(self.h, (C.c_int * 4)(*block), int(reals_per_site), int(bool(to_openqxd)), _ptr(f), _ptr(out)))
        return out.reshape(self.V, reals_per_site)

    def openqxd_gauge(self, field, to_openqxd, block, phase=False):
        torch = self.torch
        f = self._dev(field, torch.float64 if phase else torch.complex128).reshape(-1)
        nr = 1 if phase else 18
        vphys = self.dims[0] * self.dims[1] * self.dims[2] * self.dims[3]
        n_in, n_out = (vphys * 4, self.V // 2 * 8) if to_openqxd else (self.V // 2 * 8, vphys * 4)
        per = 1 if phase else 9
        assert f.numel() == n_in * per, (f.numel(), n_in * per)
        out = torch.empty(n_out * per, dtype=f.dtype, device=self.device)
        self._chk(self.lib.qxd_openqxd_gauge(self.h, (C.c_int * 4)(*block), nr, int(bool(to_openqxd)), _ptr(f), _ptr(out)))
        if to_openqxd:
            return out.reshape((self.V // 2, 8) + (() if phase else (3, 3)))
        return out.reshape(self.dims + (4,) + (() if phase else (3, 3)))

    def set_gauge_reconstruct(self, recon, prec=None):
        if prec is None:
            self._chk(self.lib.qxd_set_gauge_reconstruct(self.h, int(recon)))
        else:
            self._chk(self.lib.qxd_set_gauge_reconstruct_prec(self.h, int(prec), int(recon)))

    def set_rhs_per_thread(self, r):
        self._chk(self.lib.qxd_set_rhs_per_thread(self.h, int(r)))

    def apply_Dw_multi_packed(self, pin, pout, prec, nrhs):
        self._chk(self.lib.qxd_apply_Dw_multi_packed(self.h, prec, int(nrhs), _ptr(pin), _ptr(pout)))
        return pout

    def solve_host(self, eta_host, psi_host, tol, algo=QXD_CGNE, sloppy=QXD_F64, delta=0.0, maxiter=0):
        assert eta_host.device.type == "cpu" and psi_host.device.type == "cpu"
        info = self._info(algo, sloppy, delta, maxiter)
        rc = self._chk(self.lib.qxd_solve_host(self.h, _ptr(eta_host), _ptr(psi_host), float(tol), C.byref(info)), allow=(QXD_ENOCONV,))
        return psi_host, self._report(rc, info)

    # -- domain decomposition building blocks (row f2) ---------------------------------------------------
    def time_slabs(self):
        n, t = C.c_int(0), C.c_int(0)
        self._chk(self.lib.qxd_time_slabs(self.h, C.byref(n), C.byref(t)))
        return n.value, t.value

    def dslash_packed(self, mode, pin, pout, prec, parity_out=0, flags=0, phi=None, slabs=None):
        lo, hi = slabs if slabs is not None else (0, self.time_slabs()[0])
        self._chk(self.lib.qxd_dslash_packed(self.h, prec, mode, flags, parity_out, _ptr(pin), _ptr(phi), _ptr(pout), lo, hi))
        return pout

    def clover_apply_packed(self, pin, pout, prec, parity, inverse=False):
        self._chk(self.lib.qxd_clover_apply_packed(self.h, prec, int(inverse), parity, _ptr(pin), _ptr(pout)))
        return pout

    def face_buffer(self, prec, mu):
        n = self.lib.qxd_face_bytes(self.h, prec, mu)
        dt = self.torch.float64 if prec == QXD_F64 else self.torch.float32
        return self.torch.zeros(n // (8 if prec == QXD_F64 else 4), dtype=dt, device=self.device)

    def face_gather(self, packed, prec, parity_mask, mu, coord, sign, buf):
        self._chk(self.lib.qxd_face_gather(self.h, prec, _ptr(packed), parity_mask, mu, coord, sign, _ptr(buf)))
        return buf

    def face_scatter(self, packed, prec, parity_mask, mu, coord, shift1, buf):
        self._chk(self.lib.qxd_face_scatter(self.h, prec, _ptr(packed), parity_mask, mu, coord, shift1, _ptr(buf)))

    def halo_zero(self, packed, prec, parity_mask, mu, lo, hi):
        self._chk(self.lib.qxd_halo_zero(self.h, prec, _ptr(packed), parity_mask, mu, lo, hi))

    def blas_norm2_dev(self, x, prec, out):
        self._chk(self.lib.qxd_blas_norm2_dev(self.h, prec, _ptr(x), _ptr(out)))

    def blas_cg_xr(self, prec, num, den, p, t, x, r, rr):
        self._chk(self.lib.qxd_blas_cg_xr(self.h, prec, _ptr(num), _ptr(den), _ptr(p), _ptr(t), _ptr(x), _ptr(r), _ptr(rr)))

    def blas_cg_xr_h(self, num, den, p16, t16, x32, r32, r16, rr):
        self._chk(self.lib.qxd_blas_cg_xr_h(self.h, _ptr(num), _ptr(den), _ptr(p16), _ptr(t16), _ptr(x32), _ptr(r32), _ptr(r16), _ptr(rr)))

    def blas_cg_p_h(self, num, den, s16, p32, p16):
        self._chk(self.lib.qxd_blas_cg_p_h(self.h, _ptr(num), _ptr(den), _ptr(s16), _ptr(p32), _ptr(p16)))

    def blas_cg_p(self, prec, num, den, s, p):
        self._chk(self.lib.qxd_blas_cg_p(self.h, prec, _ptr(num), _ptr(den), _ptr(s), _ptr(p)))

    def blas_copy(self, x, y, prec):
        self._chk(self.lib.qxd_blas_copy(self.h, prec, _ptr(x), _ptr(y)))

    def blas_zero(self, x, prec):
        self._chk(self.lib.qxd_blas_zero(self.h, prec, _ptr(x)))

    def blas_convert(self, x, prec_from, y, prec_to):
        self._chk(self.lib.qxd_blas_convert(self.h, prec_from, _ptr(x), prec_to, _ptr(y)))

    def blas_acc_hi(self, x_lo, prec, x_hi):
        self._chk(self.lib.qxd_blas_acc_hi(self.h, prec, _ptr(x_lo), _ptr(x_hi)))

    def blas_sub_norm_dev(self, b, t, r, prec, rr):
        self._chk(self.lib.qxd_blas_sub_norm_dev(self.h, prec, _ptr(b), _ptr(t), _ptr(r), _ptr(rr)))

    # -- packed layout -------------------------------------------------------------------------------
    def packed_spinor_bytes(self, prec, half_only=False):
        return self.lib.qxd_packed_spinor_bytes(self.h, prec, int(half_only))

    def new_packed(self, prec, half_only=False):
        return self.torch.zeros(self.packed_spinor_bytes(prec, half_only), dtype=self.torch.uint8, device=self.device)

    def spinor_pack(self, nat, prec, packed=None):
        nat = self._dev(nat, self.torch.complex128)
        if packed is None:
            packed = self.new_packed(prec)
        self._chk(self.lib.qxd_spinor_pack(self.h, prec, _ptr(nat), _ptr(packed)))
        return packed

    def spinor_unpack(self, packed, prec):
        out = self.torch.empty(self.dims_ext + (4, 3), dtype=self.torch.complex128, device=self.device)
        self._chk(self.lib.qxd_spinor_unpack(self.h, prec, _ptr(packed), _ptr(out)))
        return out

    def apply_Dw_packed(self, pin, pout, prec):
        self._chk(self.lib.qxd_apply_Dw_packed(self.h, prec, _ptr(pin), _ptr(pout)))
        return pout

    def apply_Dhat_packed(self, pin_e, pout_e, prec, dagger=False):
        self._chk(self.lib.qxd_apply_Dhat_packed(self.h, prec, _ptr(pin_e), _ptr(pout_e), int(dagger)))
        return pout_e

    # -- BLAS-1 on packed half-lattice spinors ---------------------------------------------------------
    def blas_axpy(self, a, x, y, prec):
        self._chk(self.lib.qxd_blas_axpy(self.h, prec, float(a), _ptr(x), _ptr(y)))
        return y

    def blas_cdot(self, x, y, prec):
        out = (C.c_double * 2)()
        self._chk(self.lib.qxd_blas_cdot(self.h, prec, _ptr(x), _ptr(y), C.cast(out, C.c_void_p)))
        return complex(out[0], out[1])

    def blas_norm2(self, x, prec):
        out = C.c_double(0.0)
        self._chk(self.lib.qxd_blas_norm2(self.h, prec, _ptr(x), C.cast(C.byref(out), C.c_void_p)))
        return out.value
