"""Field-status manager (include/qxd.h "field-status manager").

An HMC trajectory changes the gauge field while kappa, q, c_sw stay.  With lazy refresh the derived fields (hopping links,
clover term and inverse) are marked stale by the setters and regenerated once, at their first use.  CPU: the host-side
state machine of the calls that need no device.  GPU: a short "trajectory" of changing gauge fields and quark parameters,
every operator application and solve compared with an oracle that was rebuilt from scratch for that field."""
import ctypes as C

import numpy as np
import pytest

import synth
from oracle import qxd_ref as R

KAPPA, CSW, CSWQ, Q = 0.12, 1.5, 1.0, 2.0 / 3.0


def test_status_calls_without_a_device():
    from paper_2502_02490_b200 import binding as B
    lib = B.load_library()
    h = C.c_void_p()
    assert lib.qxd_geometry_create(4, 4, 4, 4, 3 | 4, C.byref(h)) == 0
    st = C.c_int(-1)
    cnt = (C.c_long * 2)(-1, -1)
    assert lib.qxd_field_status(h, C.byref(st), cnt) == 0 and st.value == 0 and tuple(cnt) == (0, 0)
    assert lib.qxd_set_lazy_refresh(h, 1) == 0
    assert lib.qxd_field_status(h, C.byref(st), None) == 0 and st.value == B.QXD_FS_LAZY
    assert lib.qxd_refresh(h) == 0                         # nothing stale: no device work
    assert lib.qxd_set_lazy_refresh(h, 0) == 0
    assert lib.qxd_field_status(h, C.byref(st), None) == 0 and st.value == 0
    assert lib.qxd_field_status(h, None, None) == B.QXD_EINVAL
    assert lib.qxd_field_status(None, C.byref(st), None) == B.QXD_EINVAL
    assert lib.qxd_set_lazy_refresh(None, 1) == B.QXD_EINVAL and lib.qxd_refresh(None) == B.QXD_EINVAL
    assert lib.qxd_geometry_destroy(h) == 0


def fresh_oracle(dims, bc, U, A, kappa, q, csw, cswq):
    ref = R.Ref(*dims, bc)
    ref.gauge_load(U, A, 1.0)
    ref.set_quark(kappa, q)
    ref.clover_build(csw, cswq)
    return ref


def relerr(a, b):
    a, b = np.asarray(a).ravel(), np.asarray(b).ravel()
    return np.linalg.norm(a - b) / np.linalg.norm(b)


@pytest.mark.gpu
@pytest.mark.parametrize("dims,cstar,pairing", [((8, 4, 4, 4), 3, True), ((8, 4, 4, 4), 3, False), ((4, 4, 4, 8), 0, None)])
def test_trajectory_with_lazy_refresh(dims, cstar, pairing):
    from paper_2502_02490_b200 import binding as B
    bc = cstar | 4
    g = B.Qxd(*dims, bc, precisions=(B.QXD_F64, B.QXD_F32), pairing=pairing)
    X = g.dims_ext
    psi = synth.gaussian_spinor(X, 3)
    pe = synth.gaussian_spinor(X, 6).reshape(-1, 4, 3)[: g.V // 2]
    fields = [(synth.su3_links(dims, 0.3, 10 + k), synth.u1_field(dims, 0.3, 20 + k)) for k in range(3)]
    FS = B

    # eager default: a new gauge field invalidates what depends on it
    g.gauge_load(*fields[0], 1.0)
    g.set_quark(KAPPA, Q)
    g.clover_build(CSW, CSWQ)
    assert g.field_status() == (FS.QXD_FS_GAUGE | FS.QXD_FS_HOPLINKS | FS.QXD_FS_CLOVER, 1, 1)
    g.gauge_load(*fields[1], 1.0)
    assert g.field_status()[0] == FS.QXD_FS_GAUGE
    with pytest.raises(B.QxdError) as e:
        g.apply_Dw(psi)
    assert e.value.status == B.QXD_ESTATE

    # lazy: the setters record, the first use regenerates, once
    g.set_lazy_refresh(True)
    g.set_quark(KAPPA, Q)
    g.clover_build(CSW, CSWQ)
    lazy_stale = FS.QXD_FS_GAUGE | FS.QXD_FS_HOPLINKS_STALE | FS.QXD_FS_CLOVER_STALE | FS.QXD_FS_LAZY
    clean = FS.QXD_FS_GAUGE | FS.QXD_FS_HOPLINKS | FS.QXD_FS_CLOVER | FS.QXD_FS_LAZY
    assert g.field_status() == (lazy_stale, 1, 1)
    ref = fresh_oracle(dims, bc, *fields[1], KAPPA, Q, CSW, CSWQ)
    exp = ref.apply_Dw(psi)
    assert relerr(g.apply_Dw(psi).cpu().numpy().reshape(exp.shape), exp) < 1e-13
    assert g.field_status() == (clean, 2, 2)
    assert relerr(g.apply_Dw(psi, B.QXD_F32).cpu().numpy().reshape(exp.shape), exp) < 1e-6
    assert g.field_status() == (clean, 2, 2)

    # the trajectory: gauge_load; solve; gauge_load; solve ...  (one regeneration per field, in every bound precision)
    for k, (U, A) in enumerate(fields):
        g.gauge_load(U, A, 1.0)
        assert g.field_status() == (lazy_stale, 2 + k, 2 + k)
        ref = fresh_oracle(dims, bc, U, A, KAPPA, Q, CSW, CSWQ)
        sol, info = g.solve(psi, 1e-10, algo=B.QXD_CGNE, sloppy=B.QXD_F32)
        assert info["status"] == 0
        sol = sol.cpu().numpy().reshape(psi.shape)
        assert relerr(ref.apply_Dw(sol), psi) <= 1.05e-10       # true residual, by the oracle's operator on this field
        assert g.field_status() == (clean, 3 + k, 3 + k)
        e2 = ref.apply_Dhat(pe)
        assert relerr(g.apply_Dhat_eo(pe).cpu().numpy().reshape(e2.shape), e2) < 2e-13
        assert g.field_status() == (clean, 3 + k, 3 + k)
    n = 2 + len(fields)

    # another quark flavour on the same field: hopping links (charge) and clover term (mass, charge) follow
    g.set_quark(0.115, -1.0 / 3.0)
    assert g.field_status() == (lazy_stale, n, n)
    ref = fresh_oracle(dims, bc, *fields[-1], 0.115, -1.0 / 3.0, CSW, CSWQ)
    e2 = ref.apply_Dhat(pe, dagger=True)
    assert relerr(g.apply_Dhat_eo(pe, dagger=True).cpu().numpy().reshape(e2.shape), e2) < 2e-13
    assert g.field_status() == (clean, n + 1, n + 1)

    # new improvement coefficients: only the clover term is stale; the 12-real link format on a stale field waits too
    g.clover_build(1.2, 0.8)
    assert g.field_status() == (FS.QXD_FS_GAUGE | FS.QXD_FS_HOPLINKS | FS.QXD_FS_CLOVER_STALE | FS.QXD_FS_LAZY, n + 1, n + 1)
    ref = fresh_oracle(dims, bc, *fields[-1], 0.115, -1.0 / 3.0, 1.2, 0.8)
    got = g.clover_export(False).cpu().numpy()
    assert relerr(got, ref.clover_packed(False).reshape(got.shape)) < 1e-13
    assert g.field_status() == (clean, n + 1, n + 2)
    g.gauge_load(*fields[0], 1.0)
    g.set_gauge_reconstruct(B.QXD_RECON_12)
    assert g.field_status() == (lazy_stale, n + 1, n + 2)
    ref = fresh_oracle(dims, bc, *fields[0], 0.115, -1.0 / 3.0, 1.2, 0.8)
    exp = ref.apply_Dw(psi)
    assert relerr(g.apply_Dw(psi).cpu().numpy().reshape(exp.shape), exp) < 1e-13
    assert g.field_status() == (clean, n + 2, n + 3)

    # host-buffer call and explicit refresh; switching lazy refresh off regenerates what is stale
    g.gauge_load(*fields[1], 1.0)
    g.refresh()
    assert g.field_status() == (clean, n + 3, n + 4)
    g.gauge_load(*fields[2], 1.0)
    ref = fresh_oracle(dims, bc, *fields[2], 0.115, -1.0 / 3.0, 1.2, 0.8)
    exp = ref.apply_Dw(psi)
    import torch
    hin = torch.from_numpy(np.ascontiguousarray(psi)).pin_memory()
    hout = torch.empty_like(hin).pin_memory()
    g.apply_Dw_host(hin, hout, B.QXD_F64)
    assert relerr(hout.numpy().reshape(exp.shape), exp) < 1e-13
    assert g.field_status() == (clean, n + 4, n + 5)
    g.gauge_load(*fields[0], 1.0)
    g.set_lazy_refresh(False)
    assert g.field_status() == (clean & ~FS.QXD_FS_LAZY, n + 5, n + 6)
    g.close()
