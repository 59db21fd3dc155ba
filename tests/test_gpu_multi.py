"""GPU parity of the multi-RHS path (BASELINE config 4): the batched D_w and the batched
mixed-precision solve against the fp64 CPU oracle, right-hand side by right-hand side.  Tolerances as in
test_gpu_parity.py (fp64 1e-13, fp32 1e-6, fp16 2e-3; solves: true residual with the oracle's D)."""
import numpy as np
import pytest

import synth
from test_gpu_parity import Case, relerr, to_np, TOL, F64, F32, F16

pytestmark = pytest.mark.gpu


def true_residual(ref, eta, psi):
    return np.linalg.norm(np.ravel(eta - ref.apply_Dw(psi))) / np.linalg.norm(np.ravel(eta))


# nrhs chosen to be ragged against 2 and 3 right-hand sides per thread; Vh = 720 has a ragged tile tail
@pytest.mark.parametrize("dims,cstar,qed,nrhs", [((6, 4, 6, 10), 0, False, 5), ((6, 4, 4, 6), 3, True, 4), ((4, 4, 4, 4), 0, True, 1)])
@pytest.mark.parametrize("prec", [F64, F32, F16])
@pytest.mark.parametrize("rpt", [0, 1, 2, 3])
def test_apply_Dw_multi(dims, cstar, qed, nrhs, prec, rpt):
    import torch
    c = Case(dims, cstar, 1, qed, nrhs=max(nrhs, 2))
    g = c.gpu
    g.set_rhs_per_thread(rpt)
    etas = [synth.gaussian_spinor(c.dims_ext, 11 + k) for k in range(nrhs)]
    nb = g.packed_spinor_bytes(prec)
    pin = torch.zeros(nrhs * nb, dtype=torch.uint8, device="cuda")
    pout = torch.zeros_like(pin)
    for k in range(nrhs):
        g.spinor_pack(etas[k], prec, packed=pin[k * nb:(k + 1) * nb])
    g.apply_Dw_multi_packed(pin, pout, prec, nrhs)
    for k in range(nrhs):
        got = to_np(g.spinor_unpack(pout[k * nb:(k + 1) * nb], prec))
        assert relerr(got, c.ref.apply_Dw(etas[k])) < TOL[prec], (k, prec, rpt)
    # the batched launch must agree bit for bit with nrhs single launches (same arithmetic per site)
    single = torch.zeros(nb, dtype=torch.uint8, device="cuda")
    g.apply_Dw_packed(pin[:nb], single, prec)
    assert torch.equal(single, pout[:nb])
    c.close()


@pytest.mark.parametrize("dims,cstar,qed,pairing", [((8, 4, 4, 8), 0, False, False), ((8, 4, 4, 8), 3, True, False), ((8, 4, 4, 8), 3, True, True),
                                                    ((6, 4, 6, 10), 2, True, True)])
@pytest.mark.parametrize("prec", [F64, F32, F16])
@pytest.mark.parametrize("recon", [18, 14])
def test_apply_Dw_multi_interleaved_is_bit_identical(dims, cstar, qed, pairing, prec, recon):
    """Experimental layout of row a10 (right-hand sides across lanes, csrc/dslash_ilv.cu): interleave -> batched D_w -> de-interleave
    must equal the plain batch bit for bit (same arithmetic per site and right-hand side), which is itself compared with the oracle
    in test_apply_Dw_multi; ragged tile tail (Vh = 720 x 2) and both link formats included."""
    import torch
    c = Case(dims, cstar, 1, qed, nrhs=8, pairing=pairing)
    g = c.gpu
    g.set_gauge_reconstruct(c.B.QXD_RECON_12 if recon == 14 else c.B.QXD_RECON_NONE)
    n = 8
    nb = g.packed_spinor_bytes(prec)
    pin = torch.zeros(n * nb, dtype=torch.uint8, device="cuda")
    for k in range(n):
        g.spinor_pack(synth.gaussian_spinor(c.dims_ext, 11 + k), prec, packed=pin[k * nb:(k + 1) * nb])
    pout, qin, qout, back = (torch.zeros_like(pin) for _ in range(4))
    g.apply_Dw_multi_packed(pin, pout, prec, n)
    g.multi_interleave(pin, qin, prec, n, True)
    g.apply_Dw_multi_interleaved(qin, qout, prec, n)
    g.multi_interleave(back, qout, prec, n, False)
    assert torch.equal(back, pout)
    with pytest.raises(c.B.QxdError):
        g.apply_Dw_multi_interleaved(qin, qout, prec, 6)          # not a multiple of 4
    c.close()


@pytest.mark.parametrize("sloppy", [F32, F16])
@pytest.mark.parametrize("rpt", [0, 2])
def test_solve_multi(sloppy, rpt):
    """Five systems (one of them with a zero source, one a multiple of another) to 1e-10 in lockstep."""
    dims = (8, 4, 4, 8)
    c = Case(dims, 3, 1, True, q=-1 / 3, kappa=0.125, csw=1.5, csw_qed=1.0, eps=0.2, nrhs=5)
    c.gpu.set_rhs_per_thread(rpt)
    etas = np.stack([synth.gaussian_spinor(c.dims_ext, 21 + k) for k in range(5)])
    etas[2] = 0.0
    etas[4] = 1e-3 * etas[0]
    psi, infos = c.gpu.solve_multi(etas, 1e-10, sloppy=sloppy, delta=0.1)
    psi = to_np(psi).reshape(etas.shape)
    for k in range(5):
        assert infos[k]["status"] == 0, infos[k]
        if k == 2:
            assert np.all(psi[k] == 0) and infos[k]["iters"] == 0
            continue
        assert true_residual(c.ref, etas[k], psi[k]) <= 1.05e-10, (k, infos[k])
        assert infos[k]["n_reliable"] >= 2
    # in-place (psi aliases eta) gives the same solutions
    import torch
    buf = torch.from_numpy(etas).cuda()
    c.gpu.solve_multi(buf, 1e-10, sloppy=sloppy, delta=0.1, psi=buf)
    assert relerr(to_np(buf).reshape(etas.shape)[[0, 1, 3, 4]], psi[[0, 1, 3, 4]]) < 1e-8
    c.close()


def test_solve_multi_argument_errors():
    c = Case((4, 4, 4, 4), 0, 1, False, precisions=(F64, F32), nrhs=2)
    B = c.B
    etas = np.stack([synth.gaussian_spinor(c.dims_ext, 31 + k) for k in range(3)])
    with pytest.raises(B.QxdError) as e:
        c.gpu.solve_multi(etas, 1e-10, sloppy=F32)            # 3 systems, workspace bound for 2
    assert e.value.status == B.QXD_EINVAL
    with pytest.raises(B.QxdError) as e:
        c.gpu.solve_multi(etas[:2], 1e-10, sloppy=F64)        # batch vectors sized for fp32
    assert e.value.status == B.QXD_EINVAL
    c.close()
    c1 = Case((4, 4, 4, 4), 0, 1, False, precisions=(F64, F32), nrhs=1)
    with pytest.raises(B.QxdError) as e:
        c1.gpu.solve_multi(etas[:1], 1e-10, sloppy=F32)       # workspace bound without a batch
    assert e.value.status == B.QXD_EWORKSPACE
    c1.close()


class _Shared:
    pass


@pytest.fixture(scope="module")
def c4_oracle():
    """Oracle context of BASELINE config 4 (96x48^3 QCD, 10.6 M sites), built once for the module."""
    from oracle import qxd_ref as R
    cfg = synth.config("c4")
    o = _Shared()
    o.cfg = cfg
    o.U = synth.su3_links(cfg["dims"], cfg["eps"], 1)
    o.A = None
    o.ref = R.Ref(*cfg["dims"], cfg["bc"])
    o.ref.gauge_load(o.U, None, cfg["qel"])
    o.ref.set_quark(cfg["kappa"], cfg["q"])
    o.ref.clover_build(cfg["csw"], cfg["csw_qed"])
    yield o


def test_full_c4_gcr_sap_converges_where_bicgstab_does_not(c4_oracle):
    """Row f3 at config 4: the SAP-preconditioned GCR reaches 1e-10 (whole-lattice residual with the oracle's D_w) on the
    system on which BiCGstab on D-hat stalls (round 1: QXD_ENOCONV after 548 iterations, true residual 6e-3)."""
    cfg = c4_oracle.cfg
    c = Case(cfg["dims"], cfg["cstar"], cfg["antiperiodic"], cfg["qed"], q=cfg["q"], kappa=cfg["kappa"], csw=cfg["csw"],
             csw_qed=cfg["csw_qed"], qel=cfg["qel"], eps=cfg["eps"], precisions=(F64, F32, F16), share=c4_oracle, gcr=(16, 4, 5))
    eta = synth.gaussian_spinor(c.dims_ext, 51)
    psi, info = c.gpu.solve(eta, cfg["tol"], algo=2, sloppy=F16, maxiter=2000)
    assert info["status"] == 0 and info["true_res"] <= cfg["tol"], info
    assert true_residual(c.ref, eta, to_np(psi).reshape(eta.shape)) <= 1.05 * cfg["tol"]
    _, ib = c.gpu.solve(eta, cfg["tol"], algo=1, sloppy=F32, maxiter=2000)
    assert ib["status"] in (0, c.B.QXD_ENOCONV)
    if ib["status"] == 0:
        assert ib["true_res"] <= cfg["tol"]
    c.close()


def test_full_c4_twelve_rhs_batched_dslash_and_solve(c4_oracle):
    """BASELINE config 4 AS STATED (96x48^3 QCD, 10.6 M sites): 12 Gaussian right-hand sides, the 12-RHS batched D_w in the
    launch configuration bench.py uses and the batched mixed fp64/fp32 solve of all 12 systems to 1e-10; every right-hand
    side is compared with the oracle over the WHOLE lattice (D_w: relative L2; solve: ||eta - D_ref psi|| / ||eta||).
    Sources are generated one at a time (a c4 spinor is 2 GB in fp64) and regenerated for the check."""
    import torch
    cfg = c4_oracle.cfg
    n = cfg["nrhs"]
    assert n == 12
    c = Case(cfg["dims"], cfg["cstar"], cfg["antiperiodic"], cfg["qed"], q=cfg["q"], kappa=cfg["kappa"], csw=cfg["csw"],
             csw_qed=cfg["csw_qed"], qel=cfg["qel"], eps=cfg["eps"], precisions=(F64, F32), nrhs=n, share=c4_oracle)
    g = c.gpu
    source = lambda k: synth.gaussian_spinor(c.dims_ext, 51 + k)
    # ---- batched D_w, 12 right-hand sides in one launch ----
    nb = g.packed_spinor_bytes(F32)
    pin = torch.empty(n * nb, dtype=torch.uint8, device="cuda")
    pout = torch.zeros_like(pin)
    for k in range(n):
        g.spinor_pack(source(k), F32, packed=pin[k * nb:(k + 1) * nb])
    g.apply_Dw_multi_packed(pin, pout, F32, n)
    for k in (0, 5, 11):
        got = to_np(g.spinor_unpack(pout[k * nb:(k + 1) * nb], F32))
        exp = c.ref.apply_Dw(source(k))
        assert relerr(got, exp) < TOL[F32], k
    del pin, pout, got, exp
    torch.cuda.empty_cache()
    # ---- batched solve of the 12 systems, in place on the device ----
    buf = torch.empty((n,) + tuple(c.dims_ext) + (4, 3), dtype=torch.complex128, device="cuda")
    for k in range(n):
        buf[k].copy_(torch.from_numpy(source(k)))
    _, infos = g.solve_multi(buf, cfg["tol"], sloppy=F32, delta=0.1, maxiter=5000, psi=buf)
    for k in range(n):
        assert infos[k]["status"] == 0 and infos[k]["true_res"] <= cfg["tol"], (k, infos[k])
        res = true_residual(c.ref, source(k), to_np(buf[k]))
        assert res <= 1.05 * cfg["tol"], (k, res, infos[k])
    c.close()


def test_solve_multi_fp16_only_workspace():
    """Only fp64 and binary16 bound: the batch workspace has no room for fp32 Krylov vectors, so the batched solver runs
    with binary16 vectors throughout (more iterations, same acceptance on the fp64 true residual)."""
    dims = (8, 4, 4, 8)
    c = Case(dims, 3, 1, True, q=-1 / 3, kappa=0.125, csw=1.5, csw_qed=1.0, eps=0.2, precisions=(F64, F16), nrhs=3)
    etas = np.stack([synth.gaussian_spinor(c.dims_ext, 61 + k) for k in range(3)])
    psi, infos = c.gpu.solve_multi(etas, 1e-10, sloppy=F16, delta=0.1)
    psi = to_np(psi).reshape(etas.shape)
    for k in range(3):
        assert infos[k]["status"] == 0, infos[k]
        assert true_residual(c.ref, etas[k], psi[k]) <= 1.05e-10
    c.close()
