"""GPU parity of SURVEY.md §8(f) row f3: the Schwarz alternating procedure (SAP) and the SAP-preconditioned GCR.

The paper names the method and nothing else ("heavily preconditioned GCR ... Schwarz alternating procedure"),
so the preconditioner is checked against a step-by-step restatement of include/qxd.h's definition built from the ORACLE's
D_w (block restriction by masking, per-block minimal-residual steps, exact residual update by a full D_w apply), and the
solver through the only thing that is unique: ||eta - D_ref psi|| / ||eta|| with the oracle's D_w over the whole lattice.
"""
import ctypes as C

import numpy as np
import pytest

import synth
from test_gpu_parity import Case, relerr, to_np, F64, F32, F16

pytestmark = pytest.mark.gpu

GCR = 2


def true_residual(ref, eta, psi):
    return np.linalg.norm(np.ravel(eta) - np.ravel(ref.apply_Dw(psi))) / np.linalg.norm(np.ravel(eta))


def block_map(c):
    """(tile id, colour) of every site of the extended lattice in natural order, from the library's host-side introspection
    of its site order (qxd_site_index): a block is one 128-index tile; its colour is the parity of its box coordinates."""
    lib = c.B.load_library()
    X = c.dims_ext
    V = c.V
    tile = np.empty(V, dtype=np.int64)
    coords = np.stack(np.unravel_index(np.arange(V), X), axis=1).astype(np.int32)
    cb, par = C.c_int(0), C.c_int(0)
    for s in range(V):
        x = (C.c_int * 4)(*coords[s])
        assert lib.qxd_site_index(c.gpu.h, x, C.byref(cb), C.byref(par)) == 0
        tile[s] = cb.value >> 7
    # box of every tile on the indexed lattice (physical coordinates in the paired layout: both mirror images share a tile)
    ci = coords.astype(np.int64).copy()
    if c.gpu.cstar and c.pairing:
        ci[:, 1] %= c.dims[1]
    ntiles = tile.max() + 1
    lo = np.full((ntiles, 4), 1 << 30)
    hi = np.full((ntiles, 4), -1)
    np.minimum.at(lo, tile, ci)
    np.maximum.at(hi, tile, ci)
    ext = (hi - lo + 1)
    assert (ext == ext[0]).all() and (np.prod(ext[0]) * (2 if (c.gpu.cstar and c.pairing) else 1) == 256)
    box = lo // ext[0]
    nbox = box.max(axis=0) + 1
    colour_t = (box * (nbox > 1)).sum(axis=1) & 1
    return tile, colour_t[tile]


def sap_reference(c, tile, colour, r_in, ncy, nmr):
    """M_sap r_in as include/qxd.h defines it, with the oracle's D_w: for cy < ncy, for colour in (0, 1): on every block of the
    colour nmr minimal-residual steps on P D_w P; psi += e; r -= D_w e (exact, by a full apply)."""
    D = lambda v: c.ref.apply_Dw(v.reshape(c.psi_shape)).reshape(-1, 12)
    psi = np.zeros((c.V, 12), dtype=complex)
    r = r_in.reshape(-1, 12).astype(complex)
    ntiles = tile.max() + 1
    for _ in range(ncy):
        for col in (0, 1):
            mask = (colour == col)[:, None]
            rho = r * mask
            e = np.zeros_like(r)
            for _ in range(nmr):
                t = D(rho) * mask
                num = np.zeros(ntiles, dtype=complex)
                den = np.zeros(ntiles)
                np.add.at(num, tile, np.sum(np.conj(t) * rho, axis=1))
                np.add.at(den, tile, np.sum(np.abs(t) ** 2, axis=1))
                alpha = np.where(den > 0, num / np.where(den > 0, den, 1.0), 0.0)[tile][:, None]
                e += alpha * rho
                rho -= alpha * t
            psi += e
            r = r - D(e)
    return psi


SAP_CASES = [
    # dims, cstar, qed, pairing
    ((8, 8, 8, 8), 0, False, False),
    ((8, 8, 8, 8), 3, True, False),
    ((8, 4, 8, 8), 3, True, True),
    ((16, 8, 8, 8), 2, True, True),
]


@pytest.mark.parametrize("dims,cstar,qed,pairing", SAP_CASES)
@pytest.mark.parametrize("prec,recon", [(F32, 18), (F32, 14), (F16, 18)])
def test_sap_matches_stepwise_definition(dims, cstar, qed, pairing, prec, recon):
    import torch
    ncy, nmr = 3, 4
    c = Case(dims, cstar, 1, qed, q=-1 / 3, kappa=0.125, csw=1.5, csw_qed=1.0, eps=0.2, pairing=pairing, gcr=(4, ncy, nmr))
    c.pairing = pairing
    c.psi_shape = tuple(c.dims_ext) + (4, 3)
    g, B = c.gpu, c.B
    g.set_gauge_reconstruct(B.QXD_RECON_12 if recon == 14 else B.QXD_RECON_NONE, prec=prec)
    tile, colour = block_map(c)
    r_in = synth.gaussian_spinor(c.dims_ext, 71)
    pin = g.spinor_pack(r_in, F32)
    pout = torch.zeros_like(pin)
    g.apply_sap(pin, pout, prec)
    got = to_np(g.spinor_unpack(pout, F32)).reshape(-1, 12)
    r32 = to_np(g.spinor_unpack(pin, F32)).reshape(-1, 12)          # the input as the device holds it (rounded to fp32)
    exp = sap_reference(c, tile, colour, r32, ncy, nmr)
    # fp32 arithmetic through 2 ncy (nmr + 1) block operators; binary16 storage of links and clover blocks (reading R13)
    assert relerr(got, exp) < (1e-4 if prec == F32 else 5e-3), relerr(got, exp)
    # the preconditioner does reduce the residual substantially
    res = np.linalg.norm(r32 - c.ref.apply_Dw(got.reshape(c.psi_shape)).reshape(-1, 12)) / np.linalg.norm(r32)
    assert res < 0.3, res
    c.close()


@pytest.mark.parametrize("dims,cstar,qed,pairing", SAP_CASES + [((8, 8, 8, 8), 3, True, True)])
@pytest.mark.parametrize("sloppy", [F32, F16])
def test_gcr_solve_small(dims, cstar, qed, pairing, sloppy):
    c = Case(dims, cstar, 1, qed, q=2 / 3, kappa=0.125, csw=1.5, csw_qed=1.0, eps=0.2, pairing=pairing, gcr=(8, 4, 4))
    eta = synth.gaussian_spinor(c.dims_ext, 5)
    psi, info = c.gpu.solve(eta, 1e-10, algo=GCR, sloppy=sloppy)
    assert info["status"] == 0, info
    res = true_residual(c.ref, eta, to_np(psi).reshape(eta.shape))
    assert res <= 1.05e-10, (res, info)
    assert abs(res - info["true_res"]) <= 0.1 * res
    assert info["n_reliable"] >= 2                 # fp32 cycles cannot reach 1e-10 without fp64 restarts
    # GCR with the Schwarz preconditioner needs far fewer operator applications than CG on the normal equations
    _, icg = c.gpu.solve(eta, 1e-10, algo=0, sloppy=F32)
    assert info["iters"] < icg["iters"], (info, icg)
    c.close()


def test_gcr_argument_errors_and_zero_source():
    import torch
    c = Case((8, 8, 8, 8), 0, 1, False, precisions=(F64, F32))           # no Krylov space
    eta = synth.gaussian_spinor(c.dims_ext, 5)
    with pytest.raises(c.B.QxdError) as e:
        c.gpu.solve(eta, 1e-10, algo=GCR, sloppy=F32)
    assert e.value.status == c.B.QXD_EWORKSPACE
    c.close()
    c = Case((8, 8, 8, 8), 0, 1, False, precisions=(F64, F32), gcr=(4, 2, 4))
    with pytest.raises(c.B.QxdError) as e:
        c.gpu.solve(eta, 1e-10, algo=GCR, sloppy=F64)                     # block operator in fp64: not provided
    assert e.value.status == c.B.QXD_EINVAL
    psi, info = c.gpu.solve(np.zeros_like(eta), 1e-10, algo=GCR, sloppy=F32)
    assert info["status"] == 0 and info["iters"] == 0 and float(psi.abs().max()) == 0.0
    psi, info = c.gpu.solve(eta, 1e-10, algo=GCR, sloppy=F32, maxiter=3)
    assert info["status"] == c.B.QXD_ENOCONV and info["iters"] == 3
    res = true_residual(c.ref, eta, to_np(psi).reshape(eta.shape))
    assert abs(res - info["true_res"]) < 1e-9 and res < 1.0
    c.close()
    # a lattice with an odd number of blocks in a direction has no two-colouring: rejected, not silently wrong
    c = Case((12, 4, 4, 4), 0, 1, False, precisions=(F64, F32), gcr=(4, 2, 4))
    with pytest.raises(c.B.QxdError) as e:
        c.gpu.solve(synth.gaussian_spinor(c.dims_ext, 5), 1e-10, algo=GCR, sloppy=F32)
    assert e.value.status == c.B.QXD_EINVAL
    c.close()


@pytest.mark.parametrize("sloppy", [F32, F16])
def test_gcr_config_c2_full_size(sloppy):
    """BASELINE config 2 at full size (32x16^3 QCD+QED C*, paired layout = the library default)."""
    cfg = synth.config("c2")
    c = Case(cfg["dims"], cfg["cstar"], cfg["antiperiodic"], cfg["qed"], q=cfg["q"], kappa=cfg["kappa"], csw=cfg["csw"],
             csw_qed=cfg["csw_qed"], qel=cfg["qel"], eps=cfg["eps"], pairing=True, gcr=(16, 4, 4))
    eta = synth.gaussian_spinor(c.dims_ext, 3)
    psi, info = c.gpu.solve(eta, cfg["tol"], algo=GCR, sloppy=sloppy)
    assert info["status"] == 0, info
    assert true_residual(c.ref, eta, to_np(psi).reshape(eta.shape)) <= 1.05 * cfg["tol"]
    c.close()


# ---- second level: local-coherence deflation (qxd_set_deflation / qxd_deflation_setup / QXD_DFL_GCR) ---------------------------
DFL_GCR = 3


def _dfl_case(dims, cstar, qed, pairing, ns=8, ninv=3, nkc=12, kappa=0.125, prec=F32, nref=0, chiral=0, refk=1):
    import torch
    c = Case(dims, cstar, 1, qed, q=2 / 3, kappa=kappa, csw=1.5, csw_qed=1.0, eps=0.2, pairing=pairing, gcr=(8, 3, 4),
             deflation=(ns, ninv, nkc, nref, chiral, refk))
    g = c.gpu
    rnd = torch.cat([g.spinor_pack(synth.gaussian_spinor(c.dims_ext, 100 + i), F32) for i in range(ns)])
    g.deflation_setup(rnd, prec)
    return c, rnd


@pytest.mark.parametrize("dims,cstar,qed,pairing", SAP_CASES)
@pytest.mark.parametrize("chiral", [0, 1])
def test_deflation_subspace_and_coarse_operator(dims, cstar, qed, pairing, chiral):
    """R P = 1 on the coarse space (block-orthonormal null vectors), P R is a projector, and the stored nine-point coarse operator
    equals R D_w P applied through the (oracle-verified) fp32 D_w kernel.  chiral = 1: null vectors split by chirality (2 ns
    coarse degrees of freedom per block); then gamma5 maps the deflation space onto itself."""
    import torch
    c, _ = _dfl_case(dims, cstar, qed, pairing, chiral=chiral)
    g = c.gpu
    nb, ns, ready = g.deflation_info()
    assert ready and nb == c.V // 256 and ns == 8 * (1 + chiral)
    rng = np.random.default_rng(7)
    cc = torch.from_numpy((rng.normal(size=(nb, ns)) + 1j * rng.normal(size=(nb, ns))).astype(np.complex64)).cuda()
    fine = g.new_packed(F32)
    g.deflation_op(1, cc, fine)                                   # P c
    back = torch.empty_like(cc)
    g.deflation_op(0, fine, back)                                 # R P c
    assert float((back - cc).abs().max() / cc.abs().max()) < 2e-5
    fine2 = g.new_packed(F32)
    g.deflation_op(1, back, fine2)                                # P R P c = P c
    a, b = to_np(g.spinor_unpack(fine, F32)), to_np(g.spinor_unpack(fine2, F32))
    assert relerr(b, a) < 2e-5
    dfine = g.new_packed(F32)
    g.apply_Dw_packed(fine, dfine, F32)                           # D_w P c
    ref_c = torch.empty_like(cc)
    g.deflation_op(0, dfine, ref_c)                               # R D_w P c
    got_c = torch.empty_like(cc)
    g.deflation_op(2, cc, got_c)                                  # A_c c
    assert float((got_c - ref_c).abs().max() / ref_c.abs().max()) < 1e-4
    # and against the ORACLE's D_w: R D_ref P c with P c taken from the device
    dref = c.ref.apply_Dw(a.reshape(tuple(c.dims_ext) + (4, 3)))
    pd = g.spinor_pack(dref, F32)
    ref2 = torch.empty_like(cc)
    g.deflation_op(0, pd, ref2)
    assert float((got_c - ref2).abs().max() / ref2.abs().max()) < 1e-4
    if chiral:     # gamma5 P c = P c' with c'[2 i + chi] = (+1, -1)[chi] c[2 i + chi]   (chiral basis: gamma5 = diag(1, 1, -1, -1))
        g5 = a.reshape(tuple(c.dims_ext) + (4, 3)).copy()
        g5[..., 2:, :] *= -1
        sgn = torch.tensor([1.0, -1.0], device="cuda").repeat(ns // 2)
        g.deflation_op(1, (cc * sgn).contiguous(), fine2)
        assert relerr(to_np(g.spinor_unpack(fine2, F32)), g5) < 2e-6
    c.close()


@pytest.mark.parametrize("dims,cstar,qed,pairing", SAP_CASES)
@pytest.mark.parametrize("chiral", [0, 1])
def test_coarse_solve_even_odd(dims, cstar, qed, pairing, chiral):
    """The coarse-grid solver (GCR on the even-odd Schur form of the nine-point operator, matrices read in binary16): the
    residual b - A_c x, evaluated with the fp32 coarse operator that the previous test ties to R D_w P, falls with the number of
    steps down to the rounding of the binary16 copy; x = 0 for b = 0."""
    import torch
    res = []
    for nkc in (4, 32):
        c, _ = _dfl_case(dims, cstar, qed, pairing, ns=8, ninv=3, nkc=nkc, chiral=chiral)
        g = c.gpu
        nb, ns, _ = g.deflation_info()
        rng = np.random.default_rng(11)
        b = torch.from_numpy((rng.normal(size=(nb, ns)) + 1j * rng.normal(size=(nb, ns))).astype(np.complex64)).cuda()
        x = torch.empty_like(b)
        g.deflation_op(4, b, x)
        ax = torch.empty_like(b)
        g.deflation_op(2, x, ax)
        res.append(float(torch.linalg.vector_norm(b - ax) / torch.linalg.vector_norm(b)))
        if nkc == 4:
            z = torch.zeros_like(b)
            g.deflation_op(4, z, x)
            assert float(x.abs().max()) == 0.0
        c.close()
    assert res[0] < 0.5 and res[1] < 5e-3 and res[1] < 0.1 * res[0], res


@pytest.mark.parametrize("ns,chiral", [(2, 0), (2, 1), (16, 1), (32, 0)])
def test_coarse_level_at_the_extreme_sizes(ns, chiral):
    """The smallest and the largest coarse dimensions per block (2 and 32; CTA shapes of the coarse kernels depend on it): R P = 1,
    A_c c = R D_w P c through the fp32 D_w kernel, the coarse solver reduces the residual, and the solve converges."""
    import torch
    dims, cstar, qed, pairing = SAP_CASES[0]
    c, _ = _dfl_case(dims, cstar, qed, pairing, ns=ns, ninv=2, nkc=16, chiral=chiral)
    g = c.gpu
    nb, nc, ready = g.deflation_info()
    assert ready and nc == ns * (1 + chiral)
    rng = np.random.default_rng(3)
    cc = torch.from_numpy((rng.normal(size=(nb, nc)) + 1j * rng.normal(size=(nb, nc))).astype(np.complex64)).cuda()
    fine, back = g.new_packed(F32), torch.empty_like(cc)
    g.deflation_op(1, cc, fine)
    g.deflation_op(0, fine, back)
    assert float((back - cc).abs().max() / cc.abs().max()) < 5e-5
    dfine, ref_c, got_c = g.new_packed(F32), torch.empty_like(cc), torch.empty_like(cc)
    g.apply_Dw_packed(fine, dfine, F32)
    g.deflation_op(0, dfine, ref_c)
    g.deflation_op(2, cc, got_c)
    assert float((got_c - ref_c).abs().max() / ref_c.abs().max()) < 2e-4
    x, ax = torch.empty_like(cc), torch.empty_like(cc)
    g.deflation_op(4, cc, x)
    g.deflation_op(2, x, ax)
    assert float(torch.linalg.vector_norm(cc - ax) / torch.linalg.vector_norm(cc)) < 2e-2
    eta = synth.gaussian_spinor(c.dims_ext, 5)
    psi, info = g.solve(eta, 1e-10, algo=DFL_GCR, sloppy=F16)
    assert info["status"] == 0 and true_residual(c.ref, eta, to_np(psi).reshape(eta.shape)) <= 1.05e-10
    c.close()


def test_deflation_pays_on_a_smooth_field():
    """On links with long-range order (synth.su3_links_smooth) close to the critical hopping parameter the low modes are locally
    coherent: the deflated solver must need clearly fewer GCR steps than the plain Schwarz-preconditioned one, both reaching the
    oracle residual.  (On the white-noise links of the other cases there is nothing to deflate.)"""
    import torch
    from paper_2502_02490_b200 import binding as B
    from oracle import qxd_ref as R
    dims = (16, 16, 16, 16)
    U = synth.su3_links_smooth(dims, 0.7, 1, 4)
    eta = synth.gaussian_spinor(dims, 3)
    ns = 12
    g = B.Qxd(*dims, 4, precisions=(0, 1, 2), gcr=(16, 4, 5), deflation=(ns, 6, 12, 0))
    g.gauge_load(U, None, 1.0)
    g.set_quark(0.1295, 0.0)
    g.clover_build(1.0, 0.0)
    rnd = torch.cat([g.spinor_pack(synth.gaussian_spinor(dims, 100 + i), F32) for i in range(ns)])
    g.deflation_setup(rnd, F16)
    ref = R.Ref(*dims, 4)
    ref.gauge_load(U, None, 1.0)
    ref.set_quark(0.1295, 0.0)
    ref.clover_build(1.0, 0.0)
    steps = {}
    for algo in (GCR, DFL_GCR):
        psi, info = g.solve(eta, 1e-10, algo=algo, sloppy=F16, maxiter=2000)
        assert info["status"] == 0, info
        assert true_residual(ref, eta, to_np(psi).reshape(eta.shape)) <= 1.05e-10
        steps[algo] = info["iters"]
    assert steps[DFL_GCR] < 0.6 * steps[GCR], steps
    g.close()


@pytest.mark.parametrize("dims,cstar,qed,pairing", SAP_CASES)
@pytest.mark.parametrize("sloppy,chiral", [(F32, 0), (F16, 0), (F16, 1)])
def test_deflated_gcr_solve(dims, cstar, qed, pairing, sloppy, chiral):
    """QXD_DFL_GCR: the two-level preconditioner is a contraction on the residual (|r - D_ref M r| < |r| with the oracle's D_w),
    the solve reaches the oracle residual, and a change of the quark invalidates the setup (QXD_ESTATE) until it is redone."""
    import torch
    # refinement of the deflation space: one application of the two-level preconditioner per vector (fp32 case), an inverse
    # iteration of 3 deflated GCR steps per vector (chirality-split case), none (fp16 case)
    c, rnd = _dfl_case(dims, cstar, qed, pairing, ns=8, ninv=4, nkc=16, kappa=0.125, prec=sloppy, nref=1 if (sloppy == F32 or chiral) else 0,
                       chiral=chiral, refk=3 if chiral else 1)
    g = c.gpu
    eta = synth.gaussian_spinor(c.dims_ext, 5)
    pin = g.spinor_pack(eta, F32)
    pz = g.new_packed(F32)
    g.deflation_op(3, pin, pz)
    r32 = to_np(g.spinor_unpack(pin, F32)).reshape(eta.shape)
    z = to_np(g.spinor_unpack(pz, F32)).reshape(eta.shape)
    contraction = np.linalg.norm(r32 - c.ref.apply_Dw(z)) / np.linalg.norm(r32)
    assert contraction < 0.5, contraction
    psi, info = g.solve(eta, 1e-10, algo=DFL_GCR, sloppy=sloppy)
    assert info["status"] == 0, info
    res = true_residual(c.ref, eta, to_np(psi).reshape(eta.shape))
    assert res <= 1.05e-10, (res, info)
    g.set_quark(0.124, 2 / 3 if qed else 0.0)
    g.clover_build(1.5, 1.0 if qed else 0.0)
    assert g.deflation_info()[2] is False
    with pytest.raises(c.B.QxdError) as e:
        g.solve(eta, 1e-10, algo=DFL_GCR, sloppy=sloppy)
    assert e.value.status == c.B.QXD_ESTATE
    g.deflation_setup(rnd, sloppy)                 # redone for the new quark: usable again
    psi, info = g.solve(eta, 1e-10, algo=DFL_GCR, sloppy=sloppy)
    assert info["status"] == 0
    c.close()
