"""GPU parity: the CUDA path (through the C-ABI, paper_2502_02490_b200.binding) against the fp64 CPU
oracle, element by element on the same seeded inputs (SURVEY.md §8(d) "Parity").

Tolerances (BASELINE.json north_star):
  fp64 operator: relative L2 error <= 1e-13;  fp32: <= 1e-6;  fp16 (reading R13): <= 2e-3;
  solves: ||eta - D_ref psi|| / ||eta|| <= tol with the ORACLE's D (1e-12 for c0/c1, 1e-10 mixed).
Integer / layout work (pack -> unpack) is bit-exact.
"""
import numpy as np
import pytest

import synth
from oracle import qxd_ref as R

pytestmark = pytest.mark.gpu

F64, F32, F16 = 0, 1, 2
TOL = {F64: 1e-13, F32: 1e-6, F16: 2e-3}


def relerr(a, b):
    a = np.ravel(a)
    b = np.ravel(b)
    return np.linalg.norm(a - b) / np.linalg.norm(b)


def to_np(t):
    return t.detach().cpu().numpy()


class Case:
    """Oracle context + CUDA context on identical seeded fields."""

    def __init__(self, dims, cstar, ap, qed, q=2 / 3, kappa=0.12, csw=1.5, csw_qed=1.0, qel=1.0, eps=0.3,
                 precisions=(F64, F32, F16), tile=None, oracle_clover=True, nrhs=1, pairing=False, share=None, gcr=None, deflation=None):
        from paper_2502_02490_b200 import binding as B
        self.B = B
        bc = cstar | (ap << 2)
        self.dims = dims
        self.q = q if qed else 0.0
        self.csw_qed = csw_qed if qed else 0.0
        if share is not None:       # same fields and oracle context as another case (only the CUDA context differs)
            self.U, self.A, self.ref = share.U, share.A, share.ref
        else:
            self.U = synth.su3_links(dims, eps, 1)
            self.A = synth.u1_field(dims, 0.3, 2) if qed else None
            self.ref = R.Ref(*dims, bc)
            self.ref.gauge_load(self.U, self.A, qel)
            self.ref.set_quark(kappa, self.q)
            if oracle_clover:
                self.ref.clover_build(csw, self.csw_qed)
            else:
                self.ref.set_csw(csw, self.csw_qed)
        self.gpu = B.Qxd(*dims, bc, precisions=precisions, tile=tile, nrhs=nrhs, pairing=pairing, gcr=gcr, deflation=deflation)
        self.gpu.gauge_load(self.U, self.A, qel)
        self.gpu.set_quark(kappa, self.q)
        self.gpu.clover_build(csw, self.csw_qed)
        self.dims_ext = self.ref.dims_ext
        self.V = self.ref.V

    def close(self):
        self.gpu.close()


# dims (physical), cstar, antiperiodic, qed  -- several tiles, ragged tails (Vh % 128 != 0), L=2 edge cases
SMALL = [
    ((4, 4, 4, 4), 0, 1, False),      # BASELINE config c0
    ((4, 4, 4, 4), 0, 0, True),
    ((6, 4, 6, 10), 0, 1, True),      # Vh = 720: ragged tail, non power-of-two extents
    ((4, 2, 4, 4), 1, 1, True),
    ((4, 4, 2, 6), 2, 1, True),
    ((6, 4, 4, 6), 3, 1, True),
    ((2, 2, 2, 2), 3, 1, True),       # degenerate: forward and backward neighbour coincide
    ((8, 8, 8, 8), 3, 1, True),       # BASELINE config c1 (q = +2/3)
    # the same C* cases in the C*-paired device layout (links and clover once per physical site)
    ((4, 2, 4, 4), 1, 1, True, True),
    ((4, 4, 2, 6), 2, 1, True, True),
    ((6, 4, 4, 6), 3, 1, True, True),
    ((2, 2, 2, 2), 3, 1, True, True),
    ((8, 8, 8, 8), 3, 1, True, True),
    ((8, 4, 4, 4), 3, 0, False, True),   # QCD only, periodic in time
    # several 4^4 tiles per 16x4x4x4 block AND several blocks in time, as at c3 (b0 = 4, B0 = 16), both layouts
    ((32, 4, 4, 8), 3, 1, True, True),
    ((32, 4, 4, 8), 3, 1, True),
    ((32, 8, 4, 4), 2, 1, True, True),
]


@pytest.fixture(scope="module", params=SMALL,
                ids=lambda p: "x".join(map(str, p[0])) + f"-cstar{p[1]}ap{p[2]}{'qed' if p[3] else 'qcd'}{'-paired' if len(p) > 4 and p[4] else ''}")
def case(request):
    p = request.param
    c = Case(*p[:4], pairing=(len(p) > 4 and p[4]))
    yield c
    c.close()


def test_clover_blocks_match_oracle(case):
    """Row a3: M and M^{-1} in the PAPER.md:117 packing, fp64."""
    got = to_np(case.gpu.clover_export(False))
    exp = case.ref.clover_packed(False)
    assert relerr(got, exp) < 1e-13
    got = to_np(case.gpu.clover_export(True))
    exp = case.ref.clover_packed(True)
    assert relerr(got, exp) < 1e-12  # inverse of a 6x6 block with cond ~ 10


def test_clover_pivoted_inversion_fallback():
    """Row a3, the fallback of the block inversion: kappa is chosen so that the leading diagonal entry of one chirality
    block is ~1e-9 (4 + m0 cancels the clover diagonal there) while the block stays well conditioned.  The unpivoted
    in-register Gauss-Jordan must notice the tiny pivot and the library must redo the inversion with the partially pivoted
    kernel (qxd_clover_stats); M^{-1} is compared with the oracle's (LAPACK-style partial pivoting)."""
    from paper_2502_02490_b200 import binding as B
    dims, csw, k0 = (4, 4, 4, 4), 3.0, 0.12
    U = synth.su3_links(dims, 0.3, 1)
    ref = R.Ref(*dims, 4)
    ref.gauge_load(U, None, 1.0)
    ref.set_quark(k0, 0.0)
    ref.clover_build(csw, 0.0)
    d0 = ref.clover_packed(False)[:, :, 0] - 1.0 / (2 * k0)     # clover part of the entry [0][0] of every block
    kappa = 1.0 / (2.0 * (-d0.min() + 1e-9))                     # the most negative one is cancelled up to 1e-9
    ref.set_quark(kappa, 0.0)
    ref.clover_build(csw, 0.0)
    exp = ref.clover_packed(True)
    assert np.abs(ref.clover_packed(False)[:, :, 0]).min() < 2e-9
    g = B.Qxd(*dims, 4, precisions=(F64,))
    g.gauge_load(U, None, 1.0)
    g.set_quark(kappa, 0.0)
    g.clover_build(csw, 0.0)
    fast, pivoted = g.clover_stats()
    assert fast == 2 and pivoted == 2                             # both parities tried fast, both redone with pivoting
    got = to_np(g.clover_export(True))
    assert relerr(got, exp) < 1e-9                                # some blocks have condition number ~1e4 at this kappa
    # the ordinary case never takes the fallback
    g.set_quark(k0, 0.0)
    g.clover_build(csw, 0.0)
    assert g.clover_stats() == (4, 2)
    g.close()


@pytest.mark.parametrize("prec", [F64, F32, F16])
def test_apply_Dw(case, prec):
    """Row a4, element by element over the whole extended lattice."""
    psi = synth.gaussian_spinor(case.dims_ext, 3)
    exp = case.ref.apply_Dw(psi)
    got = to_np(case.gpu.apply_Dw(psi, prec)).reshape(exp.shape)
    assert relerr(got, exp) < TOL[prec]
    if prec == F64:
        assert np.max(np.abs(got - exp)) < 1e-12 * np.max(np.abs(exp))


@pytest.mark.parametrize("prec", [F64, F32, F16])
def test_apply_Dw_and_Dhat_reconstruct12(case, prec):
    """Rows a2/a4/a5 with the 14-real link format (rows 0, 1 + det W: 12-real reconstruct, U(1) phase and the
    antiperiodic sign carried by det W); switching the format rewrites the links and must not change any result."""
    B = case.B
    psi = synth.gaussian_spinor(case.dims_ext, 3)
    pe = synth.gaussian_spinor(case.dims_ext, 6).reshape(-1, 4, 3)[: case.V // 2]
    exp = case.ref.apply_Dw(psi)
    case.gpu.set_gauge_reconstruct(B.QXD_RECON_12)
    try:
        got = to_np(case.gpu.apply_Dw(psi, prec)).reshape(exp.shape)
        assert relerr(got, exp) < TOL[prec]
        for dagger in (False, True):
            e2 = case.ref.apply_Dhat(pe, dagger=dagger)
            g2 = to_np(case.gpu.apply_Dhat_eo(pe, prec, dagger=dagger)).reshape(e2.shape)
            assert relerr(g2, e2) < 2 * TOL[prec]
    finally:
        case.gpu.set_gauge_reconstruct(B.QXD_RECON_NONE)
    got = to_np(case.gpu.apply_Dw(psi, prec)).reshape(exp.shape)
    assert relerr(got, exp) < TOL[prec]


def test_reconstruct12_solve_and_bad_value(case):
    B = case.B
    eta = synth.gaussian_spinor(case.dims_ext, 4)
    case.gpu.set_gauge_reconstruct(B.QXD_RECON_12)
    try:
        psi, info = case.gpu.solve(eta, 1e-10, algo=B.QXD_CGNE, sloppy=F32)
        assert info["status"] == 0
        res = relerr(case.ref.apply_Dw(to_np(psi).reshape(eta.shape)), eta)
        assert res <= 1.05e-10
        with pytest.raises(B.QxdError):
            case.gpu.set_gauge_reconstruct(8)
        # per-precision format: fp16 back to 18 reals while fp64 / fp32 stay reconstructed; mixed fp64/fp16 solve
        case.gpu.set_gauge_reconstruct(B.QXD_RECON_NONE, prec=F16)
        psi, info = case.gpu.solve(eta, 1e-10, algo=B.QXD_CGNE, sloppy=F16)
        assert info["status"] == 0
        assert relerr(case.ref.apply_Dw(to_np(psi).reshape(eta.shape)), eta) <= 1.05e-10
    finally:
        case.gpu.set_gauge_reconstruct(B.QXD_RECON_NONE)


@pytest.mark.parametrize("prec", [F64, F32, F16])
@pytest.mark.parametrize("dagger", [False, True])
def test_apply_Dhat(case, prec, dagger):
    """Row a5: both fused passes of the even-odd operator and its adjoint."""
    pe = synth.gaussian_spinor(case.dims_ext, 6).reshape(-1, 4, 3)[: case.V // 2]
    exp = case.ref.apply_Dhat(pe, dagger=dagger)
    got = to_np(case.gpu.apply_Dhat_eo(pe, prec, dagger=dagger)).reshape(exp.shape)
    assert relerr(got, exp) < 2 * TOL[prec]


def test_pack_unpack_bit_exact(case):
    """Row a9: natural -> packed -> natural is the identity in fp64 (index work is bit-exact)."""
    psi = synth.gaussian_spinor(case.dims_ext, 7)
    p = case.gpu.spinor_pack(psi, F64)
    back = to_np(case.gpu.spinor_unpack(p, F64))
    assert np.array_equal(back.view(np.float64), psi.view(np.float64))
    # fp32 storage rounds each real once
    p = case.gpu.spinor_pack(psi, F32)
    back = to_np(case.gpu.spinor_unpack(p, F32))
    assert np.array_equal(back.view(np.float64), psi.view(np.float64).astype(np.float32).astype(np.float64))


def test_packed_apply_equals_natural_apply(case):
    psi = synth.gaussian_spinor(case.dims_ext, 3)
    g = case.gpu
    pin = g.spinor_pack(psi, F64)
    pout = g.new_packed(F64)
    g.apply_Dw_packed(pin, pout, F64)
    a = to_np(g.spinor_unpack(pout, F64))
    b = to_np(g.apply_Dw(psi, F64)).reshape(a.shape)
    assert np.array_equal(a, b)


@pytest.mark.parametrize("prec", [F64, F32, F16])
def test_blas(case, prec):
    """Row a6: axpy, complex dot, norm^2 on packed half-lattice spinors against numpy in fp64."""
    g = case.gpu
    x = synth.gaussian_spinor(case.dims_ext, 8)
    y = synth.gaussian_spinor(case.dims_ext, 9)
    px, py = g.spinor_pack(x, prec), g.spinor_pack(y, prec)
    # what the device actually holds (after storage rounding), even half first
    xs = to_np(g.spinor_unpack(px, prec)).reshape(-1, 12)
    ys = to_np(g.spinor_unpack(py, prec)).reshape(-1, 12)
    lat_par = np.indices(case.dims_ext).sum(axis=0).ravel() & 1
    xe, ye = xs[lat_par == 0], ys[lat_par == 0]
    hb = g.packed_spinor_bytes(prec, half_only=True)
    n2 = g.blas_norm2(px[:hb], prec)
    assert abs(n2 - np.vdot(xe, xe).real) / n2 < 1e-13
    d = g.blas_cdot(px[:hb], py[:hb], prec)
    expd = np.vdot(xe, ye)
    assert abs(d - expd) / abs(expd) < 1e-12
    g.blas_axpy(0.37, px[:hb], py[:hb], prec)
    got = to_np(g.spinor_unpack(py, prec)).reshape(-1, 12)[lat_par == 0]
    assert relerr(got, ye + 0.37 * xe) < {F64: 1e-15, F32: 2e-7, F16: 1e-3}[prec]


def test_dw_sweep_kernel_is_bit_identical():
    """The time-sweep D_w kernel (qxd_set_dw_sweep; fp32, 18-real links, extended layout) does the arithmetic of the tile kernel
    in the same order: bit-identical output for several segment lengths, with C* boundaries and a ragged last segment."""
    import torch
    for dims, cstar in (((16, 8, 8, 8), 0), ((12, 4, 8, 8), 3)):
        c = Case(dims, cstar, 1, cstar > 0, precisions=(F64, F32), pairing=False)
        psi = synth.gaussian_spinor(c.dims_ext, 3)
        pin = c.gpu.spinor_pack(psi, F32)
        ref = c.gpu.new_packed(F32)
        c.gpu.apply_Dw_packed(pin, ref, F32)
        for tseg in (2, 4, 8, 5):
            c.gpu.set_dw_sweep(tseg)
            out = c.gpu.new_packed(F32)
            c.gpu.apply_Dw_packed(pin, out, F32)
            assert torch.equal(out, ref), (dims, cstar, tseg)
        c.gpu.set_dw_sweep(0)
        assert relerr(to_np(c.gpu.spinor_unpack(ref, F32)).reshape(psi.shape), c.ref.apply_Dw(psi)) < TOL[F32]
        c.close()


def test_tiling_does_not_change_results():
    """Row a1: the tile shape only permutes sites in memory; results are identical for any legal tile."""
    dims = (4, 4, 4, 8)
    outs = []
    psi = synth.gaussian_spinor((4, 8, 4, 8), 3)
    for tile in [(1, 1, 1, 2), (2, 2, 2, 2), (4, 8, 4, 8), (1, 2, 4, 8), None]:
        c = Case(dims, 3, 1, True, precisions=(F64,), tile=tile, oracle_clover=False)
        outs.append(to_np(c.gpu.apply_Dw(psi, F64)))
        c.close()
    for o in outs[1:]:
        assert np.array_equal(o, outs[0])


# ---- solves ------------------------------------------------------------------------------------------------
def true_residual(ref, eta, psi):
    return np.linalg.norm(np.ravel(eta) - np.ravel(ref.apply_Dw(psi))) / np.linalg.norm(np.ravel(eta))


@pytest.mark.parametrize("name,q", [("c0", 0.0), ("c1", 2 / 3), ("c1", -1 / 3)])
@pytest.mark.parametrize("algo", [0, 1])
def test_solve_fp64_configs_c0_c1(name, q, algo):
    """BASELINE configs 0 and 1: fp64 even-odd CGNE / BiCGstab to 1e-12, residual checked with the oracle's D."""
    cfg = synth.config(name)
    c = Case(cfg["dims"], cfg["cstar"], cfg["antiperiodic"], cfg["qed"], q=q, kappa=cfg["kappa"], csw=cfg["csw"],
             csw_qed=cfg["csw_qed"], qel=cfg["qel"], eps=cfg["eps"], precisions=(F64,))
    eta = synth.gaussian_spinor(c.dims_ext, 3)
    psi, info = c.gpu.solve(eta, cfg["tol"], algo=algo, sloppy=F64)
    assert info["status"] == 0, info
    psi = to_np(psi).reshape(eta.shape)
    assert true_residual(c.ref, eta, psi) <= cfg["tol"] * 1.05
    assert abs(info["true_res"] - true_residual(c.ref, eta, psi)) < 0.2 * cfg["tol"]
    # the solution is unique: compare with the oracle's own solve
    ps_ref, iref = c.ref.solve(eta, cfg["tol"])
    assert iref["status"] == 0
    assert relerr(psi, ps_ref) < 1e-10
    if algo == 0:
        assert abs(info["iters"] - iref["iters"]) <= 3
    c.close()


@pytest.mark.parametrize("sloppy,algo", [(F32, 0), (F16, 0), (F32, 1), (F16, 1)])
def test_solve_mixed_precision_reliable_updates(sloppy, algo):
    """Row a7: sloppy inner iteration + fp64 reliable updates reaches the fp64 residual target."""
    dims = (8, 4, 4, 8)
    c = Case(dims, 3, 1, True, q=-1 / 3, kappa=0.125, csw=1.5, csw_qed=1.0, eps=0.2)
    eta = synth.gaussian_spinor(c.dims_ext, 5)
    psi, info = c.gpu.solve(eta, 1e-10, algo=algo, sloppy=sloppy, delta=0.1)
    assert info["status"] == 0, info
    assert info["n_reliable"] >= 2
    assert true_residual(c.ref, eta, to_np(psi).reshape(eta.shape)) <= 1.05e-10
    c.close()


def test_solve_host_pointers_and_zero_source():
    import torch
    c = Case((4, 4, 4, 4), 0, 1, False, precisions=(F64,))
    eta = synth.gaussian_spinor(c.dims_ext, 3)
    eh = torch.from_numpy(eta.copy()).pin_memory()
    ph = torch.empty_like(eh).pin_memory()
    _, info = c.gpu.solve_host(eh, ph, 1e-12)
    assert info["status"] == 0
    assert true_residual(c.ref, eta, ph.numpy()) <= 1.05e-12
    # D_w through host pointers
    oh = torch.empty_like(eh).pin_memory()
    c.gpu.apply_Dw_host(eh, oh, F64)
    assert relerr(oh.numpy(), c.ref.apply_Dw(eta)) < 1e-13
    # eta = 0 -> psi = 0, zero iterations
    z = torch.zeros_like(eh)
    _, info = c.gpu.solve_host(z, ph, 1e-12)
    assert info["status"] == 0 and info["iters"] == 0
    assert float(ph.abs().max()) == 0.0
    c.close()


@pytest.mark.parametrize("algo", [0, 1])
def test_maxiter_reports_noconv_with_best_iterate(algo):
    c = Case((4, 4, 4, 4), 0, 1, False, precisions=(F64,))
    eta = synth.gaussian_spinor(c.dims_ext, 3)
    psi, info = c.gpu.solve(eta, 1e-12, algo=algo, maxiter=3)
    assert info["status"] == c.B.QXD_ENOCONV and info["iters"] == 3
    res = true_residual(c.ref, eta, to_np(psi).reshape(eta.shape))
    assert 1e-12 < res <= 1.0          # never worse than the zero vector (BiCGstab returns its best iterate)
    assert abs(info["true_res"] - res) < 1e-10
    c.close()


def test_bicgstab_supercritical_returns_best_iterate():
    """Beyond the critical kappa BiCGstab on D-hat stalls or diverges: the call must end with QXD_ENOCONV (stagnation guard or
    maxiter), and the psi it returns must be the iterate with the smallest true residual it saw, reported truthfully."""
    c = Case((8, 4, 4, 4), 0, 1, False, kappa=0.20, csw=1.7, eps=0.3, precisions=(F64, F32))
    eta = synth.gaussian_spinor(c.dims_ext, 3)
    psi, info = c.gpu.solve(eta, 1e-10, algo=1, sloppy=F32, maxiter=1500)
    res = true_residual(c.ref, eta, to_np(psi).reshape(eta.shape))
    assert abs(info["true_res"] - res) <= 1e-9 * max(1.0, res)
    if info["status"] != 0:
        assert info["status"] == c.B.QXD_ENOCONV and res <= 1.0 + 1e-12
    c.close()


def test_error_codes():
    import torch
    from paper_2502_02490_b200 import binding as B
    with pytest.raises(B.QxdError):
        B.Qxd(4, 3, 4, 4, 0)           # odd extent
    g = B.Qxd(4, 4, 4, 4, 4, precisions=(F64,))
    psi = torch.zeros(g.V * 12, dtype=torch.complex128, device="cuda")
    with pytest.raises(B.QxdError) as e:
        g.apply_Dw(psi)                 # no gauge / clover yet
    assert e.value.status == B.QXD_ESTATE
    g.gauge_load(synth.su3_links((4, 4, 4, 4), 0.3, 1))
    with pytest.raises(B.QxdError) as e:
        g.clover_build(1.5)             # no quark yet
    assert e.value.status == B.QXD_ESTATE
    g.set_quark(0.12)
    g.clover_build(1.5)
    with pytest.raises(B.QxdError) as e:
        g.apply_Dw(psi, F32)            # precision not bound
    assert e.value.status == B.QXD_EINVAL
    g.close()


# ---- full-size checks (the configuration bench.py times) ---------------------------------------------------
# BASELINE config 3 (64x32^3, C*, QCD+QED; 4 194 304 extended sites) in BOTH device layouts -- the extended lattice the
# headline D_w line is quoted on and the C*-paired layout every benched solve runs on -- compared with the oracle over the
# WHOLE lattice (the oracle applies D_w to the full c3 field in about a second; its clover field is built once per module).
class _Shared:
    pass


@pytest.fixture(scope="module")
def c3_oracle():
    cfg = synth.config("c3")
    o = _Shared()
    o.cfg = cfg
    o.U = synth.su3_links(cfg["dims"], cfg["eps"], 1)
    o.A = synth.u1_field(cfg["dims"], 0.3, 2)
    o.ref = R.Ref(*cfg["dims"], cfg["bc"])
    o.ref.gauge_load(o.U, o.A, cfg["qel"])
    o.ref.set_quark(cfg["kappa"], cfg["q"])
    o.ref.clover_build(cfg["csw"], cfg["csw_qed"])
    o.psi = synth.gaussian_spinor(o.ref.dims_ext, 3)
    o.Dw = o.ref.apply_Dw(o.psi)
    o.pe = synth.gaussian_spinor(o.ref.dims_ext, 6).reshape(-1, 4, 3)[: o.ref.V // 2]
    o.Dhat = {False: o.ref.apply_Dhat(o.pe), True: o.ref.apply_Dhat(o.pe, dagger=True)}
    yield o


@pytest.fixture(scope="module", params=[False, True], ids=["extended", "paired"])
def full_c3_case(request, c3_oracle):
    cfg = c3_oracle.cfg
    c = Case(cfg["dims"], cfg["cstar"], cfg["antiperiodic"], cfg["qed"], q=cfg["q"], kappa=cfg["kappa"], csw=cfg["csw"],
             csw_qed=cfg["csw_qed"], qel=cfg["qel"], eps=cfg["eps"], precisions=(F64, F32, F16), pairing=request.param, share=c3_oracle,
             gcr=(16, 4, 5), deflation=(16, 8, 12, 0, 1))
    c.o = c3_oracle
    c.psi = c3_oracle.psi
    yield c
    c.close()


@pytest.mark.parametrize("recon", [18, 14])
@pytest.mark.parametrize("prec", [F64, F32, F16])
def test_full_c3_Dw_whole_lattice(full_c3_case, prec, recon):
    """Row a4 at full size in bench.py's launch configuration, both link formats: relative L2 over all 4.19 M sites."""
    c = full_c3_case
    c.gpu.set_gauge_reconstruct(c.B.QXD_RECON_12 if recon == 14 else c.B.QXD_RECON_NONE)
    try:
        got = to_np(c.gpu.apply_Dw(c.psi, prec)).reshape(c.o.Dw.shape)
    finally:
        c.gpu.set_gauge_reconstruct(c.B.QXD_RECON_NONE)
    assert relerr(got, c.o.Dw) < TOL[prec]
    if prec == F64:
        assert np.max(np.abs(got - c.o.Dw)) < 1e-12 * np.max(np.abs(c.o.Dw))


@pytest.mark.parametrize("recon", [18, 14])
@pytest.mark.parametrize("dagger", [False, True])
@pytest.mark.parametrize("prec", [F64, F32, F16])
def test_full_c3_Dhat_whole_lattice(full_c3_case, prec, dagger, recon):
    """Row a5 at full size: both fused passes of D-hat and D-hat^dagger over the whole even sublattice."""
    c = full_c3_case
    c.gpu.set_gauge_reconstruct(c.B.QXD_RECON_12 if recon == 14 else c.B.QXD_RECON_NONE)
    try:
        got = to_np(c.gpu.apply_Dhat_eo(c.o.pe, prec, dagger=dagger)).reshape(c.o.pe.shape)
    finally:
        c.gpu.set_gauge_reconstruct(c.B.QXD_RECON_NONE)
    assert relerr(got, c.o.Dhat[dagger]) < 2 * TOL[prec]


def test_full_c3_gamma5_hermiticity_property(full_c3_case):
    """Property that holds at any size: <phi, D psi> = <g5 D g5 phi, psi> on the full 64x64x32x32 lattice."""
    c = full_c3_case
    phi = synth.gaussian_spinor(c.dims_ext, 4)
    g5 = np.array([1, 1, -1, -1])[:, None]
    lhs = np.vdot(phi, to_np(c.gpu.apply_Dw(c.psi, F64)).reshape(phi.shape))
    rhs = np.vdot(g5 * to_np(c.gpu.apply_Dw(g5 * phi, F64)).reshape(phi.shape), c.psi)
    assert abs(lhs - rhs) / abs(lhs) < 1e-12


@pytest.mark.parametrize("algo,sloppy", [(0, F16), (0, F32), (1, F32), (1, F16), (2, F16), (2, F32)],
                         ids=["cgne_fp16", "cgne_fp32", "bicgstab_fp32", "bicgstab_fp16", "gcr_sap_fp16", "gcr_sap_fp32"])
def test_full_c3_benched_solves_whole_lattice_residual(full_c3_case, algo, sloppy):
    """The solves bench.py times (link formats as there: 14 reals in fp64 / fp32, 18 in fp16), on both layouts:
    ||eta - D_ref psi|| / ||eta|| <= 1e-10 with the ORACLE's D_w over the whole lattice."""
    c = full_c3_case
    B = c.B
    c.gpu.set_gauge_reconstruct(B.QXD_RECON_12)
    c.gpu.set_gauge_reconstruct(B.QXD_RECON_NONE, prec=F16)
    try:
        psi, info = c.gpu.solve(c.psi, 1e-10, algo=algo, sloppy=sloppy, delta=0.1, maxiter=5000)
    finally:
        c.gpu.set_gauge_reconstruct(B.QXD_RECON_NONE)
    assert info["status"] == 0 and info["true_res"] <= 1e-10, info
    res = true_residual(c.o.ref, c.psi, to_np(psi).reshape(c.psi.shape))
    assert res <= 1.05e-10, (res, info)
    assert abs(res - info["true_res"]) <= 0.1 * res       # the library's own fp64 residual is the oracle's


def test_full_c3_deflated_solve_whole_lattice_residual(full_c3_case):
    """The deflated SAP-GCR solve bench.py times (16 null vectors split by chirality, binary16 block operator), on both layouts:
    ||eta - D_ref psi|| / ||eta|| <= 1e-10 with the ORACLE's D_w over the whole lattice, in fewer steps than the plain SAP-GCR."""
    import torch
    c = full_c3_case
    B = c.B
    g = c.gpu
    g.set_gauge_reconstruct(B.QXD_RECON_12)
    g.set_gauge_reconstruct(B.QXD_RECON_NONE, prec=F16)
    try:
        gen = torch.Generator(device="cuda")
        gen.manual_seed(1234)
        nb = g.packed_spinor_bytes(F32)
        rnd = torch.randn(16 * nb // 4, dtype=torch.float32, device="cuda", generator=gen)     # any independent set will do
        g.deflation_setup(rnd.view(torch.uint8), F16)
        del rnd
        nblocks, ncoarse, ready = g.deflation_info()
        assert ready and ncoarse == 32 and nblocks == c.V // 256
        psi, info = g.solve(c.psi, 1e-10, algo=B.QXD_DFL_GCR, sloppy=F16, maxiter=500)
        _, plain = g.solve(c.psi, 1e-10, algo=B.QXD_GCR, sloppy=F16, maxiter=500)
    finally:
        g.set_gauge_reconstruct(B.QXD_RECON_NONE)
    assert info["status"] == 0 and info["true_res"] <= 1e-10, info
    res = true_residual(c.o.ref, c.psi, to_np(psi).reshape(c.psi.shape))
    assert res <= 1.05e-10, (res, info)
    assert info["iters"] < 0.8 * plain["iters"], (info, plain)


@pytest.mark.parametrize("prec", [F32, F16])
def test_full_c3_multi_rhs_whole_lattice(full_c3_case, prec):
    """Row a10 at full size: three right-hand sides in one batched launch, each compared with the oracle on every site."""
    import torch
    c = full_c3_case
    g = c.gpu
    if not hasattr(c.o, "multi"):
        etas = [synth.gaussian_spinor(c.dims_ext, 31), synth.gaussian_spinor(c.dims_ext, 32)]
        c.o.multi = [(c.psi, c.o.Dw)] + [(e, c.o.ref.apply_Dw(e)) for e in etas]
    nb = g.packed_spinor_bytes(prec)
    pin = torch.empty(3 * nb, dtype=torch.uint8, device="cuda")
    pout = torch.zeros_like(pin)
    for k in range(3):
        g.spinor_pack(c.o.multi[k][0], prec, packed=pin[k * nb:(k + 1) * nb])
    g.apply_Dw_multi_packed(pin, pout, prec, 3)
    for k in range(3):
        got = to_np(g.spinor_unpack(pout[k * nb:(k + 1) * nb], prec)).reshape(c.o.Dw.shape)
        assert relerr(got, c.o.multi[k][1]) < TOL[prec], k


@pytest.mark.parametrize("dims,cstar,pairing", [((12, 4, 4, 4), 0, False), ((16, 2, 4, 4), 1, False), ((16, 4, 4, 8), 3, False),
                                                ((8, 4, 4, 4), 0, False), ((16, 4, 4, 8), 3, True), ((12, 4, 4, 4), 1, True)])
@pytest.mark.parametrize("prec", [F64, F32])
def test_apply_Dw_host_pipelined_equals_device_apply(dims, cstar, pairing, prec):
    """qxd_apply_Dw_host cuts the lattice into time slabs and overlaps host<->device copies with pack / apply / unpack
    (3, 4 and 4 slabs here; the 8x4^3 case has only two and takes the unpipelined path).  Same kernels on the same
    data: the result must equal the device-pointer apply bit for bit, and the oracle within tolerance."""
    import torch
    c = Case(dims, cstar, 1, cstar > 0, precisions=(F64, F32), pairing=pairing)
    psi = synth.gaussian_spinor(c.dims_ext, 12)
    dev = to_np(c.gpu.apply_Dw(psi, prec))
    eh = torch.from_numpy(psi).pin_memory()
    oh = torch.empty_like(eh).pin_memory()
    for _ in range(2):   # twice: the second call reuses streams and events
        oh.zero_()
        c.gpu.apply_Dw_host(eh, oh, prec)
        assert np.array_equal(oh.numpy().reshape(dev.shape), dev)
    assert relerr(oh.numpy().reshape(psi.shape), c.ref.apply_Dw(psi)) < TOL[prec]
    c.close()


@pytest.mark.parametrize("sloppy", [F32, F16])
def test_solve_config_c2_full_size(sloppy):
    """BASELINE config 2 at its full size (32x16^3 QCD+QED C*, 262144 extended sites, eps 0.15, csw 1.7): mixed-precision
    even-odd CG with reliable updates to 1e-10; the true residual is recomputed with the oracle's D on the whole lattice."""
    cfg = synth.config("c2")
    c = Case(cfg["dims"], cfg["cstar"], cfg["antiperiodic"], cfg["qed"], q=cfg["q"], kappa=cfg["kappa"], csw=cfg["csw"],
             csw_qed=cfg["csw_qed"], qel=cfg["qel"], eps=cfg["eps"], precisions=(F64, F32, F16))
    eta = synth.gaussian_spinor(c.dims_ext, 3)
    psi, info = c.gpu.solve(eta, cfg["tol"], algo=0, sloppy=sloppy, delta=0.1)
    assert info["status"] == 0 and info["n_reliable"] >= 1, info
    assert true_residual(c.ref, eta, to_np(psi).reshape(eta.shape)) <= 1.05 * cfg["tol"]
    c.close()


def _random_geometries(n, seed):
    rng = np.random.default_rng(seed)
    out = []
    while len(out) < n:
        dims = tuple(int(2 * rng.integers(1, 5)) for _ in range(4))          # even extents 2..8
        cstar = int(rng.integers(0, 4))
        if np.prod(dims) * (2 if cstar else 1) > 6000:
            continue
        ap = int(rng.integers(0, 2))
        qed = bool(rng.integers(0, 2)) or cstar > 0
        pairing = bool(cstar > 0 and rng.integers(0, 2))
        out.append((dims, cstar, ap, qed, pairing))
    return out


@pytest.mark.parametrize("dims,cstar,ap,qed,pairing", _random_geometries(16, 2024),
                         ids=lambda v: "x".join(map(str, v)) if isinstance(v, tuple) else str(int(v)))
def test_random_geometries_fp64_operator_and_solve(dims, cstar, ap, qed, pairing):
    """Seeded random small geometries (even extents 2..8, every cstar, both time boundary conditions, both device layouts,
    both link formats): fp64 D_w and D-hat element by element against the oracle, and an fp64/fp32 solve to 1e-10."""
    c = Case(dims, cstar, ap, qed, q=-1 / 3, precisions=(F64, F32), pairing=pairing)
    psi = synth.gaussian_spinor(c.dims_ext, 3)
    exp = c.ref.apply_Dw(psi)
    pe = synth.gaussian_spinor(c.dims_ext, 6).reshape(-1, 4, 3)[: c.V // 2]
    for recon in (c.B.QXD_RECON_NONE, c.B.QXD_RECON_12):
        c.gpu.set_gauge_reconstruct(recon)
        assert relerr(to_np(c.gpu.apply_Dw(psi, F64)).reshape(exp.shape), exp) < 1e-13
        assert relerr(to_np(c.gpu.apply_Dhat_eo(pe, F64)).reshape(pe.shape), c.ref.apply_Dhat(pe)) < 2e-13
        assert relerr(to_np(c.gpu.apply_Dw(psi, F32)).reshape(exp.shape), exp) < 1e-6
    sol, info = c.gpu.solve(psi, 1e-10, algo=0, sloppy=F32)
    assert info["status"] == 0
    assert true_residual(c.ref, psi, to_np(sol).reshape(psi.shape)) <= 1.05e-10
    c.close()
