"""Pins of the fp64 CPU oracle against what the paper and the mathematics fix (CPU only).

The paper prints no worked operator values, so the oracle is pinned by closed
forms, invariants and brute force (BASELINE.json north_star):
free-field momentum-space closed form (apply and solve), gamma5-hermiticity, SU(3)xU(1) gauge
covariance, C* charge-conjugation symmetry, csw=0 -> Wilson, uniform abelian background,
SU(3)-formula-on-U(3)-links -> q*A-hat, PAPER.md:117 packing, and dense LU brute force.
"""
import numpy as np
import pytest

import synth
from synth.fields import FIELD_U1_TRAFO
from oracle import qxd_ref as R
import lattice_np as LN


def make_ref(dims, cstar, ap, U=None, A=None, kappa=0.12, q=0.0, csw=1.5, csw_qed=0.0, qel=1.0, eps=0.3):
    r = R.Ref(*dims, cstar | (ap << 2))
    if U is None:
        U = synth.su3_links(dims, eps, 1)
    r.gauge_load(U, A, qel)
    r.set_quark(kappa, q)
    r.clover_build(csw, csw_qed)
    return r, U


def relerr(a, b):
    return np.linalg.norm(np.ravel(a) - np.ravel(b)) / np.linalg.norm(np.ravel(b))


# ------------------------------------------------------------------------------------------
# Free field: U=1, A=0 => for psi(x) = exp(ipx) u:  D psi = [m0 + sum(1-cos p) + i sum gamma sin p] psi
# with the allowed momenta of SURVEY.md §8(c7): p0=(2n0+1)pi/T (antiperiodic) or 2 pi n0/T,
# p1 = 2 pi n1/(2 L1) [C*] , p_k = (2 pi n_k + pi (n1 mod 2) [k<=cstar]) / L_k.
# ------------------------------------------------------------------------------------------
def free_momentum(dims, cstar, ap, n):
    T, L1, L2, L3 = dims
    X1 = 2 * L1 if cstar else L1
    p = np.zeros(4)
    p[0] = (2 * n[0] + 1) * np.pi / T if ap else 2 * np.pi * n[0] / T
    p[1] = 2 * np.pi * n[1] / X1
    for k, L in ((2, L2), (3, L3)):
        tw = np.pi * (n[1] % 2) if (cstar and k <= cstar) else 0.0
        p[k] = (2 * np.pi * n[k] + tw) / L
    return p


@pytest.mark.parametrize("cstar", [0, 1, 2, 3])
@pytest.mark.parametrize("ap", [0, 1])
def test_free_field_closed_form_apply_and_solve(cstar, ap):
    dims = (6, 4, 4, 6)
    kappa, csw = 0.11, 1.3
    m0 = 1 / (2 * kappa) - 4
    U = np.zeros(dims + (4, 3, 3), dtype=complex)
    U[...] = np.eye(3)
    A = np.zeros(dims + (4,)) if cstar else None
    r, _ = make_ref(dims, cstar, ap, U=U, A=A, kappa=kappa, q=2 / 3, csw=csw, csw_qed=1.0 if cstar else 0.0)
    lat = LN.Lattice(*dims, cstar=cstar, antiperiodic=ap)
    rng = np.random.default_rng(5)
    for n in ([0, 0, 0, 0], [1, 1, 2, 1], [2, 3, 1, 5], [5, 2, 3, 2], [1, 5, 0, 3]):
        p = free_momentum(dims, cstar, ap, n)
        u = rng.normal(size=(4, 3)) + 1j * rng.normal(size=(4, 3))
        phase = np.exp(1j * (lat.coords @ p))
        psi = phase[:, None, None] * u
        Dp = (m0 + np.sum(1 - np.cos(p))) * np.eye(4) + 1j * sum(LN.GAMMA[mu] * np.sin(p[mu]) for mu in range(4))
        expect = phase[:, None, None] * (Dp @ u)
        got = r.apply_Dw(psi).reshape(lat.V, 4, 3)
        assert relerr(got, expect) < 1e-13, (cstar, ap, n)
        # closed-form inverse: [M(p) - i gamma.sin p] / [M(p)^2 + sum sin^2 p]
        Mp = m0 + np.sum(1 - np.cos(p))
        Dinv = (Mp * np.eye(4) - 1j * sum(LN.GAMMA[mu] * np.sin(p[mu]) for mu in range(4))) / (Mp**2 + np.sum(np.sin(p) ** 2))
        sol, info = r.solve(psi, 1e-13)
        assert info["status"] == 0
        assert relerr(sol.reshape(lat.V, 4, 3), phase[:, None, None] * (Dinv @ u)) < 1e-11


CASES = [
    # dims (physical), cstar, antiperiodic, qed
    ((4, 4, 4, 4), 0, 1, False),
    ((4, 4, 4, 4), 0, 0, True),
    ((4, 2, 4, 4), 1, 1, True),
    ((4, 4, 2, 4), 2, 1, True),
    ((6, 4, 4, 4), 3, 1, True),
    ((2, 2, 2, 2), 3, 1, True),
]


def setup_case(dims, cstar, ap, qed, q=2 / 3, kappa=0.12, csw=1.5, csw_qed=1.0, qel=1.0):
    U = synth.su3_links(dims, 0.3, 1)
    A = synth.u1_field(dims, 0.3, 2) if qed else None
    r, _ = make_ref(dims, cstar, ap, U=U, A=A, kappa=kappa, q=q if qed else 0.0, csw=csw, csw_qed=csw_qed if qed else 0.0, qel=qel)
    return r, U, A


@pytest.mark.parametrize("dims,cstar,ap,qed", CASES)
def test_gamma5_hermiticity(dims, cstar, ap, qed):
    r, U, A = setup_case(dims, cstar, ap, qed)
    psi = synth.gaussian_spinor(r.dims_ext, 3)
    phi = synth.gaussian_spinor(r.dims_ext, 4)
    g5 = np.array([1, 1, -1, -1])[:, None]
    lhs = np.vdot(phi, r.apply_Dw(psi))
    rhs = np.vdot(g5 * r.apply_Dw(g5 * phi), psi)
    assert abs(lhs - rhs) / abs(lhs) < 1e-13
    # D-hat on the even sublattice: <phi, Dhat psi> = <Dhat^dag phi, psi>
    pe = psi.reshape(-1, 4, 3)[: r.V // 2]
    fe = phi.reshape(-1, 4, 3)[: r.V // 2]
    lhs = np.vdot(fe, r.apply_Dhat(pe))
    rhs = np.vdot(r.apply_Dhat(fe, dagger=True), pe)
    assert abs(lhs - rhs) / abs(lhs) < 1e-13


@pytest.mark.parametrize("dims,cstar,ap,qed", CASES)
def test_gauge_covariance(dims, cstar, ap, qed):
    q, qel = -1 / 3, 0.7
    r, U, A = setup_case(dims, cstar, ap, qed, q=q, qel=qel)
    lat = LN.Lattice(*dims, cstar=cstar, antiperiodic=ap)
    Vp = int(np.prod(dims))
    Om = synth.random_su3(Vp, 11).reshape(dims + (3, 3))
    al = synth.u1_field(dims, 1.0, 12, field_id=FIELD_U1_TRAFO)[..., 0] if qed else np.zeros(dims)
    # extend Omega (mirror = conjugate) and alpha (mirror = -alpha) to the doubled lattice
    if cstar:
        Om_e = np.concatenate([Om, Om.conj()], axis=1).reshape(lat.V, 3, 3)
        al_e = np.concatenate([al, -al], axis=1).reshape(lat.V)
    else:
        Om_e, al_e = Om.reshape(lat.V, 3, 3), al.reshape(lat.V)
    Ue, Ae = lat.extend_gauge(U, A)
    Up = np.empty_like(Ue)
    Ap = None if Ae is None else np.empty_like(Ae)
    for mu in range(4):
        Om_f = lat.shift(Om_e, mu, 0)
        Up[:, mu] = LN.mm(LN.mm(Om_e, Ue[:, mu]), LN.dagm(Om_f))
        if Ae is not None:
            Ap[:, mu] = Ae[:, mu] + al_e - lat.shift(al_e, mu, 0)
    # the transformed field must again satisfy the mirror constraint; hand the physical half to the oracle
    X = lat.X
    Up4 = Up.reshape(X + (4, 3, 3))
    if cstar:
        assert np.abs(Up4[:, dims[1]:] - Up4[:, : dims[1]].conj()).max() < 1e-14
    Uphys = np.ascontiguousarray(Up4[:, : dims[1]])
    Aphys = None if Ap is None else np.ascontiguousarray(Ap.reshape(X + (4,))[:, : dims[1]])
    r2 = R.Ref(*dims, cstar | (ap << 2))
    r2.gauge_load(Uphys, Aphys, qel)
    r2.set_quark(0.12, q if qed else 0.0)
    r2.clover_build(1.5, 1.0 if qed else 0.0)
    psi = synth.gaussian_spinor(r.dims_ext, 3).reshape(lat.V, 4, 3)
    g = np.exp(1j * (q if qed else 0.0) * al_e)[:, None, None]
    psi_p = g * np.einsum("vab,vsb->vsa", Om_e, psi)
    lhs = r2.apply_Dw(psi_p).reshape(lat.V, 4, 3)
    rhs = g * np.einsum("vab,vsb->vsa", Om_e, r.apply_Dw(psi).reshape(lat.V, 4, 3))
    assert relerr(lhs, rhs) < 1e-13


@pytest.mark.parametrize("dims,cstar,ap,qed", [c for c in CASES if c[1] > 0])
def test_cstar_charge_conjugation_symmetry(dims, cstar, ap, qed):
    """(K psi)(x) = B psi(x + L1 1-hat)^*, B = gamma1 gamma3  =>  D K = K D; and M(x+L1) = B M(x)^* B^-1."""
    r, U, A = setup_case(dims, cstar, ap, qed)
    lat = LN.Lattice(*dims, cstar=cstar, antiperiodic=ap)
    B = LN.GAMMA[1] @ LN.GAMMA[3]
    for mu in range(4):
        assert np.abs(B @ LN.GAMMA[mu].conj() @ np.linalg.inv(B) - LN.GAMMA[mu]).max() < 1e-15
    X = lat.X

    def K(psi):
        p = psi.reshape(X + (4, 3))
        p = np.roll(p, -dims[1], axis=1)
        return np.einsum("ab,...bc->...ac", B, p.conj())

    psi = synth.gaussian_spinor(r.dims_ext, 3)
    assert relerr(r.apply_Dw(K(psi)), K(r.apply_Dw(psi))) < 1e-13
    B12 = np.kron(B, np.eye(3))
    for site in (0, 5, lat.V // 2 - 3):
        x = lat.coords[site].copy()
        x[1] = (x[1] + dims[1]) % X[1]
        mirror = np.ravel_multi_index(tuple(x), X)
        M, Mm = r.site_matrix(site), r.site_matrix(mirror)
        assert np.abs(Mm - B12 @ M.conj() @ np.linalg.inv(B12)).max() < 1e-13


def test_csw_zero_is_pure_wilson():
    dims = (4, 2, 4, 4)
    U = synth.su3_links(dims, 0.3, 1)
    A = synth.u1_field(dims, 0.3, 2)
    r, _ = make_ref(dims, 3, 1, U=U, A=A, kappa=0.125, q=2 / 3, csw=0.0, csw_qed=0.0)
    for s in (0, 7, 100):
        assert np.abs(r.site_matrix(s) - (4.0 + 1 / (2 * 0.125) - 4.0) * np.eye(12)).max() == 0.0
    # with csw != 0 the term is really there
    r.clover_build(1.5, 1.0)
    assert np.abs(r.site_matrix(7) - 4.0 * np.eye(12)).max() > 1e-2


def test_clover_blocks_hermitian_and_chirality_diagonal():
    r, U, A = setup_case((4, 4, 2, 4), 2, 1, True)
    off, ah = r.clover_diagnostics()
    assert off < 1e-15 and ah < 1e-14
    M = r.site_matrix(17)
    assert np.abs(M[:6, 6:]).max() == 0.0 and np.abs(M[6:, :6]).max() == 0.0
    assert np.abs(M - M.conj().T).max() < 1e-14


def test_clover_packing_paper_117():
    """First 6 reals = diagonal, then (re,im) of the strict upper triangle, row-major."""
    r, U, A = setup_case((4, 2, 4, 4), 3, 1, True)
    pk = r.clover_packed()
    pki = r.clover_packed(inverse=True)
    for site in (0, 33, r.V - 1):
        M = r.site_matrix(site)
        for c in range(2):
            blk = M[6 * c: 6 * c + 6, 6 * c: 6 * c + 6]
            inv = np.linalg.inv(blk)
            for mat, packed in ((blk, pk[site, c]), (inv, pki[site, c])):
                assert np.abs(packed[:6] - np.diag(mat).real).max() < 1e-13
                k = 6
                for i in range(6):
                    for j in range(i + 1, 6):
                        assert abs(packed[k] - mat[i, j].real) < 1e-13 and abs(packed[k + 1] - mat[i, j].imag) < 1e-13
                        k += 2
                assert k == 36


@pytest.mark.parametrize("mu,nu", [(0, 1), (0, 3), (1, 2), (2, 3), (1, 3)])
@pytest.mark.parametrize("qel", [1.0, 1 / 6])
def test_uniform_abelian_background_closed_form(mu, nu, qel):
    """A_nu(x) = Bf*x_mu  =>  Phi_{mu nu} = Bf on interior plaquettes, A-hat_{mu nu} = i sin(qel Bf)/qel, so
    M = (4+m0) - (q csw_qed/2) (sin(qel Bf)/qel) sigma_{mu nu} (x) 1  at a site whose leaves avoid the wrap."""
    dims = (6, 6, 6, 6)
    Bf, q, cq, kappa = 0.37, 2 / 3, 0.9, 0.12
    U = np.zeros(dims + (4, 3, 3), dtype=complex)
    U[...] = np.eye(3)
    A = np.zeros(dims + (4,))
    xm = np.arange(dims[mu]).reshape([-1 if d == mu else 1 for d in range(4)])
    A[..., nu] = Bf * xm
    r, _ = make_ref(dims, 0, 1, U=U, A=A, kappa=kappa, q=q, csw=1.0, csw_qed=cq, qel=qel)
    site = np.ravel_multi_index((2, 3, 2, 3), dims)
    expect = (1 / (2 * kappa)) * np.eye(12) - (q * cq / 2) * (np.sin(qel * Bf) / qel) * np.kron(LN.sigma_closed_form(mu, nu), np.eye(3))
    assert np.abs(r.site_matrix(site) - expect).max() < 1e-14


def test_su3_formula_on_u3_links_matches_qed_term_at_small_A():
    """F-hat[e^{iqA} 1] -> q A-hat (relative difference O(A^2)); fixes relative sign and normalisation of
    the two SW terms."""
    dims = (4, 4, 4, 4)
    q = 2 / 3
    errs = []
    for sigma in (0.03, 0.003):
        A = synth.u1_field(dims, sigma, 2)
        U3 = np.exp(1j * q * A)[..., None, None] * np.eye(3)
        U1 = np.zeros(dims + (4, 3, 3), dtype=complex)
        U1[...] = np.eye(3)
        ra, _ = make_ref(dims, 0, 1, U=U3, A=None, kappa=0.125, q=0.0, csw=1.0, csw_qed=0.0)
        rb, _ = make_ref(dims, 0, 1, U=U1, A=A, kappa=0.125, q=q, csw=0.0, csw_qed=1.0)
        da = ra.site_matrix(21) - 4 * np.eye(12)
        db = rb.site_matrix(21) - 4 * np.eye(12)
        errs.append(np.abs(da - db).max() / np.abs(db).max())
    assert errs[0] < 5e-3 and errs[1] < 5e-5 and errs[1] < errs[0] / 30


DENSE_CASES = [
    ((4, 4, 4, 4), 0, 1, False),
    ((4, 2, 4, 4), 3, 1, True),
    ((2, 2, 4, 2), 2, 0, True),
]


@pytest.mark.parametrize("dims,cstar,ap,qed", DENSE_CASES)
def test_dense_brute_force(dims, cstar, ap, qed):
    """Explicit matrix assembled entry by entry (tests/lattice_np.py), mat-vec, LU solve, Schur complement."""
    q, kappa, csw, cq, qel = 2 / 3, 0.12, 1.5, 1.0, 1.0
    r, U, A = setup_case(dims, cstar, ap, qed, q=q, kappa=kappa, csw=csw, csw_qed=cq, qel=qel)
    lat = LN.Lattice(*dims, cstar=cstar, antiperiodic=ap)
    Ue, Ae = lat.extend_gauge(U, A)
    D = LN.dense_Dw(lat, Ue, Ae, kappa, q if qed else 0.0, csw, cq if qed else 0.0, qel)
    psi = synth.gaussian_spinor(r.dims_ext, 3)
    got = r.apply_Dw(psi).ravel()
    assert relerr(got, D @ psi.ravel()) < 1e-14
    # sampled-site entry point
    sites = np.array([0, 3, lat.V - 1, lat.V // 2])
    assert relerr(r.apply_Dw_sites(psi, sites).reshape(4, 12), (D @ psi.ravel()).reshape(lat.V, 12)[sites]) < 1e-14
    # solve vs LU
    eta = synth.gaussian_spinor(r.dims_ext, 4)
    x_lu = np.linalg.solve(D, eta.ravel())
    x, info = r.solve(eta, 1e-13)
    assert info["status"] == 0
    assert relerr(x.ravel(), x_lu) < 1e-11
    assert np.linalg.norm(D @ x.ravel() - eta.ravel()) / np.linalg.norm(eta) < 2e-13
    # Schur complement on the even sublattice (even sites in increasing Lambda order)
    ev = np.where(lat.parity == 0)[0]
    od = np.where(lat.parity == 1)[0]
    D4 = D.reshape(lat.V, 12, lat.V, 12)
    blk = lambda a, b: D4[a][:, :, b].reshape(12 * len(a), 12 * len(b))
    Dhat = blk(ev, ev) - blk(ev, od) @ np.linalg.solve(blk(od, od), blk(od, ev))
    pe = synth.gaussian_spinor(r.dims_ext, 6).reshape(-1, 12)[: lat.V // 2]
    assert relerr(r.apply_Dhat(pe).ravel(), Dhat @ pe.ravel()) < 1e-13
    assert relerr(r.apply_Dhat(pe, dagger=True).ravel(), Dhat.conj().T @ pe.ravel()) < 1e-13


def test_invalid_geometry_rejected():
    with pytest.raises(R.RefError):
        R.Ref(4, 3, 4, 4, 0)
    with pytest.raises(R.RefError):
        R.Ref(4, 4, 4, 0, 0)


def test_range_apply_equals_full_apply():
    """The bounded-sample entry points (bench.py cpu_baseline) reproduce the full apply on their site range."""
    r, U, A = setup_case((4, 2, 4, 4), 3, 1, True)
    psi = synth.gaussian_spinor(r.dims_ext, 3)
    full = r.apply_Dw(psi).reshape(-1, 4, 3)
    lo, hi = 37, 201
    r.clover_build_range(1.5, 1.0, lo, hi)
    assert np.array_equal(r.apply_Dw_range(psi), full[lo:hi])


def test_reconstruct_identity_for_u3_links():
    """Reading R19: for every unitary W (here W = e^{i theta} U with U in SU(3), optionally times -1 for the
    antiperiodic time boundary) row 2 equals det W * conj(row 0 x row 1), and det W = e^{3 i theta} det U.  This is the
    identity the 14-real link format of the CUDA path relies on; checked here with numpy only."""
    U = synth.random_su3(64, 11)
    rng = np.random.default_rng(5)
    theta = rng.normal(0.0, 0.7, size=64)
    sign = np.where(rng.integers(0, 2, size=64) == 1, -1.0, 1.0)
    W = (sign * np.exp(1j * theta))[:, None, None] * U
    det = np.linalg.det(W)
    assert np.allclose(det, sign * np.exp(3j * theta) * np.linalg.det(U), atol=1e-13)
    assert np.allclose(np.linalg.det(U), 1.0, atol=1e-13)
    row2 = det[:, None] * np.conj(np.cross(W[:, 0, :], W[:, 1, :]))
    assert np.max(np.abs(row2 - W[:, 2, :])) < 1e-13


# ------------------------------------------------------------------------------------------
# Sign of the Sheikholeslami-Wohlert term, pinned by what "O(a)-improved" means (PAPER.md:3 title).
# Continuum: (gamma.D)^2 = D^2 + (1/2) sigma.F, so in a uniform magnetic field B the massless Dirac operator has exact zero
# modes (lowest Landau level: |B| from -D^2 cancels against sigma.F).  The Wilson term -(a/2) D^2 = -(a/2)[(gamma.D)^2 -
# (1/2) sigma.F] lifts them by (a/2)|B|; the SW term with the right sign and c_sw = 1 (tree level) puts them back up to
# O(a^2).  In lattice units (B = 2 pi k / L^2 on an L x L torus, m0 = 0) the lowest |eigenvalue| of gamma5 D_w must be
#     c_sw = +1:  O(B^2)  (falls like L^-4: ratio ~16 when L doubles)      c_sw = 0:  B/2        c_sw = -1:  B
# A flipped sign of the SW term in the oracle (reading R4: +c_sw (i/4) sigma.F-hat with F-hat = (Q - Q^dag)/8) would swap
# the first and the last line.  Nothing here restates the oracle's formula: the expected values are continuum Landau-level
# algebra.  Both SW terms are tested: the U(1) one (A-hat, csw_qed) and the SU(3) one on U(3) links e^{iA} 1.
# ------------------------------------------------------------------------------------------
def _lowest_landau_level(L, c, mode, k=1):
    """Lowest |eigenvalues| of gamma5 D_w (kappa = 1/8, i.e. m0 = 0) in the sector of zero momentum in directions 0 and 3,
    uniform flux 2 pi k through the (1,2) torus of size L x L; returns (sorted |eigenvalues|, B)."""
    dims = (2, L, L, 2)
    B = 2 * np.pi * k / L**2
    A = np.zeros(dims + (4,))
    x1 = np.arange(L).reshape(1, L, 1, 1)
    x2 = np.arange(L).reshape(1, 1, L, 1)
    A[..., 2] = B * x1                                   # A_2 = B x_1
    A[:, L - 1, :, :, 1] = (-B * L * x2)[:, 0]           # transition function on the last x_1 slice: every plaquette has angle B mod 2 pi
    one = np.zeros(dims + (4, 3, 3), dtype=complex)
    one[...] = np.eye(3)
    r = R.Ref(*dims, 0)                                  # periodic in all directions (zero-momentum sector exists)
    if mode == "u1":
        r.gauge_load(one, A, 1.0)
        r.set_quark(0.125, 1.0)
        r.clover_build(0.0, c)
    else:
        r.gauge_load(np.exp(1j * A)[..., None, None] * np.eye(3), None, 1.0)
        r.set_quark(0.125, 0.0)
        r.clover_build(c, 0.0)
    n = 12 * L * L
    M = np.zeros((n, n), dtype=complex)
    for j in range(n):                                   # the operator restricted to fields constant in x0, x3
        v = np.zeros((L * L, 12), dtype=complex)
        v[j // 12, j % 12] = 1.0
        psi = np.ascontiguousarray(np.broadcast_to(v.reshape(1, L, L, 1, 4, 3), dims + (4, 3)))
        out = r.apply_Dw(psi).reshape(2, L, L, 2, 12)
        assert np.abs(out - out[:1, :, :, :1]).max() < 1e-13
        M[:, j] = out[0, :, :, 0].reshape(-1)
    g5 = np.tile(np.repeat([1.0, 1.0, -1.0, -1.0], 3), L * L)
    ev = np.linalg.eigvalsh(g5[:, None] * M)
    return np.sort(np.abs(ev)), B


@pytest.mark.parametrize("mode", ["u1", "su3"])
def test_sw_term_sign_is_the_improving_one(mode):
    low = {}
    for L in (6, 12):
        for c in (1.0, 0.0, -1.0):
            ev, B = _lowest_landau_level(L, c, mode)
            low[L, c] = ev[0] / B
            assert ev[6] / B > 2.0                       # the six lowest-Landau-level modes are separated from the rest
    for L in (6, 12):
        assert abs(low[L, 0.0] - 0.5) < 0.02             # Wilson term alone: (a/2)|B|
        assert abs(low[L, -1.0] - 1.0) < 0.02            # wrong sign: doubled
        assert low[L, 1.0] < 0.02                        # c_sw = +1: the O(a) shift is gone
    # what is left at c_sw = +1 is O(a^2): lambda ~ B^2 ~ L^-4  (lambda/B ~ L^-2: ratio 4 when L doubles)
    assert 3.0 < low[6, 1.0] / low[12, 1.0] < 5.0
