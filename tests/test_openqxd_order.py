"""openQxD field orders (§2, §4.1): pins of the oracle (CPU) and bit-exact parity of
the CUDA reorder kernels against it (GPU).  Everything here is integer / copy work: the bar is bit-exact."""
import itertools

import numpy as np
import pytest

import synth
from oracle import openqxd_ref as O

CASES = [  # (extents, cache block)
    ((4, 4, 4, 4), (4, 4, 4, 4)),
    ((4, 4, 4, 4), (2, 2, 2, 2)),
    ((8, 4, 6, 4), (4, 2, 3, 2)),
    ((4, 8, 4, 6), (2, 4, 4, 2)),
    ((2, 2, 2, 2), (2, 2, 2, 2)),
]


@pytest.mark.parametrize("L,B", CASES)
def test_eq2_matches_the_prose_definition(L, B):
    """PAPER.md:95-97 in words: blocks lexicographic, points lexicographic inside a block, all even points first.
    Sorting the points by (parity, block index, in-block index) must give exactly the ranks of Eq. (2)."""
    pts = list(itertools.product(*(range(e) for e in L)))
    NB = [L[m] // B[m] for m in range(4)]

    def key(x):
        n = [x[m] // B[m] for m in range(4)]
        b = [x[m] % B[m] for m in range(4)]
        return (sum(x) % 2, O.lam(n, NB), O.lam(b, B))

    ranked = sorted(pts, key=key)
    for rank, x in enumerate(ranked):
        assert O.xhat(x, L, B) == rank


@pytest.mark.parametrize("L,B", CASES)
def test_eq2_is_a_bijection_with_even_points_first(L, B):
    V = int(np.prod(L))
    t = O.ipt(L, B)
    assert sorted(t.tolist()) == list(range(V))
    for x in itertools.product(*(range(e) for e in L)):
        assert (t[O.lam(x, L)] >= V // 2) == (sum(x) % 2 == 1)


def test_eq2_without_blocking_is_half_the_lexicographic_index():
    L = (4, 6, 2, 8)
    V = int(np.prod(L))
    for x in itertools.product(*(range(e) for e in L)):
        assert O.xhat(x, L, L) == O.lam(x, L) // 2 + (sum(x) % 2) * (V // 2)


def test_eq2_hand_table_2x2x2x2():
    """Worked by hand from Eq. (1), (2) for L = B = (2,2,2,2): Lambda = 8 x0 + 4 x1 + 2 x2 + x3."""
    L = (2, 2, 2, 2)
    want = {(0, 0, 0, 0): 0, (0, 0, 0, 1): 8, (0, 0, 1, 0): 9, (0, 0, 1, 1): 1, (0, 1, 0, 0): 10, (0, 1, 0, 1): 2,
            (0, 1, 1, 0): 3, (0, 1, 1, 1): 11, (1, 0, 0, 0): 12, (1, 0, 0, 1): 4, (1, 1, 1, 1): 7, (1, 1, 1, 0): 15}
    for x, v in want.items():
        assert O.xhat(x, L, L) == v


@pytest.mark.parametrize("dims,cstar", [((4, 4, 4, 4), 0), ((4, 2, 4, 4), 1), ((4, 4, 2, 4), 3), ((2, 2, 2, 2), 3)])
def test_gauge_order_round_trip_and_definition(dims, cstar):
    """8 links at odd points: every forward link of the physical lattice appears where reading R20 says,
    the mirror half is the complex conjugate, and to -> from is the identity."""
    X = O.ext_dims(dims, cstar)
    B = (2, 2, 2, 2)
    U = synth.su3_links(dims, 0.3, 1)
    ud = O.gauge_to_openqxd(U, dims, cstar, B)
    V = int(np.prod(X))
    assert ud.shape == (V // 2, 8, 3, 3)
    assert np.array_equal(O.gauge_from_openqxd(ud, dims, cstar, B), U)
    # definition, spot checks: an odd point and the even point behind it share one matrix
    for x in itertools.product(*(range(e) for e in X)):
        if sum(x) % 2 == 0:
            continue
        o = O.xhat(x, X, B) - V // 2
        for mu in range(4):
            y = O.shift(x, mu, -1, dims, cstar)
            assert sum(y) % 2 == 0
            w = U[y[0], y[1] % dims[1], y[2], y[3], mu]
            if y[1] >= dims[1]:
                w = np.conj(w)
            assert np.array_equal(ud[o, 2 * mu + 1], w)
    A = synth.u1_field(dims, 0.3, 2)
    ad = O.gauge_to_openqxd(A, dims, cstar, B, is_phase=True)
    assert np.array_equal(O.gauge_from_openqxd(ad, dims, cstar, B), A)


def test_site_record_round_trip():
    L, B = (4, 4, 6, 4), (2, 2, 3, 2)
    psi = synth.gaussian_spinor(L, 5).reshape(-1, 4, 3)
    oq = O.site_records_to_openqxd(psi, L, B)
    assert np.array_equal(O.site_records_from_openqxd(oq, L, B), psi)
    assert np.array_equal(oq[O.xhat((1, 2, 3, 1), L, B)], psi[O.lam((1, 2, 3, 1), L)])


# ---------------------------------------------------------------------------------------------------------------
# CUDA path against the oracle (bit-exact)
# ---------------------------------------------------------------------------------------------------------------
GPU_CASES = [((4, 4, 4, 4), 0, (2, 2, 2, 2)), ((8, 4, 6, 4), 0, (4, 2, 3, 2)), ((4, 2, 4, 4), 1, (2, 2, 2, 2)),
             ((6, 4, 4, 6), 3, (2, 4, 2, 2)), ((2, 2, 2, 2), 3, (2, 2, 2, 2)), ((8, 8, 8, 8), 3, (4, 4, 4, 4))]


@pytest.mark.gpu
@pytest.mark.parametrize("dims,cstar,blk", GPU_CASES)
def test_cuda_openqxd_orders_bit_exact(dims, cstar, blk):
    import torch
    from paper_2502_02490_b200 import binding as B
    g = B.Qxd(*dims, cstar | 4, precisions=(B.QXD_F64,))
    X = g.dims_ext
    V = g.V
    # index function
    xs = np.array(list(itertools.product(*(range(e) for e in X))), dtype=np.int32)
    got = g.openqxd_index(xs, blk)
    want = np.array([O.xhat(tuple(x), X, blk) for x in xs], dtype=np.int64)
    assert np.array_equal(got, want)
    # spinor and clover records, both directions
    for reals, seed in ((24, 7), (72, 8)):
        nat = synth.normal(seed, 9, np.arange(V * reals, dtype=np.uint64)).reshape(V, reals)
        oq = O.site_records_to_openqxd(nat, X, blk)
        got = g.openqxd_reorder(nat, reals, to_openqxd=True, block=blk).cpu().numpy()
        assert np.array_equal(got, oq)
        back = g.openqxd_reorder(oq, reals, to_openqxd=False, block=blk).cpu().numpy()
        assert np.array_equal(back, nat)
    # gauge field and U(1) field: 8 links at odd points <-> 4 forward links at every physical point
    U = synth.su3_links(dims, 0.3, 1)
    A = synth.u1_field(dims, 0.3, 2)
    ud = O.gauge_to_openqxd(U, dims, cstar, blk)
    ad = O.gauge_to_openqxd(A, dims, cstar, blk, is_phase=True)
    assert np.array_equal(g.openqxd_gauge(U, to_openqxd=True, block=blk).cpu().numpy().reshape(ud.shape), ud)
    assert np.array_equal(g.openqxd_gauge(ud, to_openqxd=False, block=blk).cpu().numpy().reshape(U.shape), U)
    assert np.array_equal(g.openqxd_gauge(A, to_openqxd=True, block=blk, phase=True).cpu().numpy().reshape(ad.shape), ad)
    assert np.array_equal(g.openqxd_gauge(ad, to_openqxd=False, block=blk, phase=True).cpu().numpy().reshape(A.shape), A)
    # bad block -> QXD_EINVAL
    with pytest.raises(B.QxdError):
        g.openqxd_reorder(np.zeros((V, 24)), 24, to_openqxd=True, block=(5, 2, 2, 2))
    g.close()


@pytest.mark.gpu
def test_cuda_solve_from_openqxd_fields():
    """Drop-in path of the paper's host code: gauge field, source and solution in openQxD order."""
    from paper_2502_02490_b200 import binding as B
    from oracle import qxd_ref as R
    dims, cstar, blk = (4, 4, 4, 4), 3, (2, 2, 2, 2)
    U = synth.su3_links(dims, 0.3, 1)
    A = synth.u1_field(dims, 0.3, 2)
    ud = O.gauge_to_openqxd(U, dims, cstar, blk)
    ad = O.gauge_to_openqxd(A, dims, cstar, blk, is_phase=True)
    g = B.Qxd(*dims, cstar | 4, precisions=(B.QXD_F64,))
    X = g.dims_ext
    g.gauge_load(g.openqxd_gauge(ud, to_openqxd=False, block=blk), g.openqxd_gauge(ad, to_openqxd=False, block=blk, phase=True), 1.0)
    g.set_quark(0.12, 2 / 3)
    g.clover_build(1.5, 1.0)
    eta = synth.gaussian_spinor(X, 3)
    eta_oq = O.site_records_to_openqxd(eta.reshape(-1, 24 // 2), X, blk)
    eta_nat = g.openqxd_reorder(eta_oq.view(np.float64).reshape(-1, 24), 24, to_openqxd=False, block=blk)
    psi_nat, info = g.solve(eta_nat.view(dtype=__import__("torch").complex128), 1e-12)
    assert info["status"] == 0
    psi_oq = g.openqxd_reorder(psi_nat.view(dtype=__import__("torch").float64).reshape(-1, 24), 24, to_openqxd=True, block=blk).cpu().numpy()
    psi = O.site_records_from_openqxd(psi_oq.view(np.complex128).reshape(-1, 12), X, blk).reshape(eta.shape)
    ref = R.Ref(*dims, cstar | 4)
    ref.gauge_load(U, A, 1.0)
    ref.set_quark(0.12, 2 / 3)
    ref.clover_build(1.5, 1.0)
    r = ref.apply_Dw(psi) - eta
    assert np.linalg.norm(r.ravel()) / np.linalg.norm(eta.ravel()) <= 1.05e-12
    # clover export in openQxD order = reorder of the natural-order export (PAPER.md:115-117 packing is shared)
    m_nat = g.clover_export(False)
    m_oq = g.openqxd_reorder(m_nat.reshape(-1, 72), 72, to_openqxd=True, block=blk).cpu().numpy()
    assert np.array_equal(m_oq, O.site_records_to_openqxd(ref.clover_packed(False).reshape(-1, 72), X, blk)) or \
        np.allclose(m_oq, O.site_records_to_openqxd(ref.clover_packed(False).reshape(-1, 72), X, blk), rtol=1e-13, atol=1e-13)
    g.close()
