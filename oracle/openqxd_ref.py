"""ORACLE (test infrastructure, not product): the openQxD field orders of PAPER.md §2 and §4.1, written out with
plain Python loops.  Shares no code with paper_2502_02490_b200/csrc.  Only tests/, __graft_entry__.smoke() and the
cpu_baseline leg of bench.py may import this module.

What it follows, passage by passage:
  * lexicographic index Lambda(x, L), Eq. (1), (t,x,y,z) order, x3 fastest;
  * cache blocks of extent B_mu, block-local index b_mu = x_mu mod B_mu, block index n_mu = floor(x_mu / B_mu),
    both lexicographic; even-odd ordering, even points first;
  * total index xhat = floor((V_B Lambda(n, N_B) + Lambda(b, B)) / 2) + P(x) V/2, Eq. (2)
    (the outer delimiters are garbled in the extraction; reading R14: floor);
  * spinor (x, alpha, a), a fastest: 12 consecutive complex numbers per site;
  * clover (x, +-, i): 2 x 36 reals per site;
  * gauge (x_odd, +-mu, a, b): the 8 links at every ODD point, 3x3 row-major.
    The paper defers the order of the 8 directions and which link "-mu" is to the host code's README
    (PAPER.md:123); reading R20: order +0,-0,+1,-1,+2,-2,+3,-3; entry +mu of the odd point x is U_mu(x),
    entry -mu is U_mu(x - mu), i.e. the link that ends at x.
On the extended (C*) lattice the fields obey U_mu(x + L1 e1) = U_mu(x)^*, A_mu(x + L1 e1) = -A_mu(x) and the shifted
boundary rule of DESIGN.md reading R8.

Pins (tests/test_openqxd_order.py): Eq. (2) against the prose definition (sort the points by parity, block, in-block
lexicographic index), bijectivity, even-first, the no-blocking special case floor(Lambda/2) + P V/2, and a
hand-enumerated 2x2x2x2 table.
"""
import itertools

import numpy as np


def lam(x, L):
    """Eq. (1)."""
    return ((x[0] * L[1] + x[1]) * L[2] + x[2]) * L[3] + x[3]


def parity(x):
    """P(x) = (1 - (-1)^{sum x_mu}) / 2."""
    return (x[0] + x[1] + x[2] + x[3]) & 1


def xhat(x, L, B):
    """Eq. (2)."""
    n = [x[m] // B[m] for m in range(4)]
    b = [x[m] % B[m] for m in range(4)]
    NB = [L[m] // B[m] for m in range(4)]
    VB = B[0] * B[1] * B[2] * B[3]
    V = L[0] * L[1] * L[2] * L[3]
    return (VB * lam(n, NB) + lam(b, B)) // 2 + parity(x) * (V // 2)


def ipt(L, B):
    """The mapping array of PAPER.md:105: ipt[Lambda(x, L)] = xhat."""
    out = np.empty(L[0] * L[1] * L[2] * L[3], dtype=np.int64)
    for x in itertools.product(*(range(e) for e in L)):
        out[lam(x, L)] = xhat(x, L, B)
    return out


def ext_dims(dims, cstar):
    T, L1, L2, L3 = dims
    return (T, 2 * L1 if cstar > 0 else L1, L2, L3)


def shift(x, mu, d, dims, cstar):
    """x + d*mu-hat on the extended lattice: time and direction 1 periodic (period X1), directions k in 2..cstar wrap with
    x1 -> x1 + L1 mod 2 L1 (reading R8)."""
    X = ext_dims(dims, cstar)
    y = list(x)
    y[mu] += d
    if y[mu] < 0 or y[mu] >= X[mu]:
        y[mu] %= X[mu]
        if mu >= 2 and mu <= cstar:
            y[1] = (y[1] + dims[1]) % X[1]
    return tuple(y)


def site_records_to_openqxd(nat, L, B):
    """nat[Lambda(x)][...] -> out[xhat][...] (spinor: 12 complex; clover: 2 x 36 reals)."""
    nat = np.asarray(nat)
    out = np.empty_like(nat)
    for x in itertools.product(*(range(e) for e in L)):
        out[xhat(x, L, B)] = nat[lam(x, L)]
    return out


def site_records_from_openqxd(oq, L, B):
    oq = np.asarray(oq)
    out = np.empty_like(oq)
    for x in itertools.product(*(range(e) for e in L)):
        out[lam(x, L)] = oq[xhat(x, L, B)]
    return out


def link_ext(U, x, mu, dims, cstar, is_phase):
    """U_mu(x) on the extended lattice from the physical field U[T][L1][L2][L3][4]...: mirror half = complex conjugate
    (SU(3) links) or minus (U(1) field A), reading R8."""
    L1 = dims[1]
    if x[1] < L1:
        return U[x[0], x[1], x[2], x[3], mu]
    v = U[x[0], x[1] - L1, x[2], x[3], mu]
    return -v if is_phase else np.conj(v)


def gauge_to_openqxd(U, dims, cstar, B, is_phase=False):
    """U: physical natural-order field [T][L1][L2][L3][4] (+[3][3]) -> ud[V_ext/2][8] (+[3][3]) at the odd points of the
    extended lattice, entry 2 mu = U_mu(x), entry 2 mu + 1 = U_mu(x - mu) (reading R20)."""
    X = ext_dims(dims, cstar)
    V = X[0] * X[1] * X[2] * X[3]
    ud = np.empty((V // 2, 8) + U.shape[5:], dtype=U.dtype)
    for x in itertools.product(*(range(e) for e in X)):
        if parity(x) == 0:
            continue
        o = xhat(x, X, B) - V // 2
        for mu in range(4):
            ud[o, 2 * mu] = link_ext(U, x, mu, dims, cstar, is_phase)
            ud[o, 2 * mu + 1] = link_ext(U, shift(x, mu, -1, dims, cstar), mu, dims, cstar, is_phase)
    return ud


def gauge_from_openqxd(ud, dims, cstar, B):
    """ud[V_ext/2][8]... -> physical natural-order field [T][L1][L2][L3][4]...: an odd point holds its own forward link,
    the forward link of an even point y is the -mu entry of the odd point y + mu."""
    X = ext_dims(dims, cstar)
    V = X[0] * X[1] * X[2] * X[3]
    U = np.empty(tuple(dims) + (4,) + ud.shape[2:], dtype=ud.dtype)
    for y in itertools.product(*(range(e) for e in dims)):
        for mu in range(4):
            if parity(y) == 1:
                U[y[0], y[1], y[2], y[3], mu] = ud[xhat(y, X, B) - V // 2, 2 * mu]
            else:
                z = shift(y, mu, +1, dims, cstar)
                U[y[0], y[1], y[2], y[3], mu] = ud[xhat(z, X, B) - V // 2, 2 * mu + 1]
    return U
