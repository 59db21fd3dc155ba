"""Test-only numpy helpers, written independently of oracle/ and of the CUDA path.

Used to pin the oracle (tests/test_oracle_pins.py): explicit gamma matrices typed from the
block forms of DESIGN.md reading R3, vectorised neighbour tables for the extended lattice with
shifted C* boundaries (reading R8), array-level clover construction and an entry-by-entry dense
assembler of D_w for brute-force LU checks on tiny lattices.
"""
from __future__ import annotations

import numpy as np

# --- Pauli and gamma matrices typed explicitly (reading R3 / SURVEY.md §8(c2)) -----------------
S1 = np.array([[0, 1], [1, 0]], dtype=complex)
S2 = np.array([[0, -1j], [1j, 0]], dtype=complex)
S3 = np.array([[1, 0], [0, -1]], dtype=complex)
PAULI = [None, S1, S2, S3]
Z2 = np.zeros((2, 2), dtype=complex)
I2 = np.eye(2, dtype=complex)
GAMMA = [np.block([[Z2, -I2], [-I2, Z2]])] + [np.block([[Z2, -1j * s], [1j * s, Z2]]) for s in (S1, S2, S3)]
GAMMA5 = np.diag([1, 1, -1, -1]).astype(complex)


def sigma_closed_form(mu, nu):
    """sigma_{mu nu} from the stated consequences: sigma_0k = diag(s_k,-s_k); sigma_ij = -eps_ijk diag(s_k,s_k)."""
    if mu == nu:
        return np.zeros((4, 4), dtype=complex)
    if mu > nu:
        return -sigma_closed_form(nu, mu)
    if mu == 0:
        s = PAULI[nu]
        return np.block([[s, Z2], [Z2, -s]])
    k = 6 - mu - nu  # the remaining spatial index
    eps = 1.0 if (mu, nu, k) in ((1, 2, 3), (2, 3, 1), (3, 1, 2)) else -1.0
    s = PAULI[k]
    return -eps * np.block([[s, Z2], [Z2, s]])


class Lattice:
    """Extended lattice bookkeeping with vectorised neighbour tables."""

    def __init__(self, T, L1, L2, L3, cstar=0, antiperiodic=True):
        self.phys = (T, L1, L2, L3)
        self.cstar = cstar
        self.L1 = L1
        self.antiper = bool(antiperiodic)
        self.X = (T, 2 * L1 if cstar > 0 else L1, L2, L3)
        self.V = int(np.prod(self.X))
        self.coords = np.stack(np.unravel_index(np.arange(self.V), self.X), axis=1)  # [V,4], x3 fastest
        self.parity = self.coords.sum(axis=1) & 1
        self.nbr = np.empty((4, 2, self.V), dtype=np.int64)     # [mu][0 fwd / 1 bwd][site]
        self.tcross = np.zeros((4, 2, self.V), dtype=bool)      # hop crosses the time boundary
        for mu in range(4):
            for d, step in enumerate((+1, -1)):
                y = self.coords.copy()
                c = y[:, mu] + step
                wrapped = (c < 0) | (c >= self.X[mu])
                y[:, mu] = np.mod(c, self.X[mu])
                if mu >= 2 and mu <= cstar:
                    y[wrapped, 1] = (y[wrapped, 1] + L1) % self.X[1]
                if mu == 0:
                    self.tcross[mu, d] = wrapped
                self.nbr[mu, d] = np.ravel_multi_index(tuple(y.T), self.X)

    # fields on the extended lattice, flattened over sites
    def extend_gauge(self, U, A=None):
        """U [T,L1,L2,L3,4,3,3] physical -> [V,4,3,3] extended (mirror = complex conjugate); A mirror = -A."""
        if self.cstar > 0:
            Ue = np.concatenate([U, np.conj(U)], axis=1)
            Ae = None if A is None else np.concatenate([A, -A], axis=1)
        else:
            Ue, Ae = U, A
        return Ue.reshape(self.V, 4, 3, 3), (None if Ae is None else Ae.reshape(self.V, 4))

    def shift(self, F, mu, d):
        """Field at x + mu-hat (d=0) or x - mu-hat (d=1)."""
        return F[self.nbr[mu, d]]


def mm(a, b):
    return np.einsum("...ij,...jk->...ik", a, b)


def dagm(a):
    return np.conj(np.swapaxes(a, -1, -2))


def clover_site_matrices(lat: Lattice, Ue, Ae, m0, csw, csw_qed, q, qel):
    """[V,12,12] site-diagonal matrices, by array-level shifts (independent of the oracle's per-site code)."""
    V = lat.V
    M = np.zeros((V, 12, 12), dtype=complex)
    M += (4.0 + m0) * np.eye(12)
    Umu = [Ue[:, mu] for mu in range(4)]
    for mu in range(4):
        for nu in range(mu + 1, 4):
            X = np.zeros((V, 3, 3), dtype=complex)
            if csw != 0.0:
                U_m, U_n = Umu[mu], Umu[nu]
                f, b = 0, 1
                U_n_xpm = lat.shift(U_n, mu, f)
                U_m_xpn = lat.shift(U_m, nu, f)
                U_m_xmm = lat.shift(U_m, mu, b)
                U_n_xmm = lat.shift(U_n, mu, b)
                U_m_xmmpn = lat.shift(U_m_xmm, nu, f)
                U_n_xmn = lat.shift(U_n, nu, b)
                U_m_xmn = lat.shift(U_m, nu, b)
                U_m_xmmmn = lat.shift(U_m_xmm, nu, b)
                U_n_xmmmn = lat.shift(U_n_xmm, nu, b)
                U_n_xpmmn = lat.shift(U_n_xpm, nu, b)
                Q = (mm(mm(U_m, U_n_xpm), mm(dagm(U_m_xpn), dagm(U_n)))
                     + mm(mm(U_n, dagm(U_m_xmmpn)), mm(dagm(U_n_xmm), U_m_xmm))
                     + mm(mm(dagm(U_m_xmm), dagm(U_n_xmmmn)), mm(U_m_xmmmn, U_n_xmn))
                     + mm(mm(dagm(U_n_xmn), U_m_xmn), mm(U_n_xpmmn, dagm(U_m))))
                X += csw * (Q - dagm(Q)) / 8.0
            if csw_qed != 0.0 and Ae is not None:
                A_m, A_n = Ae[:, mu], Ae[:, nu]
                Phi = A_m + lat.shift(A_n, mu, 0) - lat.shift(A_m, nu, 0) - A_n
                Phi_mm = lat.shift(Phi, mu, 1)
                s = np.sin(qel * Phi) + np.sin(qel * Phi_mm) + np.sin(qel * lat.shift(Phi, nu, 1)) + np.sin(qel * lat.shift(Phi_mm, nu, 1))
                X += (q * csw_qed * 1j * s / (4.0 * qel))[:, None, None] * np.eye(3)
            sg = sigma_closed_form(mu, nu)
            # (i/4) sum over both orderings = (i/2) sigma_{mu nu} (x) X_{mu nu}
            M += 0.5j * np.einsum("ab,vij->vaibj", sg, X).reshape(V, 12, 12)
    return M


def dense_Dw(lat: Lattice, Ue, Ae, kappa, q, csw, csw_qed, qel=1.0):
    """Dense (12V x 12V) matrix of D_w assembled block by block."""
    V = lat.V
    m0 = 1.0 / (2.0 * kappa) - 4.0
    D = np.zeros((V, 12, V, 12), dtype=complex)
    M = clover_site_matrices(lat, Ue, Ae, m0, csw, csw_qed, q, qel)
    idx = np.arange(V)
    D[idx, :, idx, :] += M
    for mu in range(4):
        W = Ue[:, mu] if Ae is None else np.exp(1j * q * Ae[:, mu])[:, None, None] * Ue[:, mu]
        Pm = np.eye(4) - GAMMA[mu]
        Pp = np.eye(4) + GAMMA[mu]
        fw = lat.nbr[mu, 0]
        sg = np.where(lat.tcross[mu, 0] & lat.antiper, -1.0, 1.0)
        for s in range(V):
            y = fw[s]
            # forward hop from s to y uses W_mu(s); the backward hop from y to s uses W_mu(s)^dag
            D[s, :, y, :] += -0.5 * sg[s] * np.kron(Pm, W[s])
            D[y, :, s, :] += -0.5 * sg[s] * np.kron(Pp, W[s].conj().T)
    return D.reshape(12 * V, 12 * V)
