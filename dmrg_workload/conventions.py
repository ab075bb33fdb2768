"""Conventions shared by every generator.

Spin orbitals: P = 2k (alpha of spatial orbital k), 2k+1 (beta), ordered along the
chain L < C1 < C2 < R.  A determinant is a+_{P1} a+_{P2} ... |vac> with P1 < P2 < ...
Site basis n in {0: vac, 1: beta, 2: alpha, 3: alpha beta},
index = 2 n_alpha + n_beta, |alpha beta> = a+_alpha a+_beta |vac>.
Quantum numbers q = (N, 2Sz).
"""
import numpy as np

SITE_Q = ((0, 0), (1, -1), (1, 1), (2, 0))  # (N, 2Sz) of site states 0..3


def site_annihilators():
    """4x4 matrices of a_alpha, a_beta in the site basis (signs local to the site)."""
    a_al = np.zeros((4, 4))
    a_be = np.zeros((4, 4))
    a_al[0, 2] = 1.0
    a_al[1, 3] = 1.0
    a_be[0, 1] = 1.0
    a_be[2, 3] = -1.0  # a_beta a+_alpha a+_beta |vac> = -|alpha>
    return a_al, a_be


def spin_of(P):
    """+1 for alpha (even spin-orbital index), -1 for beta."""
    return 1 if P % 2 == 0 else -1


class SpinOrbitalIntegrals:
    """h_PQ and V[P,Q,R,S] = <PQ||RS> from spatial h_pq, (pq|rs)  (Eq. 2).

    <PQ|RS> = (pr|qs) d(sP,sR) d(sQ,sS);  V = <PQ|RS> - <PQ|SR>.
    """

    def __init__(self, h, eri):
        self.h_sp = np.asarray(h, dtype=np.float64)
        self.eri = np.asarray(eri, dtype=np.float64)
        self.K = self.h_sp.shape[0]

    def h(self, P, Q):
        if (P ^ Q) & 1:
            return 0.0
        return float(self.h_sp[P >> 1, Q >> 1])

    def V(self, P, Q, R, S):
        p, q, r, s = P >> 1, Q >> 1, R >> 1, S >> 1
        v = 0.0
        if ((P ^ R) & 1) == 0 and ((Q ^ S) & 1) == 0:
            v += self.eri[p, r, q, s]
        if ((P ^ S) & 1) == 0 and ((Q ^ R) & 1) == 0:
            v -= self.eri[p, s, q, r]
        return float(v)

    def V_pq(self, P, Q):
        """V[P, Q, :, :] as a (2K x 2K) array over (R, S) -- the same numbers as V(), one slice at a time."""
        K = self.K
        p, q, oP, oQ = P >> 1, Q >> 1, P & 1, Q & 1
        e = self.eri[p, :, q, :]                 # e[r, s] = (pr|qs)
        out = np.zeros((2 * K, 2 * K))
        out[oP::2, oQ::2] += e                   # <PQ|RS>: spin(R) = spin(P), spin(S) = spin(Q)
        out[oQ::2, oP::2] -= e.T                 # <PQ|SR>: spin(S) = spin(P), spin(R) = spin(Q); (ps|qr) = e[s, r]
        return out

    def V_pt(self, P, T):
        """V[P, :, T, :] as a (2K x 2K) array over (Q, R)."""
        K = self.K
        p, t, oP, oT = P >> 1, T >> 1, P & 1, T & 1
        out = np.zeros((2 * K, 2 * K))
        if oP == oT:                             # <PQ|TR> = (pt|qr) d(sP,sT) d(sQ,sR)
            e = self.eri[p, t, :, :]
            out[0::2, 0::2] += e
            out[1::2, 1::2] += e
        out[oT::2, oP::2] -= self.eri[p, :, :, t].T   # <PQ|RT> = (pr|qt) d(sP,sR) d(sQ,sT); [q, r] = eri[p, r, q, t]
        return out

    def dense_h(self):
        n = 2 * self.K
        out = np.zeros((n, n))
        out[0::2, 0::2] = self.h_sp
        out[1::2, 1::2] = self.h_sp
        return out

    def dense_V(self):
        """Full antisymmetrised tensor (small K only: (2K)^4 doubles)."""
        K = self.K
        n = 2 * K
        coul = np.zeros((n, n, n, n))  # <PQ|RS>
        e = self.eri.transpose(0, 2, 1, 3)  # e[p,q,r,s] = (pr|qs)
        for sp in (0, 1):
            for sq in (0, 1):
                coul[sp::2, sq::2, sp::2, sq::2] = e
        return coul - coul.transpose(0, 1, 3, 2)
