"""Test helper: brute-force second-quantised operators in the full Fock space.

Independent of `oracle/` and of the CUDA path: Jordan-Wigner matrices built by
Kronecker products over sites (scipy.sparse), used to check the term table and the
blocking generator against the DEFINITIONS (Eq. 2; PAPER.md:131-139
Eqs. 20-24) at tiny K.
"""
import numpy as np
import scipy.sparse as sp

from dmrg_workload.conventions import SITE_Q, site_annihilators

_ZS = sp.diags([(-1.0) ** q[0] for q in SITE_Q]).tocsr()
_I4 = sp.identity(4, format="csr")


def block_annihilators(labels):
    """{P: a_P} on the Fock space of consecutive sites, site-Kronecker basis, local signs."""
    assert len(labels) % 2 == 0
    nsite = len(labels) // 2
    a_al, a_be = site_annihilators()
    out = {}
    for i in range(nsite):
        for spin, m in ((0, a_al), (1, a_be)):
            mats = [_ZS] * i + [sp.csr_matrix(m)] + [_I4] * (nsite - i - 1)
            acc = mats[0]
            for x in mats[1:]:
                acc = sp.kron(acc, x, format="csr")
            out[labels[2 * i + spin]] = acc
    return out


def block_Z(labels):
    acc = _ZS
    for _ in range(len(labels) // 2 - 1):
        acc = sp.kron(acc, _ZS, format="csr")
    return acc


def block_qnums(labels):
    """(N, 2Sz) of every basis state of the block, site-Kronecker order."""
    q = np.array(SITE_Q)
    N = q[:, 0]
    S = q[:, 1]
    for _ in range(len(labels) // 2 - 1):
        N = (N[:, None] + q[None, :, 0]).ravel()
        S = (S[:, None] + q[None, :, 1]).ravel()
    return N, S


class DenseBlock:
    """Operators of Eqs. (20)-(24) on block X from their definitions."""

    def __init__(self, labels, ints):
        self.X = list(labels)
        self.ints = ints
        self.a = block_annihilators(self.X)
        self.dim = 4 ** (len(self.X) // 2)

    def op(self, kind, p=-1, q=-1, lin=None):
        a, V, h, X = self.a, self.ints.V, self.ints.h, self.X
        z = sp.csr_matrix((self.dim, self.dim))
        if kind == "C":
            return a[p].T.tocsr()
        if kind == "A":
            return (a[p].T @ a[q].T).tocsr()
        if kind == "B":
            return (a[p].T @ a[q]).tocsr()
        if kind == "P":
            out = z
            for i, s in enumerate(X):
                for r in X[i + 1:]:
                    v = V(p, q, s, r)
                    if v:
                        out = out + v * (a[r] @ a[s])
            return out
        if kind == "Q":
            out = z
            for qq in X:
                for r in X:
                    v = V(p, qq, q, r)
                    if v:
                        out = out + v * (a[qq].T @ a[r])
            return out
        if kind == "S":
            out = z
            for qq in X:
                if h(p, qq):
                    out = out + 0.5 * h(p, qq) * a[qq]
                for i, s in enumerate(X):
                    for r in X[i + 1:]:
                        v = V(p, qq, s, r)
                        if v:
                            out = out + v * (a[qq].T @ a[r] @ a[s])
            return out
        if kind == "H":
            return hamiltonian({P: a[P] for P in X}, self.ints, self.dim)
        if kind == "LIN":
            out = z
            for s, c in lin:
                out = out + c * a[s].T
            return out
        raise ValueError(kind)


def hamiltonian(a, ints, dim):
    """Eq. (2): sum h a+a + 1/4 sum V a+a+aa over the labels of `a`."""
    labs = sorted(a)
    out = sp.csr_matrix((dim, dim))
    for p in labs:
        for q in labs:
            if ints.h(p, q):
                out = out + ints.h(p, q) * (a[p].T @ a[q])
    # 1/4 sum_{pqrs} V[pqrs] a+p a+q a_s a_r = sum_{p<q, r<s} V[pqrs] a+p a+q a_s a_r
    for i, p in enumerate(labs):
        for q in labs[i + 1:]:
            cc = a[p].T @ a[q].T
            for j, r in enumerate(labs):
                for s in labs[j + 1:]:
                    v = ints.V(p, q, r, s)
                    if v:
                        out = out + v * (cc @ a[s] @ a[r])
    return out


def full_annihilators(K):
    return block_annihilators(list(range(2 * K)))
