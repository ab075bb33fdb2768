"""Exact operators of a single spatial orbital (a 'dot' or a chain-end block).

Definitions: PAPER.md:131-139 (Eqs. 20-24) restricted to X = {2k, 2k+1}; the sums
"s<r" run over each unordered pair once.  All matrices are 4x4 in the site basis
of conventions.py with signs local to the site.
"""
import numpy as np

from .conventions import site_annihilators


class SiteOps:
    def __init__(self, k, ints):
        self.k = k
        self.ints = ints
        self.labels = (2 * k, 2 * k + 1)
        a_al, a_be = site_annihilators()
        self.ann = {2 * k: a_al, 2 * k + 1: a_be}
        self.cre = {P: m.T.copy() for P, m in self.ann.items()}

    def C(self, p):  # a+_p
        return self.cre[p]

    def D(self, p):  # a_p
        return self.ann[p]

    def A(self, p, q):  # a+_p a+_q
        return self.cre[p] @ self.cre[q]

    def B(self, p, t):  # a+_p a_t
        return self.cre[p] @ self.ann[t]

    def P(self, p, q):  # sum_{s<r in X} V[p,q,s,r] a_r a_s
        s, r = self.labels
        return self.ints.V(p, q, s, r) * (self.ann[r] @ self.ann[s])

    def Q(self, p, s):  # sum_{q,r in X} V[p,q,s,r] a+_q a_r
        out = np.zeros((4, 4), dtype=self.ints.dtype)
        for q in self.labels:
            for r in self.labels:
                v = self.ints.V(p, q, s, r)
                if v != 0.0:
                    out += v * (self.cre[q] @ self.ann[r])
        return out

    def S(self, p):  # sum_q h_pq/2 a_q + sum_{q; s<r} V[p,q,s,r] a+_q a_r a_s
        out = np.zeros((4, 4), dtype=self.ints.dtype)
        s, r = self.labels
        for q in self.labels:
            out += 0.5 * self.ints.h(p, q) * self.ann[q]
            v = self.ints.V(p, q, s, r)
            if v != 0.0:
                out += v * (self.cre[q] @ self.ann[r] @ self.ann[s])
        return out

    def H(self):  # Eq. (2) restricted to the site
        out = np.zeros((4, 4), dtype=self.ints.dtype)
        X = self.labels
        for p in X:
            for q in X:
                out += self.ints.h(p, q) * (self.cre[p] @ self.ann[q])
        for p in X:
            for q in X:
                for r in X:
                    for s in X:
                        v = self.ints.V(p, q, r, s)
                        if v != 0.0:
                            out += 0.25 * v * (self.cre[p] @ self.cre[q] @ self.ann[s] @ self.ann[r])
        return out
