"""The operator-pair term list  H = sum_mu O^L O^C1 O^C2 O^R  (Eq. 5).

The paper states only that there are O(K^2) terms built from normal and
complementary operators (Eqs. 19-24 at PAPER.md:126-139).  The list
below is DESIGN.md reading 2: the bipartition identity

  H^{XY} = H^X + H^Y + sum_{p in X}(a+_p S_p^Y + h.c.) + sum_{p in Y}(a+_p S_p^X + h.c.)
         + sum_{p<q in X}(A_pq P_pq^Y + h.c.) + sum_{p,s in X} B_ps Q_ps^Y

applied to (L u C1 | C2 u R) and then to the compound operators, re-associated so
that all O(K^2)-many terms are (two-index normal op on L) x (two-index complementary
op on R).  This module is symbolic: it emits slot descriptors and coefficients taken
from the integrals; it performs no contraction.

Storage conventions referenced here: A_pq, P_pq stored for p<q (P_qp = -P_pq);
B_pt, Q_pt stored for p<=t (B_tp = B_pt^H, Q_tp = Q_pt^H by Hermiticity of the integrals).
A 'LIN' operator is sum_s coef_s a+_s on one block; used "transposed" it is its Hermitian
conjugate sum_s conj(coef_s) a_s (the paper's "intermediates").
Throughout, a transposed use (trans flag) means the Hermitian conjugate of the stored operator:
the plain transpose for the real spin-free integrals, the conjugate transpose for the complex
integrals of a spin-orbit Hamiltonian, to which the same table applies.
"""
from collections import namedtuple

import numpy as np

from .conventions import SITE_Q
from .siteops import SiteOps

BlockOp = namedtuple("BlockOp", "side kind p q")  # side 'L'/'R'; kind H C A B P Q S LIN

ODD_KINDS = ("C", "S", "LIN")


def block_parity(op):
    return 1 if (op is not None and op[0].kind in ODD_KINDS) else 0


def dot_parity(m):
    """Parity of a 4x4 site matrix (None if the matrix is identically zero)."""
    nz = np.argwhere(m != 0.0)
    if len(nz) == 0:
        return None
    pars = {(SITE_Q[i][0] - SITE_Q[j][0]) & 1 for i, j in nz}
    assert len(pars) == 1, "site operator mixes parities"
    return pars.pop()


class Partition:
    def __init__(self, K, nL):
        self.K = K
        self.nL = nL
        self.nR = K - nL - 2
        assert self.nR >= 1 and nL >= 1
        self.L = list(range(0, 2 * nL))
        self.c = [2 * nL, 2 * nL + 1]
        self.d = [2 * nL + 2, 2 * nL + 3]
        self.R = list(range(2 * nL + 4, 2 * K))


class TermTable:
    """Symbolic term list.  Each entry: (coef, L slot, c matrix, d matrix, R slot),
    a slot being None (identity) or (BlockOp, trans)."""

    def __init__(self, part, ints):
        self.part = part
        self.ints = ints
        self.lincombs = {"L": [], "R": []}  # each: list of (label, coef)
        self._lin_index = {}
        self.terms = []
        self.tags = []
        self.complex = np.dtype(getattr(ints, "dtype", np.float64)).kind == "c"
        self.sc = SiteOps(part.nL, ints)
        self.sd = SiteOps(part.nL + 1, ints)
        self._build()

    # ---- helpers -------------------------------------------------------
    def _num(self, c):
        return complex(c) if self.complex else float(c)

    def linT(self, side, coefs):
        """Slot whose operator is sum_s coefs[s] a_s: the LIN operator sum_s conj(coefs[s]) a+_s, used transposed."""
        lin = self.lin(side, [(s, np.conj(c)) for s, c in coefs])
        return None if lin is None else (lin, True)

    def lin(self, side, coefs):
        """Register sum_s coefs[s] a+_s on `side`; returns BlockOp or None if all zero."""
        items = tuple((s, self._num(c)) for s, c in coefs if c != 0.0)
        if not items:
            return None
        key = (side, items)
        if key not in self._lin_index:
            self._lin_index[key] = len(self.lincombs[side])
            self.lincombs[side].append(list(items))
        return BlockOp(side, "LIN", self._lin_index[key], -1)

    @staticmethod
    def C(side, p):
        return BlockOp(side, "C", p, -1)

    @staticmethod
    def Pop(side, p, q):
        """P_pq as (op, sign) with stored order p<q."""
        if p < q:
            return BlockOp(side, "P", p, q), 1.0
        return BlockOp(side, "P", q, p), -1.0

    @staticmethod
    def Qop(side, p, t):
        """Q_pt as (op, trans) with stored order p<=t."""
        if p <= t:
            return BlockOp(side, "Q", p, t), False
        return BlockOp(side, "Q", t, p), True

    def add(self, tag, coef, L, c, d, R, hc):
        """L, R: None | (BlockOp, trans); c, d: None | 4x4 matrix."""
        if coef == 0.0:
            return
        I4 = np.eye(4)
        c = I4 if c is None else c
        d = I4 if d is None else d
        pc, pd = dot_parity(c), dot_parity(d)
        if pc is None or pd is None:
            return
        n_odd = block_parity(L) + pc + pd + block_parity(R)
        assert n_odd % 2 == 0, f"odd term in {tag}"
        self.terms.append((self._num(coef), L, c.copy(), d.copy(), R))
        self.tags.append(tag)
        if hc:
            sgn = -1.0 if (n_odd * (n_odd - 1) // 2) % 2 else 1.0
            Lh = None if L is None else (L[0], not L[1])
            Rh = None if R is None else (R[0], not R[1])
            self.terms.append((self._num(np.conj(coef)) * sgn, Lh, c.conj().T.copy(), d.conj().T.copy(), Rh))
            self.tags.append(tag + "+")

    # ---- the table -----------------------------------------------------
    def _build(self):
        pt, V = self.part, self.ints.V
        L, c, d, R = pt.L, pt.c, pt.d, pt.R
        c0, c1 = c
        d0, d1 = d
        sc, sd = self.sc, self.sd
        N = lambda op: (op, False)  # noqa: E731  normal use
        T = lambda op: (op, True)   # noqa: E731  transposed use
        H = lambda side: BlockOp(side, "H", -1, -1)  # noqa: E731
        S = lambda side, p: BlockOp(side, "S", p, -1)  # noqa: E731
        Cr = self.C
        add = self.add
        Ac = sc.A(c0, c1)
        Ad = sd.A(d0, d1)
        ddn = sd.D(d1) @ sd.D(d0)   # a_d1 a_d0
        ccn = sc.D(c1) @ sc.D(c0)   # a_c1 a_c0

        # G0
        add("G0", 1.0, N(H("L")), None, None, None, False)
        add("G0", 1.0, None, sc.H(), None, None, False)
        add("G0", 1.0, None, None, sd.H(), None, False)
        add("G0", 1.0, None, None, None, N(H("R")), False)
        # G1: H^{Lc} cross terms
        for p in L:
            add("G1a", 1.0, N(Cr("L", p)), sc.S(p), None, None, True)
        for p in c:
            add("G1b", -1.0, N(S("L", p)), sc.C(p), None, None, True)
        op, sg = self.Pop("L", c0, c1)
        add("G1c", sg, N(op), Ac, None, None, True)
        for p in c:
            for t in c:
                op, tr = self.Qop("L", p, t)
                add("G1d", 1.0, (op, tr), sc.B(p, t), None, None, False)
        # G2: H^{dR} cross terms
        for p in d:
            add("G2a", 1.0, None, None, sd.C(p), N(S("R", p)), True)
        for p in R:
            add("G2b", -1.0, None, None, sd.S(p), N(Cr("R", p)), True)
        op, sg = self.Pop("R", d0, d1)
        add("G2c", sg, None, None, Ad, N(op), True)
        for p in d:
            for t in d:
                op, tr = self.Qop("R", p, t)
                add("G2d", 1.0, None, None, sd.B(p, t), (op, tr), False)
        # G3: sum_{p in L u c} a+_p S_p^{dR}
        for p in L + c:
            if p in L:
                FL, Fc = N(Cr("L", p)), None
            else:
                FL, Fc = None, sc.C(p)
            add("G3a", 1.0, FL, Fc, sd.S(p), None, True)
            add("G3b", 1.0, FL, Fc, None, N(S("R", p)), True)
            for q in d:
                op, sg = self.Pop("R", p, q)
                add("G3c", sg, FL, Fc, sd.C(q), N(op), True)
            lin = self.lin("R", [(q, V(p, q, d0, d1)) for q in R])
            if lin is not None:
                add("G3d", 1.0, FL, Fc, ddn, N(lin), True)
            for t in d:
                op, tr = self.Qop("R", p, t)
                add("G3e", 1.0, FL, Fc, sd.D(t), (op, tr), True)
            for q in d:
                for t in d:
                    lin = self.linT("R", [(r, V(p, q, r, t)) for r in R])
                    if lin is not None:
                        add("G3f", 1.0, FL, Fc, sd.B(q, t), lin, True)
        # G4: sum_{p in d u R} a+_p S_p^{Lc}  (ordered: S_p^{Lc} to the left => -1)
        for p in d + R:
            if p in d:
                Gd, GR = sd.C(p), None
            else:
                Gd, GR = None, N(Cr("R", p))
            add("G4a", -1.0, N(S("L", p)), None, Gd, GR, True)
            add("G4b", -1.0, None, sc.S(p), Gd, GR, True)
            lin = self.lin("L", [(q, V(p, q, c0, c1)) for q in L])
            if lin is not None:
                add("G4c", -1.0, N(lin), ccn, Gd, GR, True)
            for q in c:
                op, sg = self.Pop("L", p, q)
                add("G4d", -1.0 * sg, N(op), sc.C(q), Gd, GR, True)
            for q in c:
                for t in c:
                    lin = self.linT("L", [(s, V(p, q, s, t)) for s in L])
                    if lin is not None:
                        add("G4e", -1.0, lin, sc.B(q, t), Gd, GR, True)
            for r in c:
                op, tr = self.Qop("L", p, r)
                add("G4f", -1.0, (op, tr), sc.D(r), Gd, GR, True)
        # G5: sum_{p<q in L u c} A_pq P_pq^{dR} + h.c.
        for i, p in enumerate(L):
            for q in L[i + 1:]:
                add("G5a", 1.0, N(BlockOp("L", "A", p, q)), None, None,
                    N(BlockOp("R", "P", p, q)), True)
        op, sg = self.Pop("L", d0, d1)
        add("G5b", sg, T(op), None, ddn, None, True)
        for t in d:
            for r in R:
                op, sg = self.Pop("L", t, r)
                add("G5c", -1.0 * sg, T(op), None, sd.D(t), T(Cr("R", r)), True)
        for p in L:
            for q in c:
                add("G5d", 1.0, N(Cr("L", p)), sc.C(q), None, N(BlockOp("R", "P", p, q)), True)
        for q in c:
            lin = self.lin("L", [(p, V(p, q, d0, d1)) for p in L])
            if lin is not None:
                add("G5e", 1.0, N(lin), sc.C(q), ddn, None, True)
        for p in L:
            for q in c:
                for t in d:
                    lin = self.linT("R", [(r, V(p, q, t, r)) for r in R])
                    if lin is not None:
                        add("G5f", -1.0, N(Cr("L", p)), sc.C(q), sd.D(t), lin, True)
        add("G5g", 1.0, None, Ac, None, N(BlockOp("R", "P", c0, c1)), True)
        add("G5h", V(c0, c1, d0, d1), None, Ac, ddn, None, True)
        for t in d:
            lin = self.linT("R", [(r, V(c0, c1, t, r)) for r in R])
            if lin is not None:
                add("G5i", -1.0, None, Ac, sd.D(t), lin, True)
        # G6: sum_{p,t in L u c} B_pt Q_pt^{dR}
        for i, p in enumerate(L):
            add("G6a", 1.0, N(BlockOp("L", "B", p, p)), None, None,
                N(BlockOp("R", "Q", p, p)), False)
            for t in L[i + 1:]:
                add("G6a", 1.0, N(BlockOp("L", "B", p, t)), None, None,
                    N(BlockOp("R", "Q", p, t)), True)
        for q in d:
            for t in d:
                op, tr = self.Qop("L", q, t)
                add("G6b", 1.0, (op, tr), None, sd.B(q, t), None, False)
        for q in d:
            for r in R:
                op, tr = self.Qop("L", q, r)
                add("G6c", 1.0, (op, tr), None, sd.C(q), T(Cr("R", r)), True)
        for p in L:
            for t in c:
                add("G6e", 1.0, N(Cr("L", p)), sc.D(t), None, N(BlockOp("R", "Q", p, t)), True)
        for t in c:
            for q in d:
                for u in d:
                    lin = self.lin("L", [(p, V(p, q, t, u)) for p in L])
                    if lin is not None:
                        add("G6f", 1.0, N(lin), sc.D(t), sd.B(q, u), None, True)
        for p in L:
            for t in c:
                for q in d:
                    lin = self.linT("R", [(r, V(p, q, t, r)) for r in R])
                    if lin is not None:
                        add("G6g", 1.0, N(Cr("L", p)), sc.D(t), sd.C(q), lin, True)
                    lin = self.lin("R", [(r, V(p, r, t, q)) for r in R])
                    if lin is not None:
                        add("G6h", -1.0, N(Cr("L", p)), sc.D(t), sd.D(q), N(lin), True)
        for p in c:
            for t in c:
                op, tr = self.Qop("R", p, t)
                add("G6i", 1.0, None, sc.B(p, t), None, (op, tr), False)
                add("G6j", 1.0, None, sc.B(p, t), sd.Q(p, t), None, False)
                for q in d:
                    lin = self.linT("R", [(r, V(p, q, t, r)) for r in R])
                    if lin is not None:
                        add("G6k", 1.0, None, sc.B(p, t), sd.C(q), lin, False)
                    lin = self.lin("R", [(r, V(p, r, t, q)) for r in R])
                    if lin is not None:
                        add("G6l", -1.0, None, sc.B(p, t), sd.D(q), N(lin), False)

    def referenced_ops(self):
        """All BlockOps used by the terms (lincombs included, their summands too)."""
        ops = {"L": set(), "R": set()}
        for _, Ls, _, _, Rs in self.terms:
            for s in (Ls, Rs):
                if s is not None:
                    ops[s[0].side].add(s[0])
        for side in ("L", "R"):
            for lc in self.lincombs[side]:
                for lab, _ in lc:
                    ops[side].add(BlockOp(side, "C", lab, -1))
        return ops
