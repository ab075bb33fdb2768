"""Inputs of one renormalization step (Eq. 8; Eqs. 15-18), as flat arrays.

A step enlarges a renormalized block by one site and projects with the site tensor A:
    [O_new]_{r'r} = sum_{l'c'} sum_{lc} zeta A^{c'}_{l'r'} [O^blk]_{l'l} [O^site]_{c'c} A^{c}_{lr}        (Eq. 8)
for every operator the new block carries.  This module is symbolic, like terms.py: for each new operator it
emits the list of product terms  coef * (block operator or identity, transposed or not) x (4x4 site matrix),
with coefficients taken from the integrals, plus the linear-combination operators ("intermediates",
PAPER.md:112) those terms refer to.  It performs no contraction.  The recursions are those of blocking.py
 written as term lists:

  side 0 (block x site, a left block growing to the right), side 1 (site x block, a right block growing to the left)
  a+_p    : p in block: a+_p x 1;                 p in site: 1 x a+_p
  A_pq    : (blk,blk) A x 1; (site,site) 1 x A;   one label each: a+ x a+   (the factor of the earlier label first)
  B_pt    : (blk,blk) B x 1; (site,site) 1 x B;   one label each: a+ x a
  H       : H x 1 + 1 x H + sum_{p in first}[a+_p x S_p + h.c.] - sum_{p in second}[S_p x a+_p + h.c.]
            + [P_{s0 s1}(blk) x A_{s0 s1}(site) + h.c.] + sum_{p,t in site} Q_pt(blk) x B_pt(site)
  S_p     : S_p x 1 + 1 x S_p + sum_q a+_q x P_pq + sum_q P_pq x a+_q + sum_t a_t x Q_pt + sum_r Q_pr x a_r
The Jordan-Wigner factor of an odd second factor, (-1)^{N(ket of the first factor)}, is NOT in the coefficients: it
is the zeta of Eq. (8), which both the oracle and the library derive from the operator parities (DESIGN.md
reading 3 restricted to two factors).  The h.c. of a product of two odd factors carries -1 (h.c. rule).

Block complementary operators are linear combinations of the block's two-index operators:
  P_pq(blk) = (LP_pq)^T,  LP_pq = sum_{s<r in blk} V[p,q,s,r] A_sr
  Q_pt(blk) = LQ1_pt + (LQ2_pt)^T,  LQ1 = sum_{q<=r} V[p,q,t,r] B_qr,  LQ2 = sum_{q>r} V[p,q,t,r] B_rq
"""
import numpy as np

from .conventions import SITE_Q, spin_of
from .siteops import SiteOps
from .store import KIND, op_charge
from .terms import BlockOp, dot_parity


class RenormProblem:
    """Flat arrays of one step (formats of include/dmrg_sigma.h):
    sec_old [n,3]; ops [nops,8] (side, kind, p, q, dN, d2Sz, first_block, nblocks) incl. LINCOMB rows;
    blocks [nblk,3]; values; lin_ptr/lin_op/lin_coef; site_ops [nsite,16], site_parity;
    sec_new [m,3]; wblocks [nw,4] (old sector, site state, new sector, offset into wvalues), wvalues;
    new_ops [k,8] (first_block / nblocks unused); term_ptr [k+1]; term_coef; term_idx [nt,3] (op or -1, trans, site op);
    new_keys: RBlock key of every new operator."""


def _store_key(op):
    k = op.kind
    if k == "H":
        return ("H",)
    if k in ("C", "S"):
        return (k, op.p)
    return (k, op.p, op.q)


class BlockShape:
    """What a step needs to know about a block when its operator VALUES live elsewhere (on the device): labels,
    sector table, and which operators it carries (RBlock keys)."""

    def __init__(self, labels, sectors, dims, op_keys):
        self.labels, self.sectors, self.dims, self.op_keys = list(labels), list(sectors), list(dims), list(op_keys)
        self.site_tensor = None


def carried_keys(labels, outside):
    """RBlock keys of the operators a block over `labels` carries: a+_p, A_pq (p<q), B_pt (p<=t), S_p (p outside), H."""
    X = sorted(labels)
    keys = [("C", p) for p in X]
    keys += [("A", p, q) for i, p in enumerate(X) for q in X[i + 1:]]
    keys += [("B", p, t) for i, p in enumerate(X) for t in X[i:]]
    keys += [("S", p) for p in outside]
    keys.append(("H",))
    return keys


def compl_P_items(X, p, q, ints, side):
    """P_pq = sum_{s<r in X} V[p,q,s,r] a_r a_s = sum V (A_sr)^T  (Eq. 22): [(BlockOp, coef, trans)]."""
    X = sorted(X)
    v = ints.V_pq(p, q)
    return [(BlockOp(side, "A", s, r), float(v[s, r]), 1) for i, s in enumerate(X) for r in X[i + 1:] if v[s, r] != 0.0]


def compl_Q_items(X, p, t, ints, side):
    """Q_pt = sum_{q,r in X} V[p,q,t,r] a+_q a_r (Eq. 23), B_qr stored for q <= r: [(BlockOp, coef, trans)]."""
    out = []
    vm = ints.V_pt(p, t)
    for q in sorted(X):
        for r in sorted(X):
            v = float(vm[q, r])
            if v != 0.0:
                out.append((BlockOp(side, "B", q, r), v, 0) if q <= r else (BlockOp(side, "B", r, q), v, 1))
    return out


def build_renorm_problem(blk, site_k, side, ints, outside_new, new_blk, structure_only=False):
    """blk: RBlock being enlarged by spatial orbital site_k; side 0: blk x site, 1: site x blk;
    outside_new: labels p for which the new block carries S_p; new_blk: the RBlock blocking.merge produced
    (its sector table and site tensor are the projection this step applies).
    structure_only: blk / new_blk are BlockShapes; no operator values are read and rp.blocks / rp.values stay empty
    (the values live in a device store whose operators are matched by (kind, p, q))."""
    so = SiteOps(site_k, ints)
    s0, s1 = so.labels
    sname = "L" if side == 0 else "R"
    X = list(blk.labels)
    rp = RenormProblem()
    rp.side = side
    # ---- old store: every carried operator of blk, then the linear combinations the terms need -------------
    stored = []
    for key in (blk.op_keys if structure_only else blk.ops):
        kind = key[0]
        p = key[1] if len(key) > 1 else -1
        q = key[2] if len(key) > 2 else -1
        stored.append(BlockOp(sname, kind, p, q))
    stored.sort(key=lambda o: (KIND[o.kind], o.p, o.q))
    sidx = {q: i for i, q in enumerate(blk.sectors)}
    op_id, ops_rows, blk_rows, vals = {}, [], [], []
    off = 0
    for op in stored:
        dq = op_charge(op)
        first = len(blk_rows)
        for (r, c), m in ([] if structure_only else sorted(blk.ops[_store_key(op)].items())):
            assert (blk.sectors[c][0] + dq[0], blk.sectors[c][1] + dq[1]) == blk.sectors[r]
            blk_rows.append((r, c, off))
            vals.append(np.ascontiguousarray(m, dtype=np.float64).ravel())
            off += m.size
        op_id[op] = len(ops_rows)
        ops_rows.append((side, KIND[op.kind], op.p, op.q, dq[0], dq[1], first, len(blk_rows) - first))
    lin_ptr, lin_op, lin_coef, lin_index = [0], [], [], {}

    def lincomb(items, dq):
        """Register sum coef * stored op; items: list of (BlockOp, coef).  Returns op id or None."""
        items = tuple((op_id[o], float(c)) for o, c in items if c != 0.0)
        if not items:
            return None
        if items not in lin_index:
            lin_index[items] = len(ops_rows)
            ops_rows.append((side, KIND["LIN"], len(lin_ptr) - 1, -1, dq[0], dq[1], 0, 0))
            for o, c in items:
                lin_op.append(o)
                lin_coef.append(c)
            lin_ptr.append(len(lin_op))
        return lin_index[items]

    def LP(p, q):   # sum_{s<r in blk} V[p,q,s,r] A_sr   (P_pq = LP^T)
        v = ints.V_pq(p, q)
        items = [(BlockOp(sname, "A", s, r), float(v[s, r])) for i, s in enumerate(X) for r in X[i + 1:]]
        return lincomb(items, (2, -(-spin_of(p) - spin_of(q))))

    def LQ(p, t):   # (LQ1, LQ2): Q_pt = LQ1 + LQ2^T
        v = ints.V_pt(p, t)
        i1 = [(BlockOp(sname, "B", q, r), float(v[q, r])) for q in X for r in X if q <= r]
        i2 = [(BlockOp(sname, "B", r, q), float(v[q, r])) for q in X for r in X if q > r]
        dq = (0, spin_of(t) - spin_of(p))
        return lincomb(i1, dq), lincomb(i2, (0, -dq[1]))

    # ---- site operators, deduplicated by value --------------------------------------------------------------
    site_index, site_ops, site_par = {}, [], []

    def sid(m):
        par = dot_parity(m)
        if par is None:
            return None
        key = m.tobytes()
        if key not in site_index:
            site_index[key] = len(site_ops)
            site_ops.append(np.array(m, dtype=np.float64).ravel().copy())
            site_par.append(par)
        return site_index[key]

    I4 = sid(np.eye(4))
    # ---- new operators and their terms --------------------------------------------------------------------
    new_rows, new_keys, term_ptr, tcoef, tidx = [], [], [0], [], []

    def emit(key, kind, p, q, dq, terms):
        for coef, bop, trans, m in terms:
            s = sid(m)
            if s is None or coef == 0.0 or bop is None:
                continue
            tcoef.append(float(coef))
            tidx.append((bop, int(trans), s))
        new_rows.append((side, KIND[kind], p, q, dq[0], dq[1], 0, 0))
        new_keys.append(key)
        term_ptr.append(len(tcoef))

    def bid(kind, p=-1, q=-1):
        return op_id[BlockOp(sname, kind, p, q)]

    ID = -1
    eye = np.eye(4)
    in_blk = set(X)
    in_site = {s0, s1}
    labs_new = sorted(in_blk | in_site)
    for p in labs_new:
        dq = (1, spin_of(p))
        emit(("C", p), "C", p, -1, dq, [(1.0, bid("C", p), 0, eye)] if p in in_blk else [(1.0, ID, 0, so.C(p))])
    for i, p in enumerate(labs_new):
        for q in labs_new[i + 1:]:
            dq = (2, spin_of(p) + spin_of(q))
            if p in in_blk and q in in_blk:
                t = [(1.0, bid("A", p, q), 0, eye)]
            elif p in in_site and q in in_site:
                t = [(1.0, ID, 0, so.A(p, q))]
            elif p in in_blk:       # side 0: a+_p(blk) x a+_q(site)
                t = [(1.0, bid("C", p), 0, so.C(q))]
            else:                   # side 1: a+_p(site) x a+_q(blk)
                t = [(1.0, bid("C", q), 0, so.C(p))]
            emit(("A", p, q), "A", p, q, dq, t)
        for q in labs_new[i:]:
            dq = (0, spin_of(p) - spin_of(q))
            if p in in_blk and q in in_blk:
                t = [(1.0, bid("B", p, q), 0, eye)]
            elif p in in_site and q in in_site:
                t = [(1.0, ID, 0, so.B(p, q))]
            elif p in in_blk:       # side 0: a+_p(blk) x a_q(site)
                t = [(1.0, bid("C", p), 0, so.D(q))]
            else:                   # side 1: a+_p(site) x a_q(blk)
                t = [(1.0, bid("C", q), 1, so.C(p))]
            emit(("B", p, q), "B", p, q, dq, t)
    # H
    t = [(1.0, bid("H"), 0, eye), (1.0, ID, 0, so.H())]
    first_is_blk = side == 0
    for p in (X if first_is_blk else [s0, s1]):     # p in the FIRST factor: a+_p x S_p + h.c.
        if first_is_blk:
            t += [(1.0, bid("C", p), 0, so.S(p)), (-1.0, bid("C", p), 1, so.S(p).T)]
        else:
            t += [(1.0, bid("S", p), 0, so.C(p)), (-1.0, bid("S", p), 1, so.D(p))]
    for p in ([s0, s1] if first_is_blk else X):     # p in the SECOND factor: -(S_p x a+_p) + h.c.
        if first_is_blk:
            t += [(-1.0, bid("S", p), 0, so.C(p)), (1.0, bid("S", p), 1, so.D(p))]
        else:
            t += [(-1.0, bid("C", p), 0, so.S(p)), (1.0, bid("C", p), 1, so.S(p).T)]
    lp = LP(s0, s1)
    As = so.A(s0, s1)
    t += [(1.0, lp, 1, As), (1.0, lp, 0, As.T)]
    for p in (s0, s1):
        for u in (s0, s1):
            q1, q2 = LQ(p, u)
            t += [(1.0, q1, 0, so.B(p, u)), (1.0, q2, 1, so.B(p, u))]
    emit(("H",), "H", -1, -1, (0, 0), t)
    # S_p
    for p in outside_new:
        dq = (-1, -spin_of(p))
        t = [(1.0, bid("S", p), 0, eye), (1.0, ID, 0, so.S(p))]
        for q in X:            # block label q with the site's complementary operators
            t += [(1.0, bid("C", q), 0, so.P(p, q)), (1.0, bid("C", q), 1, so.Q(p, q))]
        for q in (s0, s1):     # site label q with the block's complementary operators
            t += [(1.0, LP(p, q), 1, so.C(q))]
            q1, q2 = LQ(p, q)
            t += [(1.0, q1, 0, so.D(q)), (1.0, q2, 1, so.D(q))]
        emit(("S", p), "S", p, -1, dq, t)
    # ---- arrays ---------------------------------------------------------------------------------------------
    rp.sec_old = np.array([(q[0], q[1], d) for q, d in zip(blk.sectors, blk.dims)], dtype=np.int32).reshape(-1, 3)
    rp.ops = np.array(ops_rows, dtype=np.int64).reshape(-1, 8)
    rp.blocks = np.array(blk_rows, dtype=np.int64).reshape(-1, 3)
    rp.values = np.concatenate(vals) if vals else np.zeros(0)
    rp.lin_ptr = np.array(lin_ptr, dtype=np.int64)
    rp.lin_op = np.array(lin_op, dtype=np.int32)
    rp.lin_coef = np.array(lin_coef, dtype=np.float64)
    rp.site_ops = np.array(site_ops, dtype=np.float64).reshape(-1, 16)
    rp.site_parity = np.array(site_par, dtype=np.int32)
    rp.sec_new = np.array([(q[0], q[1], d) for q, d in zip(new_blk.sectors, new_blk.dims)], dtype=np.int32).reshape(-1, 3)
    wrows, wvals, woff = [], [], 0
    for i_old, n_site, r_new, m in new_blk.site_tensor:
        wrows.append((i_old, n_site, r_new, woff))
        wvals.append(np.ascontiguousarray(m, dtype=np.float64).ravel())
        woff += m.size
    rp.wblocks = np.array(wrows, dtype=np.int64).reshape(-1, 4)
    rp.wvalues = np.concatenate(wvals) if wvals else np.zeros(0)
    rp.new_ops = np.array(new_rows, dtype=np.int64).reshape(-1, 8)
    rp.new_keys = new_keys
    rp.term_ptr = np.array(term_ptr, dtype=np.int64)
    rp.term_coef = np.array(tcoef, dtype=np.float64)
    rp.term_idx = np.array(tidx, dtype=np.int32).reshape(-1, 3)
    rp.site_q = np.array(SITE_Q, dtype=np.int32)
    return rp
