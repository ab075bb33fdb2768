"""ORACLE (test infrastructure, not product code): the renormalization step, Eq. (8),

    [O_new]_{r'r} = sum_{l'c'} sum_{lc} zeta A^{c'}_{l'r'} [O^blk]_{l'l} [O^site]_{c'c} A^{c}_{lr},

written out block by block as the paper's Eqs. (15)-(18) state it, in FP64 numpy with plain loops
over symmetry blocks (np.matmul is the only library step; no blocking, fusion or reordering):
    (15) scale by the site factor [O^site]_{c'c} (a number for N, Sz symmetry)
    (16) I = [O^blk]_{L'L} . A(L C R)
    (17) I' = A(L' C' R')^T . I
    (18) O_new(R'R) = sum over (L' C' L C) and the product terms of the operator, zeta * I'.
Linear-combination operators ("intermediates") are formed first.

zeta (PAPER.md:75 names it, gives no formula; reading 3 restricted to two factors): the two factors of the
enlarged basis are ordered (first, second) = (block, site) for side 0 and (site, block) for side 1, and
    zeta = (-1)^{ parity(operator on the second factor) * N(ket state of the first factor) }.

Only tests/ and __graft_entry__.smoke() may import this.  Shares no code with the CUDA path; array formats only
(dmrg_workload/renorm_terms.py).  Pins: tests/test_oracle_renorm.py (every renormalized operator equals
E^T O_definition E with O_definition built by brute-force second quantisation, tests/fockdense.py).
"""
import numpy as np

SITE_N = (0, 1, 1, 2)
SITE_S = (0, -1, 1, 0)


def _op_blocks(rp):
    """{op id: {(row sector, col sector): matrix}} of the old store, linear combinations formed block by block."""
    out = []
    sec = rp.sec_old
    for o, row in enumerate(rp.ops):
        kind, first, nb = int(row[1]), int(row[6]), int(row[7])
        d = {}
        if kind != 7:
            for b in range(first, first + nb):
                r, c, off = (int(v) for v in rp.blocks[b])
                d[(r, c)] = rp.values[off:off + sec[r][2] * sec[c][2]].reshape(sec[r][2], sec[c][2])
        out.append(d)
    for o, row in enumerate(rp.ops):
        if int(row[1]) != 7:
            continue
        j = int(row[2])
        acc = {}
        for i in range(int(rp.lin_ptr[j]), int(rp.lin_ptr[j + 1])):
            for key, m in out[int(rp.lin_op[i])].items():
                acc[key] = acc.get(key, 0.0) + rp.lin_coef[i] * m
        out[o] = acc
    return out


def renormalize(rp):
    """Returns one dict per new operator: {(new row sector, new col sector): matrix}."""
    ops = _op_blocks(rp)
    sec_old, sec_new = rp.sec_old, rp.sec_new
    side = rp.side
    # site tensor A: sub-blocks (old sector i, site state n) -> new sector r
    sub = {}
    for i, n, r, off in (tuple(int(v) for v in w) for w in rp.wblocks):
        d, k = sec_old[i][2], sec_new[r][2]
        sub.setdefault(r, []).append((i, n, rp.wvalues[off:off + d * k].reshape(d, k)))
    new_index = {(int(s[0]), int(s[1])): r for r, s in enumerate(sec_new)}
    result = []
    for k, row in enumerate(rp.new_ops):
        dN, dS = int(row[4]), int(row[5])
        blocks = {}
        for r in range(len(sec_new)):            # ket sector R
            rp_ = new_index.get((int(sec_new[r][0]) + dN, int(sec_new[r][1]) + dS))
            if rp_ is None:
                continue                          # bra sector R' = R + charge absent
            acc = np.zeros((sec_new[rp_][2], sec_new[r][2]))
            hit = False
            for t in range(int(rp.term_ptr[k]), int(rp.term_ptr[k + 1])):
                coef = rp.term_coef[t]
                bop, trans, sop = (int(v) for v in rp.term_idx[t])
                o_site = rp.site_ops[sop].reshape(4, 4)
                p_site = int(rp.site_parity[sop])
                p_blk = int(rp.ops[bop][4]) & 1 if bop >= 0 else 0
                for (i, n, A_ket) in sub.get(r, []):             # ket sub-block (L, C)
                    for (ip, npr, A_bra) in sub.get(rp_, []):    # bra sub-block (L', C')
                        oc = o_site[npr, n]                      # Eq. (15): a number
                        if oc == 0.0:
                            continue
                        if bop < 0:
                            if ip != i:
                                continue
                            Ob = None
                        else:
                            Ob = ops[bop].get((i, ip)) if trans else ops[bop].get((ip, i))
                            if Ob is None:
                                continue
                            if trans:
                                Ob = Ob.T
                        if side == 0:    # (block, site): second factor = site, first ket = block state
                            zexp = p_site * int(sec_old[i][0])
                        else:            # (site, block): second factor = block, first ket = site state
                            zexp = p_blk * SITE_N[n]
                        zeta = -1.0 if zexp & 1 else 1.0
                        I16 = A_ket if Ob is None else Ob @ A_ket          # Eq. (16)
                        I17 = A_bra.T @ I16                                # Eq. (17)
                        acc += (coef * zeta * oc) * I17                    # Eq. (18)
                        hit = True
            if hit:
                blocks[(rp_, r)] = acc
        result.append(blocks)
    return result
