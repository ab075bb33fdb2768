"""Builds the operator store of one two-dot bond ON THE DEVICE by a chain of renormalization steps.

The paper's sweep produces the operators of a bond by renormalizing those of the previous one (Eq. 8;
Fig. 1a).  `build_bond` does that from both chain ends with seeded random site tensors
(dmrg_workload/site_tensor.py): every step is one dmrg_renormalize call, the complementary operators needed along
the way and at the bond are linear combinations formed on the device (dmrg_ops_add_lincombs / dmrg_ops_derive,
Eqs. 22-23), and the two blocks are joined without a copy (dmrg_ops_join).  This module only
marshals: term lists and coefficient tables come from dmrg_workload (symbolic), all arithmetic runs in libdmrg_sigma.
It is what replaces the direct-fill operators of cfg 3-5 by physical ones (SURVEY.md section 8(d) option (ii)).
"""
import time

import numpy as np

from dmrg_workload import blocking
from dmrg_workload.conventions import SITE_Q
from dmrg_workload.renorm_terms import BlockShape, build_renorm_problem, carried_keys, compl_P_items, compl_Q_items
from dmrg_workload.sectors import psi_layout
from dmrg_workload.site_tensor import random_site_tensor
from dmrg_workload.store import KIND, op_charge
from dmrg_workload.terms import BlockOp, Partition, TermTable, dot_parity

_KEY_KIND = {v: k for k, v in KIND.items()}


def _key_of_row(row):
    """RBlock key of an exported / declared operator row (side, kind, p, q, ...)."""
    kind = _KEY_KIND[int(row[1])]
    if kind == "H":
        return ("H",)
    if kind in ("C", "S"):
        return (kind, int(row[2]))
    return (kind, int(row[2]), int(row[3]))


def _blockop_key(op):
    if op.kind == "H":
        return ("H",)
    if op.kind in ("C", "S"):
        return (op.kind, op.p)
    return (op.kind, op.p, op.q)


def grow_block(g, side, sites, ints, K, N_tot, twoSz_tot, D, rng, tensor_provider=None, stream=None, workspace_bytes=0, log=None):
    """Grow a block over `sites` (ascending list of spatial orbitals; side 0 appends sites on the right, side 1 prepends
    them on the left, starting from the far end).  Returns (store, shape, key->op id, stats)."""
    order = list(sites) if side == 0 else list(sites)[::-1]
    sname = "L" if side == 0 else "R"
    inside = [order[0]]
    site0 = blocking.site_block(order[0], ints, [P for P in range(2 * K) if (P >> 1) != order[0]])
    shape = BlockShape(site0.labels, site0.sectors, site0.dims, list(site0.ops))
    store, ids = None, None
    stats = []
    for k in order[1:]:
        inside.append(k)
        outside = [P for P in range(2 * K) if (P >> 1) not in inside]
        labels_new = sorted(list(shape.labels) + [2 * k, 2 * k + 1])
        if tensor_provider is not None:
            new_secs, new_dims, tensor = tensor_provider(side, k)
        else:
            new_secs, new_dims, tensor = random_site_tensor(shape.sectors, shape.dims, side, len(inside), K, N_tot, twoSz_tot, D, rng)
        new_shape = BlockShape(labels_new, new_secs, new_dims, carried_keys(labels_new, outside))
        new_shape.site_tensor = tensor
        if store is None:
            # first step: the single-site block comes from the host with its values (4 states)
            rp = build_renorm_problem(site0, k, side, ints, outside, new_shape)
            empty = np.zeros((0, 3), dtype=np.int32)
            secL, secR = (rp.sec_old, empty) if side == 0 else (empty, rp.sec_old)
            store = g.OpsStore(secL, secR, rp.ops, rp.blocks, rp.values, rp.lin_ptr, rp.lin_op, rp.lin_coef)
            term_idx = rp.term_idx
        else:
            rp = build_renorm_problem(shape, k, side, ints, outside, new_shape, structure_only=True)
            nst = int(np.sum(rp.ops[:, 1] != KIND["LIN"]))
            perm = [ids[_key_of_row(r)] for r in rp.ops[:nst]]
            remap = {i: perm[i] for i in range(nst)}
            if len(rp.ops) > nst:
                lin_op = np.array([perm[o] for o in rp.lin_op], dtype=np.int32)
                first = store.add_lincombs(rp.ops[nst:], rp.lin_ptr, lin_op, rp.lin_coef)
                remap.update({nst + j: first + j for j in range(len(rp.ops) - nst)})
            term_idx = rp.term_idx.copy()
            term_idx[:, 0] = [remap[int(o)] if o >= 0 else -1 for o in term_idx[:, 0]]
        out, st = g.renormalize(store, side, rp.sec_new, rp.wblocks, rp.wvalues, rp.new_ops, rp.term_ptr, rp.term_coef, term_idx,
                                rp.site_ops, rp.site_parity, workspace_bytes=workspace_bytes, stream=stream)
        store.free()
        store = out
        ids = {key: i for i, key in enumerate(rp.new_keys)}
        shape = new_shape
        st.update(site=k, side=side, nops=len(rp.new_keys), dim=int(sum(new_dims)))
        stats.append(st)
        if log:
            log(f"  {sname} +site {k}: {len(rp.new_keys)} ops, sum d = {sum(new_dims)}, {st['flops']:.2e} flop, {st['device_ms']:.1f} ms")
    return store, shape, ids, stats


class Bond:
    """What dmrg_plan_create needs, plus the arrays that describe the problem (formats of dmrg_workload/store.py)."""


def build_bond(g, K, nL, N_tot, twoSz_tot, D, ints, seed, tensor_provider=None, stream=None, workspace_bytes=0, log=None):
    """Two-dot bond nL-1-1-(K-nL-2): renormalized L and R blocks, complementary operators, term table.
    Returns a Bond with .ops (two-sided device store), term arrays, sector tables, layout."""
    t0 = time.perf_counter()
    rng = np.random.Generator(np.random.Philox(seed + 7919))
    part = Partition(K, nL)
    L, shL, idL, stL = grow_block(g, 0, list(range(0, nL)), ints, K, N_tot, twoSz_tot, D, rng, tensor_provider, stream, workspace_bytes, log)
    R, shR, idR, stR = grow_block(g, 1, list(range(nL + 2, K)), ints, K, N_tot, twoSz_tot, D, rng, tensor_provider, stream, workspace_bytes, log)
    t_chain = time.perf_counter() - t0
    tt = TermTable(part, ints)
    ref = tt.referenced_ops()
    # ---- L: thin complementary operators P^L, Q^L appended as linear combinations of A^L, B^L ---------------
    def lin_tables(side_name, needed, ids, X, side):
        rows, ptr, lop, lco, ltr = [], [0], [], [], []
        for op in needed:
            dq = op_charge(op)
            items = compl_P_items(X, op.p, op.q, ints, side_name) if op.kind == "P" else compl_Q_items(X, op.p, op.q, ints, side_name)
            rows.append((side, KIND[op.kind], op.p, op.q, dq[0], dq[1], 0, 0))
            for bop, c, tr in items:
                lop.append(ids[_blockop_key(bop)])
                lco.append(c)
                ltr.append(tr)
            ptr.append(len(lop))
        return rows, ptr, lop, lco, ltr

    op_id = {}
    needL = sorted([o for o in ref["L"] if o.kind in ("P", "Q")], key=lambda o: (KIND[o.kind], o.p, o.q))
    for o in ref["L"]:
        if o.kind not in ("P", "Q", "LIN"):
            op_id[o] = idL[_blockop_key(o)]
    if needL:
        rows, ptr, lop, lco, ltr = lin_tables("L", needL, idL, shL.labels, 0)
        for j, r in enumerate(rows):
            rows[j] = r[:2] + (j,) + r[3:]      # p column = row of lin_ptr (labels are kept in op_id only)
        first = L.add_lincombs(np.array(rows, dtype=np.int64), ptr, lop, lco, ltr)
        for j, o in enumerate(needL):
            op_id[o] = first + j
    nL_ops = L.num_ops
    # ---- R: a new store with exactly the operators the terms use: a+, S, H copied, P, Q formed from A^R, B^R --
    needR = sorted([o for o in ref["R"] if o.kind != "LIN"], key=lambda o: (KIND[o.kind], o.p, o.q))
    rows, ptr, lop, lco, ltr = [], [0], [], [], []
    for j, op in enumerate(needR):
        dq = op_charge(op)
        rows.append((1, KIND[op.kind], j, op.q, dq[0], dq[1], 0, 0))
        if op.kind in ("P", "Q"):
            items = compl_P_items(shR.labels, op.p, op.q, ints, "R") if op.kind == "P" else compl_Q_items(shR.labels, op.p, op.q, ints, "R")
            for bop, c, tr in items:
                lop.append(idR[_blockop_key(bop)])
                lco.append(c)
                ltr.append(tr)
        else:
            lop.append(idR[_blockop_key(op)])
            lco.append(1.0)
            ltr.append(0)
        ptr.append(len(lop))
    Rd = R.derive(np.array(rows, dtype=np.int64), ptr, lop, lco, ltr)
    R.free()
    for j, o in enumerate(needR):
        op_id[o] = nL_ops + j
    ops = g.OpsStore.join(L, Rd)
    # ---- the term table's own linear combinations (sums of a+ on one block) -------------------
    rows, ptr, lop, lco = [], [0], [], []
    lin_ops = []
    for side_name, side in (("L", 0), ("R", 1)):
        for j, lc in enumerate(tt.lincombs[side_name]):
            charges = {op_charge(BlockOp(side_name, "C", lab, -1)) for lab, _ in lc}
            assert len(charges) == 1
            dq = charges.pop()
            rows.append((side, KIND["LIN"], len(ptr) - 1, -1, dq[0], dq[1], 0, 0))
            for lab, cf in lc:
                lop.append(op_id[BlockOp(side_name, "C", lab, -1)])
                lco.append(cf)
            ptr.append(len(lop))
            lin_ops.append(BlockOp(side_name, "LIN", j, -1))
    if rows:
        first = ops.add_lincombs(np.array(rows, dtype=np.int64), ptr, lop, lco)
        for j, o in enumerate(lin_ops):
            op_id[o] = first + j
    # ---- terms ----------------------------------------------------------------------------------------------
    site_index, site_ops, site_par = {}, [], []

    def site_id(m):
        key = m.tobytes()
        if key not in site_index:
            site_index[key] = len(site_ops)
            site_ops.append(m.ravel().copy())
            site_par.append(dot_parity(m))
        return site_index[key]

    site_id(np.eye(4))
    coefs, idx = [], []
    for coef, Ls, c, d, Rs in tt.terms:
        ol, tl = (-1, 0) if Ls is None else (op_id[Ls[0]], int(Ls[1]))
        orr, trr = (-1, 0) if Rs is None else (op_id[Rs[0]], int(Rs[1]))
        coefs.append(coef)
        idx.append((ol, tl, site_id(c), site_id(d), orr, trr))
    b = Bond()
    b.ops = ops
    b.secL = np.array([(q[0], q[1], d) for q, d in zip(shL.sectors, shL.dims)], dtype=np.int32).reshape(-1, 3)
    b.secR = np.array([(q[0], q[1], d) for q, d in zip(shR.sectors, shR.dims)], dtype=np.int32).reshape(-1, 3)
    b.term_coef = np.array(coefs, dtype=np.float64)
    b.term_idx = np.array(idx, dtype=np.int32).reshape(-1, 6)
    b.site_ops = np.array(site_ops, dtype=np.float64).reshape(-1, 16)
    b.site_parity = np.array(site_par, dtype=np.int32)
    b.N_tot, b.twoSz_tot = N_tot, twoSz_tot
    b.layout, b.psi_size = psi_layout([tuple(s) for s in b.secL], [tuple(s) for s in b.secR], N_tot, twoSz_tot)
    b.renorm_stats = stL + stR
    b.seconds = {"chains": t_chain, "total": time.perf_counter() - t0}
    b.meta = dict(K=K, nL=nL, nR=K - nL - 2, D=D, seed=seed, mode="GPU-renormalized")
    return b
