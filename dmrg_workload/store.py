"""Flat arrays handed to `dmrg_ops_load` / `dmrg_plan_create` and to the oracle.

Data model (include/dmrg_sigma.h; PAPER.md:126-141 for the operator store,
PAPER.md:95-99 for the block-sparse wavefunction):
  sectors  int32 [nsec,3]  (N, 2Sz, dim)                       per side
  ops      int32 [nops,8]  (side, kind, p, q, dN, d2Sz, first_block, nblocks)
  blocks   int64 [nblk,3]  (row_sector, col_sector, offset); dense row-major
           dim[row] x dim[col], row sector = col sector + charge
  values   float64 [nvalues]
  lincomb  CSR (lin_ptr, lin_op, lin_coef): op of kind LINCOMB number j is
           sum_i lin_coef[i] * ops[lin_op[i]],  lin_ptr[j] <= i < lin_ptr[j+1]
  site_ops float64 [nsite,16] row-major 4x4, site_parity int32 [nsite]
  terms    (coef f64; op_l, trans_l, dot1, dot2, op_r, trans_r int32)
"""
import numpy as np

from .conventions import SITE_Q, spin_of

KIND = {"H": 0, "C": 1, "A": 2, "B": 3, "P": 4, "Q": 5, "S": 6, "LIN": 7}


def op_charge(op, sym="NSz"):
    """(dN, d2Sz) of a stored operator; sym "N": only dN, d2Sz = 0."""
    if sym == "N":
        return (op_charge(op)[0], 0)
    k = op.kind
    if k == "H":
        return (0, 0)
    if k == "C":
        return (1, spin_of(op.p))
    if k == "A":
        return (2, spin_of(op.p) + spin_of(op.q))
    if k == "B":
        return (0, spin_of(op.p) - spin_of(op.q))
    if k == "P":
        return (-2, -spin_of(op.p) - spin_of(op.q))
    if k == "Q":
        return (0, spin_of(op.q) - spin_of(op.p))
    if k == "S":
        return (-1, -spin_of(op.p))
    raise ValueError(k)


class Problem:
    """Everything one bond needs: store arrays, terms, psi layout."""

    def __init__(self):
        self.secL = self.secR = None
        self.ops = None
        self.blocks = None
        self.values = None
        self.lin_ptr = self.lin_op = self.lin_coef = None
        self.site_ops = self.site_parity = None
        self.term_coef = self.term_idx = None
        self.N_tot = self.twoSz_tot = 0
        self.sym, self.dtype = "NSz", np.dtype(np.float64)   # "N" / complex128 for spin-orbit problems (psi_size counts complex numbers then)
        self.layout = None
        self.psi_size = 0
        self.meta = {}


def _op_sort_key(op):
    return (0 if op.side == "L" else 1, KIND[op.kind], op.p, op.q)


def _fill_normal(out, seed, nthreads=None):
    """out[:] ~ N(0,1), reproducible for a given (seed, len(out)) whatever the thread count:
    the array is cut into fixed 16 Mi-double pieces, piece i drawn from Philox(key=seed, counter block i)."""
    import os
    from concurrent.futures import ThreadPoolExecutor
    piece = 1 << 24
    n = out.shape[0]
    npieces = (n + piece - 1) // piece

    def work(i):
        g = np.random.Generator(np.random.Philox(key=seed, counter=[0, 0, 0, i + 1]))
        g.standard_normal(out=out[i * piece:min(n, (i + 1) * piece)])

    nthreads = nthreads or min(32, os.cpu_count() or 1)
    if npieces <= 1 or nthreads <= 1:
        for i in range(npieces):
            work(i)
    else:
        with ThreadPoolExecutor(nthreads) as ex:
            list(ex.map(work, range(npieces)))


def assemble(tt, secL, secR, block_values, N_tot, twoSz_tot, direct_seed=None, direct_scale=1.0):
    """Build a Problem from a TermTable.

    block_values(op, row_sector, col_sector, shape) -> ndarray or None (block absent);
    called for every stored (non-LINCOMB) op and every charge-allowed sector pair.
    block_values=None ("direct fill", cfg 3-5): every charge-allowed block is present and filled with
    seeded N(0, direct_scale^2) entries; H, B_pp and Q_pp blocks are symmetrised so that the summed
    operator stays Hermitian (the term table adds no h.c. for those)."""
    from .sectors import psi_layout
    from .terms import BlockOp, dot_parity
    sym = getattr(tt.ints, "sym", "NSz")
    dtype = np.dtype(getattr(tt.ints, "dtype", np.float64))
    pr = Problem()
    pr.sym, pr.dtype = sym, dtype
    pr.N_tot, pr.twoSz_tot = N_tot, twoSz_tot
    pr.secL = np.array(secL, dtype=np.int32).reshape(-1, 3)
    pr.secR = np.array(secR, dtype=np.int32).reshape(-1, 3)
    secs = {"L": secL, "R": secR}
    sidx = {s: {(q[0], q[1]): i for i, q in enumerate(secs[s])} for s in "LR"}
    ref = tt.referenced_ops()
    stored = sorted([o for s in "LR" for o in ref[s] if o.kind != "LIN"], key=_op_sort_key)
    op_id = {}
    ops_rows, blk_rows, vals = [], [], []
    sym_blocks = []   # direct fill: (offset, d) of square blocks to symmetrise
    off = 0
    for op in stored:
        dq = op_charge(op, sym)
        first = len(blk_rows)
        sl = secs[op.side]
        self_adjoint = op.kind == "H" or (op.kind in ("B", "Q") and op.p == op.q)
        for ic, qc in enumerate(sl):
            ir = sidx[op.side].get((qc[0] + dq[0], qc[1] + dq[1]))
            if ir is None:
                continue
            shape = (sl[ir][2], qc[2])
            if block_values is not None:
                m = block_values(op, ir, ic, shape)
                if m is None:
                    continue
                assert m.shape == shape
                vals.append(np.ascontiguousarray(m, dtype=dtype).ravel())
            elif self_adjoint:
                assert ir == ic
                sym_blocks.append((off, shape[0]))
            blk_rows.append((ir, ic, off))
            off += shape[0] * shape[1]
        op_id[op] = len(ops_rows)
        ops_rows.append((0 if op.side == "L" else 1, KIND[op.kind], op.p, op.q, dq[0], dq[1],
                         first, len(blk_rows) - first))
    if block_values is None and direct_seed is None:
        values = None   # structure only (sizing / planning without the 8-byte-per-element store)
    elif block_values is None:
        if dtype.kind == "c":   # real and imaginary parts N(0, 1/2) each: |entry|^2 has mean 1 as in the real fill
            raw = np.empty(2 * off, dtype=np.float64)
            _fill_normal(raw, int(direct_seed))
            raw *= direct_scale * np.sqrt(0.5)
            values = raw.view(np.complex128)
        else:
            values = np.empty(off, dtype=np.float64)
            _fill_normal(values, int(direct_seed))
            if direct_scale != 1.0:
                values *= direct_scale
        for o, d in sym_blocks:
            m = values[o:o + d * d].reshape(d, d)
            m[:] = (m + m.conj().T) * 0.5
    lin_ptr, lin_op, lin_coef = [0], [], []
    for side in "LR":
        for j, lc in enumerate(tt.lincombs[side]):
            op = BlockOp(side, "LIN", j, -1)
            charges = {op_charge(BlockOp(side, "C", lab, -1), sym) for lab, _ in lc}
            assert len(charges) == 1, "lincomb mixes charges"
            dq = charges.pop()
            op_id[op] = len(ops_rows)
            ops_rows.append((0 if side == "L" else 1, KIND["LIN"], len(lin_ptr) - 1, -1, dq[0], dq[1], 0, 0))
            for lab, cf in lc:
                lin_op.append(op_id[BlockOp(side, "C", lab, -1)])
                lin_coef.append(cf)
            lin_ptr.append(len(lin_op))
    pr.ops = np.array(ops_rows, dtype=np.int64).reshape(-1, 8)
    pr.blocks = np.array(blk_rows, dtype=np.int64).reshape(-1, 3)
    if block_values is not None:
        values = np.concatenate(vals) if vals else np.zeros(0, dtype=dtype)
    pr.values = values
    pr.lin_ptr = np.array(lin_ptr, dtype=np.int64)
    pr.lin_op = np.array(lin_op, dtype=np.int32)
    pr.lin_coef = np.array(lin_coef, dtype=dtype)
    # site operators, deduplicated by value
    site_index, site_ops, site_par = {}, [], []

    def site_id(m):
        m = np.ascontiguousarray(m, dtype=dtype)
        key = m.tobytes()
        if key not in site_index:
            site_index[key] = len(site_ops)
            site_ops.append(m.ravel().copy())
            site_par.append(dot_parity(m))
        return site_index[key]

    site_id(np.eye(4, dtype=dtype))
    coefs, idx = [], []
    for coef, Ls, c, d, Rs in tt.terms:
        ol, tl = (-1, 0) if Ls is None else (op_id[Ls[0]], int(Ls[1]))
        orr, trr = (-1, 0) if Rs is None else (op_id[Rs[0]], int(Rs[1]))
        coefs.append(coef)
        idx.append((ol, tl, site_id(c), site_id(d), orr, trr))
    pr.term_coef = np.array(coefs, dtype=dtype)
    pr.term_idx = np.array(idx, dtype=np.int32).reshape(-1, 6)
    pr.site_ops = np.array(site_ops, dtype=dtype).reshape(-1, 16)
    pr.site_parity = np.array(site_par, dtype=np.int32)
    pr.layout, pr.psi_size = psi_layout(secL, secR, N_tot, twoSz_tot, sym)
    pr.op_id = op_id
    pr.stored_ops = stored
    return pr


def block_values_from_rblocks(blkL, blkR, ints):
    """block_values callback serving honest renormalized blocks (blocking.py)."""
    cache = {}

    def get(op):
        if op in cache:
            return cache[op]
        b = blkL if op.side == "L" else blkR
        k = op.kind
        if k == "H":
            d = b.ops[("H",)]
        elif k == "C":
            d = b.ops[("C", op.p)]
        elif k == "A":
            d = b.ops[("A", op.p, op.q)]
        elif k == "B":
            d = b.ops[("B", op.p, op.q)]
        elif k == "S":
            d = b.ops[("S", op.p)]
        elif k == "P":
            d = b.compl_P(op.p, op.q, ints)
        elif k == "Q":
            d = b.compl_Q(op.p, op.q, ints)
        else:
            raise ValueError(k)
        cache.clear()
        cache[op] = d
        return d

    def fn(op, ir, ic, shape):
        m = get(op).get((ir, ic))
        return m

    return fn


def sectors_of(blk):
    return [(q[0], q[1], d) for q, d in zip(blk.sectors, blk.dims)]
