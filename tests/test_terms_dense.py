"""Pin of the term table (reading 2) against the definition of H (Eq. 2,
PAPER.md:43) in the full Fock space at tiny K: sum_mu zeta O^L O^C1 O^C2 O^R == H."""
import numpy as np
import pytest
import scipy.sparse as sp

import fockdense as fd
from dmrg_workload.integrals import make_integrals, make_so_integrals
from dmrg_workload.terms import Partition, TermTable, block_parity, dot_parity


def slot_matrix(slot, blk, lincombs):
    if slot is None:
        return sp.identity(blk.dim, format="csr")
    op, tr = slot
    if op.kind == "LIN":
        m = blk.op("LIN", lin=lincombs[op.side][op.p])
    else:
        m = blk.op(op.kind, op.p, op.q)
    return m.conj().T.tocsr() if tr else m   # a transposed use is the Hermitian conjugate (terms.py)


@pytest.mark.parametrize("K,nL,spin_orbit", [(4, 1, False), (5, 2, False), (5, 1, False), (6, 2, False),
                                             (4, 1, True), (5, 2, True), (5, 1, True)])
def test_term_table_reproduces_H(K, nL, spin_orbit):
    """spin_orbit: complex Hermitian integrals without spin selection rules -- the same table with
    every transposed use read as a Hermitian conjugate."""
    ints = (make_so_integrals if spin_orbit else make_integrals)(K, seed=100 + K + nL)
    part = Partition(K, nL)
    tt = TermTable(part, ints)
    bL, bR = fd.DenseBlock(part.L, ints), fd.DenseBlock(part.R, ints)
    ZL, ZR = fd.block_Z(part.L), fd.block_Z(part.R)
    Zs = fd.block_Z([0, 1])
    dim = bL.dim * 16 * bR.dim
    Hsum = sp.csr_matrix((dim, dim))
    for coef, Ls, c, d, Rs in tt.terms:
        mL = slot_matrix(Ls, bL, tt.lincombs)
        mR = slot_matrix(Rs, bR, tt.lincombs)
        pc, pd, pR = dot_parity(c), dot_parity(d), block_parity(Rs)
        # zeta: odd operator in a slot picks (-1)^(N of all slots to its left), ket side
        if (pc + pd + pR) % 2:
            mL = mL @ ZL
        mc = sp.csr_matrix(c)
        if (pd + pR) % 2:
            mc = mc @ Zs
        md = sp.csr_matrix(d)
        if pR % 2:
            md = md @ Zs
        Hsum = Hsum + coef * sp.kron(sp.kron(mL, mc), sp.kron(md, mR), format="csr")
    a = fd.full_annihilators(K)
    Href = fd.hamiltonian(a, ints, dim)
    diff = abs(Hsum - Href).max()
    assert diff < 1e-12, diff
    assert abs(Href - Href.conj().T).max() < 1e-12
    if spin_orbit:   # the coupling is really there: H is complex and does not commute with Sz
        assert abs(Href.imag).max() > 1e-3
        Sz = sum(0.5 * (1 if P % 2 == 0 else -1) * (a[P].T @ a[P]) for P in a)
        assert abs(Href @ Sz - Sz @ Href).max() > 1e-3
