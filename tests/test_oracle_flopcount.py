"""Pin of the oracle's cost counter (oracle.opair_sigma(return_stats=True)["flops"], oracle.opair_count) against a
HAND count on a two-term toy bond.  The cost measure is the paper's: a GEMM (M,K)(K,N) costs 2MNK
(Table 1 caption); per task 2 dLi dRi dRo for X = psi R^T (Eq. 11) if the R factor is
not the identity, + 2 dLo dLi dRo for L X (Eq. 12) if the L factor is not the identity.

Toy bond, target (N, 2Sz) = (2, 0):
  L sectors  0: (0, 0) dim 2     1: (1,+1) dim 3
  R sectors  0: (1,-1) dim 4     1: (2, 0) dim 5     2: (0, 0) dim 6
  site states 0 vac (0,0), 1 beta (1,-1), 2 alpha (1,+1), 3 alpha-beta (2,0)
  psi blocks (iL, c1, c2, iR) whose charges add up to (2, 0)  -- ten of them:
      iL = 0: (0,0,0,1) 2x5; (0,2,0,0), (0,0,2,0) 2x4; (0,3,0,2), (0,0,3,2), (0,1,2,2), (0,2,1,2) 2x6
      iL = 1: (1,0,0,0) 3x4; (1,1,0,2), (1,0,1,2) 3x6
  term 1:  L op of charge (+1,+1) (one block, row 1 <- col 0, 3x2) x 1 x 1 x R op of charge (-1,-1) (one block,
           row 0 <- col 1, 4x5).  Acts on psi blocks with iL = 0 and iR = 1: only (0,0,0,1), 2x5 -> out (1,0,0,0), 3x4:
             stage 1: 2 * dLi * dRi * dRo = 2*2*5*4 = 80      stage 2: 2 * dLo * dLi * dRo = 2*3*2*4 = 48     -> 128
  term 2:  identity on L x dot-1 operator diag(0,0,1,1) x 1 x R op of charge (0,0), blocks 4x4, 5x5, 6x6, used
           TRANSPOSED.  Acts on psi blocks with c1 in {2, 3}: (0,2,0,0) 2x4: 2*2*4*4 = 64; (0,3,0,2) 2x6: 2*2*6*6 = 144;
           (0,2,1,2) 2x6: 144; the identity L factor costs nothing                                          -> 352
  total: 4 tasks, 480 flops; restricted to the output block (1,0,0,0): 1 task, 128 flops.
"""
import numpy as np

import oracle
from dmrg_workload.sectors import psi_layout
from dmrg_workload.store import Problem


def toy_problem():
    pr = Problem()
    pr.N_tot, pr.twoSz_tot = 2, 0
    pr.secL = np.array([(0, 0, 2), (1, 1, 3)], dtype=np.int32)
    pr.secR = np.array([(1, -1, 4), (2, 0, 5), (0, 0, 6)], dtype=np.int32)
    # ops: (side, kind, p, q, dN, d2Sz, first_block, nblocks)
    pr.ops = np.array([(0, 1, 0, -1, 1, 1, 0, 1),        # L: a+-like, charge (+1,+1)
                       (1, 6, 0, -1, -1, -1, 1, 1),      # R: S-like, charge (-1,-1)
                       (1, 0, -1, -1, 0, 0, 2, 3)],      # R: H-like, charge (0,0)
                      dtype=np.int64)
    # blocks: (row sector, col sector, offset)
    pr.blocks = np.array([(1, 0, 0),                     # 3x2
                          (0, 1, 6),                     # 4x5
                          (0, 0, 26), (1, 1, 42), (2, 2, 67)],   # 4x4, 5x5, 6x6
                         dtype=np.int64)
    rng = np.random.default_rng(0)
    pr.values = rng.standard_normal(6 + 20 + 16 + 25 + 36)
    pr.lin_ptr = np.array([0], dtype=np.int64)
    pr.lin_op = np.zeros(0, dtype=np.int32)
    pr.lin_coef = np.zeros(0)
    pr.site_ops = np.stack([np.eye(4).ravel(), np.diag([0.0, 0.0, 1.0, 1.0]).ravel()])
    pr.site_parity = np.array([0, 0], dtype=np.int32)
    pr.term_coef = np.array([0.7, -1.3])
    # terms: (op_l, trans_l, dot1, dot2, op_r, trans_r)
    pr.term_idx = np.array([(0, 0, 0, 0, 1, 0), (-1, 0, 1, 0, 2, 1)], dtype=np.int32)
    pr.layout, pr.psi_size = psi_layout([tuple(s) for s in pr.secL], [tuple(s) for s in pr.secR], 2, 0)
    return pr


def test_flop_counter_matches_hand_count():
    pr = toy_problem()
    lay = [tuple(int(v) for v in r[:4]) for r in pr.layout]
    assert len(lay) == 10 and pr.psi_size == 10 + 2 * 8 + 4 * 12 + 12 + 2 * 18
    psi = np.random.default_rng(1).standard_normal(pr.psi_size)
    sig, st = oracle.opair_sigma(pr, psi, return_stats=True)
    assert st == {"tasks": 4, "flops": 480.0}
    assert oracle.opair_count(pr) == {"tasks": 4, "flops": 480.0}
    ob = lay.index((1, 0, 0, 0))
    assert oracle.opair_count(pr, only_out=[ob]) == {"tasks": 1, "flops": 128.0}
    _, st1 = oracle.opair_sigma(pr, psi, only_out=[ob], return_stats=True)
    assert st1 == {"tasks": 1, "flops": 128.0}
    # the counted work is the work done: exactly the blocks the hand count names are non-zero
    touched = {lay.index(b) for b in [(1, 0, 0, 0), (0, 2, 0, 0), (0, 3, 0, 2), (0, 2, 1, 2)]}
    for b, row in enumerate(pr.layout):
        o, n = int(row[6]), int(row[4] * row[5])
        assert (np.abs(sig[o:o + n]).max() > 0) == (b in touched)
    # and the values: term 1 by its formula, sigma[(1,0,0,0)] = 0.7 * zeta * L (psi R^T), zeta = +1 for N_l = 0
    Lb = pr.values[0:6].reshape(3, 2)
    Rb = pr.values[6:26].reshape(4, 5)
    i_in, i_out = lay.index((0, 0, 0, 1)), lay.index((1, 0, 0, 0))
    x = psi[int(pr.layout[i_in][6]):][:10].reshape(2, 5)
    want = 0.7 * Lb @ (x @ Rb.T)
    got = sig[int(pr.layout[i_out][6]):][:12].reshape(3, 4)
    assert np.abs(got - want).max() < 1e-14


def test_count_needs_no_values_and_matches_sigma_on_a_real_bond():
    from dmrg_workload.problem import make_direct_problem, random_psi
    pr = make_direct_problem(12, 5, 12, 0, D=60, seed=4)
    _, st = oracle.opair_sigma(pr, random_psi(pr.psi_size, 1), return_stats=True)
    assert oracle.opair_count(pr) == st
    pr0 = make_direct_problem(12, 5, 12, 0, D=60, seed=4, structure_only=True)
    assert pr0.values is None and oracle.opair_count(pr0) == st
