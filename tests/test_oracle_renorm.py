"""Pins of the renormalization oracle (oracle/renorm.py; Eq. 8, Eqs. 15-18).

(a) DEFINITION pin: chains of renormalization steps at tiny K with seeded random truncating / rotating isometries;
    every operator the oracle produces must equal E^T O_def E, where O_def is the operator of Eqs. (20)-(24)
     built by brute-force second quantisation in the block's Fock space (tests/fockdense.py,
    independent of oracle/) and E is the accumulated isometry from determinants to kept states.  A wrong zeta, a
    wrong h.c. sign, a transposed factor or a dropped term of the recursions fails it.
(b) the same numbers from the generator's own enlarge-and-project code (dmrg_workload/blocking.py, dense Kronecker
    products): two independent formulations of Eq. (8) must agree to rounding.
(c) invariants: an identity site tensor on an untruncated block reproduces the enlarged operators' spectra
    (H symmetric, B_pp symmetric), and the step is linear in the old operators.
"""
import numpy as np
import pytest

import fockdense as fd
from dmrg_workload import blocking
from dmrg_workload.integrals import make_integrals
from dmrg_workload.renorm_terms import build_renorm_problem
from oracle import renorm as oracle_renorm


def chain(side, sites, ints, K, N_tot, D, seed, rotate):
    """Yield (old block, site k, outside labels, new block) for every step of growing a block over `sites`."""
    rng = np.random.Generator(np.random.Philox(seed))
    order = list(sites) if side == 0 else list(sites)[::-1]
    inside, blk = [], None
    for k in order:
        inside.append(k)
        outside = [P for P in range(2 * K) if (P >> 1) not in inside]
        site = blocking.site_block(k, ints, [P for P in range(2 * K) if (P >> 1) != k])
        if blk is None:
            blk = site
            continue
        if side == 0:
            nb = blocking.merge(blk, site, ints, outside, K, N_tot, 0, D, rng, rotate, False, site_side="right", track=True)
        else:
            nb = blocking.merge(site, blk, ints, outside, K, N_tot, 0, D, rng, rotate, False, site_side="left", track=True)
        yield blk, k, outside, nb
        blk = nb


def kron_index(det, labels):
    sites = sorted({P >> 1 for P in labels})
    idx = 0
    for k in sites:
        idx = idx * 4 + 2 * ((det >> (2 * k)) & 1) + ((det >> (2 * k + 1)) & 1)
    return idx


def definition_blocks(nb, ints, key):
    """{(row sector, col sector): E^T O_def E} from the definitions of Eqs. (20)-(24)."""
    dense = fd.DenseBlock(sorted(nb.labels), ints)
    kind = key[0]
    O = dense.op(kind, *(key[1:] + (-1, -1))[:2]).toarray()
    idx = {s: np.array([kron_index(d, nb.labels) for d in nb.dets[s]]) for s in range(len(nb.sectors))}
    out = {}
    for r in range(len(nb.sectors)):
        for c in range(len(nb.sectors)):
            m = nb.E[r].T @ O[np.ix_(idx[r], idx[c])] @ nb.E[c]
            if np.abs(m).max() > 0:
                out[(r, c)] = m
    return out


def max_diff(a, b):
    d = 0.0
    for key in set(a) | set(b):
        x, y = a.get(key), b.get(key)
        if x is None:
            d = max(d, float(np.abs(y).max()))
        elif y is None:
            d = max(d, float(np.abs(x).max()))
        else:
            d = max(d, float(np.abs(x - y).max()))
    return d


@pytest.mark.parametrize("side,sites,K,N,D,rot,seed", [
    (0, [0, 1, 2], 5, 6, 9, False, 3),       # left block, truncated
    (0, [0, 1, 2], 5, 4, None, True, 4),     # left block, rotated, untruncated
    (1, [2, 3, 4], 5, 6, 9, False, 5),       # right block (site x block), truncated
    (1, [3, 4, 5], 6, 6, 7, True, 6),        # right block, rotated and truncated
    (0, [0, 1, 2, 3], 6, 6, 12, False, 7),   # three steps
])
def test_every_renormalized_operator_matches_its_definition(side, sites, K, N, D, rot, seed):
    ints = make_integrals(K, seed=seed)
    nsteps = 0
    for blk, k, outside, nb in chain(side, sites, ints, K, N, D, seed, rot):
        rp = build_renorm_problem(blk, k, side, ints, outside, nb)
        out = oracle_renorm.renormalize(rp)
        assert len(out) == len(rp.new_keys) == len(nb.ops)
        for key, got in zip(rp.new_keys, out):
            ref = definition_blocks(nb, ints, key)
            assert max_diff(got, ref) < 1e-12, (key, nsteps)                 # (a) the definition
            assert max_diff(got, nb.ops[key]) < 1e-12, (key, nsteps)         # (b) the generator's dense formulation
        nsteps += 1
    assert nsteps == len(sites) - 1


def test_zeta_matters_and_linearity():
    """A step without the Jordan-Wigner factor must NOT reproduce the definition (the pin can see a wrong zeta), and
    the renormalized operators are linear in the old block's operator values."""
    K, N = 5, 6
    ints = make_integrals(K, seed=9)
    blk, k, outside, nb = list(chain(0, [0, 1, 2], ints, K, N, 9, 11, False))[-1]
    rp = build_renorm_problem(blk, k, 0, ints, outside, nb)
    out = oracle_renorm.renormalize(rp)
    iA = next(i for i, key in enumerate(rp.new_keys) if key[0] == "A" and (key[1] >> 1) != k and (key[2] >> 1) == k)
    par = rp.site_parity.copy()
    rp.site_parity = np.zeros_like(par)                     # kill zeta
    bad = oracle_renorm.renormalize(rp)
    rp.site_parity = par
    assert max_diff(bad[iA], out[iA]) > 1e-3
    vals = rp.values.copy()
    rp.values = 2.5 * vals
    scaled = oracle_renorm.renormalize(rp)
    rp.values = vals
    iB = next(i for i, key in enumerate(rp.new_keys) if key[0] == "B" and (key[1] >> 1) != k and (key[2] >> 1) != k)
    assert max_diff(scaled[iB], {kk: 2.5 * v for kk, v in out[iB].items()}) < 1e-13


def test_structure_of_a_step():
    """H and B_pp come out symmetric, charges are respected, and the new sector table is what the site tensor spans."""
    K, N = 6, 6
    ints = make_integrals(K, seed=2)
    blk, k, outside, nb = list(chain(1, [3, 4, 5], ints, K, N, 8, 1, True))[-1]
    rp = build_renorm_problem(blk, k, 1, ints, outside, nb)
    out = oracle_renorm.renormalize(rp)
    sec = rp.sec_new
    for key, row, blocks in zip(rp.new_keys, rp.new_ops, out):
        for (r, c), m in blocks.items():
            assert (sec[c][0] + row[4], sec[c][1] + row[5]) == (sec[r][0], sec[r][1]), key
            assert m.shape == (sec[r][2], sec[c][2])
        if key[0] == "H" or (key[0] == "B" and key[1] == key[2]):
            for (r, c), m in blocks.items():
                assert r == c and np.abs(m - m.T).max() < 1e-13, key
    assert {int(w[2]) for w in rp.wblocks} == set(range(len(sec)))
