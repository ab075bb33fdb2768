"""Seeded problem instances: the five BASELINE.json configs and tiny pin cases."""
import numpy as np

from .blocking import build_block
from .integrals import make_integrals, make_so_integrals
from .sectors import block_sector_model
from .store import assemble, block_values_from_rblocks, sectors_of
from .terms import Partition, TermTable


def random_psi(n, seed):
    rng = np.random.Generator(np.random.Philox(seed))
    x = rng.standard_normal(n)
    return x / np.linalg.norm(x)


def random_psi_z(n, seed):
    """Complex start vector for the spin-orbit problems: n complex numbers, unit 2-norm."""
    rng = np.random.Generator(np.random.Philox(seed))
    x = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    return x / np.linalg.norm(x)


def make_blocked_problem(K, nL, N_tot, twoSz_tot=0, D=None, seed=1, banded=False, rotate=False,
                         force_dmax=True, track=False, ints=None):
    """Honest blocking (cfg 1-2, tiny pins): L = orbitals [0,nL), dots nL, nL+1, R = the rest."""
    ints = ints if ints is not None else make_integrals(K, seed, banded=banded)
    part = Partition(K, nL)
    rng = np.random.Generator(np.random.Philox(seed + 7919))
    bL = build_block("L", range(0, nL), ints, K, N_tot, twoSz_tot, D, rng, rotate, force_dmax, track)
    bR = build_block("R", range(nL + 2, K), ints, K, N_tot, twoSz_tot, D, rng, rotate, force_dmax, track)
    if nL == 1 or K - nL - 2 == 1:
        # single-site end blocks keep only sectors that can reach the target
        pass
    tt = TermTable(part, ints)
    pr = assemble(tt, sectors_of(bL), sectors_of(bR), block_values_from_rblocks(bL, bR, ints),
                  N_tot, twoSz_tot)
    pr.meta = dict(K=K, nL=nL, nR=K - nL - 2, D=D, seed=seed, mode="blocking", banded=banded)
    pr.ints, pr.part, pr.bL, pr.bR, pr.tt = ints, part, bL, bR, tt
    return pr


def make_direct_problem(K, nL, N_tot, twoSz_tot=0, D=1000, seed=1, banded=False, ints=None, structure_only=False):
    """Direct fill (cfg 3-5; DESIGN.md input recipe): integrals and the term table are the real ones,
    the sector tables follow the d_max(D) model of sectors.py, and every charge-allowed operator block
    is filled with seeded N(0, 1/d_max) entries (H, B_pp, Q_pp symmetric).  The contraction workload
    (block shapes, term list, coefficients, sparsity) is that of an honest bond at this D; the summed
    operator is Hermitian but is NOT a projected physical Hamiltonian."""
    ints = ints if ints is not None else make_integrals(K, seed, banded=banded)
    part = Partition(K, nL)
    sym = getattr(ints, "sym", "NSz")
    secL = block_sector_model(nL, K, N_tot, twoSz_tot, D, sym)
    secR = block_sector_model(K - nL - 2, K, N_tot, twoSz_tot, D, sym)
    tt = TermTable(part, ints)
    dmax = max(max(s[2] for s in secL), max(s[2] for s in secR))
    pr = assemble(tt, secL, secR, None, N_tot, twoSz_tot, direct_seed=None if structure_only else seed + 104729,
                  direct_scale=dmax ** -0.5)
    pr.meta = dict(K=K, nL=nL, nR=K - nL - 2, D=D, seed=seed, mode="direct", banded=banded)
    if pr.dtype.kind == "c":
        pr.meta["mode"] = "spin-orbit: complex, N only, direct"
    pr.ints, pr.part, pr.tt = ints, part, tt
    return pr


CONFIGS = {
    # BASELINE.json configs[0..4]; partition = centre two-dot (DESIGN.md input recipe)
    "cfg1": dict(gen="blocked", K=8, nL=3, N_tot=8, D=None, seed=1),
    "cfg2": dict(gen="blocked", K=24, nL=11, N_tot=24, D=500, seed=1),
    "cfg3": dict(gen="direct", K=36, nL=17, N_tot=36, D=1500, seed=1),
    "cfg4": dict(gen="direct", K=73, nL=35, N_tot=114, D=1000, seed=1, banded=True),
    "cfg5": dict(gen="direct", K=73, nL=35, N_tot=114, D=3000, seed=1, banded=True),
    # spin-orbit variants (not BASELINE.json configs): complex integrals without spin
    # selection rules (integrals.make_so_integrals), U(1)_N sectors only, direct fill with complex blocks
    "so2": dict(gen="direct", K=24, nL=11, N_tot=24, D=500, seed=1, spin_orbit=True),
    "so3": dict(gen="direct", K=36, nL=17, N_tot=36, D=1500, seed=1, spin_orbit=True),
}


def make_config(name, **over):
    kw = dict(CONFIGS[name])
    kw.update(over)
    gen = kw.pop("gen")
    if kw.pop("spin_orbit", False):
        kw["ints"] = make_so_integrals(kw["K"], kw["seed"], banded=kw.get("banded", False))
    return make_blocked_problem(**kw) if gen == "blocked" else make_direct_problem(**kw)


def term_subset_problem(pr, term_ids):
    """The same bond restricted to a subset of the operator-pair terms (a bounded SAMPLE of the workload for
    timing the oracle): stored operators are shared (no copy), linear-combination operators that no sampled
    term refers to are dropped and the rest renumbered.  No contraction arithmetic here."""
    import copy
    term_ids = np.asarray(term_ids, dtype=np.int64)
    q = copy.copy(pr)
    ti = np.array(pr.term_idx[term_ids], dtype=np.int32)
    ops = np.asarray(pr.ops)
    is_lin = ops[:, 1] == 7
    used = sorted({int(o) for o in ti[:, [0, 4]].ravel() if o >= 0 and is_lin[o]})
    keep = [i for i in range(len(ops)) if not is_lin[i]] + used
    remap = {old: new for new, old in enumerate(keep)}
    new_ops = ops[keep].copy()
    lin_ptr, lin_op, lin_coef = [0], [], []
    for new, old in enumerate(keep):
        if is_lin[old]:
            j = int(ops[old, 2])
            a, b = int(pr.lin_ptr[j]), int(pr.lin_ptr[j + 1])
            new_ops[new, 2] = len(lin_ptr) - 1
            lin_op += [remap[int(o)] for o in pr.lin_op[a:b]]
            lin_coef += list(pr.lin_coef[a:b])
            lin_ptr.append(len(lin_op))
    for col in (0, 4):
        ti[:, col] = [remap[int(o)] if o >= 0 else -1 for o in ti[:, col]]
    q.ops = new_ops
    q.lin_ptr = np.array(lin_ptr, dtype=np.int64)
    q.lin_op = np.array(lin_op, dtype=np.int32)
    q.lin_coef = np.array(lin_coef, dtype=pr.lin_coef.dtype)
    q.term_idx = ti
    q.term_coef = np.array(pr.term_coef[term_ids], dtype=pr.term_coef.dtype)
    return q


def determinant_map(pr):
    """For tracked tiny problems: list over psi blocks of (dets, E) with
    psi_block = E^T-projected determinant coefficients; E = kron(E_L, E_R) per block.
    Returns (all_dets sorted unique, P) with P the (ndet x psi_size) isometry from the
    renormalized two-dot basis to determinants: |psi_det> = P psi."""
    bL, bR, part = pr.bL, pr.bR, pr.part
    c0, c1 = part.c
    d0, d1 = part.d
    site_bits = lambda n, a, b: (0, 1 << b, 1 << a, (1 << a) | (1 << b))[n]  # noqa: E731
    rows, cols, vals = [], [], []
    det_index = {}
    for (iL, n1, n2, iR, dL, dR, off) in pr.layout:
        EL, ER = bL.E[iL], bR.E[iR]
        mid = site_bits(n1, c0, c1) | site_bits(n2, d0, d1)
        M = np.kron(EL, ER)  # (nl*nr) x (dL*dR), row-major psi block index i*dR + j
        k = 0
        for dl in bL.dets[iL]:
            for dr in bR.dets[iR]:
                det = dl | mid | dr
                di = det_index.setdefault(det, len(det_index))
                nz = np.nonzero(M[k])[0]
                rows += [di] * len(nz)
                cols += list(off + nz)
                vals += list(M[k, nz])
                k += 1
    dets = np.array(sorted(det_index, key=det_index.get), dtype=np.uint64)
    P = np.zeros((len(dets), pr.psi_size), dtype=np.result_type(np.float64, *[np.asarray(v).dtype for v in vals[:1]], bL.E[0].dtype if 0 in bL.E else np.float64, pr.dtype))
    P[rows, cols] = vals
    return dets, P
