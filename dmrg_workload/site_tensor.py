"""Seeded random site tensors A[k] (Eq. 3) for the renormalization chain: problem setup only.

"Block operators via seeded random quantum-number-preserving orthonormal isometries, truncated to bond dimension D"
(BASELINE.json configs): the enlarged basis |l>|c> (or |c>|r>) is grouped into (N, 2Sz) sectors, the kept dimension of
every sector follows the sector model of sectors.py (Eq. 25), and the kept states are the first columns
of a Haar-random orthogonal matrix of that sector (QR of a seeded Gaussian d x k matrix).  No operator arithmetic.
The sub-block order inside an enlarged sector is blocking._Enlarged's: (first factor sector, second factor sector)
lexicographic, first factor = block for side 0, site for side 1.
"""
import numpy as np

from .conventions import SITE_Q
from .sectors import full_dim, kept_dims


def enlarged_sectors(sectors, dims, side):
    """{q: [(i_old, n_site, row0, d)]} and the sorted list of enlarged sectors."""
    sub = {}
    pairs = [(i, n) for i in range(len(sectors)) for n in range(4)] if side == 0 else [(i, n) for n in range(4) for i in range(len(sectors))]
    for i, n in pairs:
        q = (sectors[i][0] + SITE_Q[n][0], sectors[i][1] + SITE_Q[n][1])
        sub.setdefault(q, []).append((i, n))
    out = {}
    for q in sorted(sub):
        row0, lst = 0, []
        for i, n in sub[q]:
            lst.append((i, n, row0, dims[i]))
            row0 += dims[i]
        out[q] = lst
    return out


def random_site_tensor(sectors, dims, side, m_new, K, N_tot, twoSz_tot, D, rng, force_dmax=True):
    """Returns (new_sectors, new_dims, site_tensor) with site_tensor = [(i_old, n_site, r_new, matrix d_old x d_new)]."""
    enl = enlarged_sectors(sectors, dims, side)
    qs = list(enl)
    avail = [sum(d for _, _, _, d in enl[q]) for q in qs]
    if D is None:
        keep = [a if full_dim(K - m_new, N_tot - q[0], twoSz_tot - q[1]) > 0 else 0 for q, a in zip(qs, avail)]
    else:
        keep = [int(x) for x in kept_dims(qs, avail, m_new, K, N_tot, twoSz_tot, D, force_dmax)]
    new_sectors, new_dims, tensor = [], [], []
    for q, a, k in zip(qs, avail, keep):
        if k <= 0:
            continue
        g = rng.standard_normal((a, k))
        w, _ = np.linalg.qr(g)          # a x k, orthonormal columns
        r_new = len(new_sectors)
        new_sectors.append(q)
        new_dims.append(k)
        for i, n, row0, d in enl[q]:
            tensor.append((i, n, r_new, np.ascontiguousarray(w[row0:row0 + d, :])))
    return new_sectors, new_dims, tensor
