"""Sector-dimension model for the renormalized bases (DESIGN.md input recipe).

The paper gives only d_max(D) = 0.128 D + 51.8 for the P-cluster middle bond
(Eq. 25; Table 3).  Kept states per (N, 2Sz):
d(q) ~ exp(-(N-Nbar)^2/2 s^2 - (2Sz)^2/2 (1.5 s)^2), Nbar = N_tot/K * (orbitals in
block), capped by min(available states of q, number of complementary states that
complete q to the target), water-filled to sum d = min(D, available), with s
bisected so that max d = round(0.128 D + 51.8); largest-remainder rounding.
"""
from math import comb

import numpy as np


def full_dim(m, N, twoSz, sym="NSz"):
    """Number of determinants with (N, 2Sz) on m spatial orbitals (sym "N": with N electrons, any spin)."""
    if sym == "N":
        return comb(2 * m, N) if (0 <= N <= 2 * m and twoSz == 0) else 0
    if (N + twoSz) % 2:
        return 0
    na, nb = (N + twoSz) // 2, (N - twoSz) // 2
    if na < 0 or nb < 0 or na > m or nb > m:
        return 0
    return comb(m, na) * comb(m, nb)


def dmax_target(D):
    return int(round(0.128 * D + 51.8))


def _waterfill(w, cap, total):
    """d = min(cap, lam*w) with sum d = total (real-valued)."""
    if cap.sum() <= total:
        return cap.astype(float)
    lo, hi = 0.0, 1.0
    while np.minimum(cap, hi * w).sum() < total:
        hi *= 2.0
    for _ in range(200):
        mid = 0.5 * (lo + hi)
        if np.minimum(cap, mid * w).sum() < total:
            lo = mid
        else:
            hi = mid
    return np.minimum(cap, hi * w)


def _round_lr(x, cap, total):
    """Largest-remainder rounding of x to integers summing to total, 0 <= d <= cap."""
    d = np.floor(x + 1e-12).astype(np.int64)
    rem = int(total - d.sum())
    if rem > 0:
        frac = x - d
        order = np.argsort(-frac, kind="stable")
        for i in order:
            if rem == 0:
                break
            if d[i] < cap[i]:
                d[i] += 1
                rem -= 1
    return d


def kept_dims(qs, avail, m_block, K, N_tot, twoSz_tot, D, force_dmax=True, sym="NSz"):
    """qs: list of (N, 2Sz); avail: available states per q in the (enlarged) basis.

    Returns integer kept dimensions (0 = sector dropped)."""
    qs = list(qs)
    big = 1 << 40
    avail = np.asarray([min(int(a), big) for a in avail], dtype=np.int64)
    m_rest = K - m_block
    comp = np.array([min(full_dim(m_rest, N_tot - N, twoSz_tot - s, sym), big) for (N, s) in qs], dtype=np.int64)
    cap = np.minimum(avail, comp)
    total = int(min(D, cap.sum()))
    if cap.sum() <= D:
        return cap
    Nbar = N_tot / K * m_block
    Nq = np.array([q[0] for q in qs], dtype=float)
    Sq = np.array([q[1] for q in qs], dtype=float)

    def dims_for(s):
        w = np.exp(-(Nq - Nbar) ** 2 / (2 * s * s) - Sq ** 2 / (2 * (1.5 * s) ** 2))
        w = np.maximum(w, 1e-300)
        return _waterfill(w, cap.astype(float), total)

    s = 1.0
    if force_dmax:
        tgt = dmax_target(D)
        lo, hi = 0.05, 50.0
        # larger s => flatter => smaller max
        if dims_for(hi).max() >= tgt:
            s = hi
        elif dims_for(lo).max() <= tgt:
            s = lo
        else:
            for _ in range(80):
                mid = np.sqrt(lo * hi)
                if dims_for(mid).max() > tgt:
                    lo = mid
                else:
                    hi = mid
            s = hi
    x = dims_for(s)
    return _round_lr(x, cap, total)


def block_sector_model(m_block, K, N_tot, twoSz_tot, D, sym="NSz"):
    """Final sector table of a block of m_block orbitals (direct-fill configs)."""
    qs, avail = [], []
    for N in range(0, 2 * m_block + 1):
        for s in (range(-m_block, m_block + 1) if sym == "NSz" else (0,)):
            fd = full_dim(m_block, N, s, sym)
            if fd > 0:
                qs.append((N, s))
                avail.append(fd)
    d = kept_dims(qs, avail, m_block, K, N_tot, twoSz_tot, D, sym=sym)
    return [(q[0], q[1], int(x)) for q, x in zip(qs, d) if x > 0]


def psi_layout(secL, secR, N_tot, twoSz_tot, sym="NSz"):
    """Block table of psi/sigma: rows (iL, c1, c2, iR, dL, dR, offset), sorted by
    (iR, c1, c2, iL) so that all blocks sharing q_R form one contiguous row panel
    (each block is a dense row-major dL x dR matrix)."""
    from .conventions import site_q
    SITE_Q = site_q(sym)
    idxL = {(s[0], s[1]): i for i, s in enumerate(secL)}
    rows = []
    off = 0
    for iR, (NR, SR, dR) in enumerate(secR):
        for c1 in range(4):
            for c2 in range(4):
                NL = N_tot - NR - SITE_Q[c1][0] - SITE_Q[c2][0]
                SL = twoSz_tot - SR - SITE_Q[c1][1] - SITE_Q[c2][1]
                iL = idxL.get((NL, SL))
                if iL is None:
                    continue
                dL = secL[iL][2]
                rows.append((iL, c1, c2, iR, dL, dR, off))
                off += dL * dR
    return np.array(rows, dtype=np.int64).reshape(-1, 7), off
