"""Seeded synthetic integrals (BASELINE.json configs; readings 13-14).

h_pq symmetric with std 0.1; (pq|rs) 8-fold symmetric with std 0.05, drawn on the
canonical representatives (p>=q, r>=s, pq>=rs) and mirrored; (pp|pp) += 0.5.
`banded=True` (cfg 4-5) multiplies (pq|rs) by the 8-fold symmetric envelope
exp(-(|p-r|+|p-s|+|q-r|+|q-s|)/40), which reduces to exp(-|p-r|/10) for p=q, r=s.
"""
import numpy as np

from .conventions import GeneralSpinOrbitalIntegrals, SpinOrbitalIntegrals


def make_integrals(K, seed, banded=False, h_std=0.1, eri_std=0.05, diag_shift=0.5,
                   h_scale=1.0, eri_scale=1.0):
    rng = np.random.Generator(np.random.Philox(seed))
    h = rng.standard_normal((K, K)) * h_std
    h = np.tril(h) + np.tril(h, -1).T
    npair = K * (K + 1) // 2
    tab = rng.standard_normal((npair, npair)) * eri_std
    idx = np.arange(K)
    hi = np.maximum(idx[:, None], idx[None, :])
    lo = np.minimum(idx[:, None], idx[None, :])
    pair = hi * (hi + 1) // 2 + lo  # [K,K]
    PQ = pair[:, :, None, None]
    RS = pair[None, None, :, :]
    eri = tab[np.maximum(PQ, RS), np.minimum(PQ, RS)]
    if banded:
        p, q, r, s = np.ix_(idx, idx, idx, idx)
        env = np.exp(-(np.abs(p - r) + np.abs(p - s) + np.abs(q - r) + np.abs(q - s)) / 40.0)
        eri = eri * env
    eri = np.ascontiguousarray(eri)
    for p in range(K):
        eri[p, p, p, p] += diag_shift
    return SpinOrbitalIntegrals(h * h_scale, eri * eri_scale)


def make_so_integrals(K, seed, banded=False, so_h_std=0.05, so_v_std=0.01):
    """Spin-orbit variant: the spin-free integrals of make_integrals written over spin orbitals,
    plus a seeded complex Hermitian one-body coupling that mixes the spins (std so_h_std per real / imaginary part)
    and a small complex two-body part without spin selection rules (std so_v_std), symmetrised so that
    <PQ|RS> = <QP|SR> = conj(<RS|PQ>) and then antisymmetrised.  Only N is conserved."""
    base = make_integrals(K, seed, banded=banded)
    n = 2 * K
    rng = np.random.Generator(np.random.Philox(seed + 31337))
    a = (rng.standard_normal((n, n)) + 1j * rng.standard_normal((n, n))) * so_h_std
    h = base.dense_h().astype(np.complex128) + 0.5 * (a + a.conj().T)
    g = (rng.standard_normal((n,) * 4) + 1j * rng.standard_normal((n,) * 4)) * so_v_std
    g = g + g.transpose(1, 0, 3, 2)
    g = g + g.conj().transpose(2, 3, 0, 1)
    V = base.dense_V().astype(np.complex128) + (g - g.transpose(0, 1, 3, 2))
    return GeneralSpinOrbitalIntegrals(h, V)
