"""Pins of the CPU oracle against what the paper and the mathematics fix.

O-pair (oracle.opair_sigma) is pinned to O-def (Slater-Condon dense H, Eq. 2),
which is itself pinned to an independent Jordan-Wigner construction (tests/fockdense.py)
and to closed forms.
"""
import numpy as np
import pytest

import fockdense as fd
import oracle
from oracle.davidson import davidson
from dmrg_workload.conventions import SpinOrbitalIntegrals
from dmrg_workload.integrals import make_integrals
from dmrg_workload.problem import determinant_map, make_blocked_problem, random_psi


def fci_h(pr, dets):
    return oracle.fci_dense_h(dets, 2 * pr.meta["K"], pr.ints.dense_h(), pr.ints.dense_V())


def test_slater_condon_matches_jordan_wigner():
    """O-def vs. brute-force second quantisation (independent of oracle/) at K=4, N=4, Sz=0."""
    K = 4
    ints = make_integrals(K, seed=11)
    a = fd.full_annihilators(K)
    H = fd.hamiltonian(a, ints, 4 ** K).toarray()
    N, S = fd.block_qnums(list(range(2 * K)))
    idx = np.nonzero((N == 4) & (S == 0))[0]
    # site-Kronecker index -> bit string: site k state n (2 n_alpha + n_beta)
    dets = []
    for i in idx:
        bits, x = 0, int(i)
        for k in reversed(range(K)):
            n = x % 4
            x //= 4
            if n & 2:
                bits |= 1 << (2 * k)
            if n & 1:
                bits |= 1 << (2 * k + 1)
        dets.append(bits)
    Hsc = oracle.fci_dense_h(np.array(dets, dtype=np.uint64), 2 * K, ints.dense_h(), ints.dense_V())
    assert np.abs(Hsc - H[np.ix_(idx, idx)]).max() < 1e-13
    # N, Sz conservation: H has no element leaving the sector
    mask = np.ones(4 ** K, bool)
    mask[idx] = False
    assert np.abs(H[np.ix_(mask, idx)]).max() == 0.0


@pytest.fixture(scope="module")
def cfg1():
    pr = make_blocked_problem(8, 3, 8, 0, D=None, seed=1, track=True)
    dets, P = determinant_map(pr)
    return pr, dets, P, fci_h(pr, dets)


def test_cfg1_sigma_equals_fci(cfg1):
    """Pin 1: untruncated 3-1-1-3, 4900 determinants, 196 psi blocks (BASELINE.json configs[0])."""
    pr, dets, P, H = cfg1
    assert len(dets) == 4900 and len(pr.layout) == 196 and pr.psi_size == 4900
    psi = random_psi(pr.psi_size, 5)
    sig = oracle.opair_sigma(pr, psi)
    ref = P.T @ (H @ (P @ psi))
    assert np.abs(sig - ref).max() / np.linalg.norm(ref) < 1e-13


def test_cfg1_hdiag_and_davidson(cfg1):
    """Pin 2: Davidson E0 == exact diagonalisation of the dense 4900x4900 H to 1e-9."""
    pr, dets, P, H = cfg1
    hd = oracle.opair_hdiag(pr)
    assert np.abs(hd - np.diag(P.T @ H @ P)).max() < 1e-12
    e0 = np.linalg.eigvalsh(H)[0]
    x0 = random_psi(pr.psi_size, 9)
    res = davidson(lambda v: oracle.opair_sigma(pr, v), hd, x0, max_iter=200, max_space=30, tol=1e-8)
    assert res["resid"] <= 1e-8
    assert abs(res["energy"] - e0) < 1e-9


def test_hermiticity_and_linearity(cfg1):
    """Pins 3, 9."""
    pr = cfg1[0]
    psi, phi = random_psi(pr.psi_size, 1), random_psi(pr.psi_size, 2)
    s_psi, s_phi = oracle.opair_sigma(pr, psi), oracle.opair_sigma(pr, phi)
    assert abs(phi @ s_psi - s_phi @ psi) < 1e-13
    s_mix = oracle.opair_sigma(pr, 0.3 * psi - 1.7 * phi)
    assert np.abs(s_mix - (0.3 * s_psi - 1.7 * s_phi)).max() < 1e-13


@pytest.mark.parametrize("K,nL,N,D,rot", [(6, 2, 6, 8, False), (7, 2, 6, 12, False), (7, 3, 8, 10, True),
                                          (6, 1, 4, None, True), (8, 2, 8, 30, False)])
def test_truncated_and_rotated(K, nL, N, D, rot):
    """Pins 5, 7, 11: random isometries; sigma == (E_L x E_R)^T H_FCI (E_L x E_R) psi; every
    stored operator == E^T O_exact E is implied by sigma for arbitrary integrals; interlacing."""
    pr = make_blocked_problem(K, nL, N, 0, D=D, seed=K * 10 + nL, track=True, force_dmax=False, rotate=rot)
    dets, P = determinant_map(pr)
    assert np.abs(P.T @ P - np.eye(pr.psi_size)).max() < 1e-12
    H = fci_h(pr, dets)
    psi = random_psi(pr.psi_size, 3)
    sig = oracle.opair_sigma(pr, psi)
    ref = P.T @ (H @ (P @ psi))
    assert np.abs(sig - ref).max() / np.linalg.norm(ref) < 1e-12
    Hp = P.T @ H @ P
    assert np.abs(oracle.opair_hdiag(pr) - np.diag(Hp)).max() < 1e-12
    # interlacing needs the full sector: compare with FCI over all determinants of (N, Sz=0)
    assert np.linalg.eigvalsh(Hp)[0] >= _fci_ground(K, N, pr.ints) - 1e-10


def _fci_ground(K, N, ints):
    from itertools import combinations
    na = N // 2
    dets = []
    for A in combinations(range(K), na):
        for B in combinations(range(K), N - na):
            dets.append(sum(1 << (2 * k) for k in A) | sum(1 << (2 * k + 1) for k in B))
    H = oracle.fci_dense_h(np.array(dets, dtype=np.uint64), 2 * K, ints.dense_h(), ints.dense_V())
    return np.linalg.eigvalsh(H)[0]


def test_partition_invariance():
    """Pin 6: 2-1-1-4, 3-1-1-3, 4-1-1-2 give the same determinant-basis sigma (untruncated, K=8)."""
    ints = make_integrals(8, seed=21)
    rng = np.random.default_rng(0)
    ref = None
    for nL in (2, 3, 4):
        pr = make_blocked_problem(8, nL, 8, 0, D=None, ints=ints, track=True)
        dets, P = determinant_map(pr)
        order = np.argsort(dets)
        if ref is None:
            vdet = rng.standard_normal(len(dets))
        psi = P.T[:, order] @ vdet
        sdet = (P @ oracle.opair_sigma(pr, psi))[order]
        if ref is None:
            ref = sdet
        else:
            assert np.abs(sdet - ref).max() < 1e-12


def test_closed_forms():
    """Pin 8: (i) no two-electron part: E0 = 2 * sum of the N/2 lowest eigenvalues of h;
    (ii) h = 0, only (pp|pp) = U: H diagonal with U * (#doubly occupied)."""
    K, N = 6, 6
    base = make_integrals(K, seed=4)
    ints = SpinOrbitalIntegrals(base.h_sp, np.zeros((K,) * 4))
    pr = make_blocked_problem(K, 2, N, 0, D=None, ints=ints, track=True)
    hd = oracle.opair_hdiag(pr)
    res = davidson(lambda v: oracle.opair_sigma(pr, v), hd, random_psi(pr.psi_size, 1), 300, 40, 1e-9)
    assert abs(res["energy"] - 2 * np.sort(np.linalg.eigvalsh(base.h_sp))[: N // 2].sum()) < 1e-8
    U = 0.7
    eri = np.zeros((K,) * 4)
    for p in range(K):
        eri[p, p, p, p] = U
    pr = make_blocked_problem(K, 2, N, 0, D=None, ints=SpinOrbitalIntegrals(np.zeros((K, K)), eri), track=True)
    dets, P = determinant_map(pr)
    psi = random_psi(pr.psi_size, 2)
    ndouble = np.array([sum(1 for k in range(K) if (int(d) >> (2 * k)) & 3 == 3) for d in dets])
    assert np.abs(P @ oracle.opair_sigma(pr, psi) - U * ndouble * (P @ psi)).max() < 1e-13


def test_sampled_output_blocks(cfg1):
    """only_out computes exactly the requested blocks (used for full-size sampled parity)."""
    pr = cfg1[0]
    psi = random_psi(pr.psi_size, 8)
    full = oracle.opair_sigma(pr, psi)
    part = oracle.opair_sigma(pr, psi, only_out=[3, 77])
    for b in (3, 77):
        o, n = pr.layout[b][6], pr.layout[b][4] * pr.layout[b][5]
        assert np.array_equal(part[o:o + n], full[o:o + n])
    assert np.count_nonzero(part) <= sum(pr.layout[b][4] * pr.layout[b][5] for b in (3, 77))
