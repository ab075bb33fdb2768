"""Pins of the spin-orbit (complex, U(1)_N only) oracle, oracle/zsigma.py, against what the mathematics fixes
(with spin-orbit couplings Sz is no good quantum number and the dot factors become two-by-two blocks).

Z-def (zfci_dense_h, complex Slater-Condon) <- an independent Jordan-Wigner H (tests/fockdense.py);
Z-pair (zopair_sigma / zopair_hdiag)        <- Z-def through honest blocking with complex isometries, Hermiticity,
                                               and the real oracle in the spin-free limit.
The complex term table is pinned in tests/test_terms_dense.py.
"""
import numpy as np
import pytest

import fockdense as fd
import oracle
from oracle import zsigma
from dmrg_workload.conventions import GeneralSpinOrbitalIntegrals
from dmrg_workload.integrals import make_integrals, make_so_integrals
from dmrg_workload.problem import determinant_map, make_blocked_problem, make_direct_problem, random_psi_z


def test_complex_slater_condon_matches_jordan_wigner():
    K, N = 4, 4
    ints = make_so_integrals(K, seed=12)
    a = fd.full_annihilators(K)
    H = fd.hamiltonian(a, ints, 4 ** K).toarray()
    Nq, _ = fd.block_qnums(list(range(2 * K)))
    idx = np.nonzero(Nq == N)[0]
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
    assert len(dets) == 70
    Hsc = zsigma.zfci_dense_h(np.array(dets, dtype=np.uint64), 2 * K, ints.dense_h(), ints.dense_V())
    assert np.abs(Hsc - H[np.ix_(idx, idx)]).max() < 1e-13
    assert np.abs(Hsc - Hsc.conj().T).max() < 1e-13 and np.abs(Hsc.imag).max() > 1e-3
    mask = np.ones(4 ** K, bool)
    mask[idx] = False
    assert np.abs(H[np.ix_(mask, idx)]).max() == 0.0   # N is conserved ...
    _, Sq = fd.block_qnums(list(range(2 * K)))
    assert np.abs(H[np.ix_(idx[Sq[idx] == 0], idx[Sq[idx] == 2])]).max() > 1e-3   # ... Sz is not


def _fci(pr, dets):
    return zsigma.zfci_dense_h(dets, 2 * pr.meta["K"], pr.ints.dense_h(), pr.ints.dense_V())


@pytest.mark.parametrize("K,nL,N,D,rot", [(5, 1, 4, None, False), (6, 2, 6, None, False), (6, 2, 5, None, True),
                                          (6, 2, 6, 14, False), (6, 3, 6, 12, True), (7, 2, 7, 20, False)])
def test_sigma_and_diagonal_equal_fci(K, nL, N, D, rot):
    """Untruncated: sigma == H_FCI psi over all C(2K, N) determinants; truncated / rotated by random complex
    isometries: sigma == (E_L x E_R)^H H_FCI (E_L x E_R) psi.  The diagonal likewise, and it is real."""
    ints = make_so_integrals(K, seed=31 + K + nL)
    pr = make_blocked_problem(K, nL, N, 0, D=D, seed=K * 10 + nL, track=True, force_dmax=False, rotate=rot, ints=ints)
    assert pr.sym == "N" and pr.dtype == np.complex128 and pr.values.dtype == np.complex128
    dets, P = determinant_map(pr)
    assert np.abs(P.conj().T @ P - np.eye(pr.psi_size)).max() < 1e-12
    if D is None:
        from math import comb
        assert len(dets) == comb(2 * K, N) == pr.psi_size
    H = _fci(pr, dets)
    psi = random_psi_z(pr.psi_size, 3)
    sig = zsigma.zopair_sigma(pr, psi)
    ref = P.conj().T @ (H @ (P @ psi))
    assert np.abs(sig - ref).max() / np.linalg.norm(ref) < 1e-12
    hd = zsigma.zopair_hdiag(pr)
    assert np.abs(hd.imag).max() < 1e-13
    assert np.abs(hd - np.diag(P.conj().T @ H @ P)).max() < 1e-12


def test_hermiticity_linearity_and_sampled_blocks():
    pr = make_blocked_problem(6, 2, 6, 0, D=16, seed=5, force_dmax=False, rotate=True, ints=make_so_integrals(6, seed=77))
    psi, phi = random_psi_z(pr.psi_size, 1), random_psi_z(pr.psi_size, 2)
    s_psi, s_phi = zsigma.zopair_sigma(pr, psi), zsigma.zopair_sigma(pr, phi)
    assert abs(np.vdot(phi, s_psi) - np.vdot(s_phi, psi)) < 1e-13
    c = 0.3 - 1.1j   # linear, not anti-linear
    assert np.abs(zsigma.zopair_sigma(pr, c * psi + phi) - (c * s_psi + s_phi)).max() < 1e-13
    part = zsigma.zopair_sigma(pr, psi, only_out=[1, 4])
    for b in (1, 4):
        o, n = int(pr.layout[b][6]), int(pr.layout[b][4] * pr.layout[b][5])
        assert np.array_equal(part[o:o + n], s_psi[o:o + n])
    assert np.count_nonzero(part) <= sum(int(pr.layout[b][4] * pr.layout[b][5]) for b in (1, 4))


def test_spin_free_limit_is_the_real_oracle():
    """Real spin-free integrals fed through the spin-orbit path (complex dtype, N-only sectors, two-by-two dot
    blocks) give, in the determinant basis, what the real N x Sz oracle gives."""
    K, nL, N = 6, 2, 6
    base = make_integrals(K, seed=8)
    zi = GeneralSpinOrbitalIntegrals(base.dense_h(), base.dense_V())
    prz = make_blocked_problem(K, nL, N, 0, D=None, ints=zi, track=True)
    prr = make_blocked_problem(K, nL, N, 0, D=None, ints=base, track=True)
    dz, Pz = determinant_map(prz)
    dr, Pr = determinant_map(prr)
    rng = np.random.default_rng(0)
    v = rng.standard_normal(len(dr))                      # a vector in the Sz = 0 sector
    pos = {int(d): i for i, d in enumerate(dz)}
    vz = np.zeros(len(dz), dtype=np.complex128)
    vz[[pos[int(d)] for d in dr]] = v
    sz = Pz @ zsigma.zopair_sigma(prz, Pz.conj().T @ vz)
    sr = Pr @ oracle.opair_sigma(prr, Pr.T @ v)
    assert np.abs(sz[[pos[int(d)] for d in dr]] - sr).max() < 1e-12
    rest = np.ones(len(dz), bool)
    rest[[pos[int(d)] for d in dr]] = False
    assert np.abs(sz[rest]).max() < 1e-12                 # a spin-free H does not leave the Sz sector


def test_direct_fill_is_hermitian():
    """The complex direct-fill problems (larger GPU parity cases) define a Hermitian operator."""
    pr = make_direct_problem(8, 3, 8, 0, D=40, seed=3, ints=make_so_integrals(8, seed=3))
    psi, phi = random_psi_z(pr.psi_size, 1), random_psi_z(pr.psi_size, 2)
    assert abs(np.vdot(phi, zsigma.zopair_sigma(pr, psi)) - np.vdot(zsigma.zopair_sigma(pr, phi), psi)) < 1e-12
    assert np.abs(zsigma.zopair_hdiag(pr).imag).max() < 1e-13
