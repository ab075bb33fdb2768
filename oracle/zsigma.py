"""CPU ORACLE -- test infrastructure, not product code -- for the spin-orbit variant.

With spin-orbit couplings "the spin projection is no longer a good quantum number": the Hamiltonian
of Eq. (2) is complex Hermitian, only U(1)_N is kept, and the dot factors [O]_{C1'C1}, [O]_{C2'C2} of Eqs. (9)-(10)
 are "either a scalar or a two-by-two matrix" (the N = 1 sector of a dot holds both spin states).
What is computed is still Eq. (7),

    sigma[l' c1' c2' r'] = sum_mu sum_{l c1 c2 r} zeta [O^L]_{l'l} [O^C1]_{c1'c1} [O^C2]_{c2'c2} [O^R]_{r'r} psi[l c1 c2 r],

in complex arithmetic, block by block: psi blocks are indexed by the dot STATES (c1, c2) as in the real oracle, so a
two-by-two dot block is simply two non-zero entries in a column of the 4 x 4 site matrix -- Eqs. (9)-(10) are the two
loops over (c1', c2') below -- followed by Eq. (11) X = psi_blk (O^R)^T, Eq. (12) O^L X and the sum of Eq. (13).
A "transposed" use of a stored operator is its Hermitian conjugate (dmrg_workload/terms.py); linear-combination
operators ("intermediates") are formed first.  zeta is DESIGN.md reading 3.

Plain numpy in complex128, one matmul per step, no blocking, no de-duplication, no reordering: tasks are summed into
each output block in (term, input block, c1', c2') order.  Independent of the CUDA path (never imports
paper_2311_02854_b200; array formats only, dmrg_workload/store.py).  Pins: tests/test_oracle_spinorbit.py.

  zopair_sigma, zopair_hdiag : the operator-pair contraction and its diagonal
  zfci_dense_h               : the definition, complex Slater-Condon rules (oracle/zfci.c)
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "zfci.c")
_LIB = os.path.join(_HERE, "libzfci.so")
_lib = None

SITE_N = (0, 1, 1, 2)


def build(force=False):
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-fPIC", "-shared", "-std=c11", "-o", _LIB, _SRC, "-lm"])
    return _LIB


def zfci_dense_h(dets, n, h, V):
    """Dense complex Slater-Condon Hamiltonian over the given determinants (bit strings); h [n,n], V [n,n,n,n]."""
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
    dets = np.ascontiguousarray(dets, np.uint64)
    h = np.ascontiguousarray(h, np.complex128)
    V = np.ascontiguousarray(V, np.complex128)
    assert h.shape == (n, n) and V.shape == (n, n, n, n)
    H = np.empty((len(dets), len(dets)), dtype=np.complex128)
    vp = C.c_void_p
    _lib.zfci_dense_h(vp(dets.ctypes.data), C.c_int64(len(dets)), C.c_int(n), vp(h.ctypes.data), vp(V.ctypes.data), vp(H.ctypes.data))
    return H


def _optabs(pr):
    """Per operator: {row sector: (col sector, dense block)}; LINCOMB operators sum_s coef_s op_s formed blockwise."""
    dims = {0: pr.secL[:, 2], 1: pr.secR[:, 2]}
    vals = np.asarray(pr.values, dtype=np.complex128)
    tabs = []
    for side, kind, _p, _q, _dn, _ds, first, nb in pr.ops:
        t = {}
        if kind != 7:
            for r, c, off in pr.blocks[first:first + nb]:
                dr, dc = int(dims[side][r]), int(dims[side][c])
                t[int(r)] = (int(c), vals[off:off + dr * dc].reshape(dr, dc))
        tabs.append(t)
    for o, (side, kind, j, _q, _dn, _ds, _f, _nb) in enumerate(pr.ops):
        if kind != 7:
            continue
        t = {}
        for i in range(int(pr.lin_ptr[j]), int(pr.lin_ptr[j + 1])):
            for r, (c, m) in tabs[int(pr.lin_op[i])].items():
                add = complex(pr.lin_coef[i]) * m
                t[r] = (c, t[r][1] + add) if r in t else (c, add)
        tabs[o] = t
    return tabs


def _tasks(pr, tabs, diag_only=False):
    """Every (term, psi block, dot transition): (out block, in block, L block or None, L conj-transposed?, R block or
    None, R conj-transposed?, alpha = c_mu zeta o1[c1',c1] o2[c2',c2]), in (term, in block, c1', c2') order."""
    lut = {(int(iL), int(c1), int(c2), int(iR)): b for b, (iL, c1, c2, iR, _dl, _dr, _off) in enumerate(pr.layout)}
    site = np.asarray(pr.site_ops, dtype=np.complex128).reshape(-1, 4, 4)
    par_op = [int(row[4]) & 1 for row in pr.ops]
    inv = [{c: r for r, (c, _m) in t.items()} for t in tabs]   # col sector -> row sector
    out = []
    for t in range(len(pr.term_coef)):
        ol, tl, s1, s2, orr, tr = (int(x) for x in pr.term_idx[t])
        o1, o2 = site[s1], site[s2]
        p1, p2 = int(pr.site_parity[s1]), int(pr.site_parity[s2])
        pR = par_op[orr] if orr >= 0 else 0
        for b, (iL, c1, c2, iR, _dl, _dr, _off) in enumerate(pr.layout):
            iL, c1, c2, iR = int(iL), int(c1), int(c2), int(iR)
            Lm = Rm = None
            iLo, iRo = iL, iR
            if ol >= 0:
                if not tl:
                    if iL not in inv[ol]:
                        continue
                    iLo = inv[ol][iL]
                    Lm = tabs[ol][iLo][1]
                else:
                    if iL not in tabs[ol]:
                        continue
                    iLo, Lm = tabs[ol][iL]
            if orr >= 0:
                if not tr:
                    if iR not in inv[orr]:
                        continue
                    iRo = inv[orr][iR]
                    Rm = tabs[orr][iRo][1]
                else:
                    if iR not in tabs[orr]:
                        continue
                    iRo, Rm = tabs[orr][iR]
            Nl = int(pr.secL[iL, 0])
            zexp = p1 * Nl + p2 * (Nl + SITE_N[c1]) + pR * (Nl + SITE_N[c1] + SITE_N[c2])
            zeta = -1.0 if zexp & 1 else 1.0
            for c1o in range(4):          # Eq. (10): the dot-1 factor, a scalar or a column of a two-by-two block
                v1 = o1[c1o, c1]
                if v1 == 0:
                    continue
                for c2o in range(4):      # Eq. (9): the dot-2 factor
                    v2 = o2[c2o, c2]
                    if v2 == 0:
                        continue
                    ob = lut.get((iLo, c1o, c2o, iRo))
                    if ob is None or (diag_only and ob != b):
                        continue
                    out.append((ob, b, Lm, tl, Rm, tr, complex(pr.term_coef[t]) * zeta * v1 * v2))
    return out


def _blk(pr, v, b):
    _iL, _c1, _c2, _iR, dl, dr, off = (int(x) for x in pr.layout[b])
    return v[off:off + dl * dr].reshape(dl, dr)


def zopair_sigma(pr, psi, only_out=None, return_stats=False):
    """sigma = H psi (complex128 vectors of pr.psi_size entries in the psi layout of pr.layout)."""
    psi = np.ascontiguousarray(psi, np.complex128)
    assert psi.shape == (pr.psi_size,)
    tabs = _optabs(pr)
    want = None if only_out is None or len(only_out) == 0 else set(int(b) for b in only_out)
    sigma = np.zeros(pr.psi_size, dtype=np.complex128)
    flops, done = 0.0, 0
    for ob, b, Lm, tl, Rm, tr, alpha in _tasks(pr, tabs):
        if want is not None and ob not in want:
            continue
        x = _blk(pr, psi, b)
        if Rm is None:
            X = x
        else:                                   # Eq. (11): X[i,j] = sum_k psi[i,k] (O^R as used)[j,k]
            X = x @ (Rm.conj() if tr else Rm.T)
            flops += 8.0 * x.shape[0] * x.shape[1] * X.shape[1]
        if Lm is None:
            Y = X
        else:                                   # Eq. (12): (O^L as used) X
            Y = (Lm.conj().T if tl else Lm) @ X
            flops += 8.0 * Y.shape[0] * X.shape[0] * X.shape[1]
        _blk(pr, sigma, ob)[...] += alpha * Y   # Eq. (13)
        done += 1
    if return_stats:
        return sigma, {"tasks": done, "flops": flops}   # complex GEMM = 8 M N K real flops
    return sigma


def zopair_hdiag(pr):
    """diag(H) in the psi layout (real for a Hermitian H; returned complex so that a test can check that)."""
    tabs = _optabs(pr)
    diag = np.zeros(pr.psi_size, dtype=np.complex128)
    for ob, _b, Lm, _tl, Rm, _tr, alpha in _tasks(pr, tabs, diag_only=True):
        out = _blk(pr, diag, ob)
        l = np.ones(out.shape[0]) if Lm is None else np.diagonal(Lm)
        r = np.ones(out.shape[1]) if Rm is None else np.diagonal(Rm)
        # a conj-transposed use has the conjugate diagonal
        l = l.conj() if (Lm is not None and _tl) else l
        r = r.conj() if (Rm is not None and _tr) else r
        out += alpha * np.outer(l, r)
    return diag
