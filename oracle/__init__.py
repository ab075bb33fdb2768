"""CPU ORACLE -- test infrastructure, not product code.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
may import this package.  It is independent of the CUDA path: it never imports
paper_2311_02854_b200 and shares no code with it (array formats only, see
dmrg_workload/store.py).

  opair_sigma / opair_hdiag : operator-pair contraction in plain C loops (sigma_oracle.c)
  opair_count               : the same task expansion, cost measure only (2MNK per GEMM)
  fci_dense_h               : dense Slater-Condon Hamiltonian, the definition (Eq. 2)
  davidson                  : single-root Davidson in numpy (oracle/davidson.py)

Parity pins: see tests/test_oracle_*.py and DESIGN.md "Pins".  Unpinned: the paper's
P-cluster energies (Table 5) and T_Hx curves -- inputs not available ("parity unpinned").
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "sigma_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")
_lib = None


def build(force=False):
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-std=c11",
                               "-o", _LIB, _SRC, "-lm"])
    return _LIB


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.opair_sigma.restype = C.c_int64
        _lib.opair_hdiag.restype = C.c_int64
        _lib.opair_count.restype = C.c_int64
        _lib.fci_element.restype = C.c_double
        _lib.oracle_num_threads.restype = C.c_int
    return _lib


def num_threads():
    return int(lib().oracle_num_threads())


def _p(a, t):
    return a.ctypes.data_as(C.POINTER(t))


def _problem_args(pr, need_values=True):
    a = dict(
        secL=np.ascontiguousarray(pr.secL, np.int32), secR=np.ascontiguousarray(pr.secR, np.int32),
        ops=np.ascontiguousarray(pr.ops, np.int64), blocks=np.ascontiguousarray(pr.blocks, np.int64),
        values=np.ascontiguousarray(pr.values, np.float64) if (need_values or pr.values is not None) else None,
        lin_ptr=np.ascontiguousarray(pr.lin_ptr, np.int64), lin_op=np.ascontiguousarray(pr.lin_op, np.int32),
        lin_coef=np.ascontiguousarray(pr.lin_coef, np.float64),
        site_ops=np.ascontiguousarray(pr.site_ops, np.float64),
        site_parity=np.ascontiguousarray(pr.site_parity, np.int32),
        term_coef=np.ascontiguousarray(pr.term_coef, np.float64),
        term_idx=np.ascontiguousarray(pr.term_idx, np.int32),
        layout=np.ascontiguousarray(pr.layout, np.int64))
    args = [_p(a["secL"], C.c_int32), C.c_int(len(a["secL"])), _p(a["secR"], C.c_int32), C.c_int(len(a["secR"])),
            _p(a["ops"], C.c_int64), C.c_int(len(a["ops"])), _p(a["blocks"], C.c_int64),
            _p(a["values"], C.c_double) if a["values"] is not None else None,
            _p(a["lin_ptr"], C.c_int64), _p(a["lin_op"], C.c_int32), _p(a["lin_coef"], C.c_double),
            _p(a["site_ops"], C.c_double), _p(a["site_parity"], C.c_int32), C.c_int(len(a["site_ops"])),
            _p(a["term_coef"], C.c_double), _p(a["term_idx"], C.c_int32), C.c_int64(len(a["term_coef"])),
            _p(a["layout"], C.c_int64), C.c_int64(len(a["layout"])), C.c_int64(pr.psi_size)]
    return a, args


def opair_sigma(pr, psi, only_out=None, return_stats=False):
    """sigma = H psi by the operator-pair contraction (Eq. 7; Eqs. 11-13)."""
    keep, args = _problem_args(pr)
    psi = np.ascontiguousarray(psi, np.float64)
    assert psi.shape == (pr.psi_size,)
    sigma = np.zeros(pr.psi_size)
    oo = np.ascontiguousarray(only_out if only_out is not None else [], np.int32)
    fl = C.c_double(0.0)
    n = lib().opair_sigma(*args, _p(psi, C.c_double), _p(sigma, C.c_double), _p(oo, C.c_int32),
                          C.c_int(len(oo)), C.byref(fl))
    if return_stats:
        return sigma, {"tasks": int(n), "flops": fl.value}
    return sigma


def opair_count(pr, only_out=None):
    """The oracle's cost measure without the arithmetic: {"tasks", "flops"} of the same
    (term, psi block, dot transition) expansion opair_sigma executes.  pr.values may be None."""
    keep, args = _problem_args(pr, need_values=False)
    oo = np.ascontiguousarray(only_out if only_out is not None else [], np.int32)
    fl = C.c_double(0.0)
    n = lib().opair_count(*args, _p(oo, C.c_int32), C.c_int(len(oo)), C.byref(fl))
    return {"tasks": int(n), "flops": fl.value}


def opair_hdiag(pr):
    keep, args = _problem_args(pr)
    diag = np.zeros(pr.psi_size)
    lib().opair_hdiag(*args, _p(diag, C.c_double))
    return diag


def fci_dense_h(dets, n, hso, V):
    """Dense Slater-Condon Hamiltonian over the given determinants (bit strings)."""
    dets = np.ascontiguousarray(dets, np.uint64)
    hso = np.ascontiguousarray(hso, np.float64)
    V = np.ascontiguousarray(V, np.float64)
    H = np.empty((len(dets), len(dets)))
    lib().fci_dense_h(_p(dets, C.c_uint64), C.c_int64(len(dets)), C.c_int(n), _p(hso, C.c_double),
                      _p(V, C.c_double), _p(H, C.c_double))
    return H
