"""Python binding of libdmrg_sigma.so (include/dmrg_sigma.h): argument marshalling only.

Every step of the hot path (operator store, planner, sigma kernels, Davidson) runs inside the
shared library; this module converts numpy arrays / torch tensors to the C structs and pointers.
There is no CPU fallback: if the library has not been built, importing `lib()` raises.
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libdmrg_sigma.so")

SECTOR_DT = np.dtype([("n", "<i4"), ("two_sz", "<i4"), ("dim", "<i4")], align=True)
OP_DT = np.dtype([("side", "<i4"), ("kind", "<i4"), ("p", "<i4"), ("q", "<i4"), ("dn", "<i4"), ("d2sz", "<i4"),
                  ("first_block", "<i8"), ("nblocks", "<i4"), ("reserved", "<i4")], align=True)
BLOCK_DT = np.dtype([("row_sector", "<i4"), ("col_sector", "<i4"), ("offset", "<i8")], align=True)
TERM_DT = np.dtype([("coef", "<f8"), ("op_l", "<i4"), ("trans_l", "<i4"), ("dot1", "<i4"), ("dot2", "<i4"),
                    ("op_r", "<i4"), ("trans_r", "<i4")], align=True)
PSIBLK_DT = np.dtype([("il", "<i4"), ("c1", "<i4"), ("c2", "<i4"), ("ir", "<i4"), ("dl", "<i4"), ("dr", "<i4"),
                      ("offset", "<i8")], align=True)
assert SECTOR_DT.itemsize == 12 and OP_DT.itemsize == 40 and BLOCK_DT.itemsize == 16
assert TERM_DT.itemsize == 32 and PSIBLK_DT.itemsize == 32

PLANOPT_DT = np.dtype([("workspace_bytes", "<i8"), ("copy_mode", "<i4"), ("min_split_stages", "<i4"), ("split_waves", "<f8"),
                       ("max_merged_cols", "<i4"), ("cost_order_only", "<i4"), ("split_small", "<i4"), ("release_r_store", "<i4"),
                       ("shard_rank", "<i4"), ("shard_count", "<i4"), ("tile_run_stages", "<i4"), ("reserved", "<i4", (5,))], align=True)
assert PLANOPT_DT.itemsize == 72
COPY_LDGSTS, COPY_TMA = 1, 2
WBLOCK_DT = np.dtype([("old_sector", "<i4"), ("site_state", "<i4"), ("new_sector", "<i4"), ("reserved", "<i4"), ("offset", "<i8")], align=True)
RTERM_DT = np.dtype([("coef", "<f8"), ("op", "<i4"), ("trans", "<i4"), ("site_op", "<i4"), ("reserved", "<i4")], align=True)
RENORMOPT_DT = np.dtype([("workspace_bytes", "<i8"), ("copy_mode", "<i4"), ("reserved", "<i4", (5,))], align=True)
RENORMSTATS_DT = np.dtype([("flops", "<f8"), ("device_ms", "<f8"), ("launches", "<i8"), ("jobs", "<i8"), ("tiles", "<i8"),
                           ("out_values", "<i8"), ("workspace_values", "<i8"), ("tensor_maps", "<i8")], align=True)
assert WBLOCK_DT.itemsize == 24 and RTERM_DT.itemsize == 24 and RENORMOPT_DT.itemsize == 32 and RENORMSTATS_DT.itemsize == 64

STAT_KEYS = ("tasks", "alg_flops", "s1_flops", "s2_flops", "padded_flops", "s1_jobs", "chunks", "launches",
             "plan_device_bytes", "alg_bytes", "s1_tiles", "s2_tiles", "canon_flops", "stage_flops", "tile_flops", "warp_flops",
             "xws_elems", "tensor_maps", "s1_fill", "s2_fill", "s1_stages", "s2_stages")

EXPORTS = ("dmrg_ops_load", "dmrg_ops_free", "dmrg_ops_device_bytes", "dmrg_plan_create", "dmrg_plan_create_opts", "dmrg_plan_destroy",
           "dmrg_plan_psi_size", "dmrg_plan_shard_terms", "dmrg_plan_num_psi_blocks", "dmrg_plan_psi_layout", "dmrg_plan_stat", "dmrg_sigma",
           "dmrg_sigma_host", "dmrg_hdiag", "dmrg_davidson", "dmrg_plan_set_timing", "dmrg_plan_stage_ms",
           "dmrg_fp64_peak_tflops", "dmrg_last_error", "dmrg_version",
           "dmrg_renormalize", "dmrg_ops_num_ops", "dmrg_ops_num_blocks", "dmrg_ops_num_values", "dmrg_ops_export", "dmrg_ops_sectors",
           "dmrg_ops_join", "dmrg_ops_add_lincombs", "dmrg_ops_derive",
           "dmrg_comm_unique_id", "dmrg_comm_create", "dmrg_comm_destroy", "dmrg_plan_set_comm", "dmrg_dots_static",
           "dmrg_ops_load_z", "dmrg_plan_create_z", "dmrg_ops_is_complex", "dmrg_plan_is_complex")
DOTS_STATIC_MAX_VECTORS = 32

_lib = None


class DmrgError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"libdmrg_sigma error {code}: {msg}")
        self.code = code


def lib():
    """Load the CUDA library; fails loudly when it has not been built (no fallback path exists)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_2311_02854_b200.build` "
                              "(or __graft_entry__.build()); there is no CPU fallback")
        L = C.CDLL(LIB_PATH)
        vp, i32, i64, f64 = C.c_void_p, C.c_int32, C.c_int64, C.c_double
        L.dmrg_ops_load.argtypes = [vp, i32, vp, i32, vp, i32, vp, i64, vp, i64, i32, vp, vp, vp, i32, C.POINTER(vp)]
        L.dmrg_ops_load.restype = C.c_int
        L.dmrg_ops_free.argtypes = [vp]
        L.dmrg_ops_free.restype = None
        L.dmrg_ops_device_bytes.argtypes = [vp]
        L.dmrg_ops_device_bytes.restype = i64
        L.dmrg_plan_create.argtypes = [vp, vp, i64, vp, vp, i32, i32, i32, i64, C.POINTER(vp)]
        L.dmrg_plan_create.restype = C.c_int
        L.dmrg_plan_create_opts.argtypes = [vp, vp, i64, vp, vp, i32, i32, i32, vp, C.POINTER(vp)]
        L.dmrg_plan_create_opts.restype = C.c_int
        L.dmrg_plan_destroy.argtypes = [vp]
        L.dmrg_plan_destroy.restype = None
        L.dmrg_plan_psi_size.argtypes = [vp]
        L.dmrg_plan_psi_size.restype = i64
        L.dmrg_plan_shard_terms.argtypes = [vp, vp, i64]
        L.dmrg_plan_shard_terms.restype = i64
        L.dmrg_plan_num_psi_blocks.argtypes = [vp]
        L.dmrg_plan_num_psi_blocks.restype = i64
        L.dmrg_plan_psi_layout.argtypes = [vp, vp]
        L.dmrg_plan_psi_layout.restype = C.c_int
        L.dmrg_plan_stat.argtypes = [vp, i32]
        L.dmrg_plan_stat.restype = f64
        L.dmrg_sigma.argtypes = [vp, vp, vp, vp]
        L.dmrg_sigma.restype = C.c_int
        L.dmrg_sigma_host.argtypes = [vp, vp, vp, vp]
        L.dmrg_sigma_host.restype = C.c_int
        L.dmrg_hdiag.argtypes = [vp, vp, vp]
        L.dmrg_hdiag.restype = C.c_int
        L.dmrg_davidson.argtypes = [vp, vp, i32, i32, f64, C.POINTER(f64), C.POINTER(f64), C.POINTER(i32), vp, vp]
        L.dmrg_davidson.restype = C.c_int
        L.dmrg_plan_set_timing.argtypes = [vp, i32]
        L.dmrg_plan_set_timing.restype = C.c_int
        L.dmrg_plan_stage_ms.argtypes = [vp, i32]
        L.dmrg_plan_stage_ms.restype = f64
        L.dmrg_fp64_peak_tflops.argtypes = [i32, f64, vp]
        L.dmrg_fp64_peak_tflops.restype = f64
        L.dmrg_renormalize.argtypes = [vp, i32, vp, i32, vp, i64, vp, i64, vp, i32, vp, vp, vp, vp, i32, vp, vp, C.POINTER(vp), vp]
        L.dmrg_renormalize.restype = C.c_int
        for name in ("dmrg_ops_num_ops", "dmrg_ops_num_blocks", "dmrg_ops_num_values"):
            getattr(L, name).argtypes = [vp]
            getattr(L, name).restype = i64
        L.dmrg_ops_export.argtypes = [vp, vp, vp, vp]
        L.dmrg_ops_export.restype = C.c_int
        L.dmrg_ops_sectors.argtypes = [vp, i32, vp, i32]
        L.dmrg_ops_sectors.restype = C.c_int
        L.dmrg_ops_join.argtypes = [vp, vp, C.POINTER(vp)]
        L.dmrg_ops_join.restype = C.c_int
        L.dmrg_ops_add_lincombs.argtypes = [vp, vp, i32, vp, vp, vp, vp, i32]
        L.dmrg_ops_add_lincombs.restype = C.c_int
        L.dmrg_ops_derive.argtypes = [vp, vp, i32, vp, vp, vp, vp, i32, C.POINTER(vp)]
        L.dmrg_ops_derive.restype = C.c_int
        L.dmrg_comm_unique_id.argtypes = [vp, i32]
        L.dmrg_comm_unique_id.restype = C.c_int
        L.dmrg_comm_create.argtypes = [vp, i32, i32, C.POINTER(vp)]
        L.dmrg_comm_create.restype = C.c_int
        L.dmrg_comm_destroy.argtypes = [vp]
        L.dmrg_comm_destroy.restype = None
        L.dmrg_plan_set_comm.argtypes = [vp, vp]
        L.dmrg_plan_set_comm.restype = C.c_int
        L.dmrg_ops_load_z.argtypes = L.dmrg_ops_load.argtypes
        L.dmrg_ops_load_z.restype = C.c_int
        L.dmrg_plan_create_z.argtypes = [vp, vp, vp, i64, vp, vp, i32, i32, vp, C.POINTER(vp)]
        L.dmrg_plan_create_z.restype = C.c_int
        L.dmrg_ops_is_complex.argtypes = [vp]
        L.dmrg_ops_is_complex.restype = i32
        L.dmrg_plan_is_complex.argtypes = [vp]
        L.dmrg_plan_is_complex.restype = i32
        L.dmrg_dots_static.argtypes = [vp, i64, i32, vp, i64, vp, vp]
        L.dmrg_dots_static.restype = C.c_int
        L.dmrg_last_error.restype = C.c_char_p
        L.dmrg_version.restype = C.c_char_p
        _lib = L
    return _lib


def _check(rc, allow=()):
    if rc != 0 and rc not in allow:
        raise DmrgError(rc, lib().dmrg_last_error().decode())
    return rc


def _check_count(n):
    if n < 0:
        raise DmrgError(n, lib().dmrg_last_error().decode())
    return int(n)


def _ptr(a):
    """Address of a numpy array (host) or of a torch tensor (device)."""
    if a is None:
        return None
    if isinstance(a, np.ndarray):
        return a.ctypes.data
    return a.data_ptr()


def _stream_ptr(stream):
    if stream is None:
        return None
    return getattr(stream, "cuda_stream", stream)


def _structured(rows, dt, cols):
    rows = np.asarray(rows)
    out = np.zeros(len(rows), dtype=dt)
    for name, c in cols:
        out[name] = rows[:, c]
    return out


class OpsStore:
    """dmrg_ops_load: block-sparse operator store resident in HBM."""

    def __init__(self, secL, secR, ops, blocks, values, lin_ptr, lin_op, lin_coef):
        """secL/secR: int [n,3] (N, 2Sz, dim); ops: int [nops,8] (side, kind, p, q, dN, d2Sz, first_block,
        nblocks); blocks: int [nblk,3] (row_sector, col_sector, offset); values: float64 numpy array (host)
        or CUDA torch tensor (device); lincomb CSR as in dmrg_sigma.h.  complex128 values (numpy) or a complex128 CUDA
        tensor select dmrg_ops_load_z (spin-orbit stores); lin_coef is then complex too."""
        self._h = None
        is_z = values is not None and (values.dtype == np.complex128 if isinstance(values, np.ndarray) else values.is_complex())
        is_z = is_z or (values is None and np.asarray(lin_coef).dtype.kind == "c")
        self.is_complex = bool(is_z)
        sl = _structured(np.asarray(secL).reshape(-1, 3), SECTOR_DT, (("n", 0), ("two_sz", 1), ("dim", 2)))
        sr = _structured(np.asarray(secR).reshape(-1, 3), SECTOR_DT, (("n", 0), ("two_sz", 1), ("dim", 2)))
        od = _structured(np.asarray(ops).reshape(-1, 8), OP_DT, (("side", 0), ("kind", 1), ("p", 2), ("q", 3), ("dn", 4),
                                                                  ("d2sz", 5), ("first_block", 6), ("nblocks", 7)))
        bd = _structured(np.asarray(blocks).reshape(-1, 3), BLOCK_DT, (("row_sector", 0), ("col_sector", 1), ("offset", 2)))
        on_dev = 0
        if values is None:
            nvalues = int(max((b[2] for b in np.asarray(blocks).reshape(-1, 3)), default=0)) + (1 << 40)
        elif isinstance(values, np.ndarray):
            values = np.ascontiguousarray(values, dtype=np.complex128 if is_z else np.float64)
        else:
            assert values.is_cuda and values.is_contiguous() and values.element_size() == (16 if is_z else 8)
            on_dev = 1
        lp = np.ascontiguousarray(lin_ptr, dtype=np.int64)
        lo = np.ascontiguousarray(lin_op, dtype=np.int32)
        lc = np.ascontiguousarray(lin_coef, dtype=np.complex128 if is_z else np.float64)
        if values is not None:
            nvalues = int(values.size if on_dev == 0 else values.numel())
        h = C.c_void_p()
        load = lib().dmrg_ops_load_z if is_z else lib().dmrg_ops_load
        _check(load(_ptr(sl), len(sl), _ptr(sr), len(sr), _ptr(od), len(od), _ptr(bd), len(bd),
                                   _ptr(values), nvalues, on_dev, _ptr(lp), _ptr(lo), _ptr(lc), len(lp) - 1, C.byref(h)))
        self._h = h

    @classmethod
    def _from_handle(cls, h):
        self = cls.__new__(cls)
        self._h = h
        return self

    @property
    def device_bytes(self):
        return int(lib().dmrg_ops_device_bytes(self._h))

    @property
    def num_ops(self):
        return int(lib().dmrg_ops_num_ops(self._h))

    def sectors(self, side):
        """int32 [n,3] (N, 2Sz, dim) of side 0 (L) / 1 (R)."""
        n = _check_count(lib().dmrg_ops_sectors(self._h, int(side), None, 0))
        out = np.zeros(n, dtype=SECTOR_DT)
        _check_count(lib().dmrg_ops_sectors(self._h, int(side), _ptr(out), n))
        return np.stack([out[k] for k in ("n", "two_sz", "dim")], axis=1).astype(np.int32).reshape(-1, 3)

    def export(self):
        """dmrg_ops_export: (ops int64 [nops,8], blocks int64 [nblk,3], values float64) in the dmrg_ops_load format."""
        L = lib()
        no, nb, nv = (int(f(self._h)) for f in (L.dmrg_ops_num_ops, L.dmrg_ops_num_blocks, L.dmrg_ops_num_values))
        od, bd, vals = np.zeros(no, dtype=OP_DT), np.zeros(max(nb, 1), dtype=BLOCK_DT), np.zeros(max(nv, 1))
        _check(L.dmrg_ops_export(self._h, _ptr(od), _ptr(bd), _ptr(vals)))
        ops = np.stack([od[k].astype(np.int64) for k in ("side", "kind", "p", "q", "dn", "d2sz", "first_block", "nblocks")], axis=1)
        blocks = np.stack([bd[k].astype(np.int64) for k in ("row_sector", "col_sector", "offset")], axis=1)[:nb]
        return ops.reshape(-1, 8), blocks.reshape(-1, 3), vals[:nv]

    @staticmethod
    def _lin_args(lin_ops, lin_ptr, lin_op, lin_coef, lin_trans):
        od = _structured(np.asarray(lin_ops).reshape(-1, 8), OP_DT, (("side", 0), ("kind", 1), ("p", 2), ("q", 3), ("dn", 4), ("d2sz", 5),
                                                                     ("first_block", 6), ("nblocks", 7)))
        lp = np.ascontiguousarray(lin_ptr, dtype=np.int64)
        lo = np.ascontiguousarray(lin_op, dtype=np.int32)
        lc = np.ascontiguousarray(lin_coef, dtype=np.float64)
        lt = None if lin_trans is None else np.ascontiguousarray(lin_trans, dtype=np.int32)
        assert len(lo) == len(lc) == int(lp[-1]) and (lt is None or len(lt) == len(lo))
        return od, lp, lo, lc, lt

    def add_lincombs(self, lin_ops, lin_ptr, lin_op, lin_coef, lin_trans=None):
        """dmrg_ops_add_lincombs; lin_ops int [n,8] rows as in `ops` (p = row of lin_ptr).  Returns the id of the first new operator."""
        first = self.num_ops
        od, lp, lo, lc, lt = self._lin_args(lin_ops, lin_ptr, lin_op, lin_coef, lin_trans)
        _check(lib().dmrg_ops_add_lincombs(self._h, _ptr(od), len(od), _ptr(lp), _ptr(lo), _ptr(lc), _ptr(lt), len(lp) - 1))
        return first

    def derive(self, lin_ops, lin_ptr, lin_op, lin_coef, lin_trans=None):
        """dmrg_ops_derive: a new store whose operators are the given linear combinations of this store's operators."""
        od, lp, lo, lc, lt = self._lin_args(lin_ops, lin_ptr, lin_op, lin_coef, lin_trans)
        h = C.c_void_p()
        _check(lib().dmrg_ops_derive(self._h, _ptr(od), len(od), _ptr(lp), _ptr(lo), _ptr(lc), _ptr(lt), len(lp) - 1, C.byref(h)))
        return OpsStore._from_handle(h)

    @staticmethod
    def join(left, right):
        """dmrg_ops_join: consumes both stores (their handles are cleared)."""
        h = C.c_void_p()
        _check(lib().dmrg_ops_join(left._h, right._h, C.byref(h)))
        left._h = right._h = None
        return OpsStore._from_handle(h)

    def free(self):
        if self._h is not None:
            lib().dmrg_ops_free(self._h)
            self._h = None

    def __del__(self):
        try:
            self.free()
        except Exception:
            pass


class Plan:
    """dmrg_plan_create and the calls that take a plan (dmrg_sigma, dmrg_hdiag, dmrg_davidson)."""

    def __init__(self, ops, term_coef, term_idx, site_ops, site_parity, n_total, two_sz_total, workspace_bytes=0, **options):
        """term_idx: int [nterms,6] (op_l, trans_l, dot1, dot2, op_r, trans_r).
        options: fields of dmrg_plan_options (copy_mode, split_waves, min_split_stages, max_merged_cols,
        cost_order_only, split_small, release_r_store); passing any selects dmrg_plan_create_opts."""
        self._h = None
        self.ops = ops   # keep the store alive: the plan borrows it
        self.is_complex = bool(lib().dmrg_ops_is_complex(ops._h))
        ti = np.asarray(term_idx).reshape(-1, 6)
        td = np.zeros(len(ti), dtype=TERM_DT)
        td["coef"] = np.asarray(term_coef).real.astype(np.float64)
        for name, c in (("op_l", 0), ("trans_l", 1), ("dot1", 2), ("dot2", 3), ("op_r", 4), ("trans_r", 5)):
            td[name] = ti[:, c]
        so = np.ascontiguousarray(site_ops, dtype=np.complex128 if self.is_complex else np.float64).reshape(-1, 16)
        sp = np.ascontiguousarray(site_parity, dtype=np.int32)
        h = C.c_void_p()
        if self.is_complex:   # dmrg_plan_create_z: complex coefficients and site matrices, N only
            ci = np.ascontiguousarray(np.asarray(term_coef, dtype=np.complex128).imag, dtype=np.float64)
            po = np.zeros(1, dtype=PLANOPT_DT)
            po["workspace_bytes"] = int(workspace_bytes)
            for k, v in options.items():
                if k not in PLANOPT_DT.names or k == "reserved":
                    raise TypeError(f"unknown plan option {k!r}")
                po[k] = v
            assert int(two_sz_total) == 0
            _check(lib().dmrg_plan_create_z(ops._h, _ptr(td), _ptr(ci), len(td), _ptr(so), _ptr(sp), len(so), int(n_total), _ptr(po), C.byref(h)))
        elif options:
            po = np.zeros(1, dtype=PLANOPT_DT)
            po["workspace_bytes"] = int(workspace_bytes)
            for k, v in options.items():
                if k not in PLANOPT_DT.names or k == "reserved":
                    raise TypeError(f"unknown plan option {k!r}")
                po[k] = v
            _check(lib().dmrg_plan_create_opts(ops._h, _ptr(td), len(td), _ptr(so), _ptr(sp), len(so), int(n_total),
                                               int(two_sz_total), _ptr(po), C.byref(h)))
        else:
            _check(lib().dmrg_plan_create(ops._h, _ptr(td), len(td), _ptr(so), _ptr(sp), len(so), int(n_total),
                                          int(two_sz_total), int(workspace_bytes), C.byref(h)))
        self._h = h

    @property
    def psi_size(self):
        return int(lib().dmrg_plan_psi_size(self._h))

    def shard_terms(self):
        """Indices (into the term arrays given to the constructor) of the terms this plan evaluates, in plan order."""
        n = int(lib().dmrg_plan_shard_terms(self._h, None, 0))
        out = np.zeros(max(n, 1), dtype=np.int64)
        lib().dmrg_plan_shard_terms(self._h, _ptr(out), n)
        return out[:n]

    def psi_layout(self):
        """int64 [nblk,7]: (iL, c1, c2, iR, dL, dR, offset)."""
        n = int(lib().dmrg_plan_num_psi_blocks(self._h))
        out = np.zeros(n, dtype=PSIBLK_DT)
        _check(lib().dmrg_plan_psi_layout(self._h, _ptr(out)))
        return np.stack([out[k].astype(np.int64) for k in ("il", "c1", "c2", "ir", "dl", "dr", "offset")], axis=1)

    def stats(self):
        return {k: float(lib().dmrg_plan_stat(self._h, i)) for i, k in enumerate(STAT_KEYS)}

    def sigma(self, psi, sigma, stream=None):
        """sigma = H psi; psi, sigma: CUDA float64 tensors (device pointers), asynchronous on `stream`."""
        _check(lib().dmrg_sigma(self._h, _ptr(psi), _ptr(sigma), _stream_ptr(stream)))

    def sigma_host(self, psi, sigma, stream=None):
        """The same through host numpy buffers (H2D + sigma + D2H, synchronous)."""
        assert isinstance(psi, np.ndarray) and isinstance(sigma, np.ndarray)
        assert psi.dtype == np.float64 and sigma.dtype == np.float64 and psi.flags.c_contiguous and sigma.flags.c_contiguous
        _check(lib().dmrg_sigma_host(self._h, _ptr(psi), _ptr(sigma), _stream_ptr(stream)))

    def hdiag(self, diag, stream=None):
        _check(lib().dmrg_hdiag(self._h, _ptr(diag), _stream_ptr(stream)))

    def davidson(self, x, max_iter, max_space, tol, stream=None):
        """x: CUDA float64 tensor, in: guess, out: Ritz vector.  Returns dict(energy, resid, iters, thetas, converged)."""
        e, r, it = C.c_double(), C.c_double(), C.c_int32()
        thetas = np.zeros(max_iter)
        rc = _check(lib().dmrg_davidson(self._h, _ptr(x), int(max_iter), int(max_space), float(tol), C.byref(e), C.byref(r),
                                        C.byref(it), _ptr(thetas), _stream_ptr(stream)), allow=(-5,))
        return {"energy": e.value, "resid": r.value, "iters": it.value, "thetas": thetas[:it.value].copy(),
                "converged": rc == 0}

    def set_comm(self, comm):
        """dmrg_plan_set_comm: a sharded plan's dmrg_sigma / dmrg_hdiag then end with the all-reduce over `comm`."""
        _check(lib().dmrg_plan_set_comm(self._h, comm._h if comm is not None else None))
        self._comm = comm   # keep it alive: the plan borrows it

    def set_timing(self, enable):
        _check(lib().dmrg_plan_set_timing(self._h, 1 if enable else 0))

    def stage_ms(self):
        return tuple(float(lib().dmrg_plan_stage_ms(self._h, k)) for k in (0, 1, 2))

    def destroy(self):
        if self._h is not None:
            lib().dmrg_plan_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


class Comm:
    """dmrg_comm: the NCCL communicator of the operator-parallel sigma (one process per GPU)."""

    def __init__(self, unique_id, rank, world):
        self._h = None
        uid = np.ascontiguousarray(unique_id, dtype=np.uint8)
        h = C.c_void_p()
        _check(lib().dmrg_comm_create(_ptr(uid), int(rank), int(world), C.byref(h)))
        self._h = h
        self.rank, self.world = int(rank), int(world)

    @staticmethod
    def unique_id():
        buf = np.zeros(256, dtype=np.uint8)
        n = _check_count(lib().dmrg_comm_unique_id(_ptr(buf), len(buf)))
        return buf[:n].copy()

    @classmethod
    def from_torch_distributed(cls, device=None):
        """Rank 0 creates the id, torch.distributed ships it (any backend), every rank joins on its current device."""
        import torch
        import torch.distributed as dist
        rank, world = (dist.get_rank(), dist.get_world_size()) if dist.is_initialized() else (0, 1)
        uid = cls.unique_id() if rank == 0 else np.zeros(128, dtype=np.uint8)
        if world > 1:
            dev = device if (device is not None and dist.get_backend() == "nccl") else "cpu"
            t = torch.from_numpy(uid.copy()).to(dev)
            dist.broadcast(t, 0)
            uid = t.cpu().numpy()
        return cls(uid, rank, world)

    def destroy(self):
        if self._h is not None:
            lib().dmrg_comm_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


def renormalize(store, side, sec_new, wblocks, wvalues, new_ops, term_ptr, term_coef, term_idx, site_ops, site_parity,
                workspace_bytes=0, copy_mode=0, stream=None):
    """dmrg_renormalize (Eq. 8 / Eqs. 15-18).  Array formats of dmrg_workload/renorm_terms.py: wblocks int [nw,4]
    (old sector, site state, new sector, offset), term_idx int [nt,3] (op or -1, trans, site op).
    Returns (OpsStore of the renormalized block, stats dict)."""
    sn = _structured(np.asarray(sec_new).reshape(-1, 3), SECTOR_DT, (("n", 0), ("two_sz", 1), ("dim", 2)))
    wb = _structured(np.asarray(wblocks).reshape(-1, 4), WBLOCK_DT, (("old_sector", 0), ("site_state", 1), ("new_sector", 2), ("offset", 3)))
    wv = np.ascontiguousarray(wvalues, dtype=np.float64)
    od = _structured(np.asarray(new_ops).reshape(-1, 8), OP_DT, (("side", 0), ("kind", 1), ("p", 2), ("q", 3), ("dn", 4), ("d2sz", 5),
                                                                 ("first_block", 6), ("nblocks", 7)))
    tp = np.ascontiguousarray(term_ptr, dtype=np.int64)
    ti = np.asarray(term_idx).reshape(-1, 3)
    td = np.zeros(len(ti), dtype=RTERM_DT)
    td["coef"] = np.asarray(term_coef, dtype=np.float64)
    td["op"], td["trans"], td["site_op"] = ti[:, 0], ti[:, 1], ti[:, 2]
    so = np.ascontiguousarray(site_ops, dtype=np.float64).reshape(-1, 16)
    sp = np.ascontiguousarray(site_parity, dtype=np.int32)
    opt = np.zeros(1, dtype=RENORMOPT_DT)
    opt["workspace_bytes"], opt["copy_mode"] = int(workspace_bytes), int(copy_mode)
    st = np.zeros(1, dtype=RENORMSTATS_DT)
    h = C.c_void_p()
    _check(lib().dmrg_renormalize(store._h, int(side), _ptr(sn), len(sn), _ptr(wb), len(wb), _ptr(wv), len(wv), _ptr(od), len(od),
                                  _ptr(tp), _ptr(td), _ptr(so), _ptr(sp), len(so), _ptr(opt), _stream_ptr(stream), C.byref(h), _ptr(st)))
    return OpsStore._from_handle(h), {k: (float(st[k][0]) if st.dtype[k].kind == "f" else int(st[k][0])) for k in st.dtype.names}


def dots_static(V, w, out, stream=None):
    """dmrg_dots_static: out[i] = V[i] . w for the rows of the 2-D CUDA float64 tensor V (m <= DOTS_STATIC_MAX_VECTORS);
    allocates nothing -- the per-CTA partial sums live in the library's static device scratch."""
    m, n = (1, V.shape[0]) if V.dim() == 1 else V.shape
    stride = V.stride(0) if V.dim() == 2 else n
    _check(lib().dmrg_dots_static(_ptr(V), int(stride), int(m), _ptr(w), int(n), _ptr(out), _stream_ptr(stream)))


def fp64_peak_tflops(which, ms=200.0, stream=None):
    """Measured FP64 pipe peak: which = 0 DFMA, 1 DMMA.8x8x4."""
    v = float(lib().dmrg_fp64_peak_tflops(int(which), float(ms), _stream_ptr(stream)))
    if v < 0:
        raise DmrgError(int(v), lib().dmrg_last_error().decode())
    return v


def load_problem(pr, workspace_bytes=0, values=None, structure_only=False, **options):
    """Convenience: OpsStore + Plan from a dmrg_workload Problem (array formats of dmrg_workload/store.py).
    structure_only=True plans without a device (statistics / layout only); options -> dmrg_plan_options."""
    ops = OpsStore(pr.secL, pr.secR, pr.ops, pr.blocks,
                   None if structure_only else (pr.values if values is None else values),
                   pr.lin_ptr, pr.lin_op, pr.lin_coef)
    plan = Plan(ops, pr.term_coef, pr.term_idx, pr.site_ops, pr.site_parity, pr.N_tot, pr.twoSz_tot, workspace_bytes, **options)
    return ops, plan
