"""GPU parity of the spin-orbit path (complex FP64, U(1)_N only, two-by-two dot blocks: SURVEY section 8(f) NEXT-4,
PAPER.md:97,285) through the C ABI (dmrg_ops_load_z, dmrg_plan_create_z, dmrg_sigma, dmrg_hdiag, dmrg_davidson)
against the complex oracle oracle/zsigma.py, element by element.

Bar: max|d sigma| / ||sigma||_2 <= 1e-11, Davidson energies within 1e-9 (BASELINE.json north_star), sigma bitwise
reproducible run to run.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from oracle import zsigma  # noqa: E402
from dmrg_workload.integrals import make_so_integrals  # noqa: E402
from dmrg_workload.problem import determinant_map, make_blocked_problem, make_direct_problem, random_psi_z  # noqa: E402

TOL_SIGMA = 1e-11
TOL_E = 1e-9


def _gpu():
    import paper_2311_02854_b200 as g
    if not torch.cuda.is_available():
        pytest.fail("gpu-marked test needs a CUDA device")
    return g


def _sigma_gpu(plan, psi):
    d_psi = torch.from_numpy(psi).cuda()
    d_sig = torch.empty_like(d_psi)
    plan.sigma(d_psi, d_sig, torch.cuda.current_stream())
    torch.cuda.synchronize()
    return d_sig.cpu().numpy()


def _make(kind, K, nL, N, D, seed, **kw):
    ints = make_so_integrals(K, seed=seed)
    if kind == "blocked":
        return make_blocked_problem(K, nL, N, 0, D=D, seed=seed, force_dmax=False, ints=ints, **kw)
    return make_direct_problem(K, nL, N, 0, D=D, seed=seed, ints=ints)


CASES = {
    "K5_exact_1left": dict(kind="blocked", K=5, nL=1, N=4, D=None, seed=41),
    "K6_exact": dict(kind="blocked", K=6, nL=2, N=6, D=None, seed=42),
    "K6_trunc_rot": dict(kind="blocked", K=6, nL=3, N=5, D=12, seed=43, rotate=True),
    "K7_trunc": dict(kind="blocked", K=7, nL=2, N=7, D=20, seed=44),
    "K10_direct_D80": dict(kind="direct", K=10, nL=4, N=10, D=80, seed=45),
    "K12_direct_D300_odd": dict(kind="direct", K=12, nL=5, N=11, D=300, seed=46),   # several tiles, ragged tails, split-K
}


@pytest.fixture(scope="module", params=list(CASES))
def case(request):
    g = _gpu()
    pr = _make(**CASES[request.param])
    ops, plan = g.load_problem(pr)
    yield request.param, pr, plan
    plan.destroy()
    ops.free()


def test_layout_and_sizes(case):
    _, pr, plan = case
    assert plan.is_complex and plan.psi_size == 2 * pr.psi_size   # doubles
    assert np.array_equal(plan.psi_layout(), pr.layout)           # offsets in complex numbers


def test_sigma_matches_oracle(case):
    name, pr, plan = case
    for seed in (5, 6):
        psi = random_psi_z(pr.psi_size, seed)
        ref, st = zsigma.zopair_sigma(pr, psi, return_stats=True)
        got = _sigma_gpu(plan, psi)
        err = np.abs(got - ref).max() / np.linalg.norm(ref)
        assert err <= TOL_SIGMA, (name, err)
    s = plan.stats()
    assert s["tasks"] == st["tasks"]
    assert abs(s["canon_flops"] - st["flops"]) <= 1e-9 * max(1.0, st["flops"])   # 8 M N K per complex GEMM


def test_sigma_bitwise_reproducible_and_linear(case):
    _, pr, plan = case
    psi = random_psi_z(pr.psi_size, 11)
    a = _sigma_gpu(plan, psi)
    for _ in range(2):
        assert np.array_equal(a, _sigma_gpu(plan, psi))
    b = _sigma_gpu(plan, 1j * psi)   # complex-linear, not anti-linear: H (i psi) = i H psi, exactly (a relabelling of re / im)
    assert np.abs(b - 1j * a).max() <= 1e-13 * np.abs(a).max()


def test_hdiag_matches_oracle(case):
    name, pr, plan = case
    d = torch.empty(pr.psi_size, dtype=torch.complex128, device="cuda")
    plan.hdiag(d, torch.cuda.current_stream())
    torch.cuda.synchronize()
    got = d.cpu().numpy()
    ref = zsigma.zopair_hdiag(pr).real
    assert np.array_equal(got.real, got.imag)   # the real diagonal in both slots of every pair
    assert np.abs(got.real - ref).max() <= 1e-11 * max(1.0, np.abs(ref).max()), name


def test_sigma_equals_the_definition_and_davidson_finds_the_ground_state():
    """End to end against the DEFINITION: complex Slater-Condon H over all C(12, 6) = 924 determinants of K = 6
    (untruncated 2-1-1-2): sigma == H psi, and dmrg_davidson -- unchanged, on the vector as 2n reals -- converges to
    the lowest eigenvalue of the Hermitian H with a complex eigenvector."""
    g = _gpu()
    K, N = 6, 6
    pr = make_blocked_problem(K, 2, N, 0, D=None, seed=9, track=True, ints=make_so_integrals(K, seed=19))
    dets, Pm = determinant_map(pr)
    assert len(dets) == 924 == pr.psi_size
    H = zsigma.zfci_dense_h(dets, 2 * K, pr.ints.dense_h(), pr.ints.dense_V())
    ops, plan = g.load_problem(pr)
    psi = random_psi_z(pr.psi_size, 5)
    ref = Pm.conj().T @ (H @ (Pm @ psi))
    assert np.abs(_sigma_gpu(plan, psi) - ref).max() / np.linalg.norm(ref) <= TOL_SIGMA
    e0 = np.linalg.eigvalsh(H)[0]
    x = torch.from_numpy(random_psi_z(pr.psi_size, 9)).cuda()
    res = plan.davidson(x, max_iter=400, max_space=30, tol=1e-8, stream=torch.cuda.current_stream())
    assert res["converged"] and res["resid"] <= 1e-8
    assert abs(res["energy"] - e0) < TOL_E
    xv = x.cpu().numpy()
    assert abs(np.linalg.norm(xv) - 1.0) < 1e-12
    hx = Pm.conj().T @ (H @ (Pm @ xv))
    assert np.linalg.norm(hx - e0 * xv) < 1e-7 and np.abs(xv.imag).max() > 1e-3
    plan.destroy()
    ops.free()


def test_plan_options_and_sharding():
    """copy_mode / split_small leave the complex sigma bitwise unchanged; split-K granularity, stack width and a small
    workspace (several chunks) only change rounding; the two shards of the term list add up."""
    g = _gpu()
    pr = _make("direct", 10, 4, 10, 120, 51)
    psi = random_psi_z(pr.psi_size, 2)
    ref = zsigma.zopair_sigma(pr, psi)
    nrm = np.linalg.norm(ref)
    ops, plan = g.load_problem(pr)
    base = _sigma_gpu(plan, psi)
    assert np.abs(base - ref).max() / nrm <= TOL_SIGMA
    plan.destroy()
    for opt, bitwise in ((dict(copy_mode=1), True), (dict(split_small=16), True),
                         (dict(split_waves=2000.0, min_split_stages=2), False), (dict(max_merged_cols=64), False),
                         (dict(workspace_bytes=1 << 20), False)):
        ws = opt.pop("workspace_bytes", 0)
        plan = g.Plan(ops, pr.term_coef, pr.term_idx, pr.site_ops, pr.site_parity, pr.N_tot, 0, ws, **opt)
        got = _sigma_gpu(plan, psi)
        if bitwise:
            assert np.array_equal(got, base), opt
        assert np.abs(got - ref).max() / nrm <= TOL_SIGMA, opt
        if ws:
            assert plan.stats()["chunks"] > 1
        plan.destroy()
    parts = []
    for r in range(2):
        plan = g.Plan(ops, pr.term_coef, pr.term_idx, pr.site_ops, pr.site_parity, pr.N_tot, 0, 0, shard_rank=r, shard_count=2)
        parts.append(_sigma_gpu(plan, psi))
        plan.destroy()
    assert np.abs(parts[0] + parts[1] - ref).max() / nrm <= TOL_SIGMA
    assert min(np.abs(p).max() for p in parts) > 0
    ops.free()


def test_real_and_complex_entry_points_do_not_mix():
    g = _gpu()
    pr = _make("blocked", 5, 1, 4, None, 41)
    ops, plan = g.load_problem(pr)
    td = np.zeros(len(pr.term_idx), dtype=g.TERM_DT)
    so = np.zeros((len(pr.site_ops), 16))
    import ctypes as C
    h = C.c_void_p()
    rc = g.lib().dmrg_plan_create(ops._h, td.ctypes.data, len(td), so.ctypes.data, pr.site_parity.ctypes.data, len(so), pr.N_tot, 0, 0, C.byref(h))
    assert rc == -1 and b"dmrg_plan_create_z" in g.lib().dmrg_last_error()
    with pytest.raises(g.DmrgError):
        ops.export()
    plan.destroy()
    ops.free()
