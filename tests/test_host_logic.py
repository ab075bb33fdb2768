"""CPU-only tests (-m "not gpu"): the C-ABI library loads and exports what include/dmrg_sigma.h declares, and
the host planner (structure-only operator store, no CUDA call) agrees with the oracle's own term expansion."""
import ctypes as C
import os
import re

import numpy as np
import pytest

import oracle
import paper_2311_02854_b200 as g
from dmrg_workload.problem import make_blocked_problem, make_direct_problem, random_psi

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module", autouse=True)
def built():
    from paper_2311_02854_b200 import build
    build.build()


def test_library_exports_every_declared_symbol():
    hdr = open(os.path.join(ROOT, "include", "dmrg_sigma.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(dmrg_[a-z0-9_]+)\s*\(", hdr))
    assert declared, "no prototypes found"
    L = C.CDLL(g.LIB_PATH)
    for name in declared:
        assert hasattr(L, name), f"{name} declared in the header but not exported"
    assert declared == set(g.EXPORTS), declared ^ set(g.EXPORTS)
    assert b"sm_100a" in g.lib().dmrg_version()


def test_struct_sizes_match_header():
    # the binding's numpy dtypes are the C structs of the header
    assert g.SECTOR_DT.itemsize == 12 and g.OP_DT.itemsize == 40 and g.BLOCK_DT.itemsize == 16
    assert g.TERM_DT.itemsize == 32 and g.PSIBLK_DT.itemsize == 32


CASES = {
    "cfg1": lambda: make_blocked_problem(8, 3, 8, 0, D=None, seed=1),
    "K7_trunc": lambda: make_blocked_problem(7, 3, 8, 0, D=10, seed=73, force_dmax=False, rotate=True),
    "K10_D60": lambda: make_blocked_problem(10, 4, 10, 0, D=60, seed=3),
    "direct_K12": lambda: make_direct_problem(12, 5, 12, 0, D=100, seed=1),
    "direct_K16_odd": lambda: make_direct_problem(16, 7, 15, 1, D=200, seed=2),
}


@pytest.fixture(scope="module", params=list(CASES))
def planned(request):
    pr = CASES[request.param]()
    ops, plan = g.load_problem(pr, structure_only=True)
    yield pr, ops, plan
    plan.destroy()
    ops.free()


def test_planner_layout_and_counts_match_oracle(planned):
    pr, ops, plan = planned
    assert plan.psi_size == pr.psi_size
    assert np.array_equal(plan.psi_layout(), pr.layout)
    _, st = oracle.opair_sigma(pr, random_psi(pr.psi_size, 1), return_stats=True)
    s = plan.stats()
    assert s["tasks"] == st["tasks"]                       # same (term, block, dot transition) expansion
    assert abs(s["canon_flops"] - st["flops"]) <= 1e-9 * max(1.0, st["flops"])
    # de-duplication never adds work; padding never removes it
    assert s["s1_flops"] + s["s2_flops"] <= s["canon_flops"] * (1 + 1e-12)
    assert s["padded_flops"] >= s["s1_flops"] + s["s2_flops"] - 1e-6
    assert s["chunks"] >= 1 and s["launches"] >= 1


def test_planner_chunking_is_structural(planned):
    """A tiny workspace splits the terms into many chunks without changing the executed work."""
    pr, ops, plan = planned
    small = g.Plan(ops, pr.term_coef, pr.term_idx, pr.site_ops, pr.site_parity, pr.N_tot, pr.twoSz_tot, workspace_bytes=1)
    a, b = plan.stats(), small.stats()
    assert b["chunks"] >= a["chunks"]
    assert b["tasks"] == a["tasks"] and b["canon_flops"] == a["canon_flops"]
    assert b["s2_flops"] == a["s2_flops"]
    assert b["s1_flops"] >= a["s1_flops"]        # fewer terms per chunk => fewer shared X products
    small.destroy()


def test_structure_only_store_refuses_compute(planned):
    pr, ops, plan = planned
    buf = np.zeros(pr.psi_size + 2)
    with pytest.raises(g.DmrgError) as ei:
        g._check(g.lib().dmrg_sigma(plan._h, buf.ctypes.data, buf.ctypes.data + 16, None))
    assert ei.value.code == -1
    with pytest.raises(g.DmrgError):
        g._check(g.lib().dmrg_hdiag(plan._h, buf.ctypes.data, None))


def test_argument_validation_without_gpu():
    pr = make_blocked_problem(6, 2, 6, 0, D=8, seed=62, force_dmax=False)
    ops, plan = g.load_problem(pr, structure_only=True)
    # a term that does not conserve (N, 2Sz)
    bad = pr.term_idx.copy()
    cre = next(i for i in range(len(pr.ops)) if pr.ops[i][0] == 0 and pr.ops[i][1] == 1)
    bad[0] = (cre, 0, 0, 0, -1, 0)
    with pytest.raises(g.DmrgError) as ei:
        g.Plan(ops, pr.term_coef, bad, pr.site_ops, pr.site_parity, pr.N_tot, pr.twoSz_tot)
    assert ei.value.code == -2
    # operator id out of range; left-slot operator that lives on the right block
    bad = pr.term_idx.copy()
    bad[0, 0] = len(pr.ops) + 5
    with pytest.raises(g.DmrgError) as ei:
        g.Plan(ops, pr.term_coef, bad, pr.site_ops, pr.site_parity, pr.N_tot, pr.twoSz_tot)
    assert ei.value.code == -1
    rop = next(i for i in range(len(pr.ops)) if pr.ops[i][0] == 1)
    bad = pr.term_idx.copy()
    bad[0, 0] = rop
    with pytest.raises(g.DmrgError):
        g.Plan(ops, pr.term_coef, bad, pr.site_ops, pr.site_parity, pr.N_tot, pr.twoSz_tot)
    # no psi block with these quantum numbers
    with pytest.raises(g.DmrgError):
        g.Plan(ops, pr.term_coef, pr.term_idx, pr.site_ops, pr.site_parity, 999, 0)
    # a block that violates its operator's charge is rejected at load time
    blocks = pr.blocks.copy()
    blocks[0, 0], blocks[0, 1] = blocks[0, 1], (blocks[0, 0] + 1) % len(pr.secL)
    with pytest.raises(g.DmrgError):
        g.OpsStore(pr.secL, pr.secR, pr.ops, blocks, None, pr.lin_ptr, pr.lin_op, pr.lin_coef)
    plan.destroy()
    ops.free()


def test_direct_fill_problem_is_hermitian_and_seeded():
    """Direct fill (cfg 3-5 recipe): the summed operator stays Hermitian (pin 3) and the values are a pure
    function of the seed, independent of the thread count used to draw them."""
    from dmrg_workload.store import _fill_normal
    pr = make_direct_problem(12, 5, 12, 0, D=60, seed=4)
    psi, phi = random_psi(pr.psi_size, 1), random_psi(pr.psi_size, 2)
    a, b = oracle.opair_sigma(pr, psi), oracle.opair_sigma(pr, phi)
    assert abs(phi @ a - b @ psi) < 1e-11 * np.linalg.norm(a)
    pr2 = make_direct_problem(12, 5, 12, 0, D=60, seed=4)
    assert np.array_equal(pr.values, pr2.values)
    x1, x2 = np.empty((1 << 24) + 1000), np.empty((1 << 24) + 1000)
    _fill_normal(x1, 7, nthreads=1)
    _fill_normal(x2, 7, nthreads=4)
    assert np.array_equal(x1, x2)


def test_term_subset_sampler_partitions_sigma():
    """bench.py --impl reference times the oracle on every stride-th term: the subsets must partition H."""
    from dmrg_workload.problem import term_subset_problem
    pr = make_direct_problem(12, 5, 12, 0, D=60, seed=4)
    psi = random_psi(pr.psi_size, 3)
    full = oracle.opair_sigma(pr, psi)
    n = len(pr.term_coef)
    acc = sum(oracle.opair_sigma(term_subset_problem(pr, np.arange(k, n, 4)), psi) for k in range(4))
    assert np.abs(acc - full).max() <= 1e-12 * np.linalg.norm(full)


def test_stage1_is_n_merged():
    """Stage 1 is planned as a few tall-and-wide GEMMs (R blocks stacked along N), not one GEMM per R block."""
    pr = make_direct_problem(16, 7, 16, 0, D=200, seed=3)
    ops, plan = g.load_problem(pr, structure_only=True)
    s = plan.stats()
    n_rblocks_used = len({(int(t[4]), int(t[5])) for t in pr.term_idx if t[4] >= 0})   # (R op, trans) pairs
    assert s["s1_jobs"] < 0.25 * n_rblocks_used * len(pr.secR)      # far fewer GEMMs than (op, sector) pairs
    assert s["s1_flops"] > 0 and s["padded_flops"] / (s["s1_flops"] + s["s2_flops"]) < 1.5
    plan.destroy()
    ops.free()


def test_split_small_option_only_regroups_launches():
    """dmrg_plan_options.split_small (measurement aid for ncu) moves small-block tiles into launches of their own:
    same tiles, same work, more launches."""
    pr = make_direct_problem(16, 7, 16, 0, D=200, seed=3)
    ops, plan = g.load_problem(pr, structure_only=True)
    plan16 = g.Plan(ops, pr.term_coef, pr.term_idx, pr.site_ops, pr.site_parity, pr.N_tot, pr.twoSz_tot, split_small=16)
    a, b = plan.stats(), plan16.stats()
    for k in ("s1_tiles", "s2_tiles", "s1_flops", "s2_flops", "padded_flops", "tasks", "chunks"):
        assert a[k] == b[k], k
    assert b["launches"] > a["launches"]
    plan16.destroy()
    plan.destroy()
    ops.free()


def test_plan_options_are_validated_and_structural():
    """Every policy of the planner is an explicit dmrg_plan_options field (no environment variables): split-K
    granularity and merged-stack width change the number of tiles / jobs but never the executed flops of stage 2."""
    import subprocess
    src = open(os.path.join(ROOT, "paper_2311_02854_b200", "csrc", "plan.cu")).read()
    assert "getenv" not in src
    pr = make_direct_problem(16, 7, 16, 0, D=200, seed=3)
    ops, plan = g.load_problem(pr, structure_only=True)
    a = plan.stats()
    fine = g.Plan(ops, pr.term_coef, pr.term_idx, pr.site_ops, pr.site_parity, pr.N_tot, pr.twoSz_tot, split_waves=4000.0, min_split_stages=1)
    narrow = g.Plan(ops, pr.term_coef, pr.term_idx, pr.site_ops, pr.site_parity, pr.N_tot, pr.twoSz_tot, max_merged_cols=64)
    assert fine.stats()["s2_tiles"] > a["s2_tiles"] and fine.stats()["s2_flops"] == a["s2_flops"]
    assert narrow.stats()["s1_jobs"] > a["s1_jobs"] and narrow.stats()["s1_flops"] == a["s1_flops"]
    assert a["xws_elems"] >= 2
    with pytest.raises(TypeError):
        g.Plan(ops, pr.term_coef, pr.term_idx, pr.site_ops, pr.site_parity, pr.N_tot, pr.twoSz_tot, no_such_option=1)
    for p_ in (fine, narrow, plan):
        p_.destroy()
    ops.free()


def test_tile_runs_only_regroup_stage1_tiles():
    """dmrg_plan_options.tile_run_stages hands stage-1 tiles out in runs of consecutive M tiles (one CTA, one descriptor
    fetch): the tiles, the work and the launches stay what they are; the plan holds fewer tile records."""
    pr = make_direct_problem(16, 7, 16, 0, D=200, seed=3)
    ops, plan = g.load_problem(pr, structure_only=True)
    single = g.Plan(ops, pr.term_coef, pr.term_idx, pr.site_ops, pr.site_parity, pr.N_tot, pr.twoSz_tot, tile_run_stages=1)
    longer = g.Plan(ops, pr.term_coef, pr.term_idx, pr.site_ops, pr.site_parity, pr.N_tot, pr.twoSz_tot, tile_run_stages=1000)
    a, b, c = plan.stats(), single.stats(), longer.stats()
    for k in ("s1_tiles", "s2_tiles", "s1_flops", "s2_flops", "padded_flops", "tasks", "chunks", "launches", "s1_fill", "s2_fill"):
        assert a[k] == b[k] == c[k], k
    # 64 bytes per tile record: runs shrink the descriptor tables, one tile per CTA is the largest
    assert c["plan_device_bytes"] <= a["plan_device_bytes"] < b["plan_device_bytes"]
    for p_ in (single, longer, plan):
        p_.destroy()
    ops.free()


def test_plan_is_the_same_whatever_the_thread_count():
    """Terms and chunks are planned by all host threads and merged in order: the tables (here: every statistic and the
    shard term lists) must not depend on how many threads the machine offers."""
    import subprocess
    import sys
    code = ("import sys, json; sys.path.insert(0, %r); import paper_2311_02854_b200 as g; "
            "from dmrg_workload.problem import make_direct_problem; "
            "pr = make_direct_problem(16, 7, 16, 0, D=200, seed=3); "
            "ops, plan = g.load_problem(pr, structure_only=True, workspace_bytes=1 << 22); "
            "print(json.dumps([plan.stats(), [int(t) for t in plan.shard_terms()[:50]]]))") % ROOT
    outs = []
    for cpus in ("0", None):
        cmd = [sys.executable, "-c", code] if cpus is None else ["taskset", "-c", cpus, sys.executable, "-c", code]
        outs.append(subprocess.run(cmd, check=True, capture_output=True, text=True).stdout.strip().splitlines()[-1])
    assert outs[0] == outs[1]
