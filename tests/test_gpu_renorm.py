"""GPU parity of the renormalization step (dmrg_renormalize; Eq. 8, Eqs. 15-18) against
oracle/renorm.py, through the C ABI, on the same seeded inputs: every block of every renormalized operator, element
by element, max|d| <= 1e-11 * max|O| (FP64; the two sides associate the triple product differently).  Cases: tiny
multi-step chains on both sides (1 x 1 ... ragged blocks, truncated and rotated isometries), a chain where the output
store of one step is the input of the next (dmrg_ops_add_lincombs in between), and one step at cfg 2 size (K = 24,
D = 500, several tiles per block)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from dmrg_workload.integrals import make_integrals  # noqa: E402
from dmrg_workload.renorm_terms import build_renorm_problem  # noqa: E402
from oracle import renorm as oracle_renorm  # noqa: E402
from test_oracle_renorm import chain, max_diff  # noqa: E402


def _gpu():
    import paper_2311_02854_b200 as g
    if not torch.cuda.is_available():
        pytest.fail("gpu-marked test needs a CUDA device")
    return g


def load_old_store(g, rp):
    empty = np.zeros((0, 3), dtype=np.int32)
    secL, secR = (rp.sec_old, empty) if rp.side == 0 else (empty, rp.sec_old)
    return g.OpsStore(secL, secR, rp.ops, rp.blocks, rp.values, rp.lin_ptr, rp.lin_op, rp.lin_coef)


def gpu_step(g, rp, store=None, **kw):
    own = store is None
    store = store or load_old_store(g, rp)
    out, st = g.renormalize(store, rp.side, rp.sec_new, rp.wblocks, rp.wvalues, rp.new_ops, rp.term_ptr, rp.term_coef, rp.term_idx,
                            rp.site_ops, rp.site_parity, stream=torch.cuda.current_stream(), **kw)
    if own:
        store.free()
    return out, st


def exported_blocks(out, sec_new):
    ops, blocks, values = out.export()
    res = []
    for row in ops:
        d = {}
        for b in range(int(row[6]), int(row[6] + row[7])):
            r, c, off = (int(v) for v in blocks[b])
            d[(r, c)] = values[off:off + sec_new[r][2] * sec_new[c][2]].reshape(sec_new[r][2], sec_new[c][2])
        res.append(d)
    return res


def check_against_oracle(rp, out, tol=1e-11):
    ref = oracle_renorm.renormalize(rp)
    got = exported_blocks(out, rp.sec_new)
    assert len(got) == len(ref)
    worst = 0.0
    for key, a, b in zip(rp.new_keys, got, ref):
        scale = max([1.0] + [float(np.abs(m).max()) for m in b.values()])
        assert set(a) == set(b), key                                   # the same blocks are present
        d = max_diff(a, b) / scale
        worst = max(worst, d)
        assert d <= tol, (key, d)
    return worst


@pytest.mark.parametrize("side,sites,K,N,D,rot,seed", [
    (0, [0, 1, 2], 5, 6, 9, False, 3),
    (0, [0, 1, 2, 3], 6, 6, 12, True, 7),
    (1, [2, 3, 4], 5, 6, 9, False, 5),
    (1, [3, 4, 5], 6, 6, 7, True, 6),
    (0, [0, 1, 2, 3, 4], 10, 10, 40, False, 8),
    (1, [5, 6, 7, 8, 9], 10, 10, 60, True, 9),
])
def test_renormalize_matches_oracle(side, sites, K, N, D, rot, seed):
    g = _gpu()
    ints = make_integrals(K, seed=seed)
    for blk, k, outside, nb in chain(side, sites, ints, K, N, D, seed, rot):
        rp = build_renorm_problem(blk, k, side, ints, outside, nb)
        out, st = gpu_step(g, rp)
        assert st["flops"] > 0 and st["launches"] >= 1
        assert np.array_equal(out.sectors(side), rp.sec_new)
        check_against_oracle(rp, out)
        out2, _ = gpu_step(g, rp, copy_mode=g.COPY_LDGSTS, workspace_bytes=1)   # many chunks, cp.async staging: bitwise the same
        a, b = out.export(), out2.export()
        assert all(np.array_equal(x, y) for x, y in zip(a, b))
        out.free()
        out2.free()


def test_chained_steps_stay_on_the_device():
    """The output store of one step is the input of the next one: only the linear-combination tables are added
    (dmrg_ops_add_lincombs).  The final operators are compared with the oracle chain fed by its OWN previous output."""
    g = _gpu()
    K, N, D, seed, side = 8, 8, 16, 12, 0
    ints = make_integrals(K, seed=seed)
    dev = None
    for blk, k, outside, nb in chain(side, [0, 1, 2, 3, 4], ints, K, N, D, seed, False):
        rp = build_renorm_problem(blk, k, side, ints, outside, nb)
        if dev is None:
            store = load_old_store(g, rp)
        else:
            # dev holds the stored operators in new_keys order == rp's stored-operator order? map by (kind, p, q)
            ops_dev = dev.export()[0]
            key_dev = {(int(r[1]), int(r[2]), int(r[3])): i for i, r in enumerate(ops_dev)}
            nst = int(np.sum(rp.ops[:, 1] != 7))
            perm = [key_dev[(int(r[1]), int(r[2]), int(r[3]))] for r in rp.ops[:nst]]
            lin_rows = rp.ops[nst:].copy()
            lin_op = np.array([perm[o] for o in rp.lin_op], dtype=np.int32)
            first = dev.add_lincombs(lin_rows, rp.lin_ptr, lin_op, rp.lin_coef)
            remap = {i: perm[i] for i in range(nst)}
            remap.update({nst + j: first + j for j in range(len(lin_rows))})
            ti = rp.term_idx.copy()
            ti[:, 0] = [remap[int(o)] if o >= 0 else -1 for o in ti[:, 0]]
            rp_dev_idx = ti
            store = dev
        idx = rp.term_idx if dev is None else rp_dev_idx
        out, _ = g.renormalize(store, side, rp.sec_new, rp.wblocks, rp.wvalues, rp.new_ops, rp.term_ptr, rp.term_coef, idx,
                               rp.site_ops, rp.site_parity, stream=torch.cuda.current_stream())
        store.free()
        check_against_oracle(rp, out, tol=1e-10)     # the inputs of later steps differ by earlier roundings
        dev = out
    dev.free()


def test_cfg2_size_step():
    """The last step of each side's chain at cfg 2 size (K = 24, D = 500: blocks of several tiles with ragged tails):
    every renormalized operator against the oracle, and the resulting sector tables are those of the cfg 2 bond."""
    g = _gpu()
    from dmrg_workload.problem import make_config
    pr = make_config("cfg2", track=False)
    K, nL, N = 24, 11, 24
    ints = pr.ints
    seed = 1 + 7919
    # replay the generator's chains (same Philox stream: L first, then R) to get the last step of each side
    rng = np.random.Generator(np.random.Philox(seed))
    from dmrg_workload import blocking
    last = {}
    for side, sites in ((0, list(range(0, nL))), (1, list(range(nL + 2, K)))):
        order = sites if side == 0 else sites[::-1]
        inside, blk = [], None
        for k in order:
            inside.append(k)
            outside = [P for P in range(2 * K) if (P >> 1) not in inside]
            site = blocking.site_block(k, ints, [P for P in range(2 * K) if (P >> 1) != k])
            if blk is None:
                blk = site
                continue
            args = (blk, site) if side == 0 else (site, blk)
            nb = blocking.merge(*args, ints, outside, K, N, 0, 500, rng, False, True, site_side="right" if side == 0 else "left")
            last[side] = (blk, k, outside, nb)
            blk = nb
    outs = {}
    for side in (0, 1):
        blk, k, outside, nb = last[side]
        rp = build_renorm_problem(blk, k, side, ints, outside, nb)
        out, st = gpu_step(g, rp)
        worst = check_against_oracle(rp, out)
        print(f"cfg2 side {side}: {len(rp.new_keys)} operators, {st['flops']:.3e} flop in {st['device_ms']:.2f} ms "
              f"({st['flops'] / st['device_ms'] * 1e-9:.2f} TFLOP/s), worst rel. diff {worst:.2e}")
        outs[side] = (out, rp)
    # the renormalized blocks are the cfg 2 bond's blocks: same sectors as the CPU-generated problem
    assert np.array_equal(outs[0][0].sectors(0), pr.secL) and np.array_equal(outs[1][0].sectors(1), pr.secR)
    for o, _ in outs.values():
        o.free()


def _cpu_chain_problem(K, nL, N, D, seed, force_dmax=False):
    """The CPU-blocked problem (dmrg_workload.blocking, as make_blocked_problem builds it) together with the site
    tensor of every step, so that the device chain can be driven through exactly the same projections."""
    from dmrg_workload import blocking
    from dmrg_workload.store import assemble, block_values_from_rblocks, sectors_of
    from dmrg_workload.terms import Partition, TermTable
    ints = make_integrals(K, seed)
    rng = np.random.Generator(np.random.Philox(seed + 7919))
    tensors, blocks = {}, {}
    for side, sites in ((0, list(range(0, nL))), (1, list(range(nL + 2, K)))):
        order = sites if side == 0 else sites[::-1]
        inside, blk = [], None
        for k in order:
            inside.append(k)
            outside = [P for P in range(2 * K) if (P >> 1) not in inside]
            site = blocking.site_block(k, ints, [P for P in range(2 * K) if (P >> 1) != k])
            if blk is None:
                blk = site
                continue
            args = (blk, site) if side == 0 else (site, blk)
            blk = blocking.merge(*args, ints, outside, K, N, 0, D, rng, False, force_dmax, site_side="right" if side == 0 else "left")
            tensors[(side, k)] = (blk.sectors, blk.dims, blk.site_tensor)
        blocks[side] = blk
    tt = TermTable(Partition(K, nL), ints)
    pr = assemble(tt, sectors_of(blocks[0]), sectors_of(blocks[1]), block_values_from_rblocks(blocks[0], blocks[1], ints), N, 0)
    return ints, pr, tensors


@pytest.mark.parametrize("K,nL,N,D,seed", [(8, 3, 8, 14, 31), (10, 4, 10, 40, 32), (12, 5, 12, 90, 33)])
def test_device_built_bond_gives_the_oracle_sigma(K, nL, N, D, seed):
    """End to end: both blocks grown on the device by chained dmrg_renormalize calls (the operators never leave HBM),
    complementary operators formed on the device, stores joined -- dmrg_sigma on that store equals the oracle's
    sigma on the CPU-blocked problem built through the same site tensors."""
    g = _gpu()
    import oracle
    from dmrg_workload.problem import random_psi
    from paper_2311_02854_b200 import bondgen
    ints, pr, tensors = _cpu_chain_problem(K, nL, N, D, seed)
    bond = bondgen.build_bond(g, K, nL, N, 0, D, ints, seed, tensor_provider=lambda side, k: tensors[(side, k)],
                              stream=torch.cuda.current_stream())
    assert np.array_equal(bond.secL, pr.secL) and np.array_equal(bond.secR, pr.secR) and np.array_equal(bond.layout, pr.layout)
    plan = g.Plan(bond.ops, bond.term_coef, bond.term_idx, bond.site_ops, bond.site_parity, N, 0)
    assert np.array_equal(plan.psi_layout(), pr.layout)
    for s in (5, 6):
        psi = random_psi(pr.psi_size, s)
        d = torch.from_numpy(psi).cuda()
        o = torch.empty_like(d)
        plan.sigma(d, o, torch.cuda.current_stream())
        torch.cuda.synchronize()
        ref = oracle.opair_sigma(pr, psi)
        assert np.abs(o.cpu().numpy() - ref).max() / np.linalg.norm(ref) <= 1e-10
    plan.destroy()
    bond.ops.free()
