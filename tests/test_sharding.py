"""NEXT-3, operator parallelism: the planner's term partition and the reduce of the partial sigmas.

CPU: (i) the shards of a structure-only plan partition the term list exactly and evenly (canonical cost); (ii) a gloo
world-size-2 run: every rank evaluates the ORACLE on the terms of its share and the ranks all-reduce -- the sum is the
oracle's full sigma.  GPU (one device, -m gpu): the partial sigmas of the shards, computed by dmrg_sigma one after the
other, add up to the unsharded dmrg_sigma to rounding, each R operator being needed by few shards."""
import os
import socket

import numpy as np
import pytest

torch = pytest.importorskip("torch")
import torch.multiprocessing as mp  # noqa: E402

import paper_2311_02854_b200 as g  # noqa: E402
from dmrg_workload.problem import make_direct_problem, random_psi, term_subset_problem  # noqa: E402


def _problem():
    return make_direct_problem(14, 6, 14, 0, D=120, seed=8)


@pytest.mark.parametrize("n", [2, 3, 8])
def test_shards_partition_the_terms_evenly(n):
    from paper_2311_02854_b200 import build, sharded
    build.build()
    pr = _problem()
    ops, full = g.load_problem(pr, structure_only=True)
    tot = full.stats()
    assert sorted(full.shard_terms()) == list(range(len(pr.term_coef)))
    seen, flops, tasks, nops = [], [], 0, []
    for r in range(n):
        p = g.Plan(ops, pr.term_coef, pr.term_idx, pr.site_ops, pr.site_parity, pr.N_tot, pr.twoSz_tot, shard_rank=r, shard_count=n)
        ids = p.shard_terms()
        seen += list(ids)
        st = p.stats()
        flops.append(st["canon_flops"])
        tasks += st["tasks"]
        nops.append(len(sharded.needed_ops(pr.term_idx, ids, pr.ops, pr.lin_ptr, pr.lin_op)))
        p.destroy()
    assert sorted(seen) == list(range(len(pr.term_coef)))                 # every term exactly once
    assert tasks == tot["tasks"] and abs(sum(flops) - tot["canon_flops"]) <= 1e-9 * tot["canon_flops"]
    assert max(flops) <= 1.25 * tot["canon_flops"] / n                    # balanced to within a term or two
    if n >= 3:
        assert max(nops) < 0.8 * len(pr.ops)                              # a shard needs only part of the operator store
    with pytest.raises(g.DmrgError):
        g.Plan(ops, pr.term_coef, pr.term_idx, pr.site_ops, pr.site_parity, pr.N_tot, pr.twoSz_tot, shard_rank=n, shard_count=n)
    full.destroy()
    ops.free()


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q):
    os.environ.update(RANK=str(rank), WORLD_SIZE=str(world), LOCAL_RANK=str(rank), MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), OMP_NUM_THREADS="2")
    import torch.distributed as dist
    import oracle
    from paper_2311_02854_b200 import replicas, sharded
    replicas.init("gloo")
    pr = _problem()
    ops, plan = g.load_problem(pr, structure_only=True, shard_rank=rank, shard_count=world)   # host planner only
    ids = plan.shard_terms()
    psi = random_psi(pr.psi_size, 4)
    partial = oracle.opair_sigma(term_subset_problem(pr, ids), psi)       # this rank's share, by the oracle
    t = torch.from_numpy(partial.copy())
    sharded.all_reduce_sum(t)                                             # the reduce of PAPER.md:162, gloo on CPU
    q.put((rank, len(ids), t.numpy().copy()))
    replicas.barrier()
    dist.destroy_process_group()


def test_gloo_two_ranks_reduce_to_the_full_sigma():
    import oracle
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    got = [q.get(timeout=300) for _ in range(world)]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    pr = _problem()
    ref = oracle.opair_sigma(pr, random_psi(pr.psi_size, 4))
    assert sum(n for _, n, _ in got) == len(pr.term_coef) and all(n > 0 for _, n, _ in got)
    for _, _, s in got:                                                   # every rank ends with the full sigma
        assert np.abs(s - ref).max() <= 1e-12 * np.linalg.norm(ref)


@pytest.mark.gpu
def test_gpu_partial_sigmas_add_up():
    if not torch.cuda.is_available():
        pytest.fail("gpu-marked test needs a CUDA device")
    import oracle
    pr = _problem()
    ops, full = g.load_problem(pr)
    psi = torch.from_numpy(random_psi(pr.psi_size, 4)).cuda()
    ref = torch.empty_like(psi)
    full.sigma(psi, ref, torch.cuda.current_stream())
    hd_ref = torch.empty_like(psi)
    full.hdiag(hd_ref, torch.cuda.current_stream())
    n = 4
    acc, hd = torch.zeros_like(psi), torch.zeros_like(psi)
    for r in range(n):
        p = g.Plan(ops, pr.term_coef, pr.term_idx, pr.site_ops, pr.site_parity, pr.N_tot, pr.twoSz_tot, shard_rank=r, shard_count=n)
        part, hpart = torch.empty_like(psi), torch.empty_like(psi)
        p.sigma(psi, part, torch.cuda.current_stream())
        p.hdiag(hpart, torch.cuda.current_stream())
        torch.cuda.synchronize()
        acc += part
        hd += hpart
        p.destroy()
    torch.cuda.synchronize()
    nrm = float(torch.linalg.norm(ref))
    assert float((acc - ref).abs().max()) <= 1e-13 * nrm
    assert float((hd - hd_ref).abs().max()) <= 1e-12 * max(1.0, float(hd_ref.abs().max()))
    orc = oracle.opair_sigma(pr, psi.cpu().numpy())
    assert np.abs(acc.cpu().numpy() - orc).max() <= 1e-11 * np.linalg.norm(orc)
    full.destroy()
    ops.free()


@pytest.mark.gpu
def test_gpu_comm_attached_plan_reduces_in_place():
    """dmrg_comm on one device (world size 1: the only size this box can run): the NCCL communicator is created, attached
    to a plan created as shard 0 of 1, and dmrg_sigma / dmrg_hdiag / dmrg_davidson go through ncclAllReduce on the caller's
    stream; results are those of the plain plan.  A communicator that does not match the plan's shard is refused."""
    if not torch.cuda.is_available():
        pytest.fail("gpu-marked test needs a CUDA device")
    pr = _problem()
    ops, plain = g.load_problem(pr)
    psi = torch.from_numpy(random_psi(pr.psi_size, 4)).cuda()
    ref = torch.empty_like(psi)
    plain.sigma(psi, ref, torch.cuda.current_stream())
    comm = g.Comm(g.Comm.unique_id(), 0, 1)
    p = g.Plan(ops, pr.term_coef, pr.term_idx, pr.site_ops, pr.site_parity, pr.N_tot, pr.twoSz_tot, shard_rank=0, shard_count=1)
    p.set_comm(comm)
    out = torch.empty_like(psi)
    p.sigma(psi, out, torch.cuda.current_stream())
    torch.cuda.synchronize()
    assert torch.equal(out, ref)
    x1, x2 = psi.clone(), psi.clone()
    r1 = plain.davidson(x1, max_iter=6, max_space=6, tol=0.0, stream=torch.cuda.current_stream())
    r2 = p.davidson(x2, max_iter=6, max_space=6, tol=0.0, stream=torch.cuda.current_stream())
    assert r1["energy"] == r2["energy"] and torch.equal(x1, x2)
    half = g.Plan(ops, pr.term_coef, pr.term_idx, pr.site_ops, pr.site_parity, pr.N_tot, pr.twoSz_tot, shard_rank=0, shard_count=2)
    with pytest.raises(g.DmrgError):
        half.set_comm(comm)
    half.destroy()
    p.destroy()
    comm.destroy()
    plain.destroy()
    ops.free()
