"""Operator parallelism over the GPUs of one node.

The paper distributes the O(K^2) terms mu over ranks, replicates the trial vector (NCCL broadcast) and reduces the
partial sigma vectors (NCCL reduce).  Here every rank holds the whole bond description (term list, sector tables) but
loads and plans only its share: `Plan(..., shard_rank=r, shard_count=n)` keeps one contiguous range of the planner's
term list, which is ordered by R operator, so a rank needs the complementary R operators of its range only
(`needed_ops` lists them) plus the O(K) one-index operators.  One H psi is then

    partial = dmrg_sigma(plan_r, psi)          # every rank, same psi (the Davidson vectors are replicated: all ranks
    sigma   = all_reduce(partial, SUM)         #  run the same deterministic vector algebra on the same sigma)

i.e. ONE collective of psi_size doubles (61 MB at cfg 5) per H psi over NVLink 5 / NVSwitch -- < 0.2 ms at the measured
725 GB/s bus bandwidth against ~250 ms of compute per rank at 8 GPUs.  BASELINE.json's north_star fixes the headline to one GPU
("replicas only"); this module is the sharded variant of the same path, covered on CPU by a gloo world-size-2 test
(partition + reduce against the oracle) and on one GPU by summing the shards' partial sigmas.
"""
import numpy as np


def all_reduce_sum(t):
    """Sum a tensor over the ranks of the default process group (NCCL on GPUs, gloo on CPU); no-op without one."""
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return t


def sharded_sigma(plan, psi, sigma, stream=None):
    """sigma = H psi with the terms sharded over ranks: this rank's partial product, then one all-reduce.
    psi, sigma: CUDA float64 tensors; `plan` was created with shard_rank / shard_count of this rank."""
    import torch
    plan.sigma(psi, sigma, stream)
    if stream is not None:
        with torch.cuda.stream(stream):
            all_reduce_sum(sigma)
    else:
        all_reduce_sum(sigma)
    return sigma


def needed_ops(term_idx, term_ids, ops, lin_ptr, lin_op):
    """Operator ids a shard must hold: those its terms name, plus the summands of the linear combinations among them."""
    ti = np.asarray(term_idx)[np.asarray(term_ids, dtype=np.int64)]
    used = {int(o) for o in ti[:, [0, 4]].ravel() if o >= 0}
    ops = np.asarray(ops)
    for o in list(used):
        if int(ops[o][1]) == 7:
            j = int(ops[o][2])
            used.update(int(x) for x in lin_op[int(lin_ptr[j]):int(lin_ptr[j + 1])])
    return sorted(used)
