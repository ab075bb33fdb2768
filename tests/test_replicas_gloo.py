"""N > 1 path on CPU: the replicas-only measurement protocol (barrier + max over ranks) with gloo, world size 2."""
import os
import socket

import pytest

torch = pytest.importorskip("torch")
import torch.multiprocessing as mp  # noqa: E402


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q):
    os.environ.update(RANK=str(rank), WORLD_SIZE=str(world), LOCAL_RANK=str(rank), MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    from paper_2311_02854_b200 import replicas
    assert replicas.dist_env() == (rank, world, rank)
    assert replicas.init("gloo") == world
    replicas.barrier()
    ms_local = 100.0 + 50.0 * rank            # rank 1 is the slow one
    thr, ms = replicas.job_throughput(2.0e12, ms_local, world)
    q.put((rank, thr, ms))
    replicas.barrier()
    import torch.distributed as dist
    dist.destroy_process_group()


def test_replicas_protocol_world2():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    out = sorted(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, thr, ms in out:
        assert ms == 150.0                                   # max over ranks
        assert abs(thr - 2 * 2.0e12 / 0.150) < 1e-3          # whole-job throughput, weak scaling


def test_single_process_is_identity():
    from paper_2311_02854_b200 import replicas
    thr, ms = replicas.job_throughput(1.0e12, 200.0, 1)
    assert ms == 200.0 and thr == 1.0e12 / 0.2
