"""World-size-2 gloo test of the multi-GPU plumbing (replicas only: MAX of the per-rank time)."""
import os
import socket
import sys

import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    import torch.distributed as dist
    from paper_2402_18471_b200.replicas import job_throughput, max_over_ranks, replica_seed
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    secs = 2.0 if rank == 0 else 5.0
    out.put((rank, max_over_ranks(secs, world), job_throughput(100, 10, secs, world), replica_seed(7, rank)))
    dist.barrier()
    dist.destroy_process_group()


def test_max_over_ranks_world2():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert [r[1] for r in res] == [5.0, 5.0]                 # slowest replica sets the time
    assert [r[2] for r in res] == [2 * 100 * 10 / 5.0] * 2   # whole-job units / max time
    assert [r[3] for r in res] == [7, 1007]                  # distinct replica seeds


def test_single_rank_is_identity():
    sys.path.insert(0, ROOT)
    from paper_2402_18471_b200.replicas import job_throughput, max_over_ranks
    assert max_over_ranks(1.25, 1) == 1.25
    assert job_throughput(10, 4, 2.0, 1) == 20.0
