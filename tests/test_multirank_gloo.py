"""world_size-2 gloo test (CPU) of the only cross-rank logic the benchmark has: "replicas only" -- no data-path
collective, a barrier and the MAX over ranks of the device time; whole-job value = all ranks' tokens / that."""
import os
import socket

import torch.multiprocessing as mp


def _worker(rank, world, port, q):
    import torch.distributed as dist
    from paper_2607_04181_b200 import multirank as M
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    M.barrier()
    local_ms = 10.0 if rank == 0 else 25.0                       # rank 1 is the slow replica
    value, ms_step = M.job_throughput(64, 5, local_ms)
    q.put((rank, M.world(), M.max_over_ranks(local_ms), value, ms_step))
    dist.destroy_process_group()


def test_replicas_only_aggregation_world2():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, world, mx, value, ms_step in got:
        assert world == 2 and mx == 25.0                          # every rank sees the slowest rank's time
        assert abs(value - 2 * 64 * 5 / 25e-3) < 1e-6 and abs(ms_step - 5.0) < 1e-12


def test_single_process_is_the_identity():
    from paper_2607_04181_b200 import multirank as M
    assert M.world() == 1 and M.max_over_ranks(3.5) == 3.5
    v, ms = M.job_throughput(64, 10, 2.0)
    assert abs(v - 64 * 10 / 2e-3) < 1e-6 and ms == 0.2
