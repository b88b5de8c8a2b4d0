"""N > 1 is "replicas only": independent layers per rank, no data-path collective;
the only reduction is bench.py's timing (max over ranks) and token count (sum).  Covered here
with world_size 2 on the gloo backend (CPU)."""
import os
import socket

import torch
import torch.distributed as dist
import torch.multiprocessing as mp


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    ms_local = 2.0 if rank == 0 else 5.0          # rank 1 is the straggler
    value, ms = bench.job_throughput(ms_local, 128 * 10, world, "cpu")
    r, w, _ = bench.dist_env()
    out.put((rank, value, ms, r, w))
    dist.barrier()
    dist.destroy_process_group()


def test_job_throughput_is_all_tokens_over_slowest_rank():
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(out.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, value, ms, r, w in got:
        assert (r, w) == (rank, 2)
        assert ms == 5.0                                  # max over ranks
        assert abs(value - 2 * 1280 / 5e-3) < 1e-6        # whole-job tokens / slowest time


def test_single_rank_needs_no_process_group():
    import bench
    value, ms = bench.job_throughput(4.0, 128, 1, "cpu")
    assert ms == 4.0 and abs(value - 128 / 4e-3) < 1e-9
