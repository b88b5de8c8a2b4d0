"""Expert parallelism across PROCESSES on one GPU: two ranks, each a process
with its own CUDA context and a layer context that holds only the experts it owns; the o buffers are exchanged as CUDA
IPC handles (caee_ep_ipc_export / caee_ep_ipc_open) through a gloo process group, every rank's expert kernel stores its
o rows into the home rank's buffer through the mapped peer pointer, and paper_2606_29982_b200/ep.py's EpGroup drives
the step (token all-gather, forward, group barrier, home-token combine).  The ranks only meet at host barriers — no
kernel waits for another process.  The assembled y must equal the single-device step bit for bit."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

pytestmark = pytest.mark.gpu


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _worker(rank, world, port, T, mode, out):
    try:
        _worker_body(rank, world, port, T, mode, out)
    except Exception as e:      # report instead of leaving the parent waiting for the queue
        out.put((rank, None, None, None, f"{type(e).__name__}: {e}"))
        raise


def _worker_body(rank, world, port, T, mode, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from paper_2606_29982_b200 import binding as B
    from paper_2606_29982_b200 import ep
    from paper_2606_29982_b200 import workloads as wl
    from paper_2606_29982_b200.layer import Layer
    torch.cuda.set_device(0)
    cfg = wl.scaled(wl.C3, name="R1-small", H=1024, I=384, E=64, k=4, n_group=8, topk_group=4, D=8, straggler_part=3, cost_ticks_ns=901)
    owner = ep.owner_table(cfg.E, world)
    group = {}

    def peers(ctx):           # called by Layer BEFORE the weights are set: the group is formed here
        group["g"] = ep.EpGroup(ctx, cfg.E, owner)
        return group["g"].peers

    L = Layer(cfg, seed=0, max_tokens=64, device="cuda:0", ep=(rank, world, owner, peers))
    G = group["g"]
    x = wl.hidden(cfg, T, 31, "cuda:0")                                  # the same seeded batch on every rank
    params = None if mode == "dense" else B.prune_params(B.CAEE_PRUNE_CIR, 0.8)
    lo, hi = ep.home_range(T, rank, world)
    y, (lo2, hi2) = G.step(x[lo:hi].contiguous(), T, params)
    torch.cuda.synchronize()
    mine = y[lo:hi].view(torch.int16).cpu().numpy().copy()
    dist.barrier()
    G.close()
    L.close()
    # the single-device reference, computed by rank 0 after the group is gone
    ref = None
    if rank == 0:
        L1 = Layer(cfg, seed=0, max_tokens=64, device="cuda:0")
        y1 = L1.forward(x, params)
        torch.cuda.synchronize()
        ref = y1.view(torch.int16).cpu().numpy().copy()
        L1.close()
    out.put((rank, (lo, hi), (lo2, hi2), mine, ref))
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("T,mode", [(29, "dense"), (8, "cir")])
def test_expert_parallel_two_processes_ipc(T, mode):
    world = 2
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, T, mode, out)) for r in range(world)]
    for p in procs:
        p.start()
    got = sorted((out.get(timeout=300) for _ in procs), key=lambda g: g[0])
    for g in got:
        assert g[1] is not None, f"rank {g[0]} failed: {g[4]}"
    for p in procs:
        p.join(timeout=120)
        assert p.exitcode == 0
    ref = got[0][4]
    assert ref is not None
    for rank, (lo, hi), (lo2, hi2), mine, _ in got:
        assert (lo, hi) == (lo2, hi2)
        assert np.array_equal(mine, ref[lo:hi]), f"rank {rank}: home rows differ from the single-device step"
