"""Host-side logic of expert parallelism (paper_2606_29982_b200/ep.py; PAPER.md:57,
97, 127) with world_size 2 and 3 on the gloo backend (CPU): the index conventions (home tokens, owner
table), the token all-gather with a ragged last block, the handle exchange, and the whole data flow
"dispatch -> computation -> aggregation" with the CPU oracle standing in for the device kernels: every
rank computes the rows of ITS experts (its segment of the dispatch plan), the rows travel to the
token's home rank, and the home rank's slot-order combine equals the single-device oracle bit for bit."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _tiny(T, H=16, I=8, E=8, S=1, k=3, seed=0):
    rng = np.random.default_rng(seed)
    x = rng.normal(size=(T, H)).astype(np.float32)
    W = lambda r, c: (0.3 * rng.normal(size=(r, c))).astype(np.float32)
    Wg, Wu, Wd = [W(I, H) for _ in range(E + S)], [W(I, H) for _ in range(E + S)], [W(H, I) for _ in range(E + S)]
    z = rng.normal(size=(T, E))
    s = (np.exp(z) / np.exp(z).sum(1, keepdims=True)).astype(np.float32)
    return x, Wg, Wu, Wd, s


def _worker(rank, world, port, T, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from oracle import ep_oracle
    from oracle import oracle as orc
    from paper_2606_29982_b200 import ep
    E, S, k, scale = 8, 1, 3, 2.5
    x, Wg, Wu, Wd, s = _tiny(T, E=E, S=S, k=k)
    lo, hi = ep.home_range(T, rank, world)
    # 1. the ranks' own tokens -> the step's x, on every rank
    xg = ep.gather_tokens(torch.from_numpy(x[lo:hi].copy()), T).numpy()
    ok_gather = np.array_equal(xg, x)
    xb = torch.from_numpy(x).to(torch.bfloat16)                       # the activation dtype of the UMMA paths
    ok_gather = ok_gather and torch.equal(ep.gather_tokens(xb[lo:hi].contiguous(), T), xb)
    # the handle exchange used for the o buffers
    hs = ep.exchange_bytes(bytes([rank]) * 64)
    ok_handles = [h[0] for h in hs] == list(range(world)) and all(len(h) == 64 for h in hs)
    # 2. the same batch-global decision everywhere (R40), then this rank's segment of the plan (R38)
    idx, gate = orc.route(s, None, k)
    keep = np.ones(E, np.uint8)
    keep[[1, 6]] = 0                                                     # two experts pruned: some slots re-routed
    idx, gate = orc.compensate(s, None, keep, idx, gate)
    owner = ep.owner_table(E, world)
    plan = ep_oracle.ep_plan(idx, owner, world)
    rows = []                                                            # (home, token, slot, row) of this rank's experts
    for i in range(plan["offs"][rank], plan["offs"][rank + 1]):
        t, j, e = int(plan["tok"][i]), int(plan["slot"][i]), int(plan["expert"][i])
        assert owner[e] == rank
        rows.append((ep.home_of(t, T, world), t, j, orc.expert_ffn(xg[t], Wg[e], Wu[e], Wd[e])))
    # 3. aggregation: every row goes to its token's home rank
    send = [[(t, j, r) for h, t, j, r in rows if h == dst] for dst in range(world)]
    allrows = [None] * world
    dist.all_gather_object(allrows, send)
    mine = [item for src in range(world) for item in allrows[src][rank]]
    # 4. combine at home, slot order; shared expert replicated (R39)
    back = {(t, j): r for t, j, r in mine}
    y = np.zeros((hi - lo, x.shape[1]), np.float64)
    for t in range(lo, hi):
        for j in range(k):
            if idx[t, j] >= 0:
                y[t - lo] += float(gate[t, j]) * back[(t, j)]
        y[t - lo] *= scale
        for sh in range(S):
            y[t - lo] += orc.expert_ffn(xg[t], Wg[E + sh], Wu[E + sh], Wd[E + sh])
    y_ref = orc.moe_tokens(x, list(range(lo, hi)), idx, gate, Wg, Wu, Wd, E, S, scale) if hi > lo else y
    n_expected = int(sum(1 for t in range(lo, hi) for j in range(k) if idx[t, j] >= 0))
    out.put((rank, ok_gather, ok_handles, bool(np.array_equal(y, y_ref)), len(mine) == n_expected, (lo, hi)))
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("world,T", [(2, 7), (2, 1), (3, 8)])
def test_expert_parallel_data_flow_over_gloo(world, T):
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, T, out)) for r in range(world)]
    for p in procs:
        p.start()
    got = sorted(out.get(timeout=180) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    covered = []
    for rank, ok_gather, ok_handles, ok_y, ok_count, (lo, hi) in got:
        assert ok_gather, "all-gathered x differs from the full batch"
        assert ok_handles and ok_y and ok_count
        covered += list(range(lo, hi))
    assert covered == list(range(T))                      # the home ranges tile the batch


def test_index_conventions():
    from paper_2606_29982_b200 import ep
    for T in (0, 1, 5, 8, 129):
        for world in (1, 2, 3, 8):
            ranges = [ep.home_range(T, r, world) for r in range(world)]
            assert [t for lo, hi in ranges for t in range(lo, hi)] == list(range(T))
            for r, (lo, hi) in enumerate(ranges):
                assert all(ep.home_of(t, T, world) == r for t in range(lo, hi))
                assert ep.local_token_count(T, r, world) == hi - lo
    assert list(ep.owner_table(8, 2)) == [0, 0, 0, 0, 1, 1, 1, 1]
    assert list(ep.owner_table(7, 3)) == [0, 0, 0, 1, 1, 1, 2]
