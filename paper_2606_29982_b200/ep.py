"""Expert-parallel plumbing (include/caee.h "Expert parallelism").

One process per GPU over torch.distributed.  Everything arithmetic happens in libcaee's kernels; this
module only moves bytes and pointers:

  home_range / owner_table    the index conventions of caee_set_ep (contiguous token blocks, contiguous expert
                              blocks = the cost model's partition table)
  gather_tokens               all-gather of the ranks' own tokens into the step's x (ragged last block)
  EpGroup                     set-up (o-buffer handles exchanged through the process group, opened as peer
                              memory) and the step: gather -> caee_moe_forward (o rows stored into the home ranks'
                              buffers by the expert kernel) -> group barrier -> caee_ep_combine

The host-side index logic is covered on CPU with world_size-2 gloo process groups
(tests/test_ep_gloo.py); the device path on one GPU with `world` contexts in one process that
run their slices one after the other (tests/test_gpu_parity.py::test_expert_parallel_*).
"""
import numpy as np
import torch
import torch.distributed as dist


def tokens_per_rank(T, world):
    return max(1, -(-T // world))


def home_range(T, rank, world):
    """Home tokens of `rank` in a T-token step: [lo, hi)."""
    per = tokens_per_rank(T, world)
    lo = min(T, rank * per)
    return lo, min(T, lo + per)


def home_of(t, T, world):
    return t // tokens_per_rank(T, world)


def owner_table(E, world):
    """Contiguous blocks of ceil(E / world) experts per rank (the default partition table)."""
    per = -(-E // world)
    return (np.arange(E) // per).astype(np.int32)


def local_token_count(T, rank, world):
    lo, hi = home_range(T, rank, world)
    return hi - lo


def gather_tokens(x_local, T, group=None):
    """All-gather the ranks' own token rows into x [T, H] (every rank gets the same tensor).
    Ranks hold home_range(T, rank, world) rows; the blocks are padded to tokens_per_rank for the collective."""
    world, rank = dist.get_world_size(group), dist.get_rank(group)
    per = tokens_per_rank(T, world)
    lo, hi = home_range(T, rank, world)
    assert x_local.shape[0] == hi - lo, (x_local.shape, lo, hi)
    pad = torch.zeros((per,) + tuple(x_local.shape[1:]), dtype=x_local.dtype, device=x_local.device)
    pad[: hi - lo] = x_local
    if x_local.is_cuda and dist.get_backend(group) == "nccl":
        out = torch.empty((world * per,) + tuple(x_local.shape[1:]), dtype=x_local.dtype, device=x_local.device)
        dist.all_gather_into_tensor(out, pad, group=group)
        return out[:T]
    # gloo (CPU tensors, or CUDA tensors staged through the host: gloo gathers host memory only)
    host = pad.cpu().contiguous().view(torch.uint8)      # gloo knows few element types: bytes always work
    parts = [torch.empty_like(host) for _ in range(world)]
    dist.all_gather(parts, host, group=group)
    out = torch.cat(parts).view(x_local.dtype)[:T]
    return out.to(x_local.device)


def exchange_bytes(payload: bytes, group=None):
    """Every rank's `payload` (same length everywhere), in rank order."""
    world = dist.get_world_size(group)
    out = [None] * world
    dist.all_gather_object(out, payload, group=group)
    return out


class EpGroup:
    """One rank of an expert-parallel group around a layer context (binding handle `ctx`).  Construct it BEFORE
    caee_set_weights and the rank may pass NULL for the experts it does not own (it then holds E / world routed
    experts + the shared ones)."""

    def __init__(self, ctx, E, owner=None, group=None):
        from . import binding as B
        self.B, self.ctx, self.group = B, ctx, group
        self.world, self.rank = dist.get_world_size(group), dist.get_rank(group)
        self.owner = owner_table(E, self.world) if owner is None else np.ascontiguousarray(owner, dtype=np.int32)
        mine, _ = B.caee_ep_obuf(ctx)
        handles = exchange_bytes(B.caee_ep_ipc_export(ctx), group)
        self.peers = [mine if r == self.rank else B.caee_ep_ipc_open(ctx, handles[r]) for r in range(self.world)]
        B.caee_set_ep(ctx, self.rank, self.world, self.owner, self.peers)

    def step(self, x_local, T, params=None, y=None, stats=None):
        """x_local: this rank's home tokens.  Returns y [T, H] whose home rows are this rank's output."""
        B = self.B
        x = gather_tokens(x_local, T, self.group)
        if y is None:
            y = torch.empty_like(x)
        B.caee_moe_forward(self.ctx, x, T, params, None, stats)
        self._group_barrier()                 # every rank's expert kernel (and its peer stores) is complete
        B.caee_ep_combine(self.ctx, T, y)
        self._group_barrier()                 # nobody overwrites a peer's o rows before they are combined
        lo, hi = home_range(T, self.rank, self.world)
        return y, (lo, hi)

    def _group_barrier(self):
        """All ranks' enqueued work is complete.  NCCL's barrier is ordered on the stream; any other backend synchronises
        the device first and then meets on the host."""
        if dist.get_backend(self.group) != "nccl":
            torch.cuda.synchronize()
        dist.barrier(group=self.group)
        if dist.get_backend(self.group) == "nccl":
            torch.cuda.synchronize()

    def close(self):
        for r, p in enumerate(self.peers):
            if r != self.rank:
                self.B.caee_ep_ipc_close(self.ctx, p)
        self.B.caee_set_ep(self.ctx, 0, 1, None, None)
