"""Set-up helper: one CAEE layer on a GPU from a workloads.LayerConfig, through the binding.

Only allocation and argument marshalling live here (the synthetic weights are drawn expert by
expert so that the raw copies can be dropped once the library has packed them)."""
import torch

from . import binding as B
from . import workloads as wl


class Layer:
    def __init__(self, cfg, seed=0, max_tokens=128, kernel=B.CAEE_KERNEL_AUTO, keep_raw=False, device="cuda:0",
                 cache=None, layer_id=0, weight_seed=None, ep=None):
        """cache: a caee_cache handle — the layer's routed experts then live in pinned host memory and
        are served through the LFU cache (layer_id = its key there).  weight_seed: seed of the expert
        weights when it should differ from the router's seed (layers of a synthetic multi-layer model).
        ep: (rank, world, owner, obuf_peers_fn) — expert parallelism is set up BEFORE the weights and only the
        experts the rank owns (and the shared ones) are drawn and loaded; obuf_peers_fn(ctx) returns the peers'
        o-buffer addresses (the rank's own at [rank])."""
        self.cfg, self.seed, self.device, self.max_tokens = cfg, seed, device, max_tokens
        self.weight_seed = seed if weight_seed is None else weight_seed
        torch.cuda.set_device(device)
        self.ctx = B.caee_create(B.layer_desc(cfg, max_tokens, kernel))
        self.Wr, self.b_logit, self.corr_bias = wl.router(cfg, seed, device)
        B.caee_set_router(self.ctx, self.Wr, self.b_logit, self.corr_bias)
        self.part = wl.partitions(cfg)
        B.caee_set_partitions(self.ctx, self.part, cfg.D)
        if cache is not None:
            B.caee_cache_attach(cache, self.ctx, layer_id)         # before the weights; the cache starts empty
            self.resident = wl.residency(cfg, seed) * 0
        else:
            self.resident = wl.residency(cfg, seed)
            B.caee_set_residency(self.ctx, self.resident)          # before the weights: it decides where images live
        self.ticks_res, self.ticks_miss = wl.cost_tables(cfg)
        B.caee_set_cost_table(self.ctx, self.ticks_res, self.ticks_miss)
        n = cfg.E + cfg.S
        mine = lambda e: True
        if ep is not None:
            rank, world, owner, peers_fn = ep
            B.caee_set_ep(self.ctx, rank, world, owner, peers_fn(self.ctx))
            mine = lambda e: e >= cfg.E or owner[e] == rank
        none = dict.fromkeys(("gate", "up", "down", "gate_scale", "up_scale", "down_scale"))
        raw = [wl.expert_weights(cfg, self.weight_seed, e, device) if mine(e) else none for e in range(n)]
        fp8 = cfg.w_dtype == wl.DT_E4M3
        B.caee_set_weights(self.ctx, [r["gate"] for r in raw], [r["up"] for r in raw], [r["down"] for r in raw],
                           [r["gate_scale"] for r in raw] if fp8 else None, [r["up_scale"] for r in raw] if fp8 else None,
                           [r["down_scale"] for r in raw] if fp8 else None, pack=1)
        torch.cuda.synchronize()
        # the UMMA path owns packed copies; the SIMT path keeps reading the raw tensors
        self.raw = raw if (keep_raw or B.caee_kernel_is_simt(cfg, kernel)) else None
        if self.raw is None:
            del raw
            torch.cuda.empty_cache()

    def calibrate(self, n_sizes=8, iters=20):
        """S10 on this GPU: replace the workload's formula costs by the table caee_calibrate_cost measures (HBM tier for
        resident experts, pinned-host H2D tier for misses), keeping the workload's 2x straggler partition.  Returns the
        two fits."""
        import numpy as np
        fits = B.caee_calibrate_cost(self.ctx, B.caee_calib_opts(n_sizes, iters, 0, 0, 1, 0))
        tr, tm = B.caee_get_cost_table(self.ctx, self.cfg.E)
        mult = np.where(self.part == self.cfg.straggler_part, 2, 1).astype(np.int64)
        self.ticks_res, self.ticks_miss = tr * mult, tm * mult
        B.caee_set_cost_table(self.ctx, self.ticks_res, self.ticks_miss)
        return fits

    def close(self):
        if self.ctx is not None:
            B.caee_destroy(self.ctx)
            self.ctx = None
            self.raw = None

    def forward(self, x, params=None, scores=None, y=None, stats=None, stream=None):
        """Enqueue one layer step; returns y (no synchronisation)."""
        T = x.shape[0]
        if y is None:
            y = torch.empty_like(x)
        if scores is None:
            B.caee_moe_forward(self.ctx, x, T, params, y, stats, stream)
        else:
            B.caee_moe_forward_from_scores(self.ctx, x, scores, T, params, y, stats, stream)
        return y

    def last_routing(self, T):
        idx = torch.empty(T, self.cfg.k, dtype=torch.int32, device=self.device)
        gate = torch.empty(T, self.cfg.k, dtype=torch.float32, device=self.device)
        B.caee_last_routing(self.ctx, T, idx, gate)
        torch.cuda.synchronize()
        return idx.cpu().numpy(), gate.cpu().numpy()
