"""Test/bench harness: builds a CAEE layer on the GPU from a workloads.LayerConfig through the
ctypes binding, and computes the matching oracle results on the host from the same bits.

The oracle side (oracle_*) only calls oracle/; the GPU side only calls the binding.
"""
import numpy as np
import torch

from oracle import oracle as orc
from paper_2606_29982_b200 import binding as B
from paper_2606_29982_b200.layer import Layer
from paper_2606_29982_b200 import workloads as wl

TOL = {wl.DT_F32: 1e-4, wl.DT_BF16: 2e-2, wl.DT_E4M3: 5e-2}   # x RMS(y), BASELINE.json north_star


class GpuLayer(Layer):
    def __init__(self, cfg, seed=0, max_tokens=128, kernel=B.CAEE_KERNEL_AUTO, keep_raw=True, device="cuda:0", **kw):
        super().__init__(cfg, seed, max_tokens, kernel, keep_raw, device, **kw)
        self._host = {}

    # ---- host copies of exactly the bits the GPU holds
    def host_expert(self, e):
        if e not in self._host:
            r = self.raw[e] if self.raw is not None else wl.expert_weights(self.cfg, self.weight_seed, e, self.device)
            self._host[e] = {k: wl.bits(v) for k, v in r.items()}
        return self._host[e]

    def w_eff(self):
        return orc.effective_cost(self.resident, self.ticks_res, self.ticks_miss)

    # ---- oracle pipeline on the same inputs
    def oracle_scores(self, x):
        return orc.scores(wl.bits(x), self.Wr.cpu().numpy(), self.b_logit.cpu().numpy(), self.cfg.score_fn)

    def oracle_decisions(self, s, mode=None, theta=0.0, flags=0, eps=None):
        """route -> prune -> compensate -> compact on scores s.  mode None = dense top-k.
        eps: bound on F_imp (switches the oracle's FLAG_IMP_BOUND on)."""
        c = self.cfg
        cb = None if self.corr_bias is None else self.corr_bias.cpu().numpy()
        idx, gate = orc.route(s, cb, c.k, c.n_group, c.topk_group, c.norm_topk)
        out = dict(idx0=idx.copy(), gate0=gate.copy())
        if mode is not None:
            if eps is not None:
                flags |= orc.FLAG_IMP_BOUND
            pr = orc.prune(mode, theta, flags, idx, gate, c.E, self.w_eff(), self.part, c.D, eps=0.0 if eps is None else eps)
            if mode != 0:
                idx, gate = orc.compensate(s, cb, pr["keep"], idx, gate, c.norm_topk, flags)
            out["prune"] = pr
        out["idx"], out["gate"] = idx, gate
        out["compact"] = orc.compact(idx, gate, c.E)
        return out

    def oracle_y(self, x, idx, gate, tokens, chunk=None):
        """chunk: evaluate that many tokens at a time and drop the host copies of the experts in between
        (a full-size expert is 44-88 MB on the host; 32 tokens touch up to ~200 of them)."""
        tokens = list(tokens)
        if chunk is not None and len(tokens) > chunk:
            out = []
            for i in range(0, len(tokens), chunk):
                out.append(self.oracle_y(x, idx, gate, tokens[i:i + chunk]))
                self._host.clear()
            return np.concatenate(out)
        c = self.cfg
        n = c.E + c.S
        used = set(int(e) for t in tokens for e in idx[t] if e >= 0) | set(range(c.E, n))
        tabs = {k: [None] * n for k in ("gate", "up", "down", "gate_scale", "up_scale", "down_scale")}
        for e in used:
            h = self.host_expert(e)
            for k in h:
                tabs[k][e] = h[k]
        fp8 = c.w_dtype == wl.DT_E4M3
        return orc.moe_tokens(wl.bits(x), list(tokens), idx, gate, tabs["gate"], tabs["up"], tabs["down"], c.E, c.S,
                              c.routed_scale, tabs["gate_scale"] if fp8 else None, tabs["up_scale"] if fp8 else None,
                              tabs["down_scale"] if fp8 else None)

    # ---- GPU calls (through the C ABI)
    def forward(self, x, params=None, scores=None, want_stats=False):
        stats = B.stats_buffer(self.device) if want_stats else None
        y = super().forward(x, params, scores, stats=stats)
        torch.cuda.synchronize()
        return (y, B.read_stats(stats)) if want_stats else y


def check_y(y_gpu, y_ref, tokens, tol):
    """max |y_gpu - y_oracle| <= tol * RMS(y_oracle) over the sampled tokens (oracle unrounded, R29)."""
    got = y_gpu[list(tokens)].double().cpu().numpy()
    rms = float(np.sqrt(np.mean(y_ref ** 2)))
    err = float(np.abs(got - y_ref).max())
    assert np.isfinite(got).all(), "non-finite output"
    assert err <= tol * rms, f"max|err| {err:.3e} > {tol:g} x RMS {rms:.3e} (ratio {err / rms:.3e})"
    return err / rms if rms > 0 else 0.0          # an all-pruned step without shared experts: y = 0 exactly
