"""Seeded synthetic workloads (BASELINE.json configs 1-5; recipe in DESIGN.md §4).

This module only draws random inputs and states configuration constants.  It
holds none of the method's arithmetic and is the one module that both the tests
of the CPU oracle and the CUDA path's tests / bench import.  The inputs stand in
for the paper's DeepSeek-R1 workloads: same shapes, value
distributions and routing skew, no real weights or prompts.
"""
from dataclasses import dataclass, field
from typing import Optional, Tuple

import numpy as np
import torch

SCORE_SOFTMAX, SCORE_SIGMOID = 0, 1
DT_F32, DT_BF16, DT_E4M3 = 0, 1, 2


@dataclass(frozen=True)
class LayerConfig:
    name: str
    H: int                      # hidden size
    I: int                      # SwiGLU intermediate size
    E: int                      # routed experts
    S: int                      # shared experts
    k: int                      # top-k
    n_group: int
    topk_group: int
    score_fn: int
    norm_topk: bool
    routed_scale: float
    act_dtype: int
    w_dtype: int
    D: int                      # expert partitions (the paper's "devices")
    cost_ticks_ns: int          # C~ for a resident expert, integer ns
    straggler_part: int = -1    # partition whose costs are doubled, -1 = none
    batches: Tuple[int, ...] = (1,)
    seeds: Tuple[int, ...] = (0,)
    zipf_lambda: float = 0.0    # 0 => b_logit ~ N(0, 0.5) (config 1)
    logit_offset: float = 0.0
    corr_bias_std: float = 0.0
    n_resident: int = -1        # experts resident in HBM, -1 = all (config 5: 64)
    miss_ticks_ns: int = 0      # C~ for a non-resident expert (H2D tier)

    @property
    def act_torch(self):
        return torch.float32 if self.act_dtype == DT_F32 else torch.bfloat16

    @property
    def expert_bytes(self) -> int:
        per = {DT_F32: 4, DT_BF16: 2, DT_E4M3: 1}[self.w_dtype]
        b = 3 * self.H * self.I * per
        if self.w_dtype == DT_E4M3:
            b += 3 * ((self.H + 127) // 128) * ((self.I + 127) // 128) * 4
        return b


# cost_ticks_ns: C1 = 1,572,864 B / 1 TB/s + 2 us = 3573 ns (BASELINE.json config 1);
# C2-C4 = bytes / 8 TB/s + 2 us: 4163, 13010, 7506 ns.
C1 = LayerConfig("C1-tiny-fp32", H=256, I=512, E=8, S=0, k=2, n_group=1, topk_group=1,
                 score_fn=SCORE_SOFTMAX, norm_topk=True, routed_scale=1.0, act_dtype=DT_F32,
                 w_dtype=DT_F32, D=2, cost_ticks_ns=3573, batches=(16,), seeds=(0,))
C2 = LayerConfig("C2-mid-bf16", H=2048, I=1408, E=64, S=2, k=6, n_group=1, topk_group=1,
                 score_fn=SCORE_SOFTMAX, norm_topk=True, routed_scale=1.0, act_dtype=DT_BF16,
                 w_dtype=DT_BF16, D=4, cost_ticks_ns=4163, batches=(1, 8, 32, 128),
                 seeds=(0, 1, 2, 3), zipf_lambda=0.5)
C3 = LayerConfig("C3-r1-bf16", H=7168, I=2048, E=256, S=1, k=8, n_group=8, topk_group=4,
                 score_fn=SCORE_SIGMOID, norm_topk=True, routed_scale=2.5, act_dtype=DT_BF16,
                 w_dtype=DT_BF16, D=8, cost_ticks_ns=13010, straggler_part=3,
                 batches=(1, 8, 32, 128), seeds=(0,), zipf_lambda=0.5, logit_offset=-5.0,
                 corr_bias_std=0.05)
C4 = LayerConfig("C4-r1-fp8", H=7168, I=2048, E=256, S=1, k=8, n_group=8, topk_group=4,
                 score_fn=SCORE_SIGMOID, norm_topk=True, routed_scale=2.5, act_dtype=DT_BF16,
                 w_dtype=DT_E4M3, D=8, cost_ticks_ns=7506, straggler_part=3,
                 batches=(1, 8, 32, 128, 4096), seeds=(0,), zipf_lambda=0.5, logit_offset=-5.0,
                 corr_bias_std=0.05)
C5 = LayerConfig("C5-r1-bf16-offload", H=7168, I=2048, E=256, S=1, k=8, n_group=8, topk_group=4,
                 score_fn=SCORE_SIGMOID, norm_topk=True, routed_scale=2.5, act_dtype=DT_BF16,
                 w_dtype=DT_BF16, D=8, cost_ticks_ns=13010, straggler_part=3, batches=(8, 32),
                 seeds=(0,), zipf_lambda=0.5, logit_offset=-5.0, corr_bias_std=0.05, n_resident=64,
                 miss_ticks_ns=1_603_462)
CONFIGS = {c.name.split("-")[0]: c for c in (C1, C2, C3, C4, C5)}


def scaled(cfg: LayerConfig, **kw) -> LayerConfig:
    """A copy of cfg with some fields replaced (reduced sizes for fast tests)."""
    d = {f: getattr(cfg, f) for f in cfg.__dataclass_fields__}
    d.update(kw)
    return LayerConfig(**d)


def _gen(seed: int, stream: int, device) -> torch.Generator:
    g = torch.Generator(device=device)
    g.manual_seed((seed * 1_000_003 + stream) & 0x7FFFFFFFFFFFFFFF)
    return g


def hidden(cfg: LayerConfig, T: int, seed: int, device="cpu") -> torch.Tensor:
    """x[T,H] ~ N(0,1), rounded to the activation dtype."""
    x = torch.randn(T, cfg.H, generator=_gen(seed, 1, device), device=device, dtype=torch.float32)
    return x.to(cfg.act_torch)


def zipf_rank(cfg: LayerConfig, seed: int) -> np.ndarray:
    """Popularity rank r_e in 1..E from a seeded permutation (rank 1 = most popular)."""
    rng = np.random.default_rng(seed * 7919 + 17)
    perm = rng.permutation(cfg.E)
    rank = np.empty(cfg.E, np.int64)
    rank[perm] = np.arange(1, cfg.E + 1)
    return rank


def router(cfg: LayerConfig, seed: int, device="cpu"):
    """W_r[E,H] ~ N(0,0.02) fp32; b_logit[E]; corr_bias[E] or None."""
    Wr = 0.02 * torch.randn(cfg.E, cfg.H, generator=_gen(seed, 2, device), device=device, dtype=torch.float32)
    if cfg.zipf_lambda == 0.0:
        b = 0.5 * torch.randn(cfg.E, generator=_gen(seed, 3, "cpu"), dtype=torch.float32)
    else:
        lnz = -1.1 * np.log(zipf_rank(cfg, seed).astype(np.float64))
        b = torch.from_numpy((cfg.zipf_lambda * (lnz - lnz.mean()) + cfg.logit_offset).astype(np.float32))
    cb = None
    if cfg.corr_bias_std > 0:
        cb = (cfg.corr_bias_std * torch.randn(cfg.E, generator=_gen(seed, 4, "cpu"), dtype=torch.float32)).to(device)
    return Wr, b.to(device), cb


def quantize_e4m3_blocks(w: torch.Tensor):
    """fp32 [R,C] -> (e4m3 codes as float8_e4m3fn [R,C], fp32 scales [ceil(R/128), ceil(C/128)]).

    scale = amax(block)/448, round-to-nearest-even, saturating.
    """
    R, Cc = w.shape
    br, bc = (R + 127) // 128, (Cc + 127) // 128
    pad = torch.zeros(br * 128, bc * 128, device=w.device, dtype=torch.float32)
    pad[:R, :Cc] = w
    blocks = pad.view(br, 128, bc, 128)
    amax = blocks.abs().amax(dim=(1, 3))
    scale = torch.where(amax > 0, amax / 448.0, torch.ones_like(amax))
    q = (blocks / scale[:, None, :, None]).clamp_(-448.0, 448.0).reshape(br * 128, bc * 128)[:R, :Cc]
    return q.contiguous().to(torch.float8_e4m3fn), scale.contiguous()


def expert_weights(cfg: LayerConfig, seed: int, e: int, device="cpu"):
    """Weights of expert e (routed 0..E-1, shared E..E+S-1), ~N(0,0.02), in storage dtype.

    Returns dict(gate=[I,H], up=[I,H], down=[H,I]) plus gate_scale/up_scale/down_scale for e4m3.
    """
    out = {}
    for m, (name, shape) in enumerate((("gate", (cfg.I, cfg.H)), ("up", (cfg.I, cfg.H)), ("down", (cfg.H, cfg.I)))):
        w = 0.02 * torch.randn(*shape, generator=_gen(seed, 1000 + 3 * e + m, device), device=device,
                               dtype=torch.float32)
        if cfg.w_dtype == DT_F32:
            out[name] = w
        elif cfg.w_dtype == DT_BF16:
            out[name] = w.to(torch.bfloat16)
        else:
            out[name], out[name + "_scale"] = quantize_e4m3_blocks(w)
    return out


def partitions(cfg: LayerConfig) -> np.ndarray:
    """Contiguous blocks of E/D experts (for C3-C5 these are the router's groups)."""
    return (np.arange(cfg.E) // (cfg.E // cfg.D)).astype(np.int32)


def residency(cfg: LayerConfig, seed: int) -> np.ndarray:
    """resident[e]: all ones, or the n_resident most popular experts (stands in for the LFU cache)."""
    if cfg.n_resident < 0:
        return np.ones(cfg.E, np.uint8)
    return (zipf_rank(cfg, seed) <= cfg.n_resident).astype(np.uint8)


def cost_tables(cfg: LayerConfig):
    """(ticks_resident[E], ticks_miss[E]) int64 ns; the straggler partition costs 2x."""
    mult = np.where(partitions(cfg) == cfg.straggler_part, 2, 1).astype(np.int64)
    return cfg.cost_ticks_ns * mult, cfg.miss_ticks_ns * mult


def bits(t: torch.Tensor) -> np.ndarray:
    """Exact bit pattern of a tensor as a numpy array the oracle accepts (bf16->uint16, e4m3->uint8)."""
    t = t.detach().cpu().contiguous()
    if t.dtype == torch.bfloat16:
        return t.view(torch.int16).numpy().view(np.uint16)
    if t.dtype == torch.float8_e4m3fn:
        return t.view(torch.uint8).numpy()
    return t.numpy()
