"""caee_route_noalloc (include/caee.h): S0+S1 without a context and without any allocation — the router GEMM's
split-K scratch lives in a file-scope device array — against the existing path, caee_route on a context
(PAPER.md:38-46).  pytest collects this file last on purpose (-x: a failure here hides nothing).

Same kernels, same split, same order of additions: scores, indices and gates are compared bit for bit, and the
scores also within the 1e-5 relative tolerance the route tests use.  Two calls in a row per case, the second on a
smaller batch, so that the array still holds the first call's partial sums when the second one runs."""
import numpy as np
import pytest
import torch

from paper_2606_29982_b200 import workloads as wl

pytestmark = pytest.mark.gpu

DEV = "cuda:0"
R1S = wl.scaled(wl.C3, name="R1-small", H=1024, I=384, E=64, k=4, n_group=8, topk_group=4, D=8,
                straggler_part=3, cost_ticks_ns=901)
C2S = wl.scaled(wl.C2, name="C2-small", H=512, I=256, E=16, S=2, k=3, D=4)
R1R = wl.scaled(wl.C3, name="R1-router-full", I=128)         # the full-size router: E = 256, H = 7168, groups 8/4
C1 = wl.C1                                                   # fp32 activations, softmax scores


@pytest.fixture(scope="module")
def B():
    from paper_2606_29982_b200 import binding
    return binding


def _outputs(cfg, T):
    return (torch.empty(T, cfg.E, dtype=torch.float32, device=DEV), torch.empty(T, cfg.k, dtype=torch.int32, device=DEV),
            torch.empty(T, cfg.k, dtype=torch.float32, device=DEV))


def _noalloc(B, cfg, x, T, Wr, b, cb, out):
    B.caee_route_noalloc(0, x, cfg.act_dtype, Wr, b, cb, T, cfg.H, cfg.E, cfg.k, cfg.n_group, cfg.topk_group, cfg.score_fn,
                         int(cfg.norm_topk), out[0], out[1], out[2])


def _same(a, b):
    s0, i0, g0 = (t.cpu().numpy() for t in a)
    s1, i1, g1 = (t.cpu().numpy() for t in b)
    np.testing.assert_allclose(s1, s0, rtol=1e-5, atol=1e-10)          # the route tests' tolerance
    assert np.array_equal(s1.view(np.uint32), s0.view(np.uint32))      # and, the kernels being the same, the same bits
    assert np.array_equal(i1, i0)
    assert np.array_equal(g1.view(np.uint32), g0.view(np.uint32))


@pytest.mark.parametrize("cfg,batches,fma_only", [(C2S, (33, 5), False), (R1S, (63, 8), False), (R1R, (40, 1), False),
                                                  (C1, (16, 3), False), (R1R, (128, 7), True), (R1S, (100, 2), True)],
                         ids=lambda v: getattr(v, "name", str(v)))
def test_route_noalloc_matches_the_context_path(B, cfg, batches, fma_only, monkeypatch):
    torch.cuda.set_device(DEV)
    if fma_only:   # from 64 tokens on a context takes the tensor-core router; keep it on the kernels both paths share
        monkeypatch.setenv("CAEE_ROUTER_MMA_MIN_TOKENS", "1000000")
    ctx = B.caee_create(B.layer_desc(cfg, max(batches)))
    try:
        Wr, b, cb = wl.router(cfg, 0, DEV)
        B.caee_set_router(ctx, Wr, b, cb)
        xs = [wl.hidden(cfg, T, 11 + i, DEV) for i, T in enumerate(batches)]
        refs, outs = [], []
        for x, T in zip(xs, batches):
            ref = _outputs(cfg, T)
            B.caee_route(ctx, x, T, *ref)
            refs.append(ref)
            outs.append(_outputs(cfg, T))
        torch.cuda.synchronize()
        # warm-up (module load, first launches), then the two calls in a row with the device's free memory watched
        _noalloc(B, cfg, xs[0], batches[0], Wr, b, cb, _outputs(cfg, batches[0]))
        _noalloc(B, cfg, xs[1], batches[1], Wr, b, cb, _outputs(cfg, batches[1]))
        torch.cuda.synchronize()
        free0 = torch.cuda.mem_get_info()[0]
        for x, T, out in zip(xs, batches, outs):
            _noalloc(B, cfg, x, T, Wr, b, cb, out)
        torch.cuda.synchronize()
        assert torch.cuda.mem_get_info()[0] == free0                   # nothing was allocated on the device
        for ref, out in zip(refs, outs):
            _same(ref, out)
        # scores are optional, as in caee_route
        T = batches[1]
        _, idx, gate = _outputs(cfg, T)
        B.caee_route_noalloc(0, xs[1], cfg.act_dtype, Wr, b, cb, T, cfg.H, cfg.E, cfg.k, cfg.n_group, cfg.topk_group,
                             cfg.score_fn, int(cfg.norm_topk), None, idx, gate)
        torch.cuda.synchronize()
        assert np.array_equal(idx.cpu().numpy(), refs[1][1].cpu().numpy())
    finally:
        B.caee_destroy(ctx)


def test_route_noalloc_rejects_what_does_not_fit(B):
    torch.cuda.set_device(DEV)
    cfg = R1S
    Wr, b, cb = wl.router(cfg, 0, DEV)
    T = 129                                                            # CAEE_ROUTE_NOALLOC_MAX_TOKENS = 128
    x = wl.hidden(cfg, T, 1, DEV)
    out = _outputs(cfg, T)
    out[1].fill_(-7)
    with pytest.raises(B.CaeeError) as ei:
        _noalloc(B, cfg, x, T, Wr, b, cb, out)
    assert ei.value.code == B.CAEE_ESHAPE and "128" in str(ei.value)
    torch.cuda.synchronize()
    assert bool((out[1] == -7).all())                                  # nothing was enqueued
    for bad in (dict(H=cfg.H + 4), dict(k=cfg.E + 1), dict(n_group=5), dict(act=7)):
        with pytest.raises(B.CaeeError):
            B.caee_route_noalloc(0, x, bad.get("act", cfg.act_dtype), Wr, b, cb, 8, bad.get("H", cfg.H), cfg.E,
                                 bad.get("k", cfg.k), bad.get("n_group", cfg.n_group), cfg.topk_group, cfg.score_fn,
                                 int(cfg.norm_topk), out[0], out[1], out[2])
    with pytest.raises(B.CaeeError):                                   # NULL input
        B.caee_route_noalloc(0, None, cfg.act_dtype, Wr, b, cb, 8, cfg.H, cfg.E, cfg.k, cfg.n_group, cfg.topk_group,
                             cfg.score_fn, int(cfg.norm_topk), out[0], out[1], out[2])
    # T = 0 is a no-op
    B.caee_route_noalloc(0, None, cfg.act_dtype, Wr, b, cb, 0, cfg.H, cfg.E, cfg.k, cfg.n_group, cfg.topk_group,
                         cfg.score_fn, int(cfg.norm_topk), None, None, None)
