"""Pins for oracle O7 (expert SwiGLU FFN) and O8 (combine): torch fp64 library routines,
linearity, the shared-expert concatenation identity and the e4m3 closed form.  CPU only."""
import numpy as np
import pytest
import torch
import torch.nn.functional as F

from paper_2606_29982_b200 import workloads as wl


def _mk(H, I, n, seed, dtype=torch.float32):
    g = torch.Generator().manual_seed(seed)
    Wg = [(0.05 * torch.randn(I, H, generator=g)).to(dtype) for _ in range(n)]
    Wu = [(0.05 * torch.randn(I, H, generator=g)).to(dtype) for _ in range(n)]
    Wd = [(0.05 * torch.randn(H, I, generator=g)).to(dtype) for _ in range(n)]
    return Wg, Wu, Wd


def _mlp64(x, Wg, Wu, Wd):
    x = x.double()
    return (F.silu(x @ Wg.double().T) * (x @ Wu.double().T)) @ Wd.double().T


@pytest.mark.parametrize("dtype", [torch.float32, torch.bfloat16])
def test_single_expert_is_a_swiglu_mlp(orc, dtype):
    """T=1, k=1, S=0 reduces the layer to one SwiGLU MLP (PAPER.md:40 with |K_t| = 1)."""
    H, I = 96, 160
    Wg, Wu, Wd = _mk(H, I, 1, 0, dtype)
    x = torch.randn(1, H, generator=torch.Generator().manual_seed(1)).to(dtype)
    ref = _mlp64(x[0], Wg[0], Wu[0], Wd[0]).numpy()
    o = orc.expert_ffn(wl.bits(x)[0], wl.bits(Wg[0]), wl.bits(Wu[0]), wl.bits(Wd[0]))
    np.testing.assert_allclose(o, ref, rtol=1e-11, atol=1e-14)
    y = orc.moe_tokens(wl.bits(x), [0], np.array([[0]], np.int32), np.array([[1.0]], np.float32),
                       [wl.bits(Wg[0])], [wl.bits(Wu[0])], [wl.bits(Wd[0])], E=1, S=0, routed_scale=1.0)
    np.testing.assert_allclose(y[0], ref, rtol=1e-11, atol=1e-14)


def test_combine_matches_torch_and_is_linear_in_gates(orc):
    H, I, E, S, k, T = 64, 96, 6, 2, 3, 5
    Wg, Wu, Wd = _mk(H, I, E + S, 2)
    g = torch.Generator().manual_seed(3)
    x = torch.randn(T, H, generator=g)
    idx = torch.stack([torch.randperm(E, generator=g)[:k] for _ in range(T)]).to(torch.int32)
    gate = torch.rand(T, k, generator=g)
    scale = 2.5
    ref = torch.zeros(T, H, dtype=torch.float64)
    for t in range(T):
        for j in range(k):
            e = int(idx[t, j])
            ref[t] += scale * gate[t, j].double() * _mlp64(x[t], Wg[e], Wu[e], Wd[e])
        for sh in range(S):
            ref[t] += _mlp64(x[t], Wg[E + sh], Wu[E + sh], Wd[E + sh])
    W = [[a.numpy() for a in lst] for lst in (Wg, Wu, Wd)]
    y = orc.moe_tokens(x.numpy(), np.arange(T), idx.numpy(), gate.numpy(), *W, E=E, S=S, routed_scale=scale)
    np.testing.assert_allclose(y, ref.numpy(), rtol=1e-10, atol=1e-13)
    # token subset = the same rows
    y13 = orc.moe_tokens(x.numpy(), [3, 1], idx.numpy(), gate.numpy(), *W, E=E, S=S, routed_scale=scale)
    assert np.array_equal(y13, y[[3, 1]])
    # linear in the gates and in routed_scale: y(2G) - shared = 2 (y(G) - shared)
    y0 = orc.moe_tokens(x.numpy(), np.arange(T), idx.numpy(), np.zeros_like(gate.numpy()), *W, E=E, S=S, routed_scale=scale)
    y2 = orc.moe_tokens(x.numpy(), np.arange(T), idx.numpy(), 2 * gate.numpy(), *W, E=E, S=S, routed_scale=scale)
    np.testing.assert_allclose(y2 - y0, 2 * (y - y0), rtol=1e-12, atol=1e-14)
    # an empty slot (idx = -1) contributes nothing
    idx_h = idx.numpy().copy()
    gate_h = gate.numpy().copy()
    idx_h[:, -1] = -1
    gate_z = gate.numpy().copy()
    gate_z[:, -1] = 0
    ya = orc.moe_tokens(x.numpy(), np.arange(T), idx_h, gate_h, *W, E=E, S=S, routed_scale=scale)
    yb = orc.moe_tokens(x.numpy(), np.arange(T), idx.numpy(), gate_z, *W, E=E, S=S, routed_scale=scale)
    np.testing.assert_allclose(ya, yb, rtol=1e-12, atol=1e-14)


def test_two_shared_experts_equal_one_concatenated(orc):
    """Two shared experts of width I are one of width 2I: [Wg;Wg'], [Wu;Wu'], [Wd Wd']."""
    H, I = 48, 64
    Wg, Wu, Wd = _mk(H, I, 2, 4)
    x = torch.randn(3, H, generator=torch.Generator().manual_seed(5)).numpy()
    none_idx = np.full((3, 1), -1, np.int32)
    zero = np.zeros((3, 1), np.float32)
    y2 = orc.moe_tokens(x, [0, 1, 2], none_idx, zero, [None] + [a.numpy() for a in Wg], [None] + [a.numpy() for a in Wu],
                        [None] + [a.numpy() for a in Wd], E=1, S=2, routed_scale=1.0)
    cg, cu, cd = torch.cat(Wg, 0).numpy(), torch.cat(Wu, 0).numpy(), torch.cat(Wd, 1).contiguous().numpy()
    y1 = orc.moe_tokens(x, [0, 1, 2], none_idx, zero, [None, cg], [None, cu], [None, cd], E=1, S=1, routed_scale=1.0)
    np.testing.assert_allclose(y2, y1, rtol=1e-12, atol=1e-15)


def test_e4m3_closed_form_table_vs_torch(orc):
    codes = torch.arange(256, dtype=torch.uint8)
    ref = codes.view(torch.float8_e4m3fn).double().numpy()      # library decode
    got = np.array([orc.e4m3_value(c) for c in range(256)])
    assert np.array_equal(np.isnan(ref), np.isnan(got)) and np.isnan(got).sum() == 2
    ok = ~np.isnan(ref)
    assert np.array_equal(ref[ok], got[ok])
    assert got[0x7E] == 448.0 and got[0x01] == 2.0 ** -9 and got[0x08] == 2.0 ** -6     # max, min subnormal, min normal


def test_block_scaled_e4m3_expert(orc):
    H, I = 256, 384
    g = torch.Generator().manual_seed(6)
    ws = [0.02 * torch.randn(*sh, generator=g) for sh in ((I, H), (I, H), (H, I))]
    q = [wl.quantize_e4m3_blocks(w) for w in ws]
    # dequantised exactly: code value times its 128x128 block's scale, done with library ops
    deq = [c.double() * s.double().repeat_interleave(128, 0).repeat_interleave(128, 1)[:c.shape[0], :c.shape[1]] for c, s in q]
    for w, d in zip(ws, deq):
        assert (w.double() - d).abs().max() <= 0.0625 * w.abs().max() + 1e-12           # e4m3: 3 mantissa bits
    x = torch.randn(H, generator=g).to(torch.bfloat16)
    ref = (F.silu(deq[0] @ x.double()) * (deq[1] @ x.double())) @ deq[2].T
    o = orc.expert_ffn(wl.bits(x), wl.bits(q[0][0]), wl.bits(q[1][0]), wl.bits(q[2][0]),
                       q[0][1].numpy(), q[1][1].numpy(), q[2][1].numpy())
    np.testing.assert_allclose(o, ref.numpy(), rtol=1e-10, atol=1e-14)


def test_workload_generators_are_seeded(orc):
    a = wl.expert_weights(wl.C1, 0, 3)
    b = wl.expert_weights(wl.C1, 0, 3)
    c = wl.expert_weights(wl.C1, 0, 4)
    assert torch.equal(a["gate"], b["gate"]) and not torch.equal(a["gate"], c["gate"])
    assert abs(float(a["down"].std()) - 0.02) < 2e-3
    Wr, bl, cb = wl.router(wl.C3, 0)
    assert Wr.shape == (256, 7168) and cb.shape == (256,) and abs(float(bl.mean()) + 5.0) < 1e-4
    assert wl.residency(wl.C5, 0).sum() == 64 and wl.partitions(wl.C3).max() == 7
    tr, tm = wl.cost_tables(wl.C3)
    assert tr[3 * 32] == 2 * tr[0] == 26020
