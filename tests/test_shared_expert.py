"""Shared (always-on) expert as a composition of the routed-expert path (Table 4:
"one shared expert at width 2048 plus ... routed experts at width 1024").

A SwiGLU FFN is separable along its hidden width: silu(x Wg) * (x Wu) is elementwise per hidden channel and the down
projection sums over channels, so a dense FFN of width n F equals the sum of n FFNs of width F.  The shared expert is
therefore n = 2 extra experts that EVERY token is sent to with gate weight 1 -- the same dispatch / grouped-GEMM /
combine kernels, a second small ctx, no new kernel.  (Reading: the shared expert's weights use the same quantised +
adapter format as the routed experts; the paper does not say.)"""
import numpy as np
import pytest

import oracle
import tqp_inputs as ti


def widen(b):
    return ti.bf16_bits_to_f32(b)


def always_on(T, n):
    return np.tile(np.arange(n, dtype=np.int32), (T, 1)), np.ones((T, n), np.float32)


def test_oracle_always_on_experts_equal_one_dense_ffn_of_double_width():
    """Pin: the oracle's chain with forced routing against numpy fp64 matmuls of the CONCATENATED merged weights."""
    cfg = ti.Config("shared", T=11, d=32, F=48, E=2, k=2, r=4, seed=41, lora_scale=0.5)
    inp = ti.make_inputs(cfg)
    rng = np.random.default_rng(1)
    for key in ("A_gate", "B_gate", "A_up", "B_up", "A_down", "B_down"):
        inp[key] = ti.f32_to_bf16_bits(rng.standard_normal(inp[key].shape).astype(np.float32) * 0.1)
    idx, w = always_on(cfg.T, 2)
    counts, offsets, perm, inv = oracle.dispatch(idx, cfg.E)
    assert list(counts) == [cfg.T, cfg.T]
    Ye, G, U, H = oracle.expert_fwd(inp, offsets, perm, dtype=np.float64)
    Y = oracle.combine(Ye, inv, w.astype(np.float64))
    X = widen(inp["X"]).astype(np.float64)
    cb = inp["codebook"].astype(np.float64)

    def merged(idx_, scale, A, B):
        out_dim = idx_.shape[0]
        Wdeq = (cb[idx_].reshape(out_dim, -1) * scale.astype(np.float64)[:, None]).T     # [in][out]
        return Wdeq + cfg.lora_scale * widen(A).astype(np.float64) @ widen(B).astype(np.float64)

    Wg = np.concatenate([merged(inp["idx_gate"][e], inp["scale_gate"][e], inp["A_gate"][e], inp["B_gate"][e]) for e in (0, 1)], axis=1)
    Wu = np.concatenate([merged(inp["idx_up"][e], inp["scale_up"][e], inp["A_up"][e], inp["B_up"][e]) for e in (0, 1)], axis=1)
    Wd = np.concatenate([merged(inp["idx_down"][e], inp["scale_down"][e], inp["A_down"][e], inp["B_down"][e]) for e in (0, 1)], axis=0)
    Gd = X @ Wg
    Hd = Gd / (1 + np.exp(-Gd)) * (X @ Wu)          # one dense SwiGLU of width 2 F
    np.testing.assert_allclose(Y, Hd @ Wd, rtol=1e-11, atol=1e-13)


@pytest.mark.gpu
def test_gpu_shared_expert_through_the_routed_kernels():
    """Width-2048 shared expert at d = 512 on the GPU (two always-on experts of width 1024, T = 700: several token tiles
    per expert and a ragged tail) against the oracle, forward and backward."""
    import torch
    from parity_util import assert_close, make_layer, to_np
    cfg = ti.Config("shared_gpu", T=700, d=512, F=1024, E=2, k=2, r=16, seed=42)
    inp = ti.make_inputs(cfg)
    layer, dev = make_layer(inp, training=True)
    idx_np, w_np = always_on(cfg.T, 2)
    idx, w = torch.from_numpy(idx_np).cuda(), torch.from_numpy(w_np).cuda()
    counts, offsets, perm, inv = layer.dispatch(idx)
    Ye = layer.expert_fwd(dev["X"], offsets, perm)
    Y = layer.combine(Ye, inv, w)
    dYe, _ = layer.combine_bwd(dev["dY"], Ye, inv, w, want_dw=False, perm=perm)
    dXp, grads = layer.expert_bwd(dev["X"], dYe, offsets, perm)
    dX = layer.dispatch_bwd(dXp, inv)
    torch.cuda.synchronize()
    c_r, o_r, p_r, inv_r = oracle.dispatch(idx_np, cfg.E)
    np.testing.assert_array_equal(to_np(perm), p_r)
    Ye_r, G, U, H = oracle.expert_fwd(inp, o_r, p_r)
    Y_r = oracle.combine(Ye_r, inv_r, w_np)
    assert_close("Y", to_np(Y), Y_r)
    dYe_r, _ = oracle.combine_bwd(inp["dY"], Ye_r, inv_r, w_np)
    dXp_r, g_r = oracle.expert_bwd(inp, dYe_r, G, U, H, o_r, p_r)
    assert_close("dX", to_np(dX), oracle.dispatch_bwd(dXp_r, inv_r, cfg.T, cfg.k))
    for key, val in g_r.items():
        assert_close(key, to_np(grads[key]), val)
