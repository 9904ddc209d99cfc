"""tqp_consolidate (§10.6) on the GPU against oracle/consolidate.py, and the
released-model cross-check: a dense bf16 MoE forward through the consolidated weights reproduces the layer's own
quantised-plus-adapter forward."""
import numpy as np
import pytest

import tqp_inputs as ti
from oracle import consolidate as oc

pytestmark = pytest.mark.gpu


def _f64(a):
    return (ti.bf16_bits_to_f32(a) if a.dtype == np.uint16 else a.astype(np.float32)).astype(np.float64)


CASES = [ti.Config("cons_r16", T=300, d=384, F=256, E=5, k=2, r=16, seed=51, lora_scale=0.5),
         ti.Config("cons_r32", T=64, d=256, F=640, E=3, k=1, r=32, seed=52),
         ti.CONFIGS[0]]


@pytest.mark.parametrize("cfg", CASES, ids=lambda c: c.name)
def test_consolidated_weights_match_the_oracle(cfg):
    """Every element of every pack: fp32 merge rounded once to bf16 against the fp64 definition.  Tolerance: one bf16
    rounding (2^-9 relative) + the fp32 sum of r + 1 terms, written as 2^-8 |ref| + 1e-6 max|ref|."""
    import torch
    from parity_util import make_layer
    inp = ti.make_inputs(cfg)
    rng = np.random.default_rng(cfg.seed)
    for key in ("A_gate", "B_gate", "A_up", "B_up", "A_down", "B_down"):      # a TRAINED adapter: both factors non-zero
        inp[key] = ti.f32_to_bf16_bits(rng.standard_normal(inp[key].shape).astype(np.float32) * 0.05)
    layer, dev = make_layer(inp, training=False)
    cb = _f64(inp["codebook"])
    for pi, pack in enumerate(("gate", "up", "down")):
        W = layer.consolidate(pack)
        torch.cuda.synchronize()
        Wg = W.float().cpu().numpy().astype(np.float64)
        for e in range(cfg.E):
            ref = oc.consolidate(inp["idx_" + pack][e], _f64(inp["scale_" + pack])[e], cb, _f64(inp["A_" + pack])[e],
                                 _f64(inp["B_" + pack])[e], cfg.lora_scale)
            assert Wg[e].shape == ref.shape
            err = np.abs(Wg[e] - ref)
            assert (err <= 2.0 ** -8 * np.abs(ref) + 1e-6 * np.abs(ref).max()).all(), (pack, e, err.max())
        # an expert range lands at the front of the output
        if cfg.E > 2:
            part = layer.consolidate(pi, e0=1, n_experts=2)
            assert torch.equal(part, W[1:3])


def test_dense_forward_through_consolidated_weights_matches_the_layer():
    """'A user of the released model sees a normal bf16 MoE' (L1112): route with the layer, then run each expert as three
    dense torch matmuls over the consolidated bf16 weights, and compare with the layer's grouped dequant GEMM path."""
    import torch
    from parity_util import make_layer
    cfg = ti.Config("cons_fwd", T=700, d=512, F=256, E=6, k=2, r=16, seed=53)
    inp = ti.make_inputs(cfg)
    rng = np.random.default_rng(7)
    for key in ("A_gate", "B_gate", "A_up", "B_up", "A_down", "B_down"):
        inp[key] = ti.f32_to_bf16_bits(rng.standard_normal(inp[key].shape).astype(np.float32) * 0.05)
    layer, dev = make_layer(inp, training=False)
    X, W_r = dev["X"], dev["W_r"]
    idx, w = layer.route(X, W_r, None)[:2]
    counts, offsets, perm, inv = layer.dispatch(idx)
    Ye = layer.expert_fwd(X, offsets, perm)
    Wg, Wu, Wd = (layer.consolidate(p).float() for p in ("gate", "up", "down"))
    torch.cuda.synchronize()
    offs = offsets.cpu().numpy()
    ref = torch.zeros_like(Ye, dtype=torch.float32)
    for e in range(cfg.E):
        rows = torch.arange(int(offs[e]), int(offs[e + 1]), device=X.device)
        if rows.numel() == 0:
            continue
        x = X[(perm[rows] // cfg.k).long()].float()
        g, u = x @ Wg[e].T, x @ Wu[e].T
        ref[rows] = (torch.nn.functional.silu(g) * u) @ Wd[e].T
    err = (Ye.float() - ref).abs().max().item()
    scale = ref.abs().max().item()
    relf = ((Ye.float() - ref).norm() / ref.norm()).item()
    assert err <= 2e-2 * scale and relf <= 1e-2, (err, scale, relf)
