"""GPU parity of the paper-faithful router variant and the balance controller against
oracle/router_ext.py: selection bit-exact (same fp32 logits, same fp32 biased keys, ties -> lower id), gate values
and scores to 1e-6, router gradients and the controller within fp32 rounding."""
import numpy as np
import pytest

import oracle
import tqp_inputs as ti
from oracle import router_ext as rx
from parity_util import assert_close, make_layer, to_np

pytestmark = pytest.mark.gpu


def _bias(E, seed):
    return (np.random.default_rng(seed).standard_normal(E) * 0.5).astype(np.float32)


@pytest.mark.parametrize("cfg_id,with_bias", [(0, True), (2, True), (2, False)])
def test_route_sigmoid_bit_exact_selection(cfg_id, with_bias):
    import torch
    cfg = ti.CONFIGS[cfg_id]
    inp = ti.make_inputs(cfg)
    if cfg_id == 0:
        inp["W_r"][:, 5] = inp["W_r"][:, 1]          # exact ties
    layer, dev = make_layer(inp, training=False)
    bias = _bias(cfg.E, 31) if with_bias else None
    bdev = torch.from_numpy(bias).cuda() if with_bias else None
    idx, w, sc, lg = layer.route_sigmoid(dev["X"], torch.from_numpy(inp["W_r"]).cuda(), bdev, want_logits=True)
    torch.cuda.synchronize()
    lg_ref = oracle.logits(inp["X"], inp["W_r"], None)
    np.testing.assert_array_equal(to_np(lg), lg_ref)
    i_ref, w_ref, s_ref = rx.route_sigmoid(lg_ref, bias, cfg.k)
    np.testing.assert_array_equal(to_np(idx), i_ref)
    assert np.abs(to_np(w) - w_ref).max() <= 1e-6 and np.abs(to_np(sc) - s_ref).max() <= 1e-6
    np.testing.assert_allclose(to_np(w).sum(1), 1.0, atol=2e-6)


@pytest.mark.parametrize("cfg_id,with_bias,impl", [(0, True, 2), (2, True, 0), (2, False, 2), (3, True, 2), (2, True, 3)])
def test_route_sigmoid_screened_matches_dense_and_oracle(cfg_id, with_bias, impl):
    """The screened router (csrc/route.cu) in its sigmoid variant: no logits requested -> tensor-core screen + canonical
    chains for the candidates; idx / w / s bitwise equal to the dense chain's and idx equal to the oracle's.  impl 3 forces
    the self-check to fail (the gated dense sigmoid kernels must then produce the result)."""
    import torch
    cfg = ti.CONFIGS[cfg_id]
    inp = ti.make_inputs(cfg)
    if cfg_id == 0:
        inp["W_r"][:, 5] = inp["W_r"][:, 1]          # exact ties
    layer, dev = make_layer(inp, training=False)
    bias = _bias(cfg.E, 33) if with_bias else None
    bdev = torch.from_numpy(bias).cuda() if with_bias else None
    Wd = torch.from_numpy(inp["W_r"]).cuda()
    layer.set_option("route_impl", 1)
    i1, w1, s1 = layer.route_sigmoid(dev["X"], Wd, bdev)
    assert layer.route_info() == (0, 0)
    layer.set_option("route_impl", impl)
    i2, w2, s2 = layer.route_sigmoid(dev["X"], Wd, bdev)
    assert layer.route_info() == (1, 1 if impl == 3 else 0)
    assert torch.equal(i1, i2)
    assert torch.equal(w1.view(torch.int32), w2.view(torch.int32)) and torch.equal(s1.view(torch.int32), s2.view(torch.int32))
    lg_ref = oracle.logits(inp["X"], inp["W_r"], None)
    i_ref, w_ref, s_ref = rx.route_sigmoid(lg_ref, bias, cfg.k)
    np.testing.assert_array_equal(to_np(i2), i_ref)
    assert np.abs(to_np(w2) - w_ref).max() <= 1e-6 and np.abs(to_np(s2) - s_ref).max() <= 1e-6


def test_route_sigmoid_backward_and_chain():
    """cfg 0 with sigmoid routing through the whole chain: Y against the oracle's expert path fed the oracle's routing,
    then dtopk_w -> dl -> dX, dW_r."""
    import torch
    cfg = ti.CONFIGS[0]
    inp = ti.make_inputs(cfg)
    layer, dev = make_layer(inp, training=True)
    bias = _bias(cfg.E, 32)
    idx, w, sc = layer.route_sigmoid(dev["X"], dev["W_r"], torch.from_numpy(bias).cuda())
    counts, offsets, perm, inv = layer.dispatch(idx)
    Ye = layer.expert_fwd(dev["X"], offsets, perm)
    Y = layer.combine(Ye, inv, w)
    dYe, dw = layer.combine_bwd(dev["dY"], Ye, inv, w, want_dw=True, perm=perm)
    dXp, grads = layer.expert_bwd(dev["X"], dYe, offsets, perm)
    dX = layer.dispatch_bwd(dXp, inv)
    dX_experts = dX.clone()
    dW_r = layer.route_sigmoid_bwd(dev["X"], dev["W_r"], idx, w, sc, dw, offsets, perm, dX)
    torch.cuda.synchronize()
    lg = oracle.logits(inp["X"], inp["W_r"], None)
    i_ref, w_ref, s_ref = rx.route_sigmoid(lg, bias, cfg.k)
    np.testing.assert_array_equal(to_np(idx), i_ref)
    c_ref, o_ref, p_ref, inv_ref = oracle.dispatch(i_ref, cfg.E)
    np.testing.assert_array_equal(to_np(perm), p_ref)
    Ye_ref, G, U, H = oracle.expert_fwd(inp, o_ref, p_ref)
    Y_ref = oracle.combine(Ye_ref, inv_ref, w_ref)
    assert_close("Y", to_np(Y), Y_ref)
    dYe_ref, dw_ref = oracle.combine_bwd(inp["dY"], Ye_ref, inv_ref, w_ref)
    assert_close("dtopk_w", to_np(dw), dw_ref)
    dl_ref = rx.route_sigmoid_dl(w_ref, s_ref, to_np(dw))             # the GPU's own dtopk_w isolates the router step
    dX_ref = to_np(dX_experts).astype(np.float32).copy()          # isolate the router term: start from the GPU's expert dX
    dW_ref = rx.route_bwd_from_dl(ti.bf16_bits_to_f32(inp["X"]), inp["W_r"], i_ref, dl_ref.astype(np.float32), dX_ref)
    assert_close("dW_r", to_np(dW_r), dW_ref, maxabs_tol=2e-3, relf_tol=2e-3)
    assert_close("dX", to_np(dX), dX_ref, maxabs_tol=8e-3, relf_tol=4e-3)


@pytest.mark.parametrize("mode,name", [(0, "sign"), (1, "three_tier")])
def test_bias_update_against_oracle(mode, name):
    import torch
    cfg = ti.CONFIGS[3]                                   # Zipf-skewed routing: dead experts and overloaded ones
    inp = ti.make_inputs(cfg)
    lg = oracle.logits(inp["X"][:2048], inp["W_r"], inp["logit_bias"])
    idx, _ = oracle.topk(lg, cfg.k)
    counts = np.bincount(idx.ravel(), minlength=cfg.E).astype(np.int32)
    assert (counts == 0).any() and counts.max() / counts.sum() > 0.005
    layer, _ = make_layer(ti.make_inputs(ti.CONFIGS[0]), training=False)
    layer.E = cfg.E
    import paper_2606_07404_b200 as tq
    layer2 = tq.TqpLayer(64, 128, 256, cfg.E, cfg.k, 8, training=False)
    bias0 = _bias(cfg.E, 33)
    b = torch.from_numpy(bias0.copy()).cuda()
    layer2.bias_update(torch.from_numpy(counts).cuda(), b, mode, 1e-4, cap_hi=0.005)
    torch.cuda.synchronize()
    ref = rx.bias_update(counts, bias0, name, 1e-4, cap_hi=0.005)
    np.testing.assert_allclose(to_np(b), ref, rtol=0, atol=1e-7 + 1e-5 * np.abs(ref - bias0).max())
    moved = to_np(b) - bias0
    assert (moved[counts == 0] > 0).all() and moved[np.argmax(counts)] < 0
