"""GPU parity of the routed-expert layer over a TurboQuant base (tqp_bind_weights_tq; PAPER.md
L944-948): the same chain as tests/test_gpu_parity.py, with the frozen base held as one 8-bit code per rotated
coordinate + row norms, the rotation applied once to the activations and the scalar-table look-up inside the grouped
GEMM's mainloop.

Oracle: routing / dispatch / combine from the C oracle (format-independent); the expert FFN from oracle/flush.py over
the DENSE effective weights decode(codes, norms)^T + s A B of each expert (fp64, library matmuls), i.e. the definition
with the reconstruction of L946 as the base.  Weights are drawn dense, encoded by the ORACLE's encoder, and the same
codes / norms / rotation draws / Lloyd-Max levels go to both sides."""
import numpy as np
import pytest

import oracle
import tqp_inputs as ti
from oracle import flush as ofl
from oracle import turboquant as otq
from parity_util import assert_close, assert_routing_exact, to_np

pytestmark = pytest.mark.gpu


def make_tq_inputs(cfg, adapter_std=0.01):
    inp = ti.make_inputs(cfg)
    rng = np.random.default_rng(1000 + cfg.seed)
    E, d, F, r = cfg.E, cfg.d, cfg.F, cfg.r
    spaces = {}
    for name, n in (("d", d), ("F", F)):
        spaces[name] = dict(n=n, R=otq.rotation(n, 50 + cfg.seed + n), levels=otq.lloyd_max_codebook(n, 8))
    tqw = {}
    for pack, (out_dim, sp) in dict(gate=(F, "d"), up=(F, "d"), down=(d, "F")).items():
        n = spaces[sp]["n"]
        W = rng.standard_normal((E, out_dim, n)) * 0.02 * rng.uniform(0.5, 1.5, size=(E, out_dim, 1))
        codes = np.empty((E, out_dim, n), np.uint8); norms = np.empty((E, out_dim), np.float32)
        for e in range(E):
            c, nn = otq.encode(W[e], spaces[sp]["R"], spaces[sp]["levels"])
            codes[e], norms[e] = c, nn.astype(np.float32)
        tqw[f"codes_{pack}"], tqw[f"norm_{pack}"] = codes, norms
    for key in ("A_gate", "B_gate", "A_up", "B_up", "A_down", "B_down"):
        inp[key] = ti.f32_to_bf16_bits(rng.standard_normal(inp[key].shape).astype(np.float32) * adapter_std)
    return inp, tqw, spaces


def oracle_tq_layer(inp, tqw, spaces, router_grad):
    """The layer with dense per-expert effective weights (fp64)."""
    k, E, s = inp["k"], inp["E"], inp["lora_scale"]
    w64 = lambda a: ti.bf16_bits_to_f32(a).astype(np.float64)
    X, dY = w64(inp["X"]), w64(inp["dY"])
    out = {}
    lg = oracle.logits(inp["X"], inp["W_r"], inp.get("logit_bias"), np.float32)
    out["logits"] = lg
    out["topk_idx"], out["topk_w"] = oracle.topk(lg, k)
    out["counts"], out["offsets"], out["perm"], out["inv_perm"] = oracle.dispatch(out["topk_idx"], E)
    offs, perm, inv = out["offsets"], out["perm"], out["inv_perm"]
    tw = out["topk_w"].astype(np.float64)
    N, d, F, r = X.shape[0] * k, inp["d"], inp["F"], inp["r"]
    Ye = np.zeros((N, d)); G = np.zeros((N, F)); U = np.zeros((N, F)); H = np.zeros((N, F))
    Wd = {}
    for e in range(E):
        p0, p1 = offs[e], offs[e + 1]
        Wd[e] = [ofl.dense_weights(tqw[f"codes_{pk}"][e], tqw[f"norm_{pk}"][e].astype(np.float64), w64(inp[f"A_{pk}"][e]),
                                   w64(inp[f"B_{pk}"][e]), s, spaces[sp]["R"], spaces[sp]["levels"])
                 for pk, sp in (("gate", "d"), ("up", "d"), ("down", "F"))]
        if p1 > p0:
            Ye[p0:p1], G[p0:p1], U[p0:p1], H[p0:p1] = ofl.expert_ffn(X[perm[p0:p1] // k], *Wd[e])
    out.update(Ye=Ye, G=G, U=U, H=H)
    out["Y"] = oracle.combine(Ye, inv, tw)
    dYe, dw = oracle.combine_bwd(dY, Ye, inv, tw, np.float64)
    out["dYe"], out["dtopk_w"] = dYe, dw
    dXp = np.zeros((N, d))
    g = {f"d{ab}_{pk}": np.zeros(inp[f"{ab}_{pk}"].shape) for ab in "AB" for pk in ("gate", "up", "down")}
    for e in range(E):
        p0, p1 = offs[e], offs[e + 1]
        if p1 == p0:
            continue
        x = X[perm[p0:p1] // k]
        dXp[p0:p1], dWg, dWu, dWdn = ofl.expert_ffn_bwd(x, dYe[p0:p1], G[p0:p1], U[p0:p1], H[p0:p1], *Wd[e])
        for pk, dW in (("gate", dWg), ("up", dWu), ("down", dWdn)):   # W_eff = base + s A B  =>  dA = s dW B^T, dB = s A^T dW
            g[f"dA_{pk}"][e] = s * dW @ w64(inp[f"B_{pk}"][e]).T
            g[f"dB_{pk}"][e] = s * w64(inp[f"A_{pk}"][e]).T @ dW
    out.update(g)
    out["dXp"] = dXp
    out["dX_experts"] = oracle.dispatch_bwd(dXp, inv, X.shape[0], k)
    if router_grad:
        dX = out["dX_experts"].copy()
        out["dW_r"], _ = oracle.route_bwd(X, inp["W_r"].astype(np.float64), out["topk_idx"], tw, dw, dX, np.float64)
        out["dX"] = dX
    return out


def run_gpu_tq(inp, tqw, spaces, router_grad):
    import torch
    import paper_2606_07404_b200 as tq
    from parity_util import to_dev
    layer = tq.TqpLayer(inp["T"], inp["d"], inp["F"], inp["E"], inp["k"], inp["r"], lora_scale=inp["lora_scale"], training=True)
    dev = to_dev(inp)
    sp = {}
    for name, S in spaces.items():
        n = S["n"]
        lv = torch.from_numpy(S["levels"]).cuda()
        if n & (n - 1) == 0:
            sp[name] = tq.TqSpace(n, lv, signs=torch.from_numpy(np.sign(S["R"][0] * np.sqrt(n)).astype(np.int8)).cuda())
        else:
            sp[name] = tq.TqSpace(n, lv, R=torch.from_numpy(np.ascontiguousarray(S["R"])).cuda())
    wt = {key: torch.from_numpy(v).cuda() for key, v in tqw.items()}
    wt.update({key: dev[key] for key in ("A_gate", "A_up", "B_gate", "B_up", "A_down", "B_down")})
    layer.bind_weights_tq(sp["d"], sp["F"], **wt)
    T, k, F, d = inp["T"], inp["k"], inp["F"], inp["d"]
    N = T * k
    idx, w, lg = layer.route(dev["X"], dev["W_r"], dev.get("logit_bias"), want_logits=True)
    counts, offsets, perm, inv = layer.dispatch(idx)
    Ye = layer.expert_fwd(dev["X"], offsets, perm)
    Y = layer.combine(Ye, inv, w)
    res = dict(logits=lg, topk_idx=idx, topk_w=w, counts=counts, offsets=offsets, perm=perm, inv_perm=inv, Ye=Ye, Y=Y)
    for name in ("G", "U"):
        res[name] = layer.debug_buffer(name, (N, F), torch.bfloat16).clone()
    dYe, dw = layer.combine_bwd(dev["dY"], Ye, inv, w, want_dw=True, perm=perm)
    dXp, grads = layer.expert_bwd(dev["X"], dYe, offsets, perm, dYe_unmodified=True)
    dX = layer.dispatch_bwd(dXp, inv)
    res.update(dYe=dYe, dtopk_w=dw, dX_experts=dX.clone(), **grads)
    if router_grad:
        res["dW_r"] = layer.route_bwd(dev["X"], dev["W_r"], idx, w, dw, offsets, perm, dX)
        res["dX"] = dX
    torch.cuda.synchronize()
    return {key: to_np(v) for key, v in res.items()}, layer


CASES = [
    ti.Config("tq_hadamard", T=640, d=256, F=512, E=6, k=3, r=16, seed=61, router_grad=True),
    ti.Config("tq_r32", T=300, d=512, F=256, E=5, k=2, r=32, seed=62, router_grad=True, lora_scale=0.5),
    ti.Config("tq_dense_d", T=500, d=768, F=256, E=4, k=2, r=16, seed=63, router_grad=True),     # d = 768: sign-fixed QR rotation
    ti.Config("tq_dense_F", T=400, d=256, F=768, E=4, k=2, r=16, seed=65, router_grad=True),     # F = 768: QR rotation of the hidden space
]


@pytest.mark.parametrize("cfg", CASES, ids=lambda c: c.name)
def test_tq_layer_full_chain(cfg):
    inp, tqw, spaces = make_tq_inputs(cfg, adapter_std=0.03)
    bias = np.zeros(cfg.E, np.float32); bias[1] = 2.0; bias[cfg.E - 1] = -50.0        # >256 rows on one expert, none on another
    inp["logit_bias"] = bias
    ref = oracle_tq_layer(inp, tqw, spaces, router_grad=True)
    gpu, _ = run_gpu_tq(inp, tqw, spaces, router_grad=True)
    assert_routing_exact(gpu, ref)
    assert ref["counts"].max() > 256 and ref["counts"].min() == 0
    for key in ("G", "U", "Ye", "Y", "dYe", "dtopk_w", "dX_experts", "dX", "dW_r",
                "dA_gate", "dB_gate", "dA_up", "dB_up", "dA_down", "dB_down"):
        ma, rf = assert_close(key, gpu[key], ref[key])
        print(f"{cfg.name} {key:10s} maxabs {ma:.2e} relF {rf:.2e}")
    for key in ("dA_gate", "dB_gate", "dA_up", "dB_up", "dA_down", "dB_down"):
        assert (gpu[key][cfg.E - 1] == 0).all()


def test_tq_step_host_matches_the_stepwise_calls():
    """tqp_step_host_async over a TurboQuant base (pinned host X / dY in, Y / dX out, two steps in flight): bit-identical to
    the stepwise API (same kernels, same order), including the gradients that come back through R^T."""
    import torch
    cfg = ti.Config("tq_host", T=1100, d=256, F=256, E=6, k=2, r=16, seed=64, router_grad=True)
    inp, tqw, spaces = make_tq_inputs(cfg, adapter_std=0.03)
    step, layer = run_gpu_tq(inp, tqw, spaces, router_grad=True)
    T, d = cfg.T, cfg.d
    pin = lambda a: torch.from_numpy(a.view(np.int16)).view(torch.bfloat16).pin_memory()
    Xh, dYh = pin(inp["X"]), pin(inp["dY"])
    outs = [(torch.zeros((T, d), dtype=torch.bfloat16).pin_memory(), torch.zeros((T, d), dtype=torch.bfloat16).pin_memory()) for _ in range(2)]
    grads = layer.alloc_grads()
    W_r = torch.from_numpy(inp["W_r"]).cuda()
    dW_r = torch.zeros((d, cfg.E), dtype=torch.float32, device="cuda")
    for i in range(2):
        layer.step_host_async(Xh, dYh, W_r, None, outs[i][0], outs[i][1], grads, dW_r)
    layer.step_host_wait(0)
    torch.cuda.synchronize()
    for i in range(2):
        np.testing.assert_array_equal(to_np(outs[i][0]), step["Y"])
        np.testing.assert_array_equal(to_np(outs[i][1]), step["dX"])
    np.testing.assert_array_equal(to_np(dW_r), step["dW_r"])
    for key in ("dA_gate", "dB_gate", "dA_up", "dB_up", "dA_down", "dB_down"):
        np.testing.assert_array_equal(to_np(grads[key]), step[key], err_msg=key)


def test_rebinding_between_the_two_base_formats():
    """One ctx: TurboQuant base bound, then the vector-quantised base of the same shape, then TurboQuant again.  Each bind
    must fully replace the other's state (GEMM problems, look-up tables, rotated-adapter buffers): results equal those of
    a fresh ctx bit for bit."""
    import torch
    from parity_util import make_layer, run_gpu, to_dev
    cfg = ti.Config("tq_rebind", T=300, d=256, F=256, E=4, k=2, r=16, seed=66, router_grad=False)
    inp, tqw, spaces = make_tq_inputs(cfg, adapter_std=0.03)
    fresh_tq, layer = run_gpu_tq(inp, tqw, spaces, router_grad=False)
    fresh_vq = run_gpu(inp, backward=True, router_grad=False)
    dev = to_dev(inp)
    layer.bind_weights(**{n: dev[n] for n in ("idx_gate", "idx_up", "idx_down", "scale_gate", "scale_up", "scale_down", "codebook",
                                              "A_gate", "A_up", "B_gate", "B_up", "A_down", "B_down")})

    def chain():
        idx, w = layer.route(dev["X"], dev["W_r"], None)
        counts, offsets, perm, inv = layer.dispatch(idx)
        Ye = layer.expert_fwd(dev["X"], offsets, perm)
        Y = layer.combine(Ye, inv, w)
        dYe, _ = layer.combine_bwd(dev["dY"], Ye, inv, w, want_dw=False, perm=perm)
        dXp, grads = layer.expert_bwd(dev["X"], dYe, offsets, perm, dYe_unmodified=True)
        dX = layer.dispatch_bwd(dXp, inv)
        torch.cuda.synchronize()
        return dict(Y=to_np(Y), dX_experts=to_np(dX), **{k_: to_np(v) for k_, v in grads.items()})

    got_vq = chain()
    for key in got_vq:
        np.testing.assert_array_equal(got_vq[key], fresh_vq[key], err_msg=f"VQ after TQ: {key}")
    sp = layer.spaces
    wt = {key: torch.from_numpy(v).cuda() for key, v in tqw.items()}
    wt.update({key: dev[key] for key in ("A_gate", "A_up", "B_gate", "B_up", "A_down", "B_down")})
    layer.bind_weights_tq(sp[0], sp[1], **wt)
    got_tq = chain()
    for key in got_tq:
        np.testing.assert_array_equal(got_tq[key], fresh_tq[key], err_msg=f"TQ after VQ: {key}")
