"""Helpers of the GPU parity tests: run the CUDA path through the C ABI binding, widen results to fp32 numpy, and
compare against the oracle with the tolerances BASELINE.json north_star states."""
from __future__ import annotations

import numpy as np

import tqp_inputs as ti

MAXABS_TOL = 2e-2   # max|gpu-ref| <= 2e-2 * max|ref|      (north_star)
RELF_TOL = 1e-2     # ||gpu-ref||_F <= 1e-2 * ||ref||_F     (north_star)
TOPKW_TOL = 1e-6    # abs, SURVEY §8(d)


def to_dev(inp, device="cuda:0"):
    import torch
    out = {}
    for key, v in inp.items():
        if not isinstance(v, np.ndarray):
            continue
        t = torch.from_numpy(v)
        if v.dtype == np.uint16:
            t = torch.from_numpy(v.view(np.int16)).view(torch.bfloat16)
        out[key] = t.to(device)
    return out


def to_np(t):
    import torch
    if t.dtype == torch.bfloat16:
        return t.float().cpu().numpy()
    return t.cpu().numpy()


def make_layer(inp, T_max=None, training=True, gemm_impl=0):
    import paper_2606_07404_b200 as tq
    layer = tq.TqpLayer(T_max or inp["T"], inp["d"], inp["F"], inp["E"], inp["k"], inp["r"],
                        lora_scale=inp["lora_scale"], training=training)
    layer.set_option("gemm_impl", gemm_impl)
    dev = to_dev(inp)
    layer.bind_weights(**{n: dev[n] for n in ("idx_gate", "idx_up", "idx_down", "scale_gate", "scale_up", "scale_down",
                                              "codebook", "A_gate", "A_up", "B_gate", "B_up", "A_down", "B_down")})
    return layer, dev


def run_gpu(inp, backward=True, router_grad=False, gemm_impl=0, keep_dev=False, fused_bwd=True, route_impl=0, options=None):
    """The whole chain through the C ABI; returns fp32/int numpy arrays keyed like oracle.layer().  fused_bwd: the call
    sequence bench.py times (tqp_combine_bwd with perm, tqp_expert_bwd with TQP_BWD_DYE_UNMODIFIED); False: the plain
    combine_bwd kernel and an expert_bwd that trusts nothing from earlier calls."""
    import torch
    layer, dev = make_layer(inp, training=backward, gemm_impl=gemm_impl)
    for name, value in (options or {}).items():   # any other library option (tqp_set_option)
        layer.set_option(name, value)
    T, k, F, d = inp["T"], inp["k"], inp["F"], inp["d"]
    N = T * k
    out = {}
    bias = dev.get("logit_bias")
    # the dense canonical chain (logits requested) and the call bench.py makes (no logits: the screened router where the
    # library picks it) must agree bit for bit; the rest of the chain runs on the second call's outputs
    idx_d, w_d, lg = layer.route(dev["X"], dev["W_r"], bias, want_logits=True)
    assert layer.route_info() == (0, 0)
    layer.set_option("route_impl", route_impl)
    idx, w = layer.route(dev["X"], dev["W_r"], bias)
    out_info = layer.route_info()
    assert torch.equal(idx, idx_d), "topk_idx: screened router differs from the dense chain"
    assert torch.equal(w.view(torch.int32), w_d.view(torch.int32)), "topk_w: screened router differs from the dense chain (bitwise)"
    counts, offsets, perm, inv = layer.dispatch(idx)
    Ye = layer.expert_fwd(dev["X"], offsets, perm)
    Y = layer.combine(Ye, inv, w)
    res = dict(logits=lg, topk_idx=idx, topk_w=w, counts=counts, offsets=offsets, perm=perm, inv_perm=inv, Ye=Ye, Y=Y)
    for name in ("G", "U", "H"):
        res[name] = layer.debug_buffer(name, (N, F), torch.bfloat16).clone()
    res["Xp"] = layer.debug_buffer("Xp", (N, d), torch.bfloat16).clone()
    if backward:
        fused = fused_bwd and inp["r"] in (16, 32)
        dYe, dw = layer.combine_bwd(dev["dY"], Ye, inv, w, want_dw=True, perm=perm if fused_bwd else None)
        dXp, grads = layer.expert_bwd(dev["X"], dYe, offsets, perm, dYe_unmodified=fused)
        dX = layer.dispatch_bwd(dXp, inv)
        res.update(dYe=dYe, dtopk_w=dw, dXp=dXp, dX_experts=dX.clone(), **grads)
        for name in ("dH", "dG", "dU"):
            res[name] = layer.debug_buffer(name, (N, F), torch.bfloat16).clone()
        if router_grad:
            res["dW_r"] = layer.route_bwd(dev["X"], dev["W_r"], idx, w, dw, offsets, perm, dX)
            res["dX"] = dX
    torch.cuda.synchronize()
    out = {key: to_np(v) for key, v in res.items()}
    out["route_info"] = out_info   # (screened, fallback) of the second route call
    if keep_dev:
        out["_layer"], out["_dev"], out["_res"] = layer, dev, res
    return out


def errors(gpu, ref):
    gpu = np.asarray(gpu, dtype=np.float64); ref = np.asarray(ref, dtype=np.float64)
    mx = np.abs(ref).max()
    maxabs = np.abs(gpu - ref).max() / mx if mx > 0 else np.abs(gpu - ref).max()
    nf = np.linalg.norm(ref)
    relf = np.linalg.norm(gpu - ref) / nf if nf > 0 else np.linalg.norm(gpu - ref)
    return float(maxabs), float(relf)


def assert_close(name, gpu, ref, maxabs_tol=MAXABS_TOL, relf_tol=RELF_TOL):
    assert np.isfinite(gpu).all(), f"{name}: non-finite values on the GPU side"
    maxabs, relf = errors(gpu, ref)
    assert maxabs <= maxabs_tol and relf <= relf_tol, f"{name}: maxabs/max|ref|={maxabs:.3e} relF={relf:.3e}"
    return maxabs, relf


def assert_routing_exact(gpu, ref):
    for key in ("topk_idx", "counts", "offsets", "perm", "inv_perm"):
        np.testing.assert_array_equal(gpu[key], ref[key], err_msg=key)
    np.testing.assert_array_equal(gpu["logits"], ref["logits"], err_msg="fp32 logits (canonical fmaf order, R1)")
    assert np.abs(gpu["topk_w"] - ref["topk_w"]).max() <= TOPKW_TOL
