"""TEST INFRASTRUCTURE — CPU oracle of the paper-faithful router variant and its balance controller.

Only tests/ may import this.  It shares no code with the CUDA path (paper_2606_07404_b200) and does not import it.
Plain numpy, written step by step in the paper's order:

  * PAPER.md L224 (§3.4): "Routing scores are produced by a sigmoid, expert selection is biased by a per-expert routing
    logit bias that is adjusted to equalize load, and balance is achieved by moving that bias rather than by adding a
    balancing term to the gradient" (the loss-free scheme of Wang et al. 2024).
  * PAPER.md L1075 (§10.5), L1097 (Table 29), L1516 (Table 37): the 5B/9B stages use "a sign-based update that nudges
    each expert's bias against the sign of its load error"; the 120B uses "a three-tier controller that applies a
    quadratic boost once an expert's load falls outside a target band"; gain MOE_BIAS_GAMMA 1e-4 -> 5e-5, band ceiling
    MOE_EXPERT_CAP_HI 0.005 -> 0.003.

Readings where the paper is silent (R21-R23): the bias enters the SELECTION key only (key = logit + bias;
gate values use the unbiased score); gates are normalised over the selected set, w_j = s_j / sum_i s_i; ties go to
the lower expert id; the three-tier law is  in band: gamma*sign(tau - load);  above the ceiling:
-gamma*(1 + ((load - hi)/tau)^2);  below the floor: +gamma*(1 + ((lo - load)/tau)^2),  with tau = 1/E the uniform share
and the floor lo = tau^2/hi unless given (the paper prints the ceiling only).  Parity unpinned beyond the pins in
tests/test_router_ext_pins.py: the paper prints no worked example of the controller.
"""
from __future__ import annotations

import numpy as np


def route_sigmoid(logits: np.ndarray, select_bias, k: int):
    """logits [T,E] (fp32 or fp64), select_bias [E] or None -> topk_idx [T,k] int32, topk_w [T,k], topk_s [T,k].

    Selection: the k largest keys (logit + bias), ties to the lower expert id, output in that order.
    Scores: s = sigmoid(logit) of the UNBIASED logit; gates w_j = s_j / (s_0 + ... + s_{k-1}), summed in ascending j."""
    dtype = logits.dtype
    T, E = logits.shape
    key = logits if select_bias is None else (logits + np.asarray(select_bias, dtype=dtype)[None, :]).astype(dtype)
    idx = np.empty((T, k), dtype=np.int32)
    s = np.empty((T, k), dtype=dtype)
    w = np.empty((T, k), dtype=dtype)
    one = dtype.type(1)
    for t in range(T):
        order = np.argsort(-key[t], kind="stable")[:k]          # stable: equal keys keep ascending id
        idx[t] = order
        lt = logits[t, order]
        st = one / (one + np.exp(-lt, dtype=dtype))
        tot = dtype.type(0)
        for j in range(k):
            tot = dtype.type(tot + st[j])
        s[t] = st
        w[t] = st / tot
    return idx, w, s


def route_sigmoid_dl(topk_w: np.ndarray, topk_s: np.ndarray, dtopk_w: np.ndarray) -> np.ndarray:
    """Gradient of the loss w.r.t. the SELECTED logits (selection held constant, the bias has no gradient):
    dL/ds_i = (dw_i - sum_j w_j dw_j) / S,  ds_i/dl_i = s_i (1 - s_i),  S = sum s = s_i / w_i."""
    dot = np.sum(topk_w * dtopk_w, axis=1, keepdims=True)
    return (dtopk_w - dot) * topk_w * (1 - topk_s)


def bias_update(counts, bias, mode: str, gamma: float, cap_hi: float = 0.0, cap_lo: float | None = None) -> np.ndarray:
    """One controller step over the per-expert assignment counts of a batch.  Returns the new bias (fp32).

    mode "sign"      : b_e += gamma * sign(tau - load_e)                                  (5B / 9B)
    mode "three_tier": in band as "sign"; load > hi: b_e -= gamma (1 + ((load-hi)/tau)^2);
                       load < lo: b_e += gamma (1 + ((lo-load)/tau)^2)                    (120B)"""
    counts = np.asarray(counts, dtype=np.float64)
    E = counts.shape[0]
    total = counts.sum()
    load = counts / total if total > 0 else np.zeros(E)
    tau = 1.0 / E
    delta = gamma * np.sign(tau - load)
    if mode == "three_tier":
        hi = float(cap_hi)
        lo = tau * tau / hi if cap_lo is None else float(cap_lo)
        above, below = load > hi, load < lo
        delta = np.where(above, -gamma * (1.0 + ((load - hi) / tau) ** 2), delta)
        delta = np.where(below, gamma * (1.0 + ((lo - load) / tau) ** 2), delta)
    elif mode != "sign":
        raise ValueError(mode)
    return (np.asarray(bias, dtype=np.float64) + delta).astype(np.float32)


def route_bwd_from_dl(X: np.ndarray, W_r: np.ndarray, topk_idx: np.ndarray, dl: np.ndarray, dX: np.ndarray):
    """Chain rule through logits = X W_r for the selected entries only (the router is trained):
    dX[t] += sum_j dl[t,j] W_r[:, e_j]  (in place);  returns dW_r with dW_r[:, e_j] += X[t] dl[t,j]."""
    T, k = topk_idx.shape
    dW_r = np.zeros_like(W_r, dtype=dX.dtype)
    for t in range(T):
        for j in range(k):
            e = int(topk_idx[t, j])
            dX[t] += dl[t, j] * W_r[:, e]
            dW_r[:, e] += X[t] * dl[t, j]
    return dW_r
