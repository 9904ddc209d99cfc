"""GPU parity at BASELINE.json's FULL sizes (configs 1-4, plus the paper-width shape 5), in the launch configuration bench.py times.

Routing, permutation, combine and the HBM-bound backward steps are compared over the whole tensors (the oracle is
cheap there).  The grouped expert FFN — too slow to run through the oracle for 460 experts inside a test — is compared
on a SAMPLE of experts the oracle computes one by one (largest, smallest, an empty one if any, and seeded random
ones): every routed row, every output element and every adapter-gradient element of the sampled experts."""
import numpy as np
import pytest

import oracle
import tqp_inputs as ti
from parity_util import assert_close, assert_routing_exact, run_gpu

pytestmark = pytest.mark.gpu


def sample_experts(counts, seed, n_random=3):
    nz = np.nonzero(counts)[0]
    S = {int(nz[np.argmax(counts[nz])]), int(nz[np.argmin(counts[nz])])}
    empty = np.nonzero(counts == 0)[0]
    if len(empty):
        S.add(int(empty[0]))
    rng = np.random.default_rng(seed)
    S.update(int(e) for e in rng.choice(len(counts), size=n_random, replace=False))
    return sorted(S)


def sub_problem(inp, S, offsets, perm):
    """The layer restricted to the experts in S (weights sliced, rows re-based); X stays whole."""
    sub = dict(inp)
    for key in ("idx_gate", "idx_up", "idx_down", "scale_gate", "scale_up", "scale_down",
                "A_gate", "B_gate", "A_up", "B_up", "A_down", "B_down"):
        sub[key] = np.ascontiguousarray(inp[key][S])
    sub["E"] = len(S)
    segs = [np.arange(offsets[e], offsets[e + 1]) for e in S]
    rows = np.concatenate(segs) if segs else np.zeros(0, np.int64)
    offs = np.zeros(len(S) + 1, np.int32)
    offs[1:] = np.cumsum([len(s) for s in segs])
    return sub, rows, offs, np.ascontiguousarray(perm[rows])


@pytest.mark.parametrize("cfg_id", [1, 2, 3, 4, 5])
def test_full_size_config(cfg_id):
    cfg = ti.CONFIGS[cfg_id]
    inp = ti.make_inputs(cfg)
    T, k, E, d, F = cfg.T, cfg.k, cfg.E, cfg.d, cfg.F
    gpu = run_gpu(inp, backward=cfg.backward, router_grad=cfg.router_grad, gemm_impl=0)

    # ---- routing and permutation: whole tensors, bit-exact ----
    lg = oracle.logits(inp["X"], inp["W_r"], inp["logit_bias"])
    ref = {"logits": lg}
    ref["topk_idx"], ref["topk_w"] = oracle.topk(lg, k)
    ref["counts"], ref["offsets"], ref["perm"], ref["inv_perm"] = oracle.dispatch(ref["topk_idx"], E)
    assert_routing_exact(gpu, ref)
    counts, offsets, perm, inv = ref["counts"], ref["offsets"], ref["perm"], ref["inv_perm"]
    if cfg.skew:
        print(f"cfg{cfg_id}: zero-token experts {np.mean(counts == 0):.1%}, top expert share {counts.max() / counts.sum():.2%}")
        assert (counts == 0).sum() > 0

    # ---- gather (whole tensor, exact) ----
    Xf = ti.bf16_bits_to_f32(inp["X"])
    np.testing.assert_array_equal(gpu["Xp"], Xf[perm // k])

    # ---- expert FFN forward on sampled experts ----
    S = sample_experts(counts, seed=cfg.seed)
    sub, rows, offs, perm_s = sub_problem(inp, S, offsets, perm)
    nrows = int(offs[-1])
    Ye_s, G_s, U_s, H_s = oracle.expert_fwd(sub, offs, perm_s, n_rows=nrows)
    for name, r_ in (("G", G_s), ("U", U_s), ("H", H_s), ("Ye", Ye_s)):
        assert_close(f"cfg{cfg_id} {name}[sampled experts {S}]", gpu[name][rows], r_)

    # ---- combine: whole tensor, given the GPU's own Ye (isolates the step) ----
    Y_ref = oracle.combine(gpu["Ye"], inv, ref["topk_w"])
    assert_close(f"cfg{cfg_id} Y", gpu["Y"], Y_ref, maxabs_tol=4e-3, relf_tol=3e-3)    # one bf16 rounding of the output
    if not cfg.backward:
        return

    # ---- combine backward: whole tensors ----
    dYe_ref, dw_ref = oracle.combine_bwd(inp["dY"], gpu["Ye"], inv, ref["topk_w"])
    assert_close(f"cfg{cfg_id} dYe", gpu["dYe"], dYe_ref, maxabs_tol=4e-3, relf_tol=3e-3)
    assert_close(f"cfg{cfg_id} dtopk_w", gpu["dtopk_w"], dw_ref, maxabs_tol=1e-4, relf_tol=1e-5)

    # ---- expert FFN backward on the sampled experts (oracle forward values, oracle dYe) ----
    dYe_oracle_rows = dYe_ref[rows]
    dXp_s, g_s = oracle.expert_bwd(sub, dYe_oracle_rows, G_s, U_s, H_s, offs, perm_s, n_rows=nrows)
    assert_close(f"cfg{cfg_id} dXp[sampled]", gpu["dXp"][rows], dXp_s)
    for key, val in g_s.items():
        got = gpu[key][S]
        nonempty = [i for i, e in enumerate(S) if counts[e] > 0]
        assert_close(f"cfg{cfg_id} {key}[sampled]", got[nonempty], val[nonempty])
        for i, e in enumerate(S):
            if counts[e] == 0:
                assert (got[i] == 0).all(), f"{key}: empty expert {e} must have exactly zero gradient"

    # ---- dispatch backward: whole tensor, given the GPU's dXp ----
    dX_ref = oracle.dispatch_bwd(gpu["dXp"], inv, T, k)
    assert_close(f"cfg{cfg_id} dX_experts", gpu["dX_experts"], dX_ref, maxabs_tol=4e-3, relf_tol=3e-3)

    # ---- router backward (configs 0 and 4): whole tensors, given the GPU's dtopk_w ----
    if cfg.router_grad:
        dX = dX_ref.copy()
        dW_r, _ = oracle.route_bwd(inp["X"], inp["W_r"], ref["topk_idx"], ref["topk_w"], gpu["dtopk_w"], dX)
        assert_close(f"cfg{cfg_id} dW_r", gpu["dW_r"], dW_r, maxabs_tol=1e-3, relf_tol=1e-4)
        assert_close(f"cfg{cfg_id} dX", gpu["dX"], dX, maxabs_tol=8e-3, relf_tol=4e-3)
