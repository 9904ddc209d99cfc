"""Pins of the consolidation oracle (oracle/consolidate.py; §10.6).  CPU only.

The consolidated matrix is checked against things other than its own formula: a hand-computed 2 x 8 example, the
independently written C oracle of the expert forward (x . W_eff must equal the factored g = x.Wdeq + s (x.A).B that
tqp_oracle.c computes, for every pack), and the special cases A = 0 / B = 0 (the dequantised base alone)."""
import numpy as np

import oracle
import tqp_inputs as ti
from oracle import consolidate as oc


def test_hand_computed_example():
    """in = 8, out = 2, r = 1.  Row 0 uses code 1 scaled by 2, row 1 code 0 scaled by -1; A = e_3 (only input 3),
    B = [10, 20], s = 0.5: row 0 gains 5 at column 3, row 1 gains 10 at column 3."""
    cb = np.zeros((256, 8)); cb[0] = np.arange(8); cb[1] = np.arange(8) * 10
    idx = np.array([[1], [0]], np.uint8)
    scale = np.array([2.0, -1.0])
    A = np.zeros((8, 1)); A[3, 0] = 1.0
    B = np.array([[10.0, 20.0]])
    W = oc.consolidate(idx, scale, cb, A, B, 0.5)
    exp = np.array([[0, 20, 40, 60 + 5, 80, 100, 120, 140], [0, -1, -2, -3 + 10, -4, -5, -6, -7]], float)
    np.testing.assert_array_equal(W, exp)


def _widen(inp, name):
    a = inp[name]
    if a.dtype == np.uint16:                                  # bf16 bit patterns
        return (a.astype(np.uint32) << 16).view(np.float32).astype(np.float64)
    return a.astype(np.float64)


def test_dense_forward_with_consolidated_weights_equals_the_factored_oracle():
    """An 'ordinary bf16 MoE' forward through the merged matrices must reproduce the quantised-plus-adapter forward of
    the C oracle (fp64, so only the order of summation differs)."""
    cfg = ti.CONFIGS[0]
    inp = ti.make_inputs(cfg)
    ref = oracle.layer(inp, dtype=np.float64, backward=False)
    X = _widen(inp, "X")
    cb = _widen(inp, "codebook")
    s = cfg.lora_scale
    offsets, perm = ref["offsets"], ref["perm"]
    Ye = np.zeros_like(ref["Ye"])
    for e in range(cfg.E):
        W = {}
        for pack in ("gate", "up", "down"):
            W[pack] = oc.consolidate(inp["idx_" + pack][e], _widen(inp, "scale_" + pack)[e], cb, _widen(inp, "A_" + pack)[e],
                                     _widen(inp, "B_" + pack)[e], s)
        rows = np.arange(offsets[e], offsets[e + 1])
        x = X[perm[rows] // cfg.k]
        g, u = x @ W["gate"].T, x @ W["up"].T
        h = g / (1.0 + np.exp(-g)) * u
        Ye[rows] = h @ W["down"].T
    assert np.abs(Ye - ref["Ye"]).max() <= 1e-10 * np.abs(ref["Ye"]).max()


def test_zero_adapter_leaves_the_dequantised_base():
    cfg = ti.CONFIGS[0]
    inp = ti.make_inputs(cfg)
    cb = _widen(inp, "codebook")
    e = 3
    A, B = _widen(inp, "A_gate")[e], _widen(inp, "B_gate")[e]
    base = oracle.dequant(inp["idx_gate"][e], inp["scale_gate"][e], inp["codebook"], dtype=np.float64)     # [in][out], C code
    for W in (oc.consolidate(inp["idx_gate"][e], _widen(inp, "scale_gate")[e], cb, np.zeros_like(A), B, 1.0),
              oc.consolidate(inp["idx_gate"][e], _widen(inp, "scale_gate")[e], cb, A, np.zeros_like(B), 1.0),
              oc.consolidate(inp["idx_gate"][e], _widen(inp, "scale_gate")[e], cb, A, B, 0.0)):
        np.testing.assert_array_equal(W, base.T)
    full = oc.consolidate(inp["idx_gate"][e], _widen(inp, "scale_gate")[e], cb, A, B, 2.0)
    np.testing.assert_allclose(full - base.T, 2.0 * (A @ B).T, rtol=0, atol=1e-12)
    assert np.abs(full - base.T).max() > 0
