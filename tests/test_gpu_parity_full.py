"""GPU parity at BASELINE.json's FULL sizes (configs 1-4, plus the paper-width shape 5), in the launch configuration
bench.py times, over ALL experts and end to end.

The oracle runs the whole layer once per config (`oracle.layer`, fp32, as it stands: ~45 s for cfg 2 / 3, ~2 min for
cfg 4 on the GPU box's 16 host cores) and EVERY tensor of the CUDA path is compared with the oracle's OWN value of it:
routing and permutation bit-exact, the gather exact, and G, U, H, Ye, Y, dYe, dtopk_w, dXp, dX, the six adapter
gradients (and dW_r / the router term of dX for cfg 4) within north_star's tolerance — both over the whole tensor and
PER EXPERT (every expert's rows / gradient slices on their own, so that a tile-scheduler or TMA-coordinate bug that
bites at one (expert, tile) position cannot hide in a global norm).

With TQP_PARITY_REPORT=<path> in the environment every config appends its per-tensor error rows (markdown) to that
file; profiles/r2_parity_errors.md is such a file.
"""
import os

import numpy as np
import pytest

import oracle
import tqp_inputs as ti
from parity_util import MAXABS_TOL, RELF_TOL, assert_routing_exact, run_gpu

pytestmark = pytest.mark.gpu

GRADS = ("dA_gate", "dB_gate", "dA_up", "dB_up", "dA_down", "dB_down")
# Per-expert bounds (this file's own, tighter than north_star's per-tensor statement): north_star's two bounds applied to
# every expert's block on its own.  For an expert with fewer than SMALL rows they are doubled: its adapter gradient is the
# outer product of a handful of bf16-rounded rows, the rounding errors of one row do not average out, and the per-expert
# ratio scatters around the tensor-wide 6e-3 (cfg 3 has experts with one or two rows; measured worst 1.25e-2).
SMALL = 16


def per_expert_bounds(rows):
    f = np.where(rows < SMALL, 2.0, 1.0)
    return RELF_TOL * f, MAXABS_TOL * f


def row_stats(gpu, ref, chunk=16384):
    """Per-row sum of squared error, sum of squared reference, max |error|, max |reference| (fp64 accumulation)."""
    n = ref.shape[0]
    se = np.empty(n); sr = np.empty(n); me = np.empty(n); mr = np.empty(n)
    for i in range(0, n, chunk):
        r = ref[i:i + chunk].astype(np.float64)
        dlt = gpu[i:i + chunk].astype(np.float64) - r
        se[i:i + chunk] = np.einsum("ij,ij->i", dlt, dlt)
        sr[i:i + chunk] = np.einsum("ij,ij->i", r, r)
        me[i:i + chunk] = np.abs(dlt).max(axis=1)
        mr[i:i + chunk] = np.abs(r).max(axis=1)
    return se, sr, me, mr


def check_rows(name, gpu, ref, offsets, report):
    """Whole tensor + every expert's row block of a [N][*] tensor."""
    assert np.isfinite(gpu).all(), f"{name}: non-finite values on the GPU side"
    se, sr, me, mr = row_stats(gpu, ref)
    maxabs, relf = me.max() / mr.max(), np.sqrt(se.sum() / sr.sum())
    nz = np.nonzero(np.diff(offsets))[0]
    starts = offsets[nz].astype(np.int64)
    e_relf = np.sqrt(np.add.reduceat(se, starts) / np.add.reduceat(sr, starts))
    e_maxabs = np.maximum.reduceat(me, starts) / np.maximum.reduceat(mr, starts)
    rows = np.diff(offsets)[nz]
    w = int(np.argmax(e_relf))
    report.append((name, maxabs, relf, e_maxabs.max(), e_relf.max(), f"{nz[w]} ({rows[w]} rows)"))
    assert maxabs <= MAXABS_TOL and relf <= RELF_TOL, f"{name}: maxabs/max|ref|={maxabs:.3e} relF={relf:.3e}"
    b_relf, b_maxabs = per_expert_bounds(rows)
    bad = np.nonzero((e_relf > b_relf) | (e_maxabs > b_maxabs))[0]
    assert len(bad) == 0, f"{name}: experts {nz[bad][:8]} rows {rows[bad][:8]} relF {e_relf[bad][:8]} maxabs {e_maxabs[bad][:8]}"


def check_grad(name, gpu, ref, counts, report):
    """Whole tensor + every expert's slice of a [E][*][*] adapter gradient; empty experts exactly zero."""
    assert np.isfinite(gpu).all(), f"{name}: non-finite values on the GPU side"
    E = ref.shape[0]
    g = gpu.reshape(E, -1).astype(np.float64); r = ref.reshape(E, -1).astype(np.float64)
    dlt = g - r
    se, sr = np.einsum("ij,ij->i", dlt, dlt), np.einsum("ij,ij->i", r, r)
    me, mr = np.abs(dlt).max(axis=1), np.abs(r).max(axis=1)
    maxabs, relf = me.max() / mr.max(), np.sqrt(se.sum() / sr.sum())
    nz = counts > 0
    assert (g[~nz] == 0).all() and (r[~nz] == 0).all(), f"{name}: an empty expert must have exactly zero gradient"
    e_relf = np.sqrt(se[nz] / sr[nz]); e_maxabs = me[nz] / mr[nz]
    ids = np.nonzero(nz)[0]
    rows = counts[nz]
    w = int(np.argmax(e_relf))
    report.append((name, maxabs, relf, e_maxabs.max(), e_relf.max(), f"{ids[w]} ({rows[w]} rows)"))
    assert maxabs <= MAXABS_TOL and relf <= RELF_TOL, f"{name}: maxabs/max|ref|={maxabs:.3e} relF={relf:.3e}"
    b_relf, b_maxabs = per_expert_bounds(rows)
    bad = np.nonzero((e_relf > b_relf) | (e_maxabs > b_maxabs))[0]
    assert len(bad) == 0, f"{name}: experts {ids[bad][:8]} rows {rows[bad][:8]} relF {e_relf[bad][:8]} maxabs {e_maxabs[bad][:8]}"


def check_whole(name, gpu, ref, report, maxabs_tol=MAXABS_TOL, relf_tol=RELF_TOL):
    assert np.isfinite(gpu).all(), f"{name}: non-finite values on the GPU side"
    se, sr, me, mr = row_stats(gpu.reshape(gpu.shape[0], -1), ref.reshape(ref.shape[0], -1))
    maxabs, relf = me.max() / mr.max(), np.sqrt(se.sum() / sr.sum())
    report.append((name, maxabs, relf, None, None, None))
    assert maxabs <= maxabs_tol and relf <= relf_tol, f"{name}: maxabs/max|ref|={maxabs:.3e} relF={relf:.3e}"


def write_report(cfg, report, counts, seconds):
    path = os.environ.get("TQP_PARITY_REPORT")
    lines = [f"\n### {cfg.name}: T={cfg.T} d={cfg.d} F={cfg.F} E={cfg.E} k={cfg.k} r={cfg.r}"
             f" ({'fwd+bwd' if cfg.backward else 'fwd'}{', router grad' if cfg.router_grad else ''}); "
             f"{int((counts == 0).sum())} empty experts, largest {int(counts.max())} rows; "
             f"oracle.layer {seconds:.0f} s on {oracle.num_threads()} threads\n",
             "| tensor | maxabs / max\\|ref\\| (bound 2e-2) | relF (bound 1e-2) | worst expert: maxabs | worst expert: relF | (expert) |",
             "|---|---|---|---|---|---|"]
    for name, a, b, c, d_, e in report:
        per = f"| {c:.2e} | {d_:.2e} | {e} |" if c is not None else "| — | — | — |"
        lines.append(f"| {name} | {a:.2e} | {b:.2e} {per}")
    text = "\n".join(lines) + "\n"
    print(text)
    if path:
        with open(path, "a") as f:
            f.write(text)


@pytest.mark.parametrize("cfg_id", [0, 1, 2, 3, 4, 5])
def test_full_size_config(cfg_id):
    import time
    cfg = ti.CONFIGS[cfg_id]
    inp = ti.make_inputs(cfg)
    T, k, E, d, F = cfg.T, cfg.k, cfg.E, cfg.d, cfg.F
    gpu = run_gpu(inp, backward=cfg.backward, router_grad=cfg.router_grad, gemm_impl=0)
    t0 = time.time()
    ref = oracle.layer(inp, dtype=np.float32, backward=cfg.backward, router_grad=cfg.router_grad)
    seconds = time.time() - t0

    # ---- routing and permutation: whole tensors, bit-exact ----
    assert_routing_exact(gpu, ref)
    counts, offsets, perm = ref["counts"], ref["offsets"], ref["perm"]
    if cfg.skew:
        print(f"cfg{cfg_id}: zero-token experts {np.mean(counts == 0):.1%}, top expert share {counts.max() / counts.sum():.2%}")
        assert (counts == 0).sum() > 0

    # ---- gather (whole tensor, exact) ----
    Xf = ti.bf16_bits_to_f32(inp["X"])
    np.testing.assert_array_equal(gpu["Xp"], Xf[perm // k])

    report = []
    try:
        # ---- expert FFN forward, every expert, against the oracle's own values ----
        for name in ("G", "U", "H", "Ye"):
            check_rows(name, gpu[name], ref[name], offsets, report)
        # ---- combine, end to end (the oracle's own Y, not a recombination of the GPU's Ye) ----
        check_whole("Y", gpu["Y"], ref["Y"], report)
        if cfg.backward:
            check_rows("dYe", gpu["dYe"], ref["dYe"], offsets, report)
            check_whole("dtopk_w", gpu["dtopk_w"], ref["dtopk_w"], report)
            check_rows("dXp", gpu["dXp"], ref["dXp"], offsets, report)
            for name in GRADS:
                check_grad(name, gpu[name], ref[name], counts, report)
            check_whole("dX_experts", gpu["dX_experts"], ref["dX_experts"], report)
            if cfg.router_grad:
                check_whole("dW_r", gpu["dW_r"], ref["dW_r"], report)
                check_whole("dX", gpu["dX"], ref["dX"], report)
    finally:
        write_report(cfg, report, counts, seconds)
