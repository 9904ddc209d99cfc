"""TEST INFRASTRUCTURE — CPU oracle of the periodic flush over a TurboQuant base and of the
TurboQuant-format expert layer (NEXT-2).

Only tests/ may import this.  It shares no code with the CUDA path (paper_2606_07404_b200) and does not import it.

Flush — PAPER.md L966 (§9.4): "periodically fold the adapter delta into the base, reset the adapter factors, and let
the next window accumulate a fresh low-rank increment"; L1047-1051 (§10.3): "two quantities were logged: the mean adapter
norm across the injected layers, and the share of each effective weight still coming from the frozen base rather than
the adapter delta" (Table 28).  With the adapter of L938 (rank-r A, B on each pack) and the quantiser of L944-946
(oracle/turboquant.py) the fold is the plain definition, per pack of one expert, in the paper's order:

    W        = decode(codes, norms)                       reconstruction of the base          [out][in]
    W_merged = W + s * (A . B)^T                          fold the adapter delta in           (A [in][r], B [r][out])
    codes', norms' = encode(W_merged)                     re-quantise row by row (L946)
    B' = 0, A' = A_new if given else A                    reset the adapter factors

Readings where the paper is silent (R24-R26):
  * reset: B <- 0 (the delta s.A.B vanishes, so right after a flush the layer computes what it computed before it, up to
    the quantiser's distortion); A <- freshly drawn values handed in by the caller (the method's random numbers are
    inputs), or kept;
  * "adapter norm" = || s . A . B ||_F of one pack of one expert; "base-weight share" = ||W||_F / (||W||_F + ||s.A.B||_F)
    with W the reconstruction of the base BEFORE the fold.  Parity unpinned against Table 28 (its numbers come from a
    training run); pinned by closed forms below.

Layer in the TurboQuant format — the same definition as oracle/tqp_oracle.c (L401, L938) with the reconstruction of
L946 ("looks up the codebook values and rescales by the stored norm", after rotating back) as the base weight.
"""
from __future__ import annotations

import numpy as np

from . import turboquant as tq


def flush_pack(codes, norms, A, B, s, R, codebook, A_new=None):
    """One pack of one expert.  codes [out][in] uint8, norms [out], A [in][r], B [r][out] (real numbers).
    Returns dict(codes, norms, A, B, adapter_norm, base_share, W_merged)."""
    W = tq.decode(codes, norms, R, codebook)                                  # [out][in]
    delta = float(s) * (np.asarray(A, np.float64) @ np.asarray(B, np.float64)).T
    W_merged = W + delta
    codes2, norms2 = tq.encode(W_merged, R, codebook)
    nb, na = np.linalg.norm(W), np.linalg.norm(delta)
    return dict(codes=codes2, norms=norms2, A=np.array(A_new if A_new is not None else A, np.float64),
                B=np.zeros_like(np.asarray(B, np.float64)), adapter_norm=na, base_share=nb / (nb + na) if nb + na > 0 else 1.0,
                W_merged=W_merged)


def dense_weights(codes, norms, A, B, s, R, codebook):
    """Effective weight of one pack of one expert in the "x . W" orientation [in][out]: decode(base)^T + s A B."""
    return tq.decode(codes, norms, R, codebook).T + float(s) * (np.asarray(A, np.float64) @ np.asarray(B, np.float64))


def expert_ffn(x, Wg, Wu, Wd):
    """Rows x [n][d] through one expert's dense SwiGLU FFN: returns y, g, u, h."""
    g = x @ Wg
    u = x @ Wu
    h = g / (1.0 + np.exp(-g)) * u
    return h @ Wd, g, u, h


def expert_ffn_bwd(x, dy, g, u, h, Wg, Wu, Wd):
    """Backward of expert_ffn for the INPUT and the effective weights: returns dx, dWg, dWu, dWd (all dense, fp64);
    the adapter gradients follow as dA = s dW B^T, dB = s A^T dW."""
    dh = dy @ Wd.T
    sig = 1.0 / (1.0 + np.exp(-g))
    du = dh * g * sig
    dg = dh * u * sig * (1.0 + g * (1.0 - sig))
    return dg @ Wg.T + du @ Wu.T, x.T @ dg, x.T @ du, h.T @ dy
