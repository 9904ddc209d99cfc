"""TEST INFRASTRUCTURE — CPU oracle of consolidation (component C14).

Only tests/ may import this.  It shares no code with the CUDA path (paper_2606_07404_b200) and does not import it.

PAPER.md L1110 (§10.6): "The trained adapter is merged into the base weights, the result is materialized as bf16";
L1481: "The 120B public artifact is produced by merging the trained TQP update into bf16 expert weights".  With the
adapter of L938 (§9.1: rank-r adapter on each of the three packs) and the reconstruction of L946 (§9.2) this is the
plain definition

    W_eff[in][out] = scale[out] * codebook[idx[out][in/8]][in%8] + s * sum_q A[in][q] * B[q][out]

written out here with numpy in the caller's precision (fp64 in the pins), element by element for the base and one
library matmul for the adapter product.  The result is returned in the released orientation [out][in] (one row per
output channel, the layout of the code indices) and is NOT rounded: the comparison with the bf16 artifact of the CUDA
path allows one bf16 rounding (tests/test_gpu_consolidate.py).
"""
from __future__ import annotations

import numpy as np


def consolidate(idx: np.ndarray, scale: np.ndarray, codebook: np.ndarray, A: np.ndarray, B: np.ndarray, s: float,
                dtype=np.float64) -> np.ndarray:
    """idx u8 [out][in/8], scale [out], codebook [256][8], A [in][r], B [r][out] (already widened to real numbers)
    -> W [out][in] = base + s * (A B)^T."""
    out_dim, nvec = idx.shape
    cb = np.asarray(codebook, dtype=dtype)
    sc = np.asarray(scale, dtype=dtype)
    W = np.empty((out_dim, nvec * 8), dtype=dtype)
    for o in range(out_dim):
        W[o] = sc[o] * cb[idx[o]].reshape(-1)          # row o: the nvec looked-up 8-vectors in order, rescaled
    delta = np.asarray(A, dtype=dtype) @ np.asarray(B, dtype=dtype)      # [in][out]
    return W + dtype(s) * delta.T
