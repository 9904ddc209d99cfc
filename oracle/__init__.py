"""TEST INFRASTRUCTURE — ctypes front of the CPU oracle (oracle/tqp_oracle.c).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this.
It shares no code with the CUDA path (paper_2606_07404_b200) and does not import it.

The functions mirror the steps of SURVEY.md §8(c) / DESIGN.md "Oracle": dequant, logits, topk, dispatch,
expert_fwd, combine and the four backward steps.  `dtype` selects the fp32 (np.float32) or fp64
(np.float64) instantiation of the same C text.  Storage formats are widened exactly before the call
(bf16 bit patterns -> float via a 16-bit shift, fp16 -> float via numpy), so no fp16/bf16 arithmetic
happens anywhere in the oracle.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libtqp_oracle.so")
_SRC = [os.path.join(_HERE, "tqp_oracle.c"), os.path.join(_HERE, "tqp_oracle_impl.inc")]
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (plain C, OpenMP over experts/tokens)."""
    if not force and os.path.exists(_LIB_PATH) and all(
        os.path.getmtime(_LIB_PATH) >= os.path.getmtime(s) for s in _SRC
    ):
        return _LIB_PATH
    cmd = ["gcc", "-O3", "-march=native", "-fopenmp", "-ffp-contract=off", "-shared", "-fPIC",
           "-o", _LIB_PATH, _SRC[0], "-lm"]
    subprocess.run(cmd, check=True, cwd=_HERE)
    return _LIB_PATH


def lib() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
    return _lib


def num_threads() -> int:
    return int(lib().tqp_oracle_num_threads())


def _sfx(dtype) -> str:
    return "_f32" if np.dtype(dtype) == np.float32 else "_f64"


def _p(a):
    if a is None:
        return None
    assert a.flags["C_CONTIGUOUS"]
    return a.ctypes.data_as(ctypes.c_void_p)


def _real(x, dtype):
    """Exact widening of any storage format to the oracle's REAL."""
    if x is None:
        return None
    if x.dtype == np.uint16:  # bf16 bit patterns
        x = (x.astype(np.uint32) << 16).view(np.float32)
    return np.ascontiguousarray(x, dtype=dtype)


def _i32(x):
    return np.ascontiguousarray(x, dtype=np.int32)


def _scalar(s, dtype):
    return ctypes.c_float(s) if np.dtype(dtype) == np.float32 else ctypes.c_double(s)


def dequant(idx, scale, codebook, dtype=np.float32):
    """Wdeq[in][out] of one pack of one expert; idx [out][in/8]."""
    out_dim, nvec = idx.shape
    W = np.empty((nvec * 8, out_dim), dtype=dtype)
    getattr(lib(), "tqp_oracle_dequant" + _sfx(dtype))(
        _p(np.ascontiguousarray(idx)), _p(_real(scale, dtype)), _p(_real(codebook, dtype)),
        ctypes.c_int(out_dim), ctypes.c_int(nvec * 8), _p(W))
    return W


def logits(X, W_r, bias=None, dtype=np.float32):
    X = _real(X, dtype); W_r = _real(W_r, dtype); bias = _real(bias, dtype)
    T, d = X.shape
    E = W_r.shape[1]
    out = np.empty((T, E), dtype=dtype)
    getattr(lib(), "tqp_oracle_logits" + _sfx(dtype))(_p(X), _p(W_r), _p(bias), T, d, E, _p(out))
    return out


def topk(lg, k):
    dtype = lg.dtype
    T, E = lg.shape
    idx = np.empty((T, k), dtype=np.int32)
    w = np.empty((T, k), dtype=dtype)
    getattr(lib(), "tqp_oracle_topk" + _sfx(dtype))(_p(np.ascontiguousarray(lg)), T, E, k, _p(idx), _p(w))
    return idx, w


def dispatch(topk_idx, E):
    topk_idx = _i32(topk_idx)
    T, k = topk_idx.shape
    N = T * k
    counts = np.empty(E, dtype=np.int32)
    offsets = np.empty(E + 1, dtype=np.int32)
    perm = np.empty(N, dtype=np.int32)
    inv_perm = np.empty(N, dtype=np.int32)
    lib().tqp_oracle_dispatch(_p(topk_idx), T, k, E, _p(counts), _p(offsets), _p(perm), _p(inv_perm))
    return counts, offsets, perm, inv_perm


_WKEYS = ("scale_gate", "scale_up", "scale_down", "codebook",
          "A_gate", "B_gate", "A_up", "B_up", "A_down", "B_down")


def _weights(inp, dtype):
    idx = [np.ascontiguousarray(inp[n]) for n in ("idx_gate", "idx_up", "idx_down")]
    real = [_real(inp[n], dtype) for n in _WKEYS]
    return idx, real


def expert_fwd(inp, offsets, perm, dtype=np.float32, save=True, n_rows=None):
    """Returns Ye [N,d] (and G, U, H [N,F] when save).  n_rows: number of routed rows actually present
    (offsets[E]) when the call covers a sample of experts only; default N = T*k."""
    X = _real(inp["X"], dtype)
    T, d = X.shape
    F, E, k, r = inp["F"], inp["E"], inp["k"], inp["r"]
    N = T * k if n_rows is None else n_rows
    idx, real = _weights(inp, dtype)
    Ye = np.empty((N, d), dtype=dtype)
    G = np.empty((N, F), dtype=dtype) if save else None
    U = np.empty((N, F), dtype=dtype) if save else None
    H = np.empty((N, F), dtype=dtype) if save else None
    getattr(lib(), "tqp_oracle_expert_fwd" + _sfx(dtype))(
        _p(X), T, d, F, E, k, r, _scalar(inp["lora_scale"], dtype), _p(_i32(offsets)), _p(_i32(perm)),
        *[_p(a) for a in idx], *[_p(a) for a in real], _p(Ye), _p(G), _p(U), _p(H))
    return (Ye, G, U, H) if save else Ye


def combine(Ye, inv_perm, topk_w):
    dtype = Ye.dtype
    T, k = topk_w.shape
    d = Ye.shape[1]
    Y = np.empty((T, d), dtype=dtype)
    getattr(lib(), "tqp_oracle_combine" + _sfx(dtype))(
        _p(np.ascontiguousarray(Ye)), _p(_i32(inv_perm)), _p(_real(topk_w, dtype)), T, d, k, _p(Y))
    return Y


def combine_bwd(dY, Ye, inv_perm, topk_w, dtype=np.float32):
    dY = _real(dY, dtype); Ye = _real(Ye, dtype)
    T, k = topk_w.shape
    d = dY.shape[1]
    dYe = np.empty((T * k, d), dtype=dtype)
    dw = np.empty((T, k), dtype=dtype)
    getattr(lib(), "tqp_oracle_combine_bwd" + _sfx(dtype))(
        _p(dY), _p(Ye), _p(_i32(inv_perm)), _p(_real(topk_w, dtype)), T, d, k, _p(dYe), _p(dw))
    return dYe, dw


def expert_bwd(inp, dYe, G, U, H, offsets, perm, dtype=np.float32, n_rows=None):
    """Returns dXp [N,d] and the dict of adapter gradients (fp, overwritten, zero for empty experts)."""
    X = _real(inp["X"], dtype)
    T, d = X.shape
    F, E, k, r = inp["F"], inp["E"], inp["k"], inp["r"]
    N = T * k if n_rows is None else n_rows
    idx, real = _weights(inp, dtype)
    dXp = np.empty((N, d), dtype=dtype)
    g = {
        "dA_gate": np.empty((E, d, r), dtype=dtype), "dB_gate": np.empty((E, r, F), dtype=dtype),
        "dA_up": np.empty((E, d, r), dtype=dtype), "dB_up": np.empty((E, r, F), dtype=dtype),
        "dA_down": np.empty((E, F, r), dtype=dtype), "dB_down": np.empty((E, r, d), dtype=dtype),
    }
    getattr(lib(), "tqp_oracle_expert_bwd" + _sfx(dtype))(
        _p(X), _p(_real(dYe, dtype)), _p(_real(G, dtype)), _p(_real(U, dtype)), _p(_real(H, dtype)),
        T, d, F, E, k, r, _scalar(inp["lora_scale"], dtype), _p(_i32(offsets)), _p(_i32(perm)),
        *[_p(a) for a in idx], *[_p(a) for a in real], _p(dXp),
        _p(g["dA_gate"]), _p(g["dB_gate"]), _p(g["dA_up"]), _p(g["dB_up"]), _p(g["dA_down"]), _p(g["dB_down"]))
    return dXp, g


def dispatch_bwd(dXp, inv_perm, T, k):
    dtype = dXp.dtype
    d = dXp.shape[1]
    dX = np.empty((T, d), dtype=dtype)
    getattr(lib(), "tqp_oracle_dispatch_bwd" + _sfx(dtype))(
        _p(np.ascontiguousarray(dXp)), _p(_i32(inv_perm)), T, d, k, _p(dX))
    return dX


def route_bwd(X, W_r, topk_idx, topk_w, dtopk_w, dX, dtype=np.float32):
    """Accumulates the router term into dX (in place, must be `dtype`); returns dW_r and dl [T,k]."""
    X = _real(X, dtype); W_r = _real(W_r, dtype)
    T, d = X.shape
    E = W_r.shape[1]
    k = topk_idx.shape[1]
    assert dX.dtype == np.dtype(dtype) and dX.flags["C_CONTIGUOUS"]
    dW_r = np.empty((d, E), dtype=dtype)
    dl = np.empty((T, k), dtype=dtype)
    getattr(lib(), "tqp_oracle_route_bwd" + _sfx(dtype))(
        _p(X), _p(W_r), _p(_i32(topk_idx)), _p(_real(topk_w, dtype)), _p(_real(dtopk_w, dtype)),
        T, d, E, k, _p(dX), _p(dW_r), _p(dl))
    return dW_r, dl


def layer(inp, dtype=np.float32, backward=True, router_grad=False):
    """The whole path in the order of SURVEY §3: route -> dispatch -> expert_fwd -> combine [-> backward]."""
    k, E = inp["k"], inp["E"]
    out = {}
    lg = logits(inp["X"], inp["W_r"], inp.get("logit_bias"), dtype)
    out["logits"] = lg
    out["topk_idx"], out["topk_w"] = topk(lg, k)
    out["counts"], out["offsets"], out["perm"], out["inv_perm"] = dispatch(out["topk_idx"], E)
    Ye, G, U, H = expert_fwd(inp, out["offsets"], out["perm"], dtype)
    out.update(Ye=Ye, G=G, U=U, H=H)
    out["Y"] = combine(Ye, out["inv_perm"], out["topk_w"])
    if not backward:
        return out
    T = inp["X"].shape[0]
    dYe, dw = combine_bwd(inp["dY"], Ye, out["inv_perm"], out["topk_w"], dtype)
    out["dYe"], out["dtopk_w"] = dYe, dw
    dXp, grads = expert_bwd(inp, dYe, G, U, H, out["offsets"], out["perm"], dtype)
    out["dXp"] = dXp
    out.update(grads)
    out["dX_experts"] = dispatch_bwd(dXp, out["inv_perm"], T, k)
    if router_grad:
        dX = out["dX_experts"].copy()
        out["dW_r"], out["dlogits_sel"] = route_bwd(inp["X"], inp["W_r"], out["topk_idx"], out["topk_w"], dw, dX, dtype)
        out["dX"] = dX
    return out
