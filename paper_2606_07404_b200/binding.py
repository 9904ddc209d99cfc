"""ctypes binding of include/tqp.h.  Argument marshalling only."""
from __future__ import annotations

import ctypes
import os
import re

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libtqp.so")
HEADER = os.path.join(HERE, "..", "include", "tqp.h")
_lib = None

STATUS = {0: "TQP_OK", 1: "TQP_ERR_ARG", 2: "TQP_ERR_SHAPE", 3: "TQP_ERR_ALIGN", 4: "TQP_ERR_WORKSPACE",
          5: "TQP_ERR_STATE", 6: "TQP_ERR_ARCH", 7: "TQP_ERR_CUDA"}


class TqpError(RuntimeError):
    def __init__(self, code, msg=""):
        self.code = code
        super().__init__(f"{STATUS.get(code, code)}: {msg}")


class LayerDesc(ctypes.Structure):
    _fields_ = [("T_max", ctypes.c_int32), ("d", ctypes.c_int32), ("F", ctypes.c_int32), ("E", ctypes.c_int32),
                ("k", ctypes.c_int32), ("r", ctypes.c_int32), ("vec", ctypes.c_int32), ("codes", ctypes.c_int32),
                ("lora_scale", ctypes.c_float), ("training", ctypes.c_int32)]


_WEIGHT_FIELDS = ["idx_gate", "idx_up", "idx_down", "scale_gate", "scale_up", "scale_down", "codebook",
                  "A_gate", "A_up", "B_gate", "B_up", "A_down", "B_down"]


class Weights(ctypes.Structure):
    _fields_ = [(n, ctypes.c_void_p) for n in _WEIGHT_FIELDS]


class TqSpaceC(ctypes.Structure):
    _fields_ = [("n", ctypes.c_int32), ("hadamard", ctypes.c_int32), ("signs", ctypes.c_void_p), ("R", ctypes.c_void_p),
                ("levels", ctypes.c_void_p)]


_TQ_FIELDS_A = ["codes_gate", "codes_up", "codes_down", "norm_gate", "norm_up", "norm_down"]
_TQ_FIELDS_B = ["A_gate", "A_up", "B_gate", "B_up", "A_down", "B_down"]


class TqWeightsC(ctypes.Structure):
    _fields_ = ([(n, ctypes.c_void_p) for n in _TQ_FIELDS_A] + [("space_d", TqSpaceC), ("space_F", TqSpaceC)] +
                [(n, ctypes.c_void_p) for n in _TQ_FIELDS_B])


class TqSpace:
    """tqp_tq_space holder: keeps the device tensors alive.  signs: int8 [n] (Hadamard) or R: float64 [n][n] (dense);
    levels: float64 [256].  All torch CUDA tensors."""

    def __init__(self, n, levels, signs=None, R=None):
        assert (signs is None) != (R is None)
        self.n, self.levels, self.signs, self.R = int(n), levels.contiguous(), signs, R
        self.c = TqSpaceC(self.n, 1 if signs is not None else 0, signs.data_ptr() if signs is not None else None,
                          R.data_ptr() if R is not None else None, self.levels.data_ptr())


def abi_symbols() -> list[str]:
    """Function names declared in include/tqp.h."""
    text = open(HEADER).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(tqp_[a-z_0-9]+)\s*\(", text)))


def load_library() -> ctypes.CDLL:
    """Loads libtqp.so; raises loudly if it has not been built (no fallback of any kind)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise TqpError(-1, f"{LIB_PATH} is missing: run `python -m paper_2606_07404_b200.build` (needs nvcc)")
        lib = ctypes.CDLL(LIB_PATH)
        vp, ci = ctypes.c_void_p, ctypes.c_int
        lib.tqp_create.argtypes = [ctypes.POINTER(vp), ctypes.POINTER(LayerDesc)]
        lib.tqp_destroy.argtypes = [vp]
        lib.tqp_destroy.restype = None
        lib.tqp_workspace_bytes.argtypes = [ctypes.POINTER(LayerDesc)]
        lib.tqp_workspace_bytes.restype = ctypes.c_size_t
        lib.tqp_bind_workspace.argtypes = [vp, vp, ctypes.c_size_t, vp]
        lib.tqp_bind_weights.argtypes = [vp, ctypes.POINTER(Weights), vp]
        lib.tqp_set_option.argtypes = [vp, ctypes.c_char_p, ci]
        lib.tqp_route.argtypes = [vp, ci] + [vp] * 7
        lib.tqp_route_info.argtypes = [vp, ctypes.POINTER(ci), ctypes.POINTER(ci), vp]
        lib.tqp_dispatch.argtypes = [vp, ci] + [vp] * 6
        lib.tqp_dispatch_noalloc.argtypes = [ci, ci, ci] + [vp] * 6
        lib.tqp_dispatch_noalloc_capacity.restype = ctypes.c_size_t
        lib.tqp_dispatch_noalloc_capacity.argtypes = []
        lib.tqp_dispatch_noalloc_error.restype = ctypes.c_char_p
        lib.tqp_dispatch_noalloc_error.argtypes = []
        lib.tqp_expert_fwd.argtypes = [vp, ci] + [vp] * 5
        lib.tqp_combine.argtypes = [vp, ci] + [vp] * 5
        lib.tqp_combine_bwd.argtypes = [vp, ci] + [vp] * 8
        lib.tqp_expert_bwd.argtypes = [vp, ci] + [vp] * 11 + [ci, vp]
        lib.tqp_dispatch_bwd.argtypes = [vp, ci] + [vp] * 4
        lib.tqp_route_bwd.argtypes = [vp, ci] + [vp] * 10
        lib.tqp_step_host.argtypes = [vp, ci] + [vp] * 14
        lib.tqp_step_host_async.argtypes = [vp, ci] + [vp] * 14
        lib.tqp_step_host_wait.argtypes = [vp, ci]
        lib.tqp_route_sigmoid.argtypes = [vp, ci] + [vp] * 8
        lib.tqp_route_sigmoid_bwd.argtypes = [vp, ci] + [vp] * 11
        lib.tqp_bias_update.argtypes = [vp, vp, vp, ci, ctypes.c_float, ctypes.c_float, ctypes.c_float, vp]
        lib.tqp_consolidate.argtypes = [vp, ci, ci, ci, vp, vp]
        sp, ll = ctypes.POINTER(TqSpaceC), ctypes.c_longlong
        lib.tqp_bind_weights_tq.argtypes = [vp, ctypes.POINTER(TqWeightsC), vp]
        lib.tqp_tq_levels.argtypes = [ci, ci, vp]
        lib.tqp_tq_rotation_qr.argtypes = [ci, vp, vp]
        lib.tqp_rotate.argtypes = [vp, sp, vp, ll, vp, ci, vp]
        lib.tqp_tq_encode.argtypes = [vp, sp, vp, ll, vp, vp, vp]
        lib.tqp_tq_decode.argtypes = [vp, sp, vp, vp, ll, vp, vp]
        lib.tqp_tq_flush.argtypes = [vp, sp, ci, ci, ci, ctypes.c_float, vp, vp, vp, vp, vp, vp, vp]
        lib.tqp_debug_buffer.argtypes = [vp, ctypes.c_char_p]
        lib.tqp_debug_buffer.restype = vp
        lib.tqp_gemm_time.argtypes = [vp, ctypes.POINTER(ctypes.c_float), ctypes.POINTER(ctypes.c_int)]
        lib.tqp_gemm_times.argtypes = [vp, ctypes.POINTER(ctypes.c_float), ctypes.c_int, ctypes.POINTER(ctypes.c_int)]
        lib.tqp_last_launch_count.argtypes = [vp]
        lib.tqp_status_string.argtypes = [ci]
        lib.tqp_status_string.restype = ctypes.c_char_p
        lib.tqp_last_error.argtypes = [vp]
        lib.tqp_last_error.restype = ctypes.c_char_p
        _lib = lib
    return _lib


def _desc(T_max, d, F, E, k, r, lora_scale=1.0, training=True) -> LayerDesc:
    return LayerDesc(T_max, d, F, E, k, r, 8, 256, float(lora_scale), 1 if training else 0)


def workspace_bytes(T_max, d, F, E, k, r, lora_scale=1.0, training=True) -> int:
    return int(load_library().tqp_workspace_bytes(ctypes.byref(_desc(T_max, d, F, E, k, r, lora_scale, training))))


def _ptr(t):
    return None if t is None else ctypes.c_void_p(t.data_ptr())


def dispatch_noalloc(topk_idx, E, counts, offsets, perm, inv_perm, stream=None):
    """tqp_dispatch_noalloc (include/tqp.h): the dispatch without ctx, workspace or any allocation.  ALL tensors are the
    caller's, on the current CUDA device: topk_idx int32 [T][k]; counts int32 [E]; offsets int32 [E + 1]; perm, inv_perm
    int32 [T * k].  Runs on `stream` (a torch stream; default: torch's current stream)."""
    import torch
    lib = load_library()
    T, k = topk_idx.shape
    st = stream if stream is not None else torch.cuda.current_stream(topk_idx.device)
    code = lib.tqp_dispatch_noalloc(int(T), int(k), int(E), _ptr(topk_idx), _ptr(counts), _ptr(offsets), _ptr(perm),
                                    _ptr(inv_perm), ctypes.c_void_p(st.cuda_stream))
    if code != 0:
        raise TqpError(code, (lib.tqp_dispatch_noalloc_error() or b"").decode())


def dispatch_noalloc_capacity() -> int:
    """Entries of the static scratch: ceil(T k / 256) * E must not exceed it."""
    return int(load_library().tqp_dispatch_noalloc_capacity())


def tq_levels(n: int, bits: int = 8):
    """HOST: Lloyd-Max levels of the coordinate law in dimension n (tqp_tq_levels) as a numpy float64 array."""
    import numpy as np
    out = np.empty(1 << bits, dtype=np.float64)
    code = load_library().tqp_tq_levels(int(n), int(bits), out.ctypes.data_as(ctypes.c_void_p))
    if code != 0:
        raise TqpError(code, "tqp_tq_levels")
    return out


def tq_rotation_qr(G):
    """HOST: sign-fixed Q of the QR factorisation of the Gaussian draw G (numpy float64 [n][n]) (tqp_tq_rotation_qr)."""
    import numpy as np
    G = np.ascontiguousarray(G, dtype=np.float64)
    n = G.shape[0]
    out = np.empty((n, n), dtype=np.float64)
    code = load_library().tqp_tq_rotation_qr(n, G.ctypes.data_as(ctypes.c_void_p), out.ctypes.data_as(ctypes.c_void_p))
    if code != 0:
        raise TqpError(code, "tqp_tq_rotation_qr")
    return out


class TqpLayer:
    """One routed-expert layer on the current CUDA device.  Methods carry the C names without the tqp_ prefix."""

    def __init__(self, T_max, d, F, E, k, r, lora_scale=1.0, training=True, device="cuda:0"):
        import torch
        self.torch = torch
        self.lib = load_library()
        if not torch.cuda.is_available():
            raise TqpError(6, "no CUDA device: the TQP path has no CPU fallback")
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        self.T_max, self.d, self.F, self.E, self.k, self.r = T_max, d, F, E, k, r
        self.training = training
        self.desc = _desc(T_max, d, F, E, k, r, lora_scale, training)
        self.ctx = ctypes.c_void_p()
        self._check(self.lib.tqp_create(ctypes.byref(self.ctx), ctypes.byref(self.desc)))
        nbytes = int(self.lib.tqp_workspace_bytes(ctypes.byref(self.desc)))
        self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
        self._check(self.lib.tqp_bind_workspace(self.ctx, _ptr(self.workspace), nbytes, self._stream()))
        self.weights = None

    def __del__(self):
        try:
            if getattr(self, "ctx", None):
                self.lib.tqp_destroy(self.ctx)
                self.ctx = None
        except Exception:
            pass

    def _stream(self):
        return ctypes.c_void_p(self.torch.cuda.current_stream(self.device).cuda_stream)

    def _check(self, code):
        if code != 0:
            msg = self.lib.tqp_last_error(self.ctx).decode() if self.ctx else ""
            raise TqpError(code, msg)

    def set_option(self, name: str, value: int):
        self._check(self.lib.tqp_set_option(self.ctx, name.encode(), int(value)))

    def bind_weights(self, **w):
        """w: device tensors named as tqp_weights' fields (uint8 codes, fp16 scales/codebook, bf16 adapters)."""
        self.weights = {n: w[n].contiguous() for n in _WEIGHT_FIELDS}
        ws = Weights(*[self.weights[n].data_ptr() for n in _WEIGHT_FIELDS])
        self._check(self.lib.tqp_bind_weights(self.ctx, ctypes.byref(ws), self._stream()))

    def bind_weights_tq(self, space_d, space_F, **w):
        """TurboQuant base: codes_* uint8, norm_* fp32, bf16 adapters (tqp_tq_weights' fields); spaces are TqSpace objects."""
        self.weights = {n: w[n].contiguous() for n in _TQ_FIELDS_A + _TQ_FIELDS_B}
        self.spaces = (space_d, space_F)
        ws = TqWeightsC(*([self.weights[n].data_ptr() for n in _TQ_FIELDS_A] + [space_d.c, space_F.c] +
                          [self.weights[n].data_ptr() for n in _TQ_FIELDS_B]))
        self._check(self.lib.tqp_bind_weights_tq(self.ctx, ctypes.byref(ws), self._stream()))

    # ---- forward ----
    def route(self, X, W_r, logit_bias=None, want_logits=False):
        t = self.torch
        T = X.shape[0]
        idx = t.empty((T, self.k), dtype=t.int32, device=self.device)
        w = t.empty((T, self.k), dtype=t.float32, device=self.device)
        lg = t.empty((T, self.E), dtype=t.float32, device=self.device) if want_logits else None
        self._check(self.lib.tqp_route(self.ctx, T, _ptr(X), _ptr(W_r), _ptr(logit_bias), _ptr(idx), _ptr(w), _ptr(lg),
                                       self._stream()))
        return (idx, w, lg) if want_logits else (idx, w)

    def route_info(self):
        """(screened, fallback) of the last route() on this layer: see tqp_route_info in include/tqp.h."""
        a, b = ctypes.c_int(0), ctypes.c_int(0)
        self._check(self.lib.tqp_route_info(self.ctx, ctypes.byref(a), ctypes.byref(b), self._stream()))
        return a.value, b.value

    def dispatch(self, topk_idx):
        t = self.torch
        T = topk_idx.shape[0]
        N = T * self.k
        counts = t.empty(self.E, dtype=t.int32, device=self.device)
        offsets = t.empty(self.E + 4, dtype=t.int32, device=self.device)[: self.E + 1]
        perm = t.empty(N, dtype=t.int32, device=self.device)
        inv = t.empty(N, dtype=t.int32, device=self.device)
        self._check(self.lib.tqp_dispatch(self.ctx, T, _ptr(topk_idx), _ptr(counts), _ptr(offsets), _ptr(perm), _ptr(inv),
                                          self._stream()))
        return counts, offsets, perm, inv

    def expert_fwd(self, X, offsets, perm, out=None):
        t = self.torch
        T = X.shape[0]
        Ye = out if out is not None else t.empty((T * self.k, self.d), dtype=t.bfloat16, device=self.device)
        self._check(self.lib.tqp_expert_fwd(self.ctx, T, _ptr(X), _ptr(offsets), _ptr(perm), _ptr(Ye), self._stream()))
        return Ye

    def combine(self, Ye, inv_perm, topk_w, out=None):
        t = self.torch
        T = topk_w.shape[0]
        Y = out if out is not None else t.empty((T, self.d), dtype=t.bfloat16, device=self.device)
        self._check(self.lib.tqp_combine(self.ctx, T, _ptr(Ye), _ptr(inv_perm), _ptr(topk_w), _ptr(Y), self._stream()))
        return Y

    # ---- backward ----
    def combine_bwd(self, dY, Ye, inv_perm, topk_w, want_dw=True, out=None, perm=None):
        """perm (the array dispatch returned) selects the fused row-gather path, see tqp.h."""
        t = self.torch
        T = topk_w.shape[0]
        dYe = out if out is not None else t.empty((T * self.k, self.d), dtype=t.bfloat16, device=self.device)
        dw = t.empty((T, self.k), dtype=t.float32, device=self.device) if want_dw else None
        self._check(self.lib.tqp_combine_bwd(self.ctx, T, _ptr(dY), _ptr(Ye), _ptr(inv_perm), _ptr(perm), _ptr(topk_w),
                                             _ptr(dYe), _ptr(dw), self._stream()))
        return dYe, dw

    def alloc_grads(self):
        t = self.torch
        E, d, F, r = self.E, self.d, self.F, self.r
        mk = lambda *s: t.empty(s, dtype=t.float32, device=self.device)
        return {"dA_gate": mk(E, d, r), "dB_gate": mk(E, r, F), "dA_up": mk(E, d, r), "dB_up": mk(E, r, F),
                "dA_down": mk(E, F, r), "dB_down": mk(E, r, d)}

    def expert_bwd(self, X, dYe, offsets, perm, grads=None, out=None, dYe_unmodified=False):
        """dYe_unmodified=True passes TQP_BWD_DYE_UNMODIFIED (dYe is the untouched output of the preceding fused combine_bwd)."""
        t = self.torch
        T = X.shape[0]
        g = grads if grads is not None else self.alloc_grads()
        dXp = out if out is not None else t.empty((T * self.k, self.d), dtype=t.bfloat16, device=self.device)
        self._check(self.lib.tqp_expert_bwd(self.ctx, T, _ptr(X), _ptr(dYe), _ptr(offsets), _ptr(perm), _ptr(dXp),
                                            _ptr(g["dA_gate"]), _ptr(g["dB_gate"]), _ptr(g["dA_up"]), _ptr(g["dB_up"]),
                                            _ptr(g["dA_down"]), _ptr(g["dB_down"]), 1 if dYe_unmodified else 0,
                                            self._stream()))
        return dXp, g

    def dispatch_bwd(self, dXp, inv_perm, out=None):
        t = self.torch
        T = dXp.shape[0] // self.k
        dX = out if out is not None else t.empty((T, self.d), dtype=t.bfloat16, device=self.device)
        self._check(self.lib.tqp_dispatch_bwd(self.ctx, T, _ptr(dXp), _ptr(inv_perm), _ptr(dX), self._stream()))
        return dX

    def route_bwd(self, X, W_r, topk_idx, topk_w, dtopk_w, offsets, perm, dX):
        t = self.torch
        T = X.shape[0]
        dW_r = t.empty((self.d, self.E), dtype=t.float32, device=self.device)
        self._check(self.lib.tqp_route_bwd(self.ctx, T, _ptr(X), _ptr(W_r), _ptr(topk_idx), _ptr(topk_w), _ptr(dtopk_w),
                                           _ptr(offsets), _ptr(perm), _ptr(dX), _ptr(dW_r), self._stream()))
        return dW_r

    # ---- paper-faithful router variant and balance controller ----
    def route_sigmoid(self, X, W_r, select_bias=None, want_logits=False):
        t = self.torch
        T = X.shape[0]
        idx = t.empty((T, self.k), dtype=t.int32, device=self.device)
        w = t.empty((T, self.k), dtype=t.float32, device=self.device)
        sc = t.empty((T, self.k), dtype=t.float32, device=self.device)
        lg = t.empty((T, self.E), dtype=t.float32, device=self.device) if want_logits else None
        self._check(self.lib.tqp_route_sigmoid(self.ctx, T, _ptr(X), _ptr(W_r), _ptr(select_bias), _ptr(idx), _ptr(w),
                                               _ptr(sc), _ptr(lg), self._stream()))
        return (idx, w, sc, lg) if want_logits else (idx, w, sc)

    def route_sigmoid_bwd(self, X, W_r, topk_idx, topk_w, topk_s, dtopk_w, offsets, perm, dX):
        t = self.torch
        T = X.shape[0]
        dW_r = t.empty((self.d, self.E), dtype=t.float32, device=self.device)
        self._check(self.lib.tqp_route_sigmoid_bwd(self.ctx, T, _ptr(X), _ptr(W_r), _ptr(topk_idx), _ptr(topk_w),
                                                   _ptr(topk_s), _ptr(dtopk_w), _ptr(offsets), _ptr(perm), _ptr(dX),
                                                   _ptr(dW_r), self._stream()))
        return dW_r

    def bias_update(self, counts, bias, mode, gamma, cap_hi=0.0, cap_lo=0.0):
        self._check(self.lib.tqp_bias_update(self.ctx, _ptr(counts), _ptr(bias), int(mode), float(gamma), float(cap_hi),
                                             float(cap_lo), self._stream()))
        return bias

    def consolidate(self, pack, e0=0, n_experts=None, out=None):
        """Merged bf16 weights [n_experts][out][in] of pack 0 (gate) / 1 (up) / 2 (down) for experts e0 .. e0 + n_experts."""
        pack = {"gate": 0, "up": 1, "down": 2}.get(pack, pack)
        n = self.E - e0 if n_experts is None else n_experts
        out_dim, in_dim = (self.d, self.F) if pack == 2 else (self.F, self.d)
        if out is None:
            out = self.torch.empty((n, out_dim, in_dim), dtype=self.torch.bfloat16, device=self.device)
        self._check(self.lib.tqp_consolidate(self.ctx, int(pack), int(e0), int(n), _ptr(out), self._stream()))
        return out

    # ---- TurboQuant-MSE base ----
    def rotate(self, space, X, inverse=False, out=None):
        t = self.torch
        Y = out if out is not None else t.empty_like(X)
        self._check(self.lib.tqp_rotate(self.ctx, ctypes.byref(space.c), _ptr(X), X.shape[0], _ptr(Y), 1 if inverse else 0, self._stream()))
        return Y

    def tq_encode(self, space, W):
        """W fp32 [rows][n] -> (codes uint8 [rows][n], norms fp32 [rows])."""
        t = self.torch
        rows = W.shape[0]
        codes = t.empty((rows, space.n), dtype=t.uint8, device=self.device)
        norms = t.empty((rows,), dtype=t.float32, device=self.device)
        self._check(self.lib.tqp_tq_encode(self.ctx, ctypes.byref(space.c), _ptr(W), rows, _ptr(codes), _ptr(norms), self._stream()))
        return codes, norms

    def tq_decode(self, space, codes, norms):
        t = self.torch
        rows = codes.shape[0]
        W = t.empty((rows, space.n), dtype=t.float32, device=self.device)
        self._check(self.lib.tqp_tq_decode(self.ctx, ctypes.byref(space.c), _ptr(codes), _ptr(norms), rows, _ptr(W), self._stream()))
        return W

    def tq_flush(self, space, codes, norms, A, B, lora_scale, A_new=None):
        """In place on codes [E][out][n], norms [E][out], A [E][n][r], B [E][r][out]; returns telemetry fp32 [E][2]."""
        t = self.torch
        E, out_dim, r = codes.shape[0], codes.shape[1], A.shape[2]
        tele = t.empty((E, 2), dtype=t.float32, device=self.device)
        self._check(self.lib.tqp_tq_flush(self.ctx, ctypes.byref(space.c), E, out_dim, r, float(lora_scale), _ptr(codes), _ptr(norms),
                                          _ptr(A), _ptr(B), _ptr(A_new), _ptr(tele), self._stream()))
        return tele

    def step_host(self, X_host, dY_host, W_r, logit_bias, Y_host, dX_host, grads, dW_r=None):
        """Whole forward+backward through HOST (pinned) X/dY/Y/dX buffers; grads / dW_r stay on the device."""
        T = X_host.shape[0]
        g = grads
        self._check(self.lib.tqp_step_host(self.ctx, T, _ptr(X_host), _ptr(dY_host), _ptr(W_r), _ptr(logit_bias),
                                           _ptr(Y_host), _ptr(dX_host), _ptr(g["dA_gate"]), _ptr(g["dB_gate"]),
                                           _ptr(g["dA_up"]), _ptr(g["dB_up"]), _ptr(g["dA_down"]), _ptr(g["dB_down"]),
                                           _ptr(dW_r), self._stream()))

    def step_host_async(self, X_host, dY_host, W_r, logit_bias, Y_host, dX_host, grads, dW_r=None):
        """step_host without the final wait: returns once everything is enqueued (at most two steps in flight; the host
        buffers of a step belong to the library until step_host_wait has returned for it)."""
        T = X_host.shape[0]
        g = grads
        self._check(self.lib.tqp_step_host_async(self.ctx, T, _ptr(X_host), _ptr(dY_host), _ptr(W_r), _ptr(logit_bias),
                                                 _ptr(Y_host), _ptr(dX_host), _ptr(g["dA_gate"]), _ptr(g["dB_gate"]),
                                                 _ptr(g["dA_up"]), _ptr(g["dB_up"]), _ptr(g["dA_down"]), _ptr(g["dB_down"]),
                                                 _ptr(dW_r), self._stream()))

    def step_host_wait(self, age=0):
        """Blocks until the latest (age 0) or the previous (age 1) asynchronous step has delivered its host outputs."""
        self._check(self.lib.tqp_step_host_wait(self.ctx, int(age)))

    def gemm_time(self):
        """(summed grouped-GEMM device ms, launches) since the last call; needs set_option('time_gemm', 1)."""
        ms, n = ctypes.c_float(), ctypes.c_int()
        self._check(self.lib.tqp_gemm_time(self.ctx, ctypes.byref(ms), ctypes.byref(n)))
        return float(ms.value), int(n.value)

    def gemm_times(self, cap=4096):
        """Per-launch grouped-GEMM device times (ms) since the last call."""
        arr = (ctypes.c_float * cap)()
        n = ctypes.c_int()
        self._check(self.lib.tqp_gemm_times(self.ctx, arr, cap, ctypes.byref(n)))
        return [float(arr[i]) for i in range(min(cap, n.value))]

    # ---- introspection ----
    def last_launch_count(self) -> int:
        return int(self.lib.tqp_last_launch_count(self.ctx))

    def debug_buffer(self, name, shape, dtype):
        """A torch view of a workspace tensor (tests only)."""
        t = self.torch
        ptr = self.lib.tqp_debug_buffer(self.ctx, name.encode())
        if not ptr:
            raise KeyError(name)
        off = ptr - self.workspace.data_ptr()
        n = 1
        for s in shape:
            n *= s
        nbytes = n * t.empty((), dtype=dtype).element_size()
        return self.workspace[off: off + nbytes].view(dtype).view(*shape)
