"""Pins of the flush oracle and of the TurboQuant-format expert FFN oracle (oracle/flush.py; §9.4,
L1047-1061 §10.3 / Table 28, L944-946 §9.2).  CPU only.

Pinned against things other than the oracle's own formulas: a hand-computed n = 2 example (tests/golden/p14_*), the closed
form of a flush with a zero adapter (codes unchanged, norm scaled by the length of the looked-up level vector), the
quantiser's distortion computed by independent quadrature and TurboQuant's stated bound sqrt(3) pi / 2 * 4^-b, function
preservation of the layer across a flush, and torch autograd (an independent differentiation routine) for the backward."""
import os

import numpy as np
import pytest
from scipy import integrate

from oracle import flush as fl
from oracle import turboquant as tq


def _golden():
    vals = {}
    for line in open(os.path.join(os.path.dirname(__file__), "golden", "p14_flush_worked_example.txt")):
        line = line.split("#")[0].strip()
        if "=" in line:
            key, v = line.split("=")
            vals[key.strip()] = np.array([float(t) for t in v.split()])
    return vals


def test_p14_hand_example_n2_one_bit():
    g = _golden()
    cb = tq.lloyd_max_codebook(2, 1)
    np.testing.assert_allclose(cb, [-g["level"][0], g["level"][0]], atol=1e-12)      # +-2/pi, the arcsine law's E|y|
    R = tq.hadamard(2) / np.sqrt(2.0)                                                 # signs (+1, +1)
    codes, norms = tq.encode(g["w"][None, :], R, cb)
    np.testing.assert_array_equal(codes[0], g["codes"])
    np.testing.assert_allclose(norms, g["norm"], rtol=1e-15)
    np.testing.assert_allclose(tq.decode(codes, norms, R, cb)[0], g["decoded"], atol=1e-12)
    out = fl.flush_pack(codes, norms, A=np.array([[1.0], [0.0]]), B=np.array([[2.0]]), s=0.5, R=R, codebook=cb)
    np.testing.assert_allclose(out["W_merged"][0], g["merged"], atol=1e-12)
    np.testing.assert_allclose(out["norms"], g["norm_new"], rtol=1e-12)
    np.testing.assert_array_equal(out["codes"][0], g["codes_new"])
    np.testing.assert_allclose(out["adapter_norm"], g["adapter_norm"], rtol=1e-12)
    np.testing.assert_allclose(out["base_share"], g["base_share"], rtol=1e-6)
    assert (out["B"] == 0).all() and (out["A"] == [[1.0], [0.0]]).all()                # B reset, A kept when no new draw is given


def _random_pack(n_in, n_out, r, seed, bits=8, adapter_std=0.02):
    rng = np.random.default_rng(seed)
    R = tq.rotation(n_in, seed + 1000)            # not the generator state W is drawn from
    cb = tq.lloyd_max_codebook(n_in, bits)
    W = rng.standard_normal((n_out, n_in)) * 0.02
    codes, norms = tq.encode(W, R, cb)
    A = rng.standard_normal((n_in, r)) * adapter_std
    B = rng.standard_normal((r, n_out)) * adapter_std
    return dict(W=W, R=R, cb=cb, codes=codes, norms=norms, A=A, B=B)


@pytest.mark.parametrize("n_in", [64, 48])       # signed Hadamard / sign-fixed QR
def test_flush_with_zero_adapter_keeps_the_codes(n_in):
    """B = 0: W_merged is the reconstruction itself, a vector ON the codebook; re-encoding it returns the same codes and
    norm' = norm * |levels[codes]| (the looked-up vector is not exactly of unit length)."""
    p = _random_pack(n_in, 40, 4, seed=3)
    out = fl.flush_pack(p["codes"], p["norms"], p["A"], np.zeros_like(p["B"]), 1.0, p["R"], p["cb"])
    np.testing.assert_array_equal(out["codes"], p["codes"])
    np.testing.assert_allclose(out["norms"], p["norms"] * np.linalg.norm(p["cb"][p["codes"]], axis=1), rtol=1e-12)
    assert out["adapter_norm"] == 0.0 and out["base_share"] == 1.0


def test_requantisation_error_is_the_quantisers_distortion():
    """|| decode(flush) - W_merged ||^2 / ||W_merged||^2 per row ~ n * E[(y - Q(y))^2] of the coordinate law (computed here
    by quadrature, independently of the oracle) and below TurboQuant's bound sqrt(3) pi / 2 * 4^-b."""
    n, bits = 256, 8
    p = _random_pack(n, 600, 8, seed=7, bits=bits, adapter_std=0.05)
    out = fl.flush_pack(p["codes"], p["norms"], p["A"], p["B"], 0.7, p["R"], p["cb"])
    rec = tq.decode(out["codes"], out["norms"], p["R"], p["cb"])
    rel2 = np.sum((rec - out["W_merged"]) ** 2, axis=1) / np.sum(out["W_merged"] ** 2, axis=1)
    cb = p["cb"]
    b = np.concatenate(([-1.0], 0.5 * (cb[:-1] + cb[1:]), [1.0]))
    logc = 0.0
    dens = lambda y: (1.0 - y * y) ** ((n - 3) / 2.0)
    z = integrate.quad(dens, -1, 1, epsabs=0, epsrel=1e-12, points=[-0.3, 0.3])[0]
    D = sum(integrate.quad(lambda y: (y - cb[j]) ** 2 * dens(y), b[j], b[j + 1], epsabs=0, epsrel=1e-10)[0] for j in range(len(cb))) / z
    assert abs(rel2.mean() / (n * D) - 1.0) < 0.1
    assert rel2.mean() < np.sqrt(3.0) * np.pi / 2.0 * 4.0 ** (-bits)
    assert rel2.max() < 8.0 * n * D                # rows with a coordinate in an outer (overload) cell


def test_flush_preserves_the_function_up_to_the_distortion():
    """after the fold and the reset the expert computes what it computed before, up to the quantiser's
    distortion: x . (base' + 0) vs x . (base + s A B)."""
    p = _random_pack(128, 96, 8, seed=11, adapter_std=0.05)
    s = 0.5
    out = fl.flush_pack(p["codes"], p["norms"], p["A"], p["B"], s, p["R"], p["cb"])
    before = fl.dense_weights(p["codes"], p["norms"], p["A"], p["B"], s, p["R"], p["cb"])
    after = fl.dense_weights(out["codes"], out["norms"], out["A"], out["B"], s, p["R"], p["cb"])
    x = np.random.default_rng(0).standard_normal((50, 128))
    err = np.linalg.norm(x @ after - x @ before) / np.linalg.norm(x @ before)
    assert 1e-3 < err < 1.5e-2                      # ~ sqrt(4.15e-5) = 6.4e-3 at 8 bits, and not zero
    delta = np.linalg.norm(s * p["A"] @ p["B"])
    assert delta > 20 * np.linalg.norm(after - before)    # the fold moved the base by far more than the re-quantisation error
    np.testing.assert_allclose(out["adapter_norm"], delta, rtol=1e-12)
    nb = np.linalg.norm(tq.decode(p["codes"], p["norms"], p["R"], p["cb"]))
    np.testing.assert_allclose(out["base_share"], nb / (nb + delta), rtol=1e-12)


def test_repeated_flushes_accumulate_rank():
    """The point of the flush (L966): each window adds a rank-r increment to the base; after k windows with independent
    adapters the cumulative update has rank ~ k r."""
    p = _random_pack(64, 64, 2, seed=13, adapter_std=0.3)
    rng = np.random.default_rng(1)
    base0 = tq.decode(p["codes"], p["norms"], p["R"], p["cb"])
    codes, norms = p["codes"], p["norms"]
    for _ in range(4):
        A, B = rng.standard_normal((64, 2)) * 0.3, rng.standard_normal((2, 64)) * 0.3
        out = fl.flush_pack(codes, norms, A, B, 1.0, p["R"], p["cb"])
        codes, norms = out["codes"], out["norms"]
    sv = np.linalg.svd(tq.decode(codes, norms, p["R"], p["cb"]) - base0, compute_uv=False)
    assert sv[7] > 10 * sv[8]                       # 4 windows x rank 2 = 8 dominant directions; the rest is quantisation noise


def test_expert_ffn_backward_against_torch_autograd():
    torch = pytest.importorskip("torch")
    rng = np.random.default_rng(5)
    n, d, F = 7, 12, 20
    x, dy = rng.standard_normal((n, d)), rng.standard_normal((n, d))
    Wg, Wu, Wd = rng.standard_normal((d, F)) * 0.3, rng.standard_normal((d, F)) * 0.3, rng.standard_normal((F, d)) * 0.3
    y, g, u, h = fl.expert_ffn(x, Wg, Wu, Wd)
    dx, dWg, dWu, dWd = fl.expert_ffn_bwd(x, dy, g, u, h, Wg, Wu, Wd)
    t = [torch.tensor(a, dtype=torch.float64, requires_grad=True) for a in (x, Wg, Wu, Wd)]
    yt = (torch.nn.functional.silu(t[0] @ t[1]) * (t[0] @ t[2])) @ t[3]
    np.testing.assert_allclose(y, yt.detach().numpy(), rtol=1e-12, atol=1e-14)
    (yt * torch.tensor(dy)).sum().backward()
    for got, ref in zip((dx, dWg, dWu, dWd), t):
        np.testing.assert_allclose(got, ref.grad.numpy(), rtol=1e-11, atol=1e-13)
