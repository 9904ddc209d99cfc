"""GPU parity of the TurboQuant-MSE pieces (tqp_tq_encode / tqp_tq_decode / tqp_rotate / tqp_tq_flush; SURVEY §8(f) NEXT-2,
NEXT-4; Table 28) against oracle/turboquant.py and oracle/flush.py, through the C ABI.

Codes are integer work: bit-exact against the oracle (both sides decide in fp64), except that a rotated coordinate
within 1e-9 / sqrt(n) of a cell boundary (where the two fp64 evaluation orders may legitimately round to different
sides) may differ by one code -- such coordinates are counted and must be rare.  Norms: fp32 rounding of the fp64 norm.
Reconstruction and rotated activations: float tolerance.  The rotation draws (signs, Gaussian matrix) and the Lloyd-Max
levels are inputs from the oracle side, identical for both."""
import numpy as np
import pytest

import tqp_inputs as ti
from oracle import flush as ofl
from oracle import turboquant as otq

pytestmark = pytest.mark.gpu


def _space(n, seed):
    import torch
    import paper_2606_07404_b200 as tq
    R = otq.rotation(n, seed)
    levels = otq.lloyd_max_codebook(n, 8)
    lv = torch.from_numpy(levels).cuda()
    if n & (n - 1) == 0:
        signs = np.sign(R[0] * np.sqrt(n)).astype(np.int8)             # R = H diag(s) / sqrt(n), H[0] = 1
        sp = tq.TqSpace(n, lv, signs=torch.from_numpy(signs).cuda())
    else:
        sp = tq.TqSpace(n, lv, R=torch.from_numpy(np.ascontiguousarray(R)).cuda())
    return sp, R, levels


def _layer():
    import paper_2606_07404_b200 as tq
    return tq.TqpLayer(64, 128, 128, 4, 2, 16)        # any ctx: the TurboQuant calls do not depend on the layer shape


def _check_codes(got, ref, Y, levels, n):
    bounds = 0.5 * (levels[:-1] + levels[1:])
    diff = np.nonzero(got != ref)
    if len(diff[0]):
        y = Y[diff]
        near = np.abs(y[:, None] - bounds[None, :]).min(axis=1)
        assert (near < 1e-9 / np.sqrt(n)).all() and (np.abs(got[diff].astype(int) - ref[diff].astype(int)) == 1).all()
    assert len(diff[0]) <= 1e-6 * got.size + 1
    return len(diff[0])


@pytest.mark.parametrize("n", [64, 1024, 4096, 192, 2560])
def test_encode_decode_against_the_oracle(n):
    import torch
    layer = _layer()
    sp, R, levels = _space(n, seed=100 + n)
    rows = 700 if n <= 1024 else 300
    rng = np.random.default_rng(n)
    W = (rng.standard_normal((rows, n)) * 0.02).astype(np.float32)
    W[5] = 0.0                                                            # a zero row
    W[6] *= 1e-6
    codes_ref, norms_ref = otq.encode(W.astype(np.float64), R, levels)
    codes, norms = layer.tq_encode(sp, torch.from_numpy(W).cuda())
    torch.cuda.synchronize()
    codes, norms = codes.cpu().numpy(), norms.cpu().numpy()
    np.testing.assert_array_equal(norms, norms_ref.astype(np.float32))
    U = np.divide(W.astype(np.float64), norms_ref[:, None], out=np.zeros((rows, n)), where=norms_ref[:, None] > 0)
    nd = _check_codes(codes, codes_ref, U @ R.T, levels, n)
    print(f"n={n}: {nd} of {codes.size} codes differ (boundary cases)")
    # reconstruction (L946) from the oracle's codes and the stored fp32 norms
    rec = layer.tq_decode(sp, torch.from_numpy(codes_ref).cuda(), torch.from_numpy(norms_ref.astype(np.float32)).cuda()).cpu().numpy()
    rec_ref = otq.decode(codes_ref, norms_ref.astype(np.float32).astype(np.float64), R, levels)
    np.testing.assert_allclose(rec, rec_ref, rtol=2e-6, atol=1e-9)
    err = np.linalg.norm(rec_ref - W) / np.linalg.norm(W)
    assert 3e-3 < err < 1e-2                                              # 8-bit distortion ~ 6.4e-3


@pytest.mark.parametrize("n", [64, 1024, 4096, 2560])
def test_rotate_activations(n):
    import torch
    layer = _layer()
    sp, R, _ = _space(n, seed=7)
    rows = 333
    X = ti.f32_to_bf16_bits(np.random.default_rng(1).standard_normal((rows, n)).astype(np.float32))
    Xf = ti.bf16_bits_to_f32(X).astype(np.float64)
    Xd = torch.from_numpy(X.view(np.int16)).view(torch.bfloat16).cuda()
    Y = layer.rotate(sp, Xd)
    Yf = Y.float().cpu().numpy()
    ref = Xf @ R.T
    tol = 4e-3 if n & (n - 1) == 0 else 6e-3                              # one bf16 rounding of the result (+ bf16 R when dense)
    assert np.linalg.norm(Yf - ref) / np.linalg.norm(ref) < tol
    Z = layer.rotate(sp, Y, inverse=True).float().cpu().numpy()          # R^T R = I up to the roundings
    assert np.linalg.norm(Z - Xf) / np.linalg.norm(Xf) < 2 * tol
    back = layer.rotate(sp, Xd, inverse=True).float().cpu().numpy()
    assert np.linalg.norm(back - Xf @ R) / np.linalg.norm(Xf) < tol


@pytest.mark.parametrize("n,out_dim,r,s", [(1024, 96, 16, 1.0), (256, 200, 8, 0.5), (192, 64, 32, 2.0), (2560, 48, 16, 1.0)])
def test_flush_against_the_oracle(n, out_dim, r, s):
    import torch
    layer = _layer()
    sp, R, levels = _space(n, seed=31)
    E = 3
    rng = np.random.default_rng(n + r)
    bf = lambda a: ti.f32_to_bf16_bits(a.astype(np.float32))
    W = rng.standard_normal((E, out_dim, n)) * 0.02
    A = bf(rng.standard_normal((E, n, r)) * 0.03)
    B = bf(rng.standard_normal((E, r, out_dim)) * 0.03)
    A_new = bf(rng.standard_normal((E, n, r)) * 0.01)
    codes0 = np.empty((E, out_dim, n), np.uint8); norms0 = np.empty((E, out_dim), np.float32)
    for e in range(E):
        c, nn = otq.encode(W[e], R, levels)
        codes0[e], norms0[e] = c, nn.astype(np.float32)                  # the stored norm is fp32
    t16 = lambda a: torch.from_numpy(a.view(np.int16)).view(torch.bfloat16).cuda()
    codes = torch.from_numpy(codes0.copy()).cuda(); norms = torch.from_numpy(norms0.copy()).cuda()
    Ad, Bd = t16(A.copy()), t16(B.copy())
    tele = layer.tq_flush(sp, codes, norms, Ad, Bd, s, A_new=t16(A_new))
    torch.cuda.synchronize()
    Af, Bf = ti.bf16_bits_to_f32(A).astype(np.float64), ti.bf16_bits_to_f32(B).astype(np.float64)
    ndiff = 0
    for e in range(E):
        ref = ofl.flush_pack(codes0[e], norms0[e].astype(np.float64), Af[e], Bf[e], s, R, levels)
        got_c = codes[e].cpu().numpy()
        ndiff += _check_codes(got_c, ref["codes"], (ref["W_merged"] / np.linalg.norm(ref["W_merged"], axis=1, keepdims=True)) @ R.T, levels, n)
        np.testing.assert_allclose(norms[e].cpu().numpy(), ref["norms"], rtol=2e-7)
        np.testing.assert_allclose(tele[e, 0].item(), ref["adapter_norm"], rtol=1e-6)
        np.testing.assert_allclose(tele[e, 1].item(), ref["base_share"], rtol=1e-6)
        assert 0.5 < ref["base_share"] < 0.999                              # the adapter delta is a visible part of the weight
    assert (Bd.float() == 0).all()                                           # reset: B <- 0, A <- the fresh draw
    np.testing.assert_array_equal(Ad.view(torch.int16).cpu().numpy().view(np.uint16), A_new)
    print(f"flush n={n}: {ndiff} codes differ at cell boundaries")


def test_error_codes():
    import torch
    import paper_2606_07404_b200 as tq
    layer = _layer()
    lv = torch.zeros(256, dtype=torch.float64, device="cuda")
    sg = torch.ones(192, dtype=torch.int8, device="cuda")
    X = torch.zeros((4, 192), dtype=torch.bfloat16, device="cuda")
    with pytest.raises(tq.TqpError) as e:                       # signed Hadamard needs a power-of-two width
        layer.rotate(tq.TqSpace(192, lv, signs=sg), X)
    assert e.value.code == 2
    with pytest.raises(tq.TqpError) as e:                       # width not a multiple of 64
        layer.rotate(tq.TqSpace(100, lv, signs=sg), X)
    assert e.value.code == 2
    sp, _, _ = _space(128, 3)
    big = tq.TqpLayer(64, 128, 128, 4, 2, 8)                    # r = 8: the TurboQuant-format layer needs r in {16, 32}
    z8 = lambda *s: torch.zeros(s, dtype=torch.uint8, device="cuda")
    zf = lambda *s: torch.zeros(s, dtype=torch.float32, device="cuda")
    zb = lambda *s: torch.zeros(s, dtype=torch.bfloat16, device="cuda")
    w = dict(codes_gate=z8(4, 128, 128), codes_up=z8(4, 128, 128), codes_down=z8(4, 128, 128), norm_gate=zf(4, 128), norm_up=zf(4, 128),
             norm_down=zf(4, 128), A_gate=zb(4, 128, 8), A_up=zb(4, 128, 8), B_gate=zb(4, 8, 128), B_up=zb(4, 8, 128), A_down=zb(4, 128, 8),
             B_down=zb(4, 8, 128))
    with pytest.raises(tq.TqpError) as e:
        big.bind_weights_tq(sp, sp, **w)
    assert e.value.code == 2
    with pytest.raises(tq.TqpError) as e:                       # flush: rank out of range
        layer.tq_flush(sp, z8(1, 8, 128), zf(1, 8), zb(1, 128, 64), zb(1, 64, 8), 1.0)
    assert e.value.code == 1
