"""Pins of the NEXT-1 oracle (oracle/router_ext.py): the paper-faithful sigmoid router with a selection-only bias
 and the loss-free bias controllers (L1075, L1097 Table 29).  CPU only.

Each pin checks the oracle against something other than itself: a brute-force selection, closed forms, invariances
the mathematics fixes, central finite differences in fp64, and hand-computed controller steps."""
import itertools

import numpy as np
import pytest

from oracle import router_ext as rx


def _rand_logits(T, E, seed, dtype=np.float64):
    return np.random.default_rng(seed).standard_normal((T, E)).astype(dtype)


def test_selection_matches_brute_force_with_ties_and_bias():
    """Brute force over ALL k-subsets on tiny inputs: the selected set maximises the sum of keys, and among equal keys
    the lower id wins; duplicated columns create exact ties."""
    E, k = 7, 3
    lg = _rand_logits(9, E, 1, np.float32)
    lg[:, 5] = lg[:, 2]                      # exact ties between experts 2 and 5
    lg[3, :] = 0.25                          # a row of all-equal logits -> experts 0,1,2
    bias = np.array([0.0, 0.5, 0.0, -0.5, 0.0, 0.0, 0.25], np.float32)
    idx, w, s = rx.route_sigmoid(lg, bias, k)
    key = (lg + bias[None, :]).astype(np.float32)
    for t in range(lg.shape[0]):
        best = max(itertools.combinations(range(E), k), key=lambda c: (sum(float(key[t, e]) for e in c), [-e for e in c]))
        assert sorted(idx[t]) == sorted(best)
        ks = key[t, idx[t]]
        assert all(ks[j] > ks[j + 1] or (ks[j] == ks[j + 1] and idx[t, j] < idx[t, j + 1]) for j in range(k - 1))
    assert list(idx[3]) == [1, 6, 0]          # all logits equal: bias decides, then the lower id


def test_bias_moves_selection_but_never_the_gate_values():
    lg = _rand_logits(64, 16, 2, np.float32)
    idx0, w0, s0 = rx.route_sigmoid(lg, None, 4)
    idx1, w1, s1 = rx.route_sigmoid(lg, np.full(16, 3.0, np.float32), 4)      # a constant bias changes nothing
    np.testing.assert_array_equal(idx0, idx1)
    np.testing.assert_array_equal(w0, w1)
    bias = np.zeros(16, np.float32); bias[11] = 50.0                            # expert 11 is now always selected first ...
    idx2, w2, s2 = rx.route_sigmoid(lg, bias, 4)
    assert (idx2[:, 0] == 11).all()
    sig = 1.0 / (1.0 + np.exp(-lg[:, 11].astype(np.float64)))
    np.testing.assert_allclose(s2[:, 0], sig, rtol=1e-6)                         # ... with its UNBIASED score as the gate value


def test_gates_closed_forms():
    lg = _rand_logits(32, 8, 3)
    idx, w, s = rx.route_sigmoid(lg, None, 8)                                    # k = E: w = sigmoid(l) / sum sigmoid(l)
    sig = 1.0 / (1.0 + np.exp(-lg))
    ref = np.take_along_axis(sig / sig.sum(1, keepdims=True), idx.astype(np.int64), axis=1)
    np.testing.assert_allclose(w, ref, rtol=1e-12)
    idx1, w1, s1 = rx.route_sigmoid(lg, None, 1)                                 # k = 1: w = 1, the arg-max expert
    np.testing.assert_array_equal(w1, np.ones_like(w1))
    np.testing.assert_array_equal(idx1[:, 0], lg.argmax(1))
    idx3, w3, s3 = rx.route_sigmoid(lg, None, 3)
    np.testing.assert_allclose(w3.sum(1), 1.0, rtol=1e-12)
    assert (w3 > 0).all() and (s3 > 0).all() and (s3 < 1).all()
    assert (np.diff(s3, axis=1) <= 0).all()                                       # no bias: scores descend with the logits


def test_logit_gradient_against_finite_differences():
    """L = sum_j w_j c_j with fixed c and a selection that does not change under the perturbation."""
    rng = np.random.default_rng(4)
    T, E, k, h = 6, 10, 4, 1e-6
    lg = rng.standard_normal((T, E)) * 2.0
    c = rng.standard_normal((T, k))
    idx, w, s = rx.route_sigmoid(lg, None, k)
    dl = rx.route_sigmoid_dl(w, s, c)
    srt = np.sort(lg, axis=1)
    assert (srt[:, -k] - srt[:, -k - 1]).min() > 1e-3                             # the top-k gap dwarfs h
    for t in range(T):
        for j in range(k):
            e = idx[t, j]
            lp, lm = lg.copy(), lg.copy()
            lp[t, e] += h; lm[t, e] -= h
            ip, wp, _ = rx.route_sigmoid(lp, None, k); im, wm, _ = rx.route_sigmoid(lm, None, k)
            assert (ip[t] == idx[t]).all() and (im[t] == idx[t]).all()
            fd = (np.dot(wp[t], c[t]) - np.dot(wm[t], c[t])) / (2 * h)
            assert abs(fd - dl[t, j]) <= 1e-7 * max(1.0, abs(fd))
    np.testing.assert_allclose(dl.sum(1) * 0 + np.sum(dl / (w * (1 - s)) * w, axis=1), 0.0, atol=1e-12)   # sum_j w_j (c_j - dot) = 0


def test_fp32_and_fp64_agree():
    lg = _rand_logits(128, 32, 5, np.float32)
    i32, w32, s32 = rx.route_sigmoid(lg, None, 6)
    i64, w64, s64 = rx.route_sigmoid(lg.astype(np.float64), None, 6)
    np.testing.assert_array_equal(i32, i64)
    assert np.abs(w32 - w64).max() < 5e-7 and np.abs(s32 - s64).max() < 5e-7


def test_sign_controller_by_hand():
    """Wang et al.'s update as the paper words it: against the sign of the load error, nothing when on target."""
    counts = np.array([30, 10, 20, 20])                     # loads 0.375, 0.125, 0.25, 0.25; tau = 0.25
    b = rx.bias_update(counts, np.zeros(4, np.float32), "sign", 1e-4)
    np.testing.assert_array_equal(b, np.array([-1e-4, 1e-4, 0.0, 0.0], np.float32))
    b2 = rx.bias_update(np.array([5, 5, 5, 5]), np.full(4, 0.5, np.float32), "sign", 1e-4)
    np.testing.assert_array_equal(b2, np.full(4, 0.5, np.float32))


def test_three_tier_controller_by_hand():
    """E = 4, tau = 0.25, ceiling hi = 0.3 -> floor lo = tau^2/hi = 0.20833.  Loads 0.40 (above), 0.10 (below),
    0.28 and 0.22 (in band).  Hand-computed boosts: ((0.40-0.30)/0.25)^2 = 0.16; ((0.208333-0.10)/0.25)^2 = 0.187778."""
    counts = np.array([40, 10, 28, 22])
    g = 1e-3
    b = rx.bias_update(counts, np.zeros(4, np.float32), "three_tier", g, cap_hi=0.3)
    exp = np.array([-g * 1.16, g * (1 + (0.0625 / 0.3 - 0.10) ** 2 / 0.0625), -g, g])
    np.testing.assert_allclose(b, exp.astype(np.float32), rtol=1e-6)
    # continuity of the law at the band edges and monotone strength outside the band
    hi = 0.3
    just_in = rx.bias_update(np.array([300, 700 / 3, 700 / 3, 700 / 3]), np.zeros(4, np.float32), "three_tier", g, cap_hi=hi)
    assert just_in[0] == np.float32(-g)
    far = rx.bias_update(np.array([60, 14, 13, 13]), np.zeros(4, np.float32), "three_tier", g, cap_hi=hi)
    near = rx.bias_update(np.array([35, 22, 22, 21]), np.zeros(4, np.float32), "three_tier", g, cap_hi=hi)
    assert far[0] < near[0] < 0
    with pytest.raises(ValueError):
        rx.bias_update(counts, np.zeros(4, np.float32), "nope", g)


def test_controller_drives_a_skewed_router_towards_balance():
    """Closed loop on synthetic logits with a strong per-expert offset: iterating route -> counts -> bias_update with the
    paper's 120B settings (scaled gain) must shrink the maximum load and revive the dead experts."""
    rng = np.random.default_rng(6)
    T, E, k = 2048, 32, 4
    offs = np.linspace(-2.0, 2.0, E).astype(np.float32)
    lg = (rng.standard_normal((T, E)).astype(np.float32) + offs[None, :])
    bias = np.zeros(E, np.float32)
    idx, _, _ = rx.route_sigmoid(lg, bias, k)
    c0 = np.bincount(idx.ravel(), minlength=E)
    for _ in range(200):
        idx, _, _ = rx.route_sigmoid(lg, bias, k)
        counts = np.bincount(idx.ravel(), minlength=E)
        bias = rx.bias_update(counts, bias, "three_tier", 2e-2, cap_hi=1.5 / E)
    c1 = np.bincount(rx.route_sigmoid(lg, bias, k)[0].ravel(), minlength=E)
    assert c1.max() < 0.5 * c0.max() and c1.min() > 4 * max(1, c0.min())


def test_router_chain_gradients_against_finite_differences():
    """L(X, W_r) = sum_t sum_j w_j(X W_r)[t] c[t,j]: dX and dW_r from route_sigmoid_dl + route_bwd_from_dl against
    central differences in fp64 (selection unchanged under the perturbation)."""
    rng = np.random.default_rng(8)
    T, d, E, k, h = 5, 7, 9, 3, 1e-6
    X = rng.standard_normal((T, d)); W = rng.standard_normal((d, E)); c = rng.standard_normal((T, k))

    def loss(Xv, Wv, idx_ref=None):
        idx, w, s = rx.route_sigmoid(Xv @ Wv, None, k)
        if idx_ref is not None:
            assert (idx == idx_ref).all()
        return float(np.sum(w * c)), idx, w, s

    _, idx, w, s = loss(X, W)
    dl = rx.route_sigmoid_dl(w, s, c)
    dX = np.zeros_like(X)
    dW = rx.route_bwd_from_dl(X, W, idx, dl, dX)
    for (t, i) in [(0, 0), (2, 3), (4, 6)]:
        Xp, Xm = X.copy(), X.copy(); Xp[t, i] += h; Xm[t, i] -= h
        fd = (loss(Xp, W, idx)[0] - loss(Xm, W, idx)[0]) / (2 * h)
        assert abs(fd - dX[t, i]) <= 1e-6 * max(1.0, abs(fd))
    for (i, e) in [(0, int(idx[0, 0])), (3, int(idx[1, 1])), (6, int(idx[4, 2]))]:
        Wp, Wm = W.copy(), W.copy(); Wp[i, e] += h; Wm[i, e] -= h
        fd = (loss(X, Wp, idx)[0] - loss(X, Wm, idx)[0]) / (2 * h)
        assert abs(fd - dW[i, e]) <= 1e-6 * max(1.0, abs(fd))
    unsel = np.setdiff1d(np.arange(E), idx.ravel())
    assert (dW[:, unsel] == 0).all()
