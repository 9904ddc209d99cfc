"""Pins of the TurboQuant MSE oracle (oracle/turboquant.py; §9.2).  CPU only.

Pinned against things other than its own formulas: the Lloyd-Max conditions checked with an independent numerical
quadrature, Max's (1960) textbook levels of the Gaussian quantiser (the n -> infinity limit of the coordinate law),
the distortion values TurboQuant's own paper states for 1-4 bits, orthogonality and the Monte-Carlo law of a rotated
coordinate, and exact reconstruction of vectors that lie on the codebook."""
import numpy as np
import pytest
from scipy import integrate, stats

from oracle import turboquant as tq


def test_coordinate_law_matches_sampled_sphere_points():
    rng = np.random.default_rng(0)
    n = 64
    x = rng.standard_normal((200000, n))
    y = x[:, 0] / np.linalg.norm(x, axis=1)
    for q in (-0.3, -0.1, 0.0, 0.05, 0.2):
        assert abs(tq.coord_cdf(q, n) - np.mean(y <= q)) < 4e-3
    assert abs(np.var(y) - 1.0 / n) < 2e-4                      # E y^2 = 1/n on the unit sphere


@pytest.mark.parametrize("n,bits", [(16, 2), (128, 3), (1024, 4)])
def test_lloyd_max_conditions_by_quadrature(n, bits):
    """Every level is the conditional mean of its cell (trapezoid-free: scipy.integrate.quad on the density written out
    here independently) and the levels are symmetric."""
    c = tq.lloyd_max_codebook(n, bits)
    assert len(c) == 1 << bits and (np.diff(c) > 0).all()
    np.testing.assert_allclose(c, -c[::-1], atol=1e-10)
    dens = lambda y: (1.0 - y * y) ** ((n - 3) / 2.0)
    b = np.concatenate(([-1.0], 0.5 * (c[:-1] + c[1:]), [1.0]))
    for j in range(len(c)):
        num = integrate.quad(lambda y: y * dens(y), b[j], b[j + 1], epsabs=0, epsrel=1e-11)[0]
        den = integrate.quad(dens, b[j], b[j + 1], epsabs=0, epsrel=1e-11)[0]
        assert abs(num / den - c[j]) < 1e-8


@pytest.mark.parametrize("n", [64, 1024])
def test_lloyd_max_conditions_at_8_bits(n):
    """The 8-bit codebook the TQP base uses.  A plain Lloyd loop stopped by an iteration cap is NOT at the
    fixed point here (round 2 found the oracle's first version 4e-3 / sqrt(n) off, condition violated by 6e-7): every level
    must be its cell's conditional mean to 1e-11 / sqrt(n)."""
    c = tq.lloyd_max_codebook(n, 8)
    assert len(c) == 256 and (np.diff(c) > 0).all()
    dens = lambda y: (1.0 - y * y) ** ((n - 3) / 2.0)
    b = np.concatenate(([-1.0], 0.5 * (c[:-1] + c[1:]), [1.0]))
    for j in range(0, 256, 3):
        num = integrate.quad(lambda y: y * dens(y), b[j], b[j + 1], epsabs=0, epsrel=1e-12)[0]
        den = integrate.quad(dens, b[j], b[j + 1], epsabs=0, epsrel=1e-12)[0]
        assert abs(num / den - c[j]) * np.sqrt(n) < 1e-10, j


def test_large_dimension_limit_is_max_gaussian_quantiser():
    """sqrt(n) * levels -> the Lloyd-Max levels of N(0, 1): 1 bit +-0.7979 (= sqrt(2/pi)), 2 bits +-0.4528, +-1.510,
    3 bits +-0.2451, +-0.7560, +-1.344, +-2.152 (Max 1960, Table I)."""
    n = 1 << 16
    s = np.sqrt(n)
    np.testing.assert_allclose(tq.lloyd_max_codebook(n, 1) * s, [-0.7979, 0.7979], atol=2e-4)
    np.testing.assert_allclose(tq.lloyd_max_codebook(n, 2) * s, [-1.510, -0.4528, 0.4528, 1.510], atol=1.5e-3)
    np.testing.assert_allclose(tq.lloyd_max_codebook(n, 3)[4:] * s, [0.2451, 0.7560, 1.344, 2.152], atol=2e-3)


def test_rotations_are_orthogonal_and_seeded():
    for n in (64, 48):                                          # signed Hadamard / sign-fixed QR
        R = tq.rotation(n, 1337)
        np.testing.assert_allclose(R @ R.T, np.eye(n), atol=1e-12)
        np.testing.assert_array_equal(R, tq.rotation(n, 1337))
        assert np.abs(R - tq.rotation(n, 1338)).max() > 0.1
    R = tq.rotation(64, 5)
    assert np.allclose(np.abs(R), 1.0 / 8.0)                    # Hadamard entries are +-1/sqrt(n)
    H = tq.hadamard(8)
    assert (H @ H.T == 8 * np.eye(8)).all() and (H[0] == 1).all() and (H[:, 0] == 1).all()


def test_distortion_matches_the_values_turboquant_reports():
    """Zandieh et al. 2025 state D_mse(b) ~ 0.36, 0.117, 0.03, 0.009 for b = 1..4 on unit vectors (and the bound
    sqrt(3) pi / 2 * 4^-b); these are the rounded mean-square errors of Max's Gaussian quantisers with 2, 4, 8, 16
    levels (Max 1960, Table I: 0.3634, 0.1175, 0.03454, 0.009497), which the per-coordinate error times n tends to.
    Monte Carlo over random rows, both rotation kinds."""
    rng = np.random.default_rng(3)
    expect = {1: 0.3634, 2: 0.1175, 3: 0.03454, 4: 0.009497}
    for n in (256, 192):
        R = tq.rotation(n, 7)
        W = rng.standard_normal((400, n)) * rng.uniform(0.1, 10.0, (400, 1))
        for bits, d_ref in expect.items():
            cb = tq.lloyd_max_codebook(n, bits)
            codes, norms = tq.encode(W, R, cb)
            Wh = tq.decode(codes, norms, R, cb)
            d = np.mean(np.sum((W - Wh) ** 2, axis=1) / norms ** 2)
            assert abs(d - d_ref) < 0.03 * d_ref, (n, bits, d)
            assert d <= np.sqrt(3) * np.pi / 2 * 4.0 ** -bits


def test_eight_bit_round_trip_properties():
    """The paper's setting: 8 bits.  Vectors that lie on the codebook are reproduced exactly (up to rounding), the code of
    a reconstruction is the code itself, norms are stored exactly, a zero row decodes to zero."""
    n = 128
    R = tq.rotation(n, 11)
    cb = tq.lloyd_max_codebook(n, 8)
    assert len(cb) == 256
    rng = np.random.default_rng(4)
    W = rng.standard_normal((50, n))
    W[7] = 0.0
    codes, norms = tq.encode(W, R, cb)
    assert codes.dtype == np.uint8
    np.testing.assert_allclose(norms, np.linalg.norm(W, axis=1), rtol=1e-15)
    Wh = tq.decode(codes, norms, R, cb)
    assert (Wh[7] == 0).all()
    rel = np.linalg.norm(W - Wh, axis=1)[norms > 0] / norms[norms > 0]
    assert rel.max() < 0.02                                      # 8-bit scalar codes: ~1 % relative error per row
    # a reconstruction is not a unit vector any more, so re-encoding renormalises it; its direction must still quantise
    # to the same codes wherever the coordinate is not within rounding of a cell boundary
    codes2, norms2 = tq.encode(Wh, R, cb)
    same = np.mean(codes2[norms > 0] == codes[norms > 0])
    assert same > 0.97
    # exact fixed point: a vector built FROM the levels, normalised, keeps every code
    pick = rng.integers(100, 156, (20, n))
    Y = cb[pick]
    scale = np.linalg.norm(Y, axis=1)
    # choose rows whose norm is 1 within 2 %: then renormalising moves no coordinate across a boundary except by chance
    V = (Y @ R)
    c3, n3 = tq.encode(V, R, cb)
    Yn = Y / scale[:, None]
    bounds = 0.5 * (cb[:-1] + cb[1:])
    np.testing.assert_array_equal(c3, np.searchsorted(bounds, Yn, side="left"))
    np.testing.assert_allclose(n3, scale, rtol=1e-12)
