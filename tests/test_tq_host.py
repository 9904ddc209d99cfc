"""Host-side pieces of the TurboQuant path inside libtqp.so (no GPU needed): the library's own Lloyd-Max solver and its
own sign-fixed QR against the oracle's (oracle/turboquant.py).  The two sides share no code: the library integrates the
coordinate law with Gauss-Legendre panels and starts from Gaussian quantiles, the oracle uses scipy's incomplete beta
function and starts from the law's own quantiles; the library orthogonalises by Gram-Schmidt, the oracle calls LAPACK's
Householder QR.  Lloyd-Max of a log-concave density has one fixed point and the sign-fixed Q is unique, so they must agree."""
import numpy as np
import pytest

import paper_2606_07404_b200 as tq
from oracle import turboquant as otq


@pytest.mark.parametrize("n,bits", [(64, 8), (1024, 8), (2560, 8), (4096, 8), (256, 4)])
def test_library_lloyd_max_levels_match_the_oracle(n, bits):
    mine = tq.tq_levels(n, bits)
    ref = otq.lloyd_max_codebook(n, bits)
    assert (np.diff(mine) > 0).all()
    np.testing.assert_allclose(mine, -mine[::-1], atol=0)
    # both iterate to a fixed point with a tolerance; the scale of the levels is 1 / sqrt(n)
    assert np.abs(mine - ref).max() * np.sqrt(n) < 2e-8
    # same cells for any coordinate that is not within 1e-8 / sqrt(n) of a boundary
    b_m, b_r = 0.5 * (mine[:-1] + mine[1:]), 0.5 * (ref[:-1] + ref[1:])
    y = np.random.default_rng(0).standard_normal(200000) / np.sqrt(n)
    assert (np.searchsorted(b_m, y, side="left") != np.searchsorted(b_r, y, side="left")).sum() == 0


@pytest.mark.parametrize("n", [48, 320])
def test_library_qr_rotation_matches_the_oracle(n):
    seed = 77
    G = np.random.default_rng(seed).standard_normal((n, n))         # the same draw oracle.turboquant.rotation makes
    mine = tq.tq_rotation_qr(G)
    ref = otq.rotation(n, seed)
    np.testing.assert_allclose(mine @ mine.T, np.eye(n), atol=1e-12)
    np.testing.assert_allclose(mine, ref, atol=1e-10)


def test_host_argument_errors():
    lib = tq.load_library()
    assert lib.tqp_tq_levels(4, 8, None) == 1          # NULL output
    with pytest.raises(tq.TqpError):
        tq.tq_levels(4, 8)                              # n < 8
    with pytest.raises(tq.TqpError):
        tq.tq_levels(64, 9)
