"""TEST INFRASTRUCTURE — CPU oracle of the TurboQuant MSE quantiser (component C10).

Only tests/ may import this.  It shares no code with the CUDA path (paper_2606_07404_b200) and does not import it.
No CUDA kernel uses this format yet: the oracle and its pins are committed first, as the build order requires.

PAPER.md L944-946 (§9.2), step by step in the paper's order:
  "For a weight vector, the quantizer separates scale from direction, normalizes the vector and stores its norm,
   applies a seeded random orthogonal rotation, and then quantizes each rotated coordinate independently against a
   scalar codebook. ... After a random orthogonal rotation the coordinates of a unit vector are distributed like the
   coordinates of a random point on the sphere, which is a known law, a shifted Beta distribution on the interval, so
   the Lloyd-Max scalar codebook for a given dimension and bit width can be computed analytically from that law ...
   The rotation is a signed Hadamard transform when the dimension is a power of two and a QR rotation from a Gaussian
   matrix with sign fixing otherwise.  Reconstruction looks up the codebook values and rescales by the stored norm."
  L946: "The base is held at 8-bit weight precision, with the per-expert weight packs quantized row by row."
  The one-bit residual (inner-product) variant "was not used; TQP uses the MSE path only".

Readings where the paper is silent (to be listed in DESIGN.md with the CUDA path):
  * coordinate law of a uniform point on S^{n-1}:  f_n(y) = C (1 - y^2)^((n-3)/2) on [-1, 1]  (y = 2 B - 1 with
    B ~ Beta((n-1)/2, (n-1)/2): the "shifted Beta");
  * Lloyd-Max = the fixed point of  boundaries = midpoints of neighbouring levels,  level = E[y | cell]  under f_n,
    started from the equal-probability quantiles, reached by a few Lloyd sweeps followed by Newton's method on the same
    equations; levels ascending, codes 0 .. 2^b - 1;
  * a coordinate on a cell boundary takes the LOWER code (searchsorted side="left" on the boundaries);
  * signed Hadamard: R = H_n diag(s) / sqrt(n), H_n the Sylvester matrix, s in {-1, +1}^n from
    numpy.random.default_rng(seed); QR: Q of a default_rng(seed) standard-normal n x n matrix, columns multiplied by
    sign(diag(R_qr)) (the usual fix that makes Q Haar-distributed);
  * a zero row is stored as norm 0 with the code of the level nearest 0 (the lower of the two middle levels).
"""
from __future__ import annotations

import numpy as np
from scipy import special


# ---- coordinate law -----------------------------------------------------------------------------------------------
def coord_cdf(y, n: int):
    """P(Y <= y) for one coordinate of a uniform point on S^{n-1}."""
    a = (n - 1) / 2.0
    return special.betainc(a, a, (np.asarray(y, dtype=np.float64) + 1.0) / 2.0)


def _partial_mean(lo, hi, n: int):
    """integral of y f_n(y) over [lo, hi]:  closed form  C [ -(1-y^2)^((n-1)/2) / (n-1) ]  (antiderivative of y (1-y^2)^((n-3)/2))."""
    a = (n - 1) / 2.0
    logc = special.gammaln(n / 2.0) - special.gammaln((n - 1) / 2.0) - 0.5 * np.log(np.pi)      # C = Gamma(n/2) / (sqrt(pi) Gamma((n-1)/2))
    def g(y):
        t = 1.0 - np.minimum(np.asarray(y, dtype=np.float64) ** 2, 1.0)
        with np.errstate(divide="ignore"):
            return -np.exp(logc + a * np.log(t) - np.log(n - 1.0))          # t = 0 at y = +-1: exp(-inf) = 0
    return g(hi) - g(lo)


def lloyd_max_codebook(n: int, bits: int, tol: float = 1e-15, max_iter: int = 100) -> np.ndarray:
    """The 2^bits Lloyd-Max levels of the coordinate law in dimension n (ascending, fp64): the point where every level is
    the conditional mean of its cell and every boundary the midpoint of its two levels.

    The plain Lloyd sweep (boundaries <- midpoints, levels <- cell means) contracts towards that point only linearly, and
    at 8 bits far too slowly (after 20 000 sweeps the levels were still 4e-3 / sqrt(n) away and the Lloyd-Max condition
    held to 6e-7 only), so after a few sweeps the same equations  F_j(c) = c_j - E[y | cell_j(c)] = 0  are solved by
    Newton's method.  Cell j depends on c_{j-1}, c_j, c_{j+1} only, so the Jacobian is tridiagonal:
        d E[y | cell] / d(upper boundary) =  f(b_up) (b_up - E) / mass,   d E / d(lower boundary) = -f(b_lo) (b_lo - E) / mass,
    and each boundary moves by half of either neighbouring level.  tests/test_turboquant_pins.py checks the result against
    the Lloyd-Max conditions with an independent quadrature at 8 bits."""
    from scipy.linalg import solve_banded
    L = 1 << bits
    a = (n - 1) / 2.0
    logc = special.gammaln(n / 2.0) - special.gammaln((n - 1) / 2.0) - 0.5 * np.log(np.pi)
    pdf = lambda y: np.exp(logc + (n - 3) / 2.0 * np.log1p(-np.minimum(y * y, 1.0 - 1e-300)))
    # start: conditional means of the equal-probability cells
    q = np.linspace(0.0, 1.0, L + 1)
    b = 2.0 * special.betaincinv(a, a, q) - 1.0
    b[0], b[-1] = -1.0, 1.0
    c = _partial_mean(b[:-1], b[1:], n) / np.diff(coord_cdf(b, n))

    def cells(c):
        b = np.concatenate(([-1.0], 0.5 * (c[:-1] + c[1:]), [1.0]))
        mass = np.diff(coord_cdf(b, n))
        return b, mass, _partial_mean(b[:-1], b[1:], n) / mass

    for _ in range(20):                                   # a few plain Lloyd sweeps
        c = cells(c)[2]
    for _ in range(max_iter):
        b, mass, cen = cells(c)
        F = c - cen
        fb = pdf(b[1:-1])                                 # density at the interior boundaries b_1 .. b_{L-1}
        dup = np.zeros(L); dlo = np.zeros(L)
        dup[:-1] = fb * (b[1:-1] - cen[:-1]) / mass[:-1]  # d cen_j / d b_{j+1}
        dlo[1:] = -fb * (b[1:-1] - cen[1:]) / mass[1:]    # d cen_j / d b_j
        ab = np.zeros((3, L))
        ab[1] = 1.0 - 0.5 * (dup + dlo)                   # dF_j / dc_j
        ab[0, 1:] = -0.5 * dup[:-1]                       # dF_j / dc_{j+1}
        ab[2, :-1] = -0.5 * dlo[1:]                       # dF_j / dc_{j-1}
        step = solve_banded((1, 1), ab, -F)
        c = c + step
        if np.max(np.abs(step)) < tol * max(1.0, np.sqrt(n)) / np.sqrt(n):
            break
    return c


# ---- rotation -----------------------------------------------------------------------------------------------------
def hadamard(n: int) -> np.ndarray:
    assert n & (n - 1) == 0 and n > 0
    H = np.ones((1, 1))
    while H.shape[0] < n:
        H = np.block([[H, H], [H, -H]])
    return H


def rotation(n: int, seed: int) -> np.ndarray:
    """The seeded orthogonal matrix R (y = R u)."""
    rng = np.random.default_rng(seed)
    if n & (n - 1) == 0:
        s = rng.integers(0, 2, n) * 2.0 - 1.0
        return hadamard(n) * s[None, :] / np.sqrt(n)
    Q, Rr = np.linalg.qr(rng.standard_normal((n, n)))
    return Q * np.sign(np.diag(Rr))[None, :]


# ---- encode / decode ----------------------------------------------------------------------------------------------
def encode(W: np.ndarray, R: np.ndarray, codebook: np.ndarray):
    """Rows of W [rows][n] -> (codes uint8/uint16 [rows][n], norms fp64 [rows])."""
    W = np.asarray(W, dtype=np.float64)
    norms = np.sqrt(np.sum(W * W, axis=1))
    U = np.divide(W, norms[:, None], out=np.zeros_like(W), where=norms[:, None] > 0)
    Y = U @ R.T
    bounds = 0.5 * (codebook[:-1] + codebook[1:])
    codes = np.searchsorted(bounds, Y, side="left")
    return codes.astype(np.uint8 if len(codebook) <= 256 else np.uint16), norms


def decode(codes: np.ndarray, norms: np.ndarray, R: np.ndarray, codebook: np.ndarray) -> np.ndarray:
    """Reconstruction: look the levels up, rotate back, rescale by the stored norm."""
    Yh = codebook[codes.astype(np.int64)]
    return (Yh @ R) * np.asarray(norms, dtype=np.float64)[:, None]
