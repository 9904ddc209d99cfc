"""Host-side check of the selection rule the screened router relies on (csrc/route.cu): if every
approximate logit is within delta of the exact one, then the experts with a >= (k-th largest a) - 2 delta contain the exact
top-k under the order (-logit, id) -- ties included -- so running the canonical chain on those candidates only and taking
the top-k among them gives the dense result.  No GPU, no oracle: plain numpy, adversarial perturbations."""
import numpy as np
import pytest


def exact_topk(l, k):
    order = np.lexsort((np.arange(l.size), -l))       # by -logit, then id
    return order[:k]


def candidates(a, k, delta):
    """As the kernel: the window is 2 delta plus a rounding slack relative to tau (the kernel takes 1e-6 |tau| in fp32 and
    inflates delta by 1 %): in exact arithmetic the worst case sits exactly ON the boundary, tau - 2 delta."""
    tau = np.sort(a)[::-1][k - 1]
    return np.nonzero(a >= tau - 2.0 * delta - 1e-9 * (abs(tau) + delta))[0]


@pytest.mark.parametrize("E,k", [(8, 2), (64, 8), (460, 12), (1024, 32)])
def test_candidates_contain_the_exact_topk(E, k):
    rng = np.random.default_rng(E * 100 + k)
    for trial in range(300):
        l = rng.standard_normal(E)
        if trial % 3 == 0:                             # exact ties around the selection boundary
            srt = np.sort(l)[::-1]
            l[rng.integers(0, E, size=4)] = srt[k - 1]
        delta = 10.0 ** rng.uniform(-4, -0.5)
        for mode in range(4):
            if mode == 0:
                e = rng.uniform(-delta, delta, E)
            elif mode == 1:                            # push the true top-k down and everything else up (worst case)
                e = np.full(E, delta)
                e[exact_topk(l, k)] = -delta
            elif mode == 2:
                e = np.where(rng.random(E) < 0.5, delta, -delta)
            else:
                e = np.zeros(E)
            a = l + e
            cand = candidates(a, k, delta)
            top = exact_topk(l, k)
            assert np.isin(top, cand).all(), (trial, mode)
            # and the top-k among the candidates, taken on the EXACT values, is the dense result (order included)
            sub = cand[np.lexsort((cand, -l[cand]))][:k]
            np.testing.assert_array_equal(sub, top)


def test_rule_is_tight_in_the_factor_two():
    """With a window of only one delta the rule can lose a member of the top-k: the 2 is needed."""
    l = np.array([1.0, 0.9, 0.0])
    delta = 0.06
    a = l + np.array([delta, -delta, 0.0])             # a = [1.06, 0.84, 0]; k = 1, exact top-1 = expert 0: fine
    assert 0 in candidates(a, 1, delta)
    l = np.array([1.0, 1.05, 0.0])                     # exact top-1 = expert 1
    a = l + np.array([delta, -delta, 0.0])             # a = [1.06, 0.99, 0]: tau = 1.06, tau - delta = 1.0 > a[1]
    tau = a.max()
    assert not (a[1] >= tau - delta)                   # a one-delta window would drop the true winner
    assert 1 in candidates(a, 1, delta)                # the two-delta window keeps it
