"""Random-shape parity of the whole chain against the oracle: a fixed set of seeds drawn from the shape space the
library accepts (T 1..3000, d and F multiples of 128, E 1..200, k 1..16, r in {8, 16, 32}, half of them with a logit
bias that floods one expert and empties another).  The hand-picked cases elsewhere cover the known corner cases; this
one looks for the unknown ones (tile / stage / ring boundaries that only some combination of sizes hits)."""
import numpy as np
import pytest

import tqp_inputs as ti
from test_gpu_parity import check_all

pytestmark = pytest.mark.gpu


def _case(seed, big):
    rng = np.random.default_rng(seed)
    d = int(rng.choice([128, 256, 384, 512, 768, 1024]))
    F = int(rng.choice([128, 256, 384, 512]))
    E = int(rng.integers(1, 201 if big else 41))
    k = int(rng.integers(1, min(E, 16 if big else 8) + 1))
    r = int(rng.choice([8, 16, 32]))
    T = int(rng.integers(1, 3000 if big else 1200))
    cfg = ti.Config(f"fuzz{seed}", T=T, d=d, F=F, E=E, k=k, r=r, seed=seed, router_grad=bool(T * k >= 64))
    inp = ti.make_inputs(cfg)
    if rng.random() < 0.5 and E >= 3:
        bias = np.zeros(E, np.float32)
        bias[int(rng.integers(0, E))] = 2.5
        bias[int(rng.integers(0, E))] = -50.0
        inp["logit_bias"] = bias
    return cfg, inp


# Seeds: the contiguous ranges 1000-1004 (small shapes) and 5000-5004 (big shapes), chosen without looking at results,
# plus the non-contiguous seeds of round 1 (1017, 1020, 1036, 5012, 5016, 5025, 5028; their selection rule was not recorded),
# kept as regression cases.
SEEDS = sorted({(s, False) for s in (1000, 1001, 1002, 1003, 1004, 1017, 1020, 1036)} |
               {(s, True) for s in (5000, 5001, 5002, 5003, 5004, 5012, 5016, 5025, 5028)})


@pytest.mark.parametrize("seed,big", SEEDS)
def test_random_shape_matches_the_oracle(seed, big):
    cfg, inp = _case(seed, big)
    check_all(inp, backward=True, router_grad=cfg.router_grad, gemm_impl=0)
