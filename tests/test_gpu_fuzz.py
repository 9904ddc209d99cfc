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


# The screened router is the library's choice only for large E and T (tqp_route_info); here it is FORCED (route_impl = 2) on
# random shapes -- few experts, k close to E, a flooded and an emptied expert, T far below one 128-token tile -- and
# run_gpu asserts its topk_idx / topk_w bitwise against the dense chain before the rest of the layer runs on them.
# Seeds 1100-1103 and 5100-5103: the first four of either range of a one-off sweep over 1100-1139 / 5100-5139 (80 shapes, all
# green on the B200) that was run once when the router was written.
@pytest.mark.parametrize("seed,big", [(s, False) for s in range(1100, 1104)] + [(s, True) for s in range(5100, 5104)])
def test_random_shape_through_the_forced_screened_router(seed, big):
    from parity_util import assert_close, assert_routing_exact, run_gpu
    from test_gpu_parity import BWD_KEYS, FWD_KEYS, RG_KEYS, oracle_ref
    cfg, inp = _case(seed, big)
    ref = oracle_ref(inp, True, cfg.router_grad)
    gpu = run_gpu(inp, backward=True, router_grad=cfg.router_grad, route_impl=2)
    assert gpu["route_info"][0] == 1
    assert_routing_exact(gpu, ref)
    for key in FWD_KEYS + BWD_KEYS + (RG_KEYS if cfg.router_grad else ()):
        assert_close(key, gpu[key], ref[key])
