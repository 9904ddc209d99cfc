"""tqp_dispatch_noalloc: the dispatch for callers that cannot allocate (include/tqp.h).  Its scratch is a static __device__
array inside the library; the caller passes inputs and outputs only.  Integer work, so the bar is bit-exact: counts,
offsets, perm and inv_perm must equal the existing path's (tqp_dispatch through a ctx and a workspace) and the oracle's.
Four calls in a row on the same stream -- the second SMALLER, with other shapes, so that it runs over the first call's
left-overs in the shared array, the last a repeat of the first.  Collected last on purpose (pytest -x).
Passes alone in a fresh process (the first call does the one-time symbol look-up) and after the rest of the suite."""
import numpy as np
import pytest

import oracle

pytestmark = pytest.mark.gpu


def _existing_path(topk_idx_dev, T, E, k):
    import paper_2606_07404_b200 as tq
    layer = tq.TqpLayer(T, 128, 128, E, k, 8, training=False)
    counts, offsets, perm, inv = layer.dispatch(topk_idx_dev)
    return [x.clone() for x in (counts, offsets, perm, inv)]


def _routing(T, E, k, seed, skew):
    """k distinct experts per token; skewed draws leave some experts empty and crowd others."""
    rng = np.random.default_rng(seed)
    p = 1.0 / np.arange(1, E + 1) ** (1.3 if skew else 0.0)
    p /= p.sum()
    g = rng.gumbel(size=(T, E)) + np.log(p)[None, :]
    return np.argsort(-g, axis=1)[:, :k].astype(np.int32)


CASES = [  # T, E, k, skew: a full-size routing (cfg 4: 768 chunks), then a small ragged one, then a mid one with E = 1024
    (16384, 460, 12, False),
    (777, 37, 5, True),
    (3001, 1024, 8, True),
]


def test_dispatch_noalloc_matches_the_existing_path_on_calls_in_a_row():
    import torch
    import paper_2606_07404_b200 as tq
    dev = torch.device("cuda:0")
    inputs = [torch.from_numpy(_routing(T, E, k, 100 + i, skew)).to(dev) for i, (T, E, k, skew) in enumerate(CASES)]
    outs = []
    order = [0, 1, 2, 0]                      # back to back on one stream; the last repeats the first over stale scratch
    for ci in order:
        T, E, k, _ = CASES[ci]
        o = dict(counts=torch.full((E,), -7, dtype=torch.int32, device=dev), offsets=torch.full((E + 1,), -7, dtype=torch.int32, device=dev),
                 perm=torch.full((T * k,), -7, dtype=torch.int32, device=dev), inv_perm=torch.full((T * k,), -7, dtype=torch.int32, device=dev))
        outs.append(o)
    w = [torch.empty(n, dtype=torch.int32, device=dev) for n in (8, 9, 64, 64)]
    tq.dispatch_noalloc(torch.zeros((32, 2), dtype=torch.int32, device=dev), 8, *w)   # first call of the process: symbol look-up, module load
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    for ci, o in zip(order, outs):
        T, E, k, _ = CASES[ci]
        tq.dispatch_noalloc(inputs[ci], E, o["counts"], o["offsets"], o["perm"], o["inv_perm"])
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= free0, "the calls must not have taken device memory"
    for ci, o in zip(order, outs):
        T, E, k, skew = CASES[ci]
        ref = _existing_path(inputs[ci], T, E, k)
        for name, r in zip(("counts", "offsets", "perm", "inv_perm"), ref):
            assert torch.equal(o[name], r), f"case {ci} {name}: differs from tqp_dispatch"
        c_ref, o_ref, p_ref, i_ref = oracle.dispatch(inputs[ci].cpu().numpy(), E)
        np.testing.assert_array_equal(o["counts"].cpu().numpy(), c_ref)
        np.testing.assert_array_equal(o["offsets"].cpu().numpy(), o_ref)
        np.testing.assert_array_equal(o["perm"].cpu().numpy(), p_ref)
        np.testing.assert_array_equal(o["inv_perm"].cpu().numpy(), i_ref)
        if E == 1024:
            assert (o["counts"] == 0).any() and o["counts"].max() > 1024    # empty and multi-chunk experts in one call


def test_dispatch_noalloc_rejects_what_does_not_fit():
    import torch
    import paper_2606_07404_b200 as tq
    dev = torch.device("cuda:0")
    cap = tq.dispatch_noalloc_capacity()
    assert cap == 1 << 20
    E, k = 1024, 8
    T = (cap // E + 1) * 256 // k            # ceil(T k / 256) * E just past the capacity
    idx = torch.zeros((T, k), dtype=torch.int32, device=dev)
    bufs = [torch.empty(n, dtype=torch.int32, device=dev) for n in (E, E + 1, T * k, T * k)]
    with pytest.raises(tq.TqpError) as e:
        tq.dispatch_noalloc(idx, E, *bufs)
    assert e.value.code == 2 and "exceeds the static scratch" in str(e.value)
    with pytest.raises(tq.TqpError) as e:
        tq.dispatch_noalloc(idx[:16], 2000, *bufs)     # E > 1024
    assert e.value.code == 1
    with pytest.raises(tq.TqpError) as e:
        tq.dispatch_noalloc(idx[:16], 4, *bufs)        # k > E
    assert e.value.code == 1
    # the largest shape that fits still works after the rejections
    T_ok = cap // E * 256 // k
    idx_ok = torch.from_numpy(_routing(T_ok, E, k, 9, False)).to(dev)
    tq.dispatch_noalloc(idx_ok, E, bufs[0], bufs[1], bufs[2][:T_ok * k], bufs[3][:T_ok * k])
    torch.cuda.synchronize()
    c_ref, o_ref, p_ref, i_ref = oracle.dispatch(idx_ok.cpu().numpy(), E)
    np.testing.assert_array_equal(bufs[0].cpu().numpy(), c_ref)
    np.testing.assert_array_equal(bufs[2][:T_ok * k].cpu().numpy(), p_ref)
