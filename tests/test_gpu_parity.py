"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element, on seeded inputs.
Bit-exact for routing/permutation; max-abs <= 2e-2*max|ref| and relative Frobenius <= 1e-2 for floats (north_star)."""
import numpy as np
import pytest

import oracle
import tqp_inputs as ti
from parity_util import assert_close, assert_routing_exact, errors, run_gpu

pytestmark = pytest.mark.gpu

FWD_KEYS = ("Xp", "G", "U", "H", "Ye", "Y")
BWD_KEYS = ("dYe", "dXp", "dX_experts", "dA_gate", "dB_gate", "dA_up", "dB_up", "dA_down", "dB_down")
RG_KEYS = ("dtopk_w", "dW_r", "dX")


def oracle_ref(inp, backward, router_grad):
    ref = oracle.layer(inp, dtype=np.float32, backward=backward, router_grad=router_grad)
    ref["Xp"] = ti.bf16_bits_to_f32(inp["X"])[ref["perm"] // inp["k"]]
    return ref


def check_all(inp, backward, router_grad, gemm_impl, report=None):
    ref = oracle_ref(inp, backward, router_grad)
    gpu = run_gpu(inp, backward=backward, router_grad=router_grad, gemm_impl=gemm_impl)
    assert_routing_exact(gpu, ref)
    keys = FWD_KEYS + (BWD_KEYS if backward else ()) + (RG_KEYS if router_grad else ())
    errs = {}
    for key in keys:
        errs[key] = errors(gpu[key], ref[key])
    if report is not None:
        report.update(errs)
    for key in keys:
        assert_close(key, gpu[key], ref[key])
    return gpu, ref


MID = ti.Config("mid_ragged", T=640, d=256, F=384, E=6, k=3, r=16, seed=21, router_grad=True)
MID32 = ti.Config("mid_r32", T=300, d=384, F=256, E=5, k=2, r=32, seed=22, router_grad=True)


def _skewed(cfg):
    """Same recipe, plus a logit bias that sends >256 rows to one expert and none to another (several tiles per
    expert, a ragged tail, an empty expert)."""
    inp = ti.make_inputs(cfg)
    bias = np.zeros(cfg.E, np.float32)
    bias[1] = 2.0
    bias[cfg.E - 1] = -50.0
    inp["logit_bias"] = bias
    return inp


@pytest.mark.parametrize("gemm_impl", [1, 2, 0], ids=["scaffold", "tcgen05_1cta", "tcgen05"])
def test_cfg0_tiny_full_chain(gemm_impl):
    cfg = ti.CONFIGS[0]
    inp = ti.make_inputs(cfg)
    check_all(inp, backward=True, router_grad=True, gemm_impl=gemm_impl)


@pytest.mark.parametrize("gemm_impl", [1, 2, 3, 0],
                         ids=["scaffold", "tcgen05_1cta", "tcgen05_2cta_smemA", "tcgen05"])
@pytest.mark.parametrize("cfg", [MID, MID32], ids=lambda c: c.name)
def test_mid_ragged_multi_tile(cfg, gemm_impl):
    inp = _skewed(cfg)
    gpu, ref = check_all(inp, backward=True, router_grad=True, gemm_impl=gemm_impl)
    assert ref["counts"].max() > 256 and ref["counts"].min() == 0
    for key in ("dA_gate", "dB_gate", "dA_up", "dB_up", "dA_down", "dB_down"):
        assert (gpu[key][cfg.E - 1] == 0).all()        # empty expert: exactly zero gradients


# d % 256 == 0 with r = 32: the TMA-gather projections (rows_gather_proj_kernel) in their rank-32 instantiations, two
# 256-column stages per row, whole and ragged 128-row items, an expert with several tiles and an empty one
MID32_D512 = ti.Config("mid_r32_d512", T=700, d=512, F=256, E=5, k=2, r=32, seed=23, router_grad=True)


@pytest.mark.parametrize("cfg", [MID, MID32_D512], ids=lambda c: c.name)
def test_two_runs_are_bitwise_identical(cfg):
    """No atomics and no run-dependent order anywhere on the path (persistent kernels walk fixed item sequences, weight
    gradients are summed in segment order): the same inputs must give the same bits, ragged tiles included.  A write
    past an expert's last row by the TMA scatter, or a race on a shared-memory stage, would show up here."""
    inp = _skewed(cfg)
    a = run_gpu(inp, backward=True, router_grad=True)
    b = run_gpu(inp, backward=True, router_grad=True)
    assert a.keys() == b.keys()
    for key in a:
        assert np.array_equal(np.asarray(a[key]), np.asarray(b[key])), key


@pytest.mark.parametrize("cfg", [MID, MID32_D512], ids=lambda c: c.name)
def test_dgu_projection_and_dB_in_one_pass_forced_and_off(cfg):
    """rows_proj_wgrad_kernel (dG . B^T with (x.A)^T dG from one pass over dG, same for dU) against the separate passes it
    replaces, on a skewed batch where one expert owns several tiles (per-tile partials + ordered reduction), several own one
    tile (direct write) and one owns none (zeroed): option fuse_dgu = 1 (the default), 0 switches it off.  Both must match the
    oracle; between the two only the fp32 summation order of dB differs."""
    inp = _skewed(cfg)
    ref = oracle_ref(inp, True, False)
    res = {}
    for mode in (0, 1):
        gpu = run_gpu(inp, backward=True, options={"fuse_dgu": mode})
        for key in BWD_KEYS:
            assert_close(f"{key} (fuse_dgu={mode})", gpu[key], ref[key])
        for key in ("dB_gate", "dB_up"):
            assert (gpu[key][cfg.E - 1] == 0).all()
        res[mode] = gpu
    assert ref["counts"].max() > 256 and ref["counts"].min() == 0
    for key in ("dB_gate", "dB_up", "dA_gate", "dA_up", "dXp"):
        _, relf = errors(res[1][key], res[0][key])
        assert relf <= 1e-5, f"{key}: the two paths differ by relF {relf:.2e}"


def test_gathered_projections_rank32_multi_stage():
    inp = _skewed(MID32_D512)
    gpu, ref = check_all(inp, backward=True, router_grad=True, gemm_impl=0)
    assert ref["counts"].max() > 256 and ref["counts"].min() == 0


def test_tile_list_covers_every_row_once():
    """The grouped GEMMs draw items from a global counter in tile-list order.  Host-logic check of the device-built list
    under heavy skew: every routed row of every expert is covered exactly once, tiles hold at most 256 rows, tiles of
    one expert have equal size in multiples of 16 (but the last), experts ascend (a fixed order, hence reproducible)."""
    import torch
    from parity_util import make_layer
    cfg = ti.Config("tiles", T=3000, d=128, F=128, E=40, k=4, r=16, seed=55)
    inp = ti.make_inputs(cfg)
    bias = np.zeros(cfg.E, np.float32); bias[3] = 3.0; bias[7] = 1.5; bias[11] = -50.0
    inp["logit_bias"] = bias
    layer, dev = make_layer(inp, training=False)
    idx, w = layer.route(dev["X"], dev["W_r"], dev["logit_bias"])
    counts, offsets, perm, inv = layer.dispatch(idx)
    torch.cuda.synchronize()
    counts, offsets = counts.cpu().numpy(), offsets.cpu().numpy()
    nt = int(layer.debug_buffer("num_tiles", (1,), torch.int32).item())
    tiles = layer.debug_buffer("tiles", (nt, 4), torch.int32).cpu().numpy()
    assert counts.max() > 1024 and counts.min() == 0
    covered = np.zeros(cfg.N, np.int32)
    for e, row0, rows, _ in tiles:
        assert 0 <= rows <= 256 and offsets[e] <= row0 and row0 + rows <= offsets[e + 1]
        covered[row0:row0 + rows] += 1
    assert (covered == 1).all()
    assert (np.diff(tiles[:, 0]) >= 0).all(), "experts ascend"
    for e in np.unique(tiles[:, 0]):
        r = tiles[tiles[:, 0] == e, 2]
        assert (r[:-1] == r[0]).all() and r[0] % 16 == 0 or len(r) == 1
    assert nt == sum((c + 255) // 256 for c in counts)


def test_no_write_outside_the_buffers_guard_regions():
    """compute-sanitizer is closed on this pool (profiles/r2_sanitizer.md), so this is the suite's own bounds check: every
    caller-owned output tensor and the bound workspace sit between 4 KB guard regions filled with a canary pattern; after
    the whole forward + backward chain on a skewed, ragged batch (TMA scatter of ragged tiles, over-reading 16-row groups,
    persistent kernels with dynamic work lists) every guard byte must be untouched and the results must still be right."""
    import ctypes
    import torch
    from parity_util import to_dev
    import paper_2606_07404_b200 as tq
    inp = _skewed(MID32_D512)
    cfg = MID32_D512
    ref = oracle_ref(inp, True, True)
    G = 4096
    guards = []

    def guarded(shape, dtype):
        n = int(np.prod(shape)) * torch.empty((), dtype=dtype).element_size()
        pad = (-n) % 16
        raw = torch.full((G + n + pad + G,), 0xAB, dtype=torch.uint8, device="cuda")
        guards.append((raw, n))
        return raw[G:G + n].view(dtype).view(*shape)

    layer = tq.TqpLayer(cfg.T, cfg.d, cfg.F, cfg.E, cfg.k, cfg.r, lora_scale=cfg.lora_scale, training=True)
    nbytes = tq.workspace_bytes(cfg.T, cfg.d, cfg.F, cfg.E, cfg.k, cfg.r, cfg.lora_scale, True)
    ws = guarded((nbytes,), torch.uint8)
    layer.workspace = ws
    layer._check(layer.lib.tqp_bind_workspace(layer.ctx, ctypes.c_void_p(ws.data_ptr()), nbytes, layer._stream()))
    dev = to_dev(inp)
    layer.bind_weights(**{n: dev[n] for n in ("idx_gate", "idx_up", "idx_down", "scale_gate", "scale_up", "scale_down",
                                              "codebook", "A_gate", "A_up", "B_gate", "B_up", "A_down", "B_down")})
    T, k, d, F, E, r = cfg.T, cfg.k, cfg.d, cfg.F, cfg.E, cfg.r
    N = T * k
    bf = torch.bfloat16
    Ye, dYe, dXp = guarded((N, d), bf), guarded((N, d), bf), guarded((N, d), bf)
    Y, dX = guarded((T, d), bf), guarded((T, d), bf)
    grads = {"dA_gate": guarded((E, d, r), torch.float32), "dB_gate": guarded((E, r, F), torch.float32),
             "dA_up": guarded((E, d, r), torch.float32), "dB_up": guarded((E, r, F), torch.float32),
             "dA_down": guarded((E, F, r), torch.float32), "dB_down": guarded((E, r, d), torch.float32)}
    idx, w = layer.route(dev["X"], dev["W_r"], dev["logit_bias"])
    counts, offsets, perm, inv = layer.dispatch(idx)
    layer.expert_fwd(dev["X"], offsets, perm, out=Ye)
    layer.combine(Ye, inv, w, out=Y)
    _, dw = layer.combine_bwd(dev["dY"], Ye, inv, w, want_dw=True, out=dYe, perm=perm)
    layer.expert_bwd(dev["X"], dYe, offsets, perm, grads=grads, out=dXp, dYe_unmodified=True)
    layer.dispatch_bwd(dXp, inv, out=dX)
    dW_r = layer.route_bwd(dev["X"], dev["W_r"], idx, w, dw, offsets, perm, dX)
    torch.cuda.synchronize()
    for raw, n in guards:
        assert (raw[:G] == 0xAB).all() and (raw[G + n + ((-n) % 16):] == 0xAB).all(), "a guard region was written"
    from parity_util import to_np
    assert_close("Y", to_np(Y), ref["Y"])
    assert_close("dX", to_np(dX), ref["dX"])
    for key, g in grads.items():
        assert_close(key, to_np(g), ref[key])


def test_zero_scale_channels():
    """The forward GEMMs apply the channel scale in the fp32 epilogue and feed the adapter row divided by it; a channel
    whose scale is exactly 0 (a zero weight row) must still get its adapter term and produce no NaN / Inf."""
    inp = _skewed(MID)
    for key in ("scale_gate", "scale_up", "scale_down"):
        sc = inp[key].copy()
        sc[:, 3] = 0; sc[1, 100:140] = 0; sc[2, -1] = 0
        inp[key] = sc
    rng = np.random.default_rng(9)
    for key in ("A_gate", "B_gate", "A_up", "B_up", "A_down", "B_down"):
        inp[key] = ti.f32_to_bf16_bits(rng.standard_normal(inp[key].shape).astype(np.float32) * 0.05)
    gpu, ref = check_all(inp, backward=True, router_grad=True, gemm_impl=0)
    assert np.abs(ref["G"][:, 3]).max() > 0        # the adapter alone drives these channels


def test_routing_ties_lower_id_wins():
    cfg = ti.CONFIGS[0]
    inp = ti.make_inputs(cfg)
    inp["W_r"][:, 5] = inp["W_r"][:, 1]      # duplicate router columns -> exact ties
    inp["W_r"][:, 6] = inp["W_r"][:, 1]
    ref = oracle_ref(inp, False, False)
    gpu = run_gpu(inp, backward=False, gemm_impl=1)
    assert_routing_exact(gpu, ref)


def test_error_codes_on_device():
    import torch
    import paper_2606_07404_b200 as tq
    layer = tq.TqpLayer(64, 128, 256, 8, 2, 8)
    X = torch.zeros(64, 128, dtype=torch.bfloat16, device="cuda")
    W = torch.zeros(128, 8, device="cuda")
    idx, w = layer.route(X, W)
    counts, offsets, perm, inv = layer.dispatch(idx)
    with pytest.raises(tq.TqpError) as e:
        layer.expert_fwd(X, offsets, perm)            # no weights bound
    assert e.value.code == 5
    with pytest.raises(tq.TqpError) as e:
        layer.route(X[:0], W)                          # T == 0
    assert e.value.code == 1
    with pytest.raises(tq.TqpError) as e:
        layer.route(torch.zeros(65 * 128 + 1, dtype=torch.bfloat16, device="cuda")[1:].view(65, 128)[:64], W)
    assert e.value.code == 3                           # misaligned pointer


@pytest.mark.parametrize("cfg", [ti.CONFIGS[0], MID], ids=lambda c: c.name)
def test_step_host_end_to_end(cfg):
    """tqp_step_host (pinned host X/dY in, Y/dX out, copies overlapped with compute on internal streams) against the
    oracle; called twice so that a stale event or buffer from the first call would show."""
    import torch
    from parity_util import make_layer, to_np
    inp = _skewed(cfg) if cfg is MID else ti.make_inputs(cfg)
    ref = oracle_ref(inp, True, True)
    layer, dev = make_layer(inp, training=True)
    T, d = inp["T"], inp["d"]
    Xh, dYh = dev["X"].cpu().pin_memory(), dev["dY"].cpu().pin_memory()
    Yh = torch.zeros((T, d), dtype=torch.bfloat16).pin_memory()
    dXh = torch.zeros((T, d), dtype=torch.bfloat16).pin_memory()
    grads = layer.alloc_grads()
    dW_r = torch.zeros((d, inp["E"]), dtype=torch.float32, device="cuda")
    for _ in range(2):
        Yh.zero_(); dXh.zero_()
        layer.step_host(Xh, dYh, dev["W_r"], dev.get("logit_bias"), Yh, dXh, grads, dW_r)
    assert_close("Y", to_np(Yh), ref["Y"])
    assert_close("dX", to_np(dXh), ref["dX"])
    assert_close("dW_r", to_np(dW_r), ref["dW_r"])
    for key in ("dA_gate", "dB_gate", "dA_up", "dB_up", "dA_down", "dB_down"):
        assert_close(key, to_np(grads[key]), ref[key])


def test_step_host_async_three_steps_in_a_pipeline():
    """tqp_step_host_async / tqp_step_host_wait: three steps with alternating inputs enqueued back to back (two in flight,
    so the uploads of a step travel under the previous step's kernels and use the other staging set); every step's Y and
    dX must be that step's own, and the gradients those of the last step."""
    import torch
    from parity_util import make_layer, to_np
    inpA = _skewed(MID)
    inpB = dict(inpA)
    other = ti.make_inputs(ti.Config("mid_other", T=MID.T, d=MID.d, F=MID.F, E=MID.E, k=MID.k, r=MID.r, seed=97, router_grad=True))
    inpB["X"], inpB["dY"] = other["X"], other["dY"]
    refA, refB = oracle_ref(inpA, True, True), oracle_ref(inpB, True, True)
    layer, dev = make_layer(inpA, training=True)
    T, d = inpA["T"], inpA["d"]

    def pinned(a):
        return torch.from_numpy(a.view(np.int16)).view(torch.bfloat16).pin_memory()

    host = {"A": (pinned(inpA["X"]), pinned(inpA["dY"])), "B": (pinned(inpB["X"]), pinned(inpB["dY"]))}
    outs = [(torch.zeros((T, d), dtype=torch.bfloat16).pin_memory(), torch.zeros((T, d), dtype=torch.bfloat16).pin_memory())
            for _ in range(3)]
    grads = layer.alloc_grads()
    dW_r = torch.zeros((d, inpA["E"]), dtype=torch.float32, device="cuda")
    order = ["A", "B", "A"]
    refs = {"A": refA, "B": refB}
    for i, which in enumerate(order):
        layer.step_host_async(host[which][0], host[which][1], dev["W_r"], dev.get("logit_bias"), outs[i][0], outs[i][1], grads, dW_r)
        if i >= 1:
            layer.step_host_wait(1)
            assert_close(f"Y[{i - 1}]", to_np(outs[i - 1][0]), refs[order[i - 1]]["Y"])
            assert_close(f"dX[{i - 1}]", to_np(outs[i - 1][1]), refs[order[i - 1]]["dX"])
    layer.step_host_wait(0)
    assert_close("Y[2]", to_np(outs[2][0]), refA["Y"])
    assert_close("dX[2]", to_np(outs[2][1]), refA["dX"])
    assert_close("dW_r", to_np(dW_r), refA["dW_r"])
    for key in ("dA_gate", "dB_gate", "dA_up", "dB_up", "dA_down", "dB_down"):
        assert_close(key, to_np(grads[key]), refA[key])
    assert np.abs(refA["Y"] - refB["Y"]).max() > 0.1 * np.abs(refA["Y"]).max()     # the two inputs really differ


@pytest.mark.parametrize("T", [1025, 2050])
@pytest.mark.parametrize("chunks", [4, 1, 0])
def test_step_host_chunked_upload_is_bitwise_the_stepwise_api(T, chunks):
    """the path behind the e2e number at T >= 1024.  X goes up and is routed in four ragged token chunks
    (T = 1025 -> 260 + 260 + 260 + 245, T = 2050 -> 516 x 3 + 502), or in one piece when the previous step is still running;
    both branches are pinned through the option "host_chunks" and must give, bit for bit, what the stepwise API gives
    (same kernels, same order of every sum), for Y, dX and all gradients; two async steps in flight."""
    import torch
    from parity_util import make_layer, to_np
    cfg = ti.Config(f"host_T{T}", T=T, d=256, F=256, E=12, k=3, r=16, seed=40 + T, router_grad=True)
    inp = ti.make_inputs(cfg)
    step = run_gpu(inp, backward=True, router_grad=True)
    layer, dev = make_layer(inp, training=True)
    layer.set_option("host_chunks", chunks)
    d = cfg.d
    Xh, dYh = dev["X"].cpu().pin_memory(), dev["dY"].cpu().pin_memory()
    outs = [(torch.zeros((T, d), dtype=torch.bfloat16).pin_memory(), torch.zeros((T, d), dtype=torch.bfloat16).pin_memory())
            for _ in range(3)]
    grads = layer.alloc_grads()
    dW_r = torch.zeros((d, cfg.E), dtype=torch.float32, device="cuda")
    for i in range(3):
        layer.step_host_async(Xh, dYh, dev["W_r"], None, outs[i][0], outs[i][1], grads, dW_r)
        if i >= 1:
            layer.step_host_wait(1)
    layer.step_host_wait(0)
    for i in range(3):
        np.testing.assert_array_equal(to_np(outs[i][0]), step["Y"], err_msg=f"Y of step {i}")
        np.testing.assert_array_equal(to_np(outs[i][1]), step["dX"], err_msg=f"dX of step {i}")
    np.testing.assert_array_equal(to_np(dW_r), step["dW_r"])
    for key in ("dA_gate", "dB_gate", "dA_up", "dB_up", "dA_down", "dB_down"):
        np.testing.assert_array_equal(to_np(grads[key]), step[key], err_msg=key)
    ref = oracle_ref(inp, True, True)
    assert_close("Y", to_np(outs[2][0]), ref["Y"])
    assert_close("dX", to_np(outs[2][1]), ref["dX"])


def test_layer_reuse_smaller_batch_and_foreign_dYe():
    """One ctx, two calls: a full batch, then a smaller batch with different data (stale workspace rows, tile list and
    cached dispatch pointers must not leak), and an expert_bwd fed a dYe tensor that did NOT come from the fused
    tqp_combine_bwd of this step (the library must then project it itself)."""
    import torch
    from parity_util import make_layer, to_dev, to_np
    big = _skewed(MID)
    layer, dev = make_layer(big, training=True)
    for _ in range(2):   # warm the ctx with the big batch (fused combine_bwd path, cached Zd)
        idx, w = layer.route(dev["X"], dev["W_r"], dev.get("logit_bias"))
        counts, offsets, perm, inv = layer.dispatch(idx)
        Ye = layer.expert_fwd(dev["X"], offsets, perm)
        dYe, _ = layer.combine_bwd(dev["dY"], Ye, inv, w, want_dw=False, perm=perm)
        layer.expert_bwd(dev["X"], dYe, offsets, perm, dYe_unmodified=True)
    small_cfg = ti.Config("small_after_big", T=200, d=MID.d, F=MID.F, E=MID.E, k=MID.k, r=MID.r, seed=77)
    small = ti.make_inputs(small_cfg)
    for key in ("idx_gate", "idx_up", "idx_down", "scale_gate", "scale_up", "scale_down", "codebook",
                "A_gate", "A_up", "B_gate", "B_up", "A_down", "B_down"):
        small[key] = big[key]                      # same bound weights
    ref = oracle_ref(small, True, False)
    sd = to_dev(small)
    idx, w = layer.route(sd["X"], sd["W_r"], None)
    counts, offsets, perm, inv = layer.dispatch(idx)
    Ye = layer.expert_fwd(sd["X"], offsets, perm)
    Y = layer.combine(Ye, inv, w)
    dYe_fused, dw = layer.combine_bwd(sd["dY"], Ye, inv, w, want_dw=True, perm=perm)
    dYe_foreign = dYe_fused.clone()                # a different tensor: the cached projection must not be trusted
    import paper_2606_07404_b200 as tq
    with pytest.raises(tq.TqpError) as e:          # vouching for a tensor the fused combine_bwd did not write is refused
        layer.expert_bwd(sd["X"], dYe_foreign, offsets, perm, dYe_unmodified=True)
    assert e.value.code == 5
    dXp, grads = layer.expert_bwd(sd["X"], dYe_foreign, offsets, perm)
    dX = layer.dispatch_bwd(dXp, inv)
    torch.cuda.synchronize()
    np.testing.assert_array_equal(to_np(idx), ref["topk_idx"])
    np.testing.assert_array_equal(to_np(perm), ref["perm"])
    assert_close("Y", to_np(Y), ref["Y"])
    assert_close("dYe", to_np(dYe_fused), ref["dYe"])
    assert_close("dtopk_w", to_np(dw), ref["dtopk_w"])
    assert_close("dX_experts", to_np(dX), ref["dX_experts"])
    for key in ("dA_gate", "dB_gate", "dA_up", "dB_up", "dA_down", "dB_down"):
        assert_close(key, to_np(grads[key]), ref[key])


def test_dYe_edited_in_place_between_combine_bwd_and_expert_bwd():
    """a caller that adds something to dYe in place (a shared-expert or auxiliary gradient) between the fused
    tqp_combine_bwd and tqp_expert_bwd passes flags = 0; the adapter projection left by combine_bwd must then NOT be
    used.  Checked against the oracle's expert_bwd on the edited dYe.  Also: the unfused path (perm = NULL) gives the same
    dYe bits as the fused one."""
    import torch
    from parity_util import make_layer, to_np
    inp = _skewed(MID)
    ref = oracle_ref(inp, True, False)
    layer, dev = make_layer(inp, training=True)
    idx, w = layer.route(dev["X"], dev["W_r"], dev.get("logit_bias"))
    counts, offsets, perm, inv = layer.dispatch(idx)
    Ye = layer.expert_fwd(dev["X"], offsets, perm)
    dYe_plain, dw_plain = layer.combine_bwd(dev["dY"], Ye, inv, w, want_dw=True)             # perm = NULL
    dYe, dw = layer.combine_bwd(dev["dY"], Ye, inv, w, want_dw=True, perm=perm)              # fused
    assert torch.equal(dYe_plain, dYe) and torch.equal(dw_plain, dw)
    extra = torch.randn_like(dYe, dtype=torch.float32).mul_(0.5).to(torch.bfloat16)
    dYe.add_(extra)                                                                          # in-place edit
    dXp, grads = layer.expert_bwd(dev["X"], dYe, offsets, perm)                              # flags = 0
    torch.cuda.synchronize()
    dYe_ref = to_np(dYe)
    dXp_ref, g_ref = oracle.expert_bwd(inp, dYe_ref, ref["G"], ref["U"], ref["H"], ref["offsets"], ref["perm"])
    assert_close("dXp", to_np(dXp), dXp_ref)
    for key in ("dA_gate", "dB_gate", "dA_up", "dB_up", "dA_down", "dB_down"):
        assert_close(key, to_np(grads[key]), g_ref[key])


@pytest.mark.parametrize("lora_scale,r", [(0.5, 16), (2.0, 32), (0.25, 8)])
def test_lora_scale_not_one_full_chain(lora_scale, r):
    """the whole chain including all six adapter gradients at lora_scale != 1 with adapters large
    enough (N(0, 0.1), as pin P7) that a dropped or doubled factor s in the forward, in dA / dB or in the adapter term of
    dX is far outside the tolerance (`tqp_layer_desc.lora_scale`)."""
    cfg = ti.Config(f"mid_ls{lora_scale}_r{r}", T=640, d=256, F=384, E=6, k=3, r=r, seed=24, router_grad=True, lora_scale=lora_scale)
    inp = _skewed(cfg)
    rng = np.random.default_rng(5)
    for key in ("A_gate", "B_gate", "A_up", "B_up", "A_down", "B_down"):
        inp[key] = ti.f32_to_bf16_bits(rng.standard_normal(inp[key].shape).astype(np.float32) * 0.1)
    gpu, ref = check_all(inp, backward=True, router_grad=True, gemm_impl=0)
    base = oracle.layer(dict(inp, lora_scale=0.0), dtype=np.float32, backward=False)["Y"]
    assert np.linalg.norm(ref["Y"] - base) > 0.3 * np.linalg.norm(base)      # the adapter term is a large part of Y
    one = oracle.layer(dict(inp, lora_scale=1.0), dtype=np.float32, backward=True, router_grad=True)
    for key in ("Y", "dX", "dA_gate", "dB_down"):                            # and s = 1 would be far outside the tolerance
        assert np.linalg.norm(one[key] - ref[key]) > 0.05 * np.linalg.norm(ref[key]), key


EDGE = [
    ti.Config("edge_T1", T=1, d=128, F=128, E=4, k=2, r=16, seed=31),   # 2 dot products: dtopk_w too ill-conditioned to compare
    ti.Config("edge_k_eq_E", T=37, d=256, F=128, E=4, k=4, r=16, seed=32, router_grad=True),
    ti.Config("edge_E1", T=50, d=128, F=256, E=1, k=1, r=32, seed=33, router_grad=True),
    ti.Config("edge_k1_many_empty", T=9, d=128, F=128, E=64, k=1, r=16, seed=34, router_grad=True),
    ti.Config("edge_max_E_k", T=96, d=128, F=128, E=1024, k=32, r=16, seed=35, router_grad=True),   # API maxima of E and k
]


@pytest.mark.parametrize("cfg", EDGE, ids=lambda c: c.name)
def test_degenerate_shapes(cfg):
    """A single token, k = E (every expert selected, softmax over all logits), one expert, and far more experts than
    assignments (most experts empty): full chain against the oracle."""
    inp = ti.make_inputs(cfg)
    check_all(inp, backward=True, router_grad=cfg.router_grad, gemm_impl=0)
