#!/usr/bin/env python
"""bench.py — expert-layer fwd+bwd throughput of the TQP routed-expert layer on B200 (BASELINE.json metric).

A "step" is one pass of the whole hot path (route -> dispatch -> expert_fwd -> combine ->
combine_bwd -> expert_bwd -> dispatch_bwd [-> route_bwd]) over one synthetic batch of the 120B-shaped config.

    python bench.py --gpus 1 --steps 20 --warmup 5            # our CUDA path (default workload: configs[2])
    python bench.py --impl reference --steps 3 --warmup 1     # the CPU oracle on a bounded sample (reference arm)
    torchrun ... bench.py --gpus N ...                        # N independent batches, no collective (weak scaling)

Prints ONE JSON line on rank 0.  Inputs are seeded synthetic tensors (tqp_inputs.py); they are far larger than L2
(code indices 452 MB + permuted rows 503 MB per step at configs[2]), so no explicit L2 flush is needed.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)
import tqp_inputs as ti  # noqa: E402

METRIC = "expert-layer fwd+bwd tokens/s (TQP routed-expert layer, 120B shape)"


def flops(cfg, T):
    """Algorithmic work of one fwd+bwd step; the avoided frozen-weight gradient is not counted."""
    N = T * cfg.k
    base = 12.0 * N * cfg.d * cfg.F                      # 3 packs x (fwd + dX) x 2 flop/MAC
    lora = 18.0 * N * cfg.r * (cfg.d + cfg.F)            # fwd, activation-grad, weight-grad of the adapters
    router = 2.0 * T * cfg.d * cfg.E
    gemm = base + 6.0 * N * cfg.r * (cfg.d + cfg.F)      # what the grouped-GEMM kernels themselves execute
    if not cfg.backward:                                 # forward-only config (configs[1]): half of the base, a third of the adapters
        base, lora, gemm = base / 2, lora / 3, gemm / 2
    return dict(total=base + lora + router, base=base, lora=lora, router=router, gemm=gemm)


# roofline.traffic is NOT measured by this run (ncu cannot run inside a timed bench): it is dram__bytes_read.sum +
# dram__bytes_write.sum per grouped-GEMM launch (average over the launches of one step) copied from the committed
# `ncu --set full` capture named beside it; None for workloads without a capture.
NCU_GEMM_TRAFFIC = {"cfg2_120b": (1.063e9, "profiles/r2_gemm_ncu.md"), "cfg3_120b_skew": (0.970e9, "profiles/r2_gemm_ncu.md"),
                    "cfg4_120b_mb": (1.925e9, "profiles/r2_gemm_ncu.md")}
GEMM_IMPL_NAMES = {0: "tcgen05 CTA pairs, weight operand in TMEM (gemm_tcgen05_ts2)", 1: "CUDA-core scaffold",
                   2: "tcgen05 one CTA per tile, smem weight operand", 3: "tcgen05 CTA pairs, smem weight operand"}


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        p = json.load(open(path))
        return dict(tensor_burst=p["bf16_tflops"], tensor_sustained=p["bf16_tflops_sustained"], hbm=p["hbm_gbs"],
                    source="measured (MEASURED_PEAKS.json)")
    return dict(tensor_burst=1590.0, tensor_sustained=1400.0, hbm=6650.0, source="fallback (B200_PROFILING.md)")


class ClockSampler(threading.Thread):
    """Samples SM clocks and throttle reasons while the timed region runs (NVML every ~5 ms; nvidia-smi as fallback)."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.mhz, self.reasons, self.max_mhz, self.stop_flag = index, [], set(), None, False
        self.nvml = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nvml = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self.nvml = None

    def _sample_nvml(self):
        n = self.nvml
        self.mhz.append(float(n.nvmlDeviceGetClockInfo(self.h, n.NVML_CLOCK_SM)))
        bits = n.nvmlDeviceGetCurrentClocksEventReasons(self.h) if hasattr(n, "nvmlDeviceGetCurrentClocksEventReasons") \
            else n.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
        table = {"hw_slowdown": 0x8, "sw_thermal_slowdown": 0x20, "hw_thermal_slowdown": 0x40, "sw_power_cap": 0x4}
        for name, bit in table.items():
            if bits & bit:
                self.reasons.add(name)

    def _sample_smi(self):
        out = subprocess.run(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits"],
                             capture_output=True, text=True, timeout=5).stdout
        r = [c.strip() for c in out.strip().split(",")]
        if len(r) == 6 and r[0].isdigit():
            self.mhz.append(float(r[0]))
            self.max_mhz = float(r[1])
            for i, name in enumerate(["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]):
                if r[2 + i] == "Active":
                    self.reasons.add(name)

    def run(self):
        while not self.stop_flag:
            try:
                if self.nvml is not None:
                    self._sample_nvml()
                    time.sleep(0.005)
                else:
                    self._sample_smi()
                    time.sleep(0.05)
            except Exception:
                time.sleep(0.05)

    def summary(self):
        if not self.mhz:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": [], "samples": 0}
        return {"sm_mhz": float(np.median(self.mhz)), "sm_min_mhz": float(min(self.mhz)), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.mhz),
                "source": "nvml" if self.nvml is not None else "nvidia-smi"}


def rank_config(cfg, rank):
    """Weak scaling: every rank owns an independent batch of the same shape (its own seed); no data-path collective."""
    import dataclasses
    return dataclasses.replace(cfg, seed=cfg.seed + 1000 * rank)


def max_over_ranks(ms, dist, device):
    """Device time of the slowest rank (the contract's 'max over ranks')."""
    if dist is None:
        return ms
    import torch
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(world, tokens_per_rank, steps, ms):
    return world * tokens_per_rank * steps / (ms / 1e3)


def oracle_step(inp, cfg):
    import oracle
    return oracle.layer(inp, dtype=np.float32, backward=True, router_grad=cfg.router_grad)


def time_oracle(cfg, T_sample, steps, warmup):
    import oracle
    oracle.build()
    inp = ti.make_inputs(cfg, T=T_sample)
    for _ in range(warmup):
        oracle_step(inp, cfg)
    t0 = time.perf_counter()
    for _ in range(steps):
        oracle_step(inp, cfg)
    dt = (time.perf_counter() - t0) / max(steps, 1)
    return dict(value=T_sample / dt, unit="tokens/s", cores=oracle.num_threads(), kind="oracle",
                sample=f"T={T_sample} of {cfg.T} tokens, all {cfg.E} experts (each dequantised once per pass), "
                       f"{'fwd+bwd' if cfg.backward else 'fwd+bwd (the GPU arm of this config is forward only)'}, fp32, "
                       f"{steps} step(s) of {dt:.2f} s",
                seconds_per_step=dt, gflops=flops(cfg, T_sample)["total"] / dt / 1e9)


def run_reference(args, cfg):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    T_s = args.ref_tokens
    cb = time_oracle(cfg, T_s, args.steps, args.warmup)
    line = {
        "impl": "reference", "metric": METRIC, "value": cb["value"], "unit": "tokens/s", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": cb["seconds_per_step"] * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": cfg.name, "T": cfg.T, "d": cfg.d, "F": cfg.F, "E": cfg.E, "k": cfg.k, "r": cfg.r,
                   "sample_tokens": T_s},
        "cpu_baseline": {k: cb[k] for k in ("value", "unit", "cores", "kind", "sample")},
        "e2e": {"value": cb["value"], "unit": "tokens/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def bind_tq_synthetic(tq, torch, layer, cfg, inp, up, dev):
    """--format tq: a TurboQuant base of the same shape.  Input recipe: rotation = signed
    Hadamard with seeded signs for power-of-two widths, else the library's sign-fixed QR of a seeded Gaussian draw; levels
    = the library's Lloyd-Max solver; codes drawn i.i.d. from the coordinate law (a N(0, 1/n) draw put into its Lloyd-Max
    cell -- what encoding Gaussian weight rows gives, without holding fp32 weights of 100B-scale packs); norms =
    0.02 sqrt(n) U(0.5, 1.5); adapters as in the vector-quantised recipe."""
    rng = np.random.default_rng(20_000 + cfg.seed)
    gen = torch.Generator(device=dev); gen.manual_seed(30_000 + cfg.seed)
    spaces = {}
    for n in {cfg.d, cfg.F}:
        lv = tq.tq_levels(n, 8)
        lvd = torch.from_numpy(lv).to(dev)
        if n & (n - 1) == 0:
            signs = torch.from_numpy((rng.integers(0, 2, n) * 2 - 1).astype(np.int8)).to(dev)
            spaces[n] = tq.TqSpace(n, lvd, signs=signs)
        else:
            R = tq.tq_rotation_qr(rng.standard_normal((n, n)))
            spaces[n] = tq.TqSpace(n, lvd, R=torch.from_numpy(R).to(dev))
        spaces[n].bounds = torch.from_numpy((0.5 * (lv[:-1] + lv[1:])).astype(np.float32)).to(dev)
    w = {}
    for pack, (out_dim, n) in dict(gate=(cfg.F, cfg.d), up=(cfg.F, cfg.d), down=(cfg.d, cfg.F)).items():
        codes = torch.empty((cfg.E, out_dim, n), dtype=torch.uint8, device=dev)
        for e0 in range(0, cfg.E, 16):
            y = torch.randn((min(16, cfg.E - e0), out_dim, n), generator=gen, device=dev) * (1.0 / np.sqrt(n))
            codes[e0:e0 + y.shape[0]] = torch.bucketize(y, spaces[n].bounds).to(torch.uint8)
        w[f"codes_{pack}"] = codes
        w[f"norm_{pack}"] = (torch.rand((cfg.E, out_dim), generator=gen, device=dev) + 0.5) * (0.02 * np.sqrt(n))
    for key in ("A_gate", "A_up", "B_gate", "B_up", "A_down", "B_down"):
        w[key] = up(inp[key])
    layer.bind_weights_tq(spaces[cfg.d], spaces[cfg.F], **w)
    return w, spaces


def run_ours(args, cfg):
    import torch
    import paper_2606_07404_b200 as tq

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local}"))
    dev = torch.device(f"cuda:{local}")
    torch.cuda.set_device(dev)

    # each rank owns an independent batch of the same shape (weak scaling, no data-path collective)
    inp = ti.make_inputs(rank_config(cfg, rank))
    T, k, d = cfg.T, cfg.k, cfg.d
    layer = tq.TqpLayer(T, cfg.d, cfg.F, cfg.E, cfg.k, cfg.r, lora_scale=cfg.lora_scale, training=True, device=str(dev))
    if args.gemm_impl:
        layer.set_option("gemm_impl", args.gemm_impl)
    if args.route_impl:
        layer.set_option("route_impl", args.route_impl)
    for kv in args.opt:   # any other library option (tqp_set_option), e.g. --opt fuse_dgu=0
        name, _, val = kv.partition("=")
        layer.set_option(name, int(val))

    def up(a):
        t = torch.from_numpy(a.view(np.int16)).view(torch.bfloat16) if a.dtype == np.uint16 else torch.from_numpy(a)
        return t.to(dev)

    wnames = ("idx_gate", "idx_up", "idx_down", "scale_gate", "scale_up", "scale_down", "codebook",
              "A_gate", "A_up", "B_gate", "B_up", "A_down", "B_down")
    if args.format == "tq":
        tq_keep = bind_tq_synthetic(tq, torch, layer, cfg, inp, up, dev)   # noqa: F841  (keeps the device tensors alive)
    else:
        layer.bind_weights(**{n: up(inp[n]) for n in wnames})
    X, dY, W_r = up(inp["X"]), up(inp["dY"]), up(inp["W_r"])
    bias = up(inp["logit_bias"]) if inp["logit_bias"] is not None else None
    N = T * k
    bf = torch.bfloat16
    Ye = torch.empty((N, d), dtype=bf, device=dev); dYe = torch.empty_like(Ye); dXp = torch.empty_like(Ye)
    Y = torch.empty((T, d), dtype=bf, device=dev); dX = torch.empty_like(Y)
    grads = layer.alloc_grads()
    launches = [0]

    def step():
        n = 0
        idx, w = layer.route(X, W_r, bias); n += layer.last_launch_count()
        counts, offsets, perm, inv = layer.dispatch(idx); n += layer.last_launch_count()
        layer.expert_fwd(X, offsets, perm, out=Ye); n += layer.last_launch_count()
        layer.combine(Ye, inv, w, out=Y); n += layer.last_launch_count()
        if not cfg.backward:
            launches[0] = n
            return
        _, dw = layer.combine_bwd(dY, Ye, inv, w, want_dw=cfg.router_grad, out=dYe, perm=perm); n += layer.last_launch_count()
        layer.expert_bwd(X, dYe, offsets, perm, grads=grads, out=dXp, dYe_unmodified=cfg.r in (16, 32)); n += layer.last_launch_count()
        layer.dispatch_bwd(dXp, inv, out=dX); n += layer.last_launch_count()
        if cfg.router_grad:
            layer.route_bwd(X, W_r, idx, w, dw, offsets, perm, dX); n += layer.last_launch_count()
        launches[0] = n

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        step()
    sampler = ClockSampler(local)
    barrier()
    sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(args.steps):
        step()
    e1.record()
    barrier()
    ms = e0.elapsed_time(e1)
    screened, fallback = layer.route_info()   # of the last timed step (outside the timed region: it synchronises)
    router_desc = ("screened: tcgen05 approximate logits + canonical fp32 chain for the candidates (bit-identical top-k)"
                   + (", FALLBACK to the dense chain taken" if fallback else "")) if screened else "dense canonical fp32 chain"
    # second pass of the same K steps with every grouped-GEMM launch bracketed by CUDA events on its own stream
    # (tqp_gemm_time); the headline time above carries no such events.  The clock sampler covers both passes.
    layer.set_option("time_gemm", 1)
    for _ in range(args.steps):
        step()
    barrier()
    sampler.stop_flag = True
    gemm_each = layer.gemm_times()
    gemm_ms, gemm_launches = float(sum(gemm_each)), len(gemm_each)
    layer.set_option("time_gemm", 0)
    ms = max_over_ranks(ms, dist, dev)
    ms_per_step = ms / args.steps
    value = whole_job_value(world, T, args.steps, ms)

    # ---- end to end through the C ABI with HOST buffers (H2D + whole chain + D2H inside the timed region) ----
    e2e = None
    if not args.no_e2e and cfg.backward:   # tqp_step_host runs forward + backward
        Xh = X.cpu().pin_memory(); dYh = dY.cpu().pin_memory()
        Yh = torch.empty((T, d), dtype=bf).pin_memory(); dXh = torch.empty((T, d), dtype=bf).pin_memory()
        dW_r = torch.empty((d, cfg.E), dtype=torch.float32, device=dev) if cfg.router_grad else None
        # Steps are issued through tqp_step_host_async with two in flight, the way a training loop with a prefetching data
        # loader calls it: the next step's X / dY upload travels under this step's kernels and this step's dX download
        # under the next forward pass.  Every step still copies its own inputs up and its own Y / dX down (separate pinned
        # output buffers per in-flight step); the timed region ends when the last step's outputs are on the host.
        Yh2 = torch.empty((T, d), dtype=bf).pin_memory(); dXh2 = torch.empty((T, d), dtype=bf).pin_memory()
        outs = [(Yh, dXh), (Yh2, dXh2)]
        for _ in range(min(args.warmup, 3)):
            layer.step_host(Xh, dYh, W_r, bias, Yh, dXh, grads, dW_r)
        barrier()
        t_host0 = time.perf_counter()
        e0.record()
        for i in range(args.steps):
            layer.step_host_async(Xh, dYh, W_r, bias, outs[i & 1][0], outs[i & 1][1], grads, dW_r)
            if i >= 1:
                layer.step_host_wait(1)
        layer.step_host_wait(0)
        e1.record()
        torch.cuda.synchronize()
        t_host1 = time.perf_counter()
        barrier()
        ems = max(e0.elapsed_time(e1), (t_host1 - t_host0) * 1e3)   # the copy streams are not torch's: the host clock bounds them
        ems = max_over_ranks(ems, dist, dev)
        nb = T * d * 2
        # the same loop with one blocking call per step (tqp_step_host), for comparison
        barrier()
        e0.record()
        for _ in range(args.steps):
            layer.step_host(Xh, dYh, W_r, bias, Yh, dXh, grads, dW_r)
        e1.record()
        barrier()
        sms = max_over_ranks(e0.elapsed_time(e1), dist, dev)
        e2e = {"value": whole_job_value(world, T, args.steps, ems), "unit": "tokens/s", "h2d_bytes_per_step": 2 * nb,
               "d2h_bytes_per_step": 2 * nb, "ms_per_step": ems / args.steps,
               "mode": "tqp_step_host_async, two steps in flight (copies of a step overlap its neighbours' kernels)",
               "blocking_call_value": whole_job_value(world, T, args.steps, sms), "blocking_call_ms_per_step": sms / args.steps}

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return
    fl = flops(cfg, T)
    pk = peaks()
    gemm_ms_step = gemm_ms / args.steps
    gemm_tflops = fl["gemm"] / (gemm_ms_step / 1e3) / 1e12 if gemm_ms_step > 0 else 0.0
    nl = 4 if cfg.backward else 2
    traffic = NCU_GEMM_TRAFFIC.get(cfg.name, (None, None)) if args.format == "vq" else (None, None)
    line = {
        "metric": METRIC, "value": value, "unit": "tokens/s", "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "bf16",
        "data": "synthetic",
        "config": {"workload": cfg.name + ("_tq" if args.format == "tq" else ""), "T": T, "d": cfg.d, "F": cfg.F, "E": cfg.E, "k": cfg.k, "r": cfg.r,
                   "passes": ("fwd+bwd" if cfg.backward else "fwd") + ("+router_grad" if cfg.router_grad else ""), "routing": "zipf1.1" if cfg.skew else "near-uniform",
                   "l2": f"inputs larger than L2 ({3 * cfg.E * cfg.d * cfg.F / 8 / 1e6:.0f} MB code indices + "
                         f"{T * cfg.k * cfg.d * 2 / 1e6:.0f} MB permuted rows per step), no flush",
                   "base_format": "TurboQuant-MSE 8-bit scalar codes + row norms, rotated space (PAPER.md L944-948)" if args.format == "tq"
                   else "vector-quantised, 8-vectors / 256-entry codebook / fp16 channel scales (BASELINE.json)",
                   "gemm_impl": GEMM_IMPL_NAMES.get(args.gemm_impl, str(args.gemm_impl)), "router": router_desc, "parallelism": f"replicas x{world}, no collective"},
        "tflops": world * fl["total"] / (ms_per_step / 1e3) / 1e12,
        "frac_of_bf16_peak": {"measured_burst": fl["total"] / (ms_per_step / 1e3) / 1e12 / pk["tensor_burst"],
                              "measured_sustained": fl["total"] / (ms_per_step / 1e3) / 1e12 / pk["tensor_sustained"],
                              "datasheet_2250": fl["total"] / (ms_per_step / 1e3) / 1e12 / 2250.0},
        "clocks": sampler.summary(),
        "e2e": e2e,
        "gpu_launches": launches[0] * args.steps,
        # the primary denominator is the MEASURED BURST bf16 peak; sustained and datasheet beside it
        "roofline": {"kernel": "grouped dequant GEMM gemm_tcgen05_ts2_kernel (4 launches/step: gate+up, down, dH, dXp)", "bound": "tensor",
                     "achieved": gemm_tflops, "peak": pk["tensor_burst"], "unit": "TFLOP/s",
                     "frac": gemm_tflops / pk["tensor_burst"], "frac_of_sustained": gemm_tflops / pk["tensor_sustained"],
                     "frac_of_datasheet_2250": gemm_tflops / 2250.0, "peak_source": pk["source"] + ", burst bf16 (bf16_tflops)",
                     "gemm_ms_per_step": gemm_ms_step, "gemm_share_of_step": gemm_ms_step / ms_per_step,
                     "gemm_launches": gemm_launches, "flops_per_step": fl["gemm"],
                     "flops_per_launch": fl["gemm"] / (4.0 if cfg.backward else 2.0),
                     "launch_ms": [float(np.mean(gemm_each[i::nl])) for i in range(nl)] if gemm_each else [],
                     "traffic": traffic[0], "traffic_source": traffic[1]},
    }
    if world == 1 and not args.no_cpu_baseline:
        # one full oracle pass over the workload's own batch where that takes about a minute; capped at
        # 8192 tokens (cfg 4 would need ~2 min); --cpu-tokens overrides
        cb = time_oracle(cfg, args.cpu_tokens if args.cpu_tokens > 0 else min(cfg.T, 8192), 1, 0)
        line["cpu_baseline"] = {k: cb[k] for k in ("value", "unit", "cores", "kind", "sample")}
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=2, help="index into BASELINE.json configs (2 = 120B shape, fwd+bwd)")
    ap.add_argument("--gemm-impl", type=int, default=0)
    ap.add_argument("--opt", action="append", default=[], metavar="NAME=INT", help="library option passed to tqp_set_option (repeatable)")
    ap.add_argument("--route-impl", type=int, default=0, help="0 library's choice, 1 dense fp32 chain, 2 screened router (see tqp_route_info)")
    ap.add_argument("--format", default="vq", choices=["vq", "tq"], help="frozen-base format: BASELINE.json's VQ (default) or TurboQuant-MSE")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-tokens", type=int, default=0, help="tokens of the cpu_baseline oracle pass (0: the whole batch, at most 8192)")
    ap.add_argument("--ref-tokens", type=int, default=256, help="tokens per step of the --impl reference arm")
    args = ap.parse_args()
    cfg = ti.CONFIGS[args.config]
    if args.impl == "reference":
        run_reference(args, cfg)
    else:
        run_ours(args, cfg)


if __name__ == "__main__":
    main()
