#!/usr/bin/env python
"""bench.py -- MoE layer fwd+bwd throughput on B200 through the C ABI (BASELINE.json metric).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config NAME] [--impl reference]

One "step" = moe_layer_fwd + moe_layer_bwd (every row of SURVEY.md §8a) over one batch of synthetic input.
Prints ONE JSON line (rank 0).  `value` = algorithmic TFLOP/s (18*T*K*H*F + shared + router flops, S20)
with inputs resident in HBM; `e2e` = the same through moe_layer_step_host with pinned HOST activations
(H2D of X, dY and D2H of Y, dX inside the timed region).  Multi-GPU: replicas only: each rank
runs the same layer on its own batch, no data-path collective, weak scaling.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

import workloads as wl  # noqa: E402

METRIC = "moe_layer_fwd_bwd_tflops"
UNIT = "TFLOP/s"
NOMINAL = {"bf16_tflops": 2250.0, "hbm_gbs": 8000.0}
NOMINAL_FP8_OVER_BF16 = 2.0   # B200_PROFILING.md: 4.5 vs 2.25 PFLOP/s dense; the fp8 peak is ASSUMED = measured bf16 x 2


def load_traffic(workload):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of each stage's kernel, read from profiles/traffic.json
    (written by `python ncu_summary.py` from an `ncu --set full` capture; it names the capture).
    Returns ({stage: bytes}, source string) or ({}, None) when no capture of this workload is tracked."""
    path = os.path.join(ROOT, "profiles", "traffic.json")
    try:
        rec = json.load(open(path)).get(workload)
    except (OSError, ValueError):
        rec = None
    if not rec:
        return {}, None
    return rec.get("stages", {}), rec.get("source")


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        p = json.load(open(path))
        return {"hbm_gbs": p["hbm_gbs"], "bf16_burst": p["bf16_tflops"], "bf16_sustained": p["bf16_tflops_sustained"],
                "source": "measured (MEASURED_PEAKS.json)"}
    return {"hbm_gbs": 6650.0, "bf16_burst": 1590.0, "bf16_sustained": 1400.0, "source": "fallback (B200_PROFILING.md)"}


def pick_config(name):
    cfg = wl.CONFIGS.get(name) or wl.SMALL_CONFIGS.get(name)
    if cfg is None:
        raise SystemExit(f"unknown config {name}; have {sorted(wl.CONFIGS) + sorted(wl.SMALL_CONFIGS)}")
    if cfg.dtype != wl.DTYPE_FP32:
        cfg = cfg.replace(row_align=int(os.environ.get("MOE_BENCH_ROW_ALIGN", "128")))   # tensor-core path: expert groups start at multiples of 128 rows
    return cfg


# ----------------------------------------------------------------------------------------------------
# the oracle leg (cpu_baseline and --impl reference): a bounded sample of the same workload
# ----------------------------------------------------------------------------------------------------

def oracle_sample(cfg, budget_s=15.0, max_experts=None):
    """Oracle routing over all T tokens, then the oracle's expert FFN fwd+bwd (fp64) for experts 0..n-1 on the
    rows routed to them, until `budget_s` of CPU time is spent.  Returns (flops, seconds, description)."""
    from oracle import moe_oracle as orc
    X, Wr, bias, dY = wl.gen_X(cfg), wl.gen_Wr(cfg), wl.gen_bias(cfg), wl.gen_dY(cfg)
    t0 = time.perf_counter()
    z = orc.router_logits(X, Wr)
    idx, w = orc.route(z, bias, cfg)
    counts, offsets, p2f, f2p = orc.permute_maps(idx, cfg.E, 1)
    Xp = orc.permute_rows(X, p2f, cfg.K)
    t_route = time.perf_counter() - t0
    flops = 2.0 * cfg.T * cfg.H * cfg.E
    spent, n, rows = t_route, 0, 0
    for e in range(cfg.E if max_experts is None else min(cfg.E, max_experts)):
        Wg, Wu, Wd = wl.gen_expert_weights(cfg, e)            # generation is not timed
        r0, r1 = int(offsets[e]), int(offsets[e]) + int(counts[e])
        if r1 == r0:
            continue
        t0 = time.perf_counter()
        g, u, a, y = orc.expert_ffn_fwd(Xp[r0:r1], Wg, Wu, Wd)
        tok = p2f[r0:r1] // cfg.K
        dy = dY[tok].astype(np.float64) * w.reshape(-1)[p2f[r0:r1]][:, None]
        orc.expert_ffn_bwd(dy, Xp[r0:r1], g, u, a, Wg, Wu, Wd)
        spent += time.perf_counter() - t0
        flops += 18.0 * (r1 - r0) * cfg.H * cfg.F
        n += 1
        rows += r1 - r0
        if spent > budget_s:
            break
    return flops, spent, f"oracle routing of all {cfg.T} tokens + expert FFN fwd+bwd (fp64) of experts 0..{n - 1} ({rows} routed rows)"


def blas_threads():
    try:
        from threadpoolctl import threadpool_info
        return max([i.get("num_threads", 1) for i in threadpool_info()] or [os.cpu_count()])
    except Exception:
        return os.cpu_count()


def run_reference(args, cfg):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    for _ in range(max(0, min(args.warmup, 1))):
        oracle_sample(cfg, budget_s=1.0, max_experts=1)
    budget = max(2.0, min(12.0, 120.0 / max(1, args.steps)))
    tot_f = tot_t = 0.0
    desc = ""
    for _ in range(args.steps):
        f, t, desc = oracle_sample(cfg, budget_s=budget)
        tot_f += f
        tot_t += t
    val = tot_f / tot_t / 1e12
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": tot_t / args.steps * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": cfg.name, "T": cfg.T, "H": cfg.H, "E": cfg.E, "K": cfg.K, "F": cfg.F},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": blas_threads(), "kind": "oracle", "sample": desc},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))


# ----------------------------------------------------------------------------------------------------
# the CUDA arm
# ----------------------------------------------------------------------------------------------------

class ClockSampler(threading.Thread):
    """Samples SM clock, power and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index, period=0.01):
        super().__init__(daemon=True)
        self.period, self.samples, self.reasons, self.stop_flag = period, [], set(), False
        self.max_mhz, self.power = None, []
        try:
            import pynvml as nv
            nv.nvmlInit()
            self.nv, self.h = nv, nv.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = nv.nvmlDeviceGetMaxClockInfo(self.h, nv.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def run(self):
        if self.nv is None:
            return
        nv = self.nv
        names = {"hw_slowdown": 0x8, "sw_power_cap": 0x4, "hw_thermal_slowdown": 0x40, "sw_thermal_slowdown": 0x20,
                 "hw_power_brake_slowdown": 0x80}
        while not self.stop_flag:
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                self.power.append(nv.nvmlDeviceGetPowerUsage(self.h) / 1000.0)
                r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            time.sleep(self.period)

    def result(self):
        s = sorted(self.samples)
        return {"sm_mhz": (s[len(s) // 2] if s else None), "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(s), "power_w_max": (max(self.power) if self.power else None)}


def max_over_ranks(ms, world, device="cuda"):
    """Replicas only: the job's step time is the slowest replica's."""
    if world <= 1:
        return ms
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def replica_seed(cfg, rank):
    """Each replica runs the same layer on its own batch."""
    return cfg.replace(seed=cfg.seed + rank)


def stage_flops(cfg):
    """Algorithmic flops per stage per step (S20)."""
    r = cfg.T * cfg.K * cfg.H * cfg.F
    s = cfg.T * cfg.H * cfg.F_shared
    return {"gemm1_swiglu": 4 * r, "gemm2": 2 * r, "dgrad_down_swiglu": 2 * r, "dgrad_gateup": 4 * r, "wgrad": 6 * r,
            "shared_fwd": 6 * s, "shared_bwd": 12 * s, "router_gemm": 2 * cfg.T * cfg.H * cfg.E}


def stage_bytes(cfg):
    """Algorithmic HBM bytes per stage per step: every operand read once, every result written once.
    GEMM stages: activations at 2 bytes (fp8 fprop/dgrad operands at 1 byte + fp32 scales), weights once per step."""
    b = 4 if cfg.dtype == wl.DTYPE_FP32 else 2
    T, H, E, K, F, TK = cfg.T, cfg.H, cfg.E, cfg.K, cfg.F, cfg.T * cfg.K
    fp8 = cfg.dtype == wl.DTYPE_FP8
    ab = 1 if fp8 else b                       # bytes per element of an fprop / dgrad GEMM operand
    sc = (lambda rows, cols: rows * (cols // 128) * 4) if fp8 else (lambda rows, cols: 0)
    W = E * H * F
    return {"route": T * E * 4 + TK * 8, "maps": 3 * TK * 4, "permute": T * H * b + TK * H * b + TK * 4,
            "combine": TK * H * b + T * H * b + TK * 8, "combine_bwd": 2 * TK * H * b + T * H * b + TK * 12,
            "dx_combine": TK * H * b + T * H * b + TK * 4,
            "gemm1_swiglu": TK * H * ab + sc(TK, H) + 2 * W * ab + TK * 3 * F * b,      # Xp, Wg, Wu -> gu, a
            "gemm2": TK * F * ab + sc(TK, F) + W * ab + TK * H * b,                      # a, Wd -> y
            "dgrad_down_swiglu": TK * H * ab + sc(TK, H) + W * ab + TK * 2 * F * b + TK * 2 * F * b,   # dy, Wd, gu -> dgu
            "dgrad_gateup": TK * 2 * F * ab + sc(TK, 2 * F) + 2 * W * ab + TK * H * b,   # dgu, Wg, Wu -> dXp
            "wgrad": TK * (2 * H + 3 * F) * b + 3 * W * b}                               # dy, a, dgu, Xp -> dWd, dWg, dWu


def roof(flops, byts, sec, peak_tflops, peak_gbs):
    """Roofline of one stage: which roof binds (the larger of flops/peak and bytes/peak) and the achieved fraction of it."""
    t_tensor, t_hbm = flops / (peak_tflops * 1e12), byts / (peak_gbs * 1e9)
    bound = "tensor" if t_tensor >= t_hbm else "hbm"
    return bound, max(t_tensor, t_hbm) / sec


def time_standalone_movers(moe, lb, cfg, stream, iters=20):
    """"the standalone moe_permute / moe_unpermute_combine are what the GB/s metric measures even if
    moe_layer_fwd fuses the gather".  moe_route + moe_permute (histogram, scan, maps, row gather) from the layer's logits,
    and moe_unpermute_combine on the result, each timed per call with CUDA events on the launching stream; a 512 MB
    buffer is overwritten between calls (outside the events) so that every call starts with a cold L2."""
    import torch
    b = 4 if cfg.dtype == wl.DTYPE_FP32 else 2
    T, H, E, K, TK = cfg.T, cfg.H, cfg.E, cfg.K, cfg.T * cfg.K
    R = lb.R
    z = lb.ctx_view("z").clone()
    i32 = lambda *sh: torch.empty(*sh, dtype=torch.int32, device="cuda")
    idx, w = i32(T, K), torch.empty(T, K, dtype=torch.float32, device="cuda")
    counts, offsets, p2f, f2p = i32(E), i32(E + 1), i32(R), i32(TK)
    Xp = torch.empty(R, H, dtype=lb.X.dtype, device="cuda")
    Y = torch.empty_like(lb.X)
    flush = torch.empty(512 << 20, dtype=torch.uint8, device="cuda")
    def rp():
        moe.moe_route(lb.ccfg, z, lb.bias, idx, w, stream)
        moe.moe_permute(lb.ccfg, lb.X, idx, counts, offsets, p2f, f2p, Xp, lb.ws, stream)

    def cb():
        moe.moe_unpermute_combine(lb.ccfg, Xp, w, f2p, None, Y, stream)

    rp(); cb()
    torch.cuda.synchronize()
    # each call sequence is captured once and replayed, so the six small launches of route + permute are not separated
    # by host launch gaps (the layer itself is timed the same way)
    g_rp, g_cb = torch.cuda.CUDAGraph(), torch.cuda.CUDAGraph()
    with torch.cuda.graph(g_rp):
        moe.moe_route(lb.ccfg, z, lb.bias, idx, w)
        moe.moe_permute(lb.ccfg, lb.X, idx, counts, offsets, p2f, f2p, Xp, lb.ws)
    with torch.cuda.graph(g_cb):
        moe.moe_unpermute_combine(lb.ccfg, Xp, w, f2p, None, Y)
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(4)]
    t_rp, t_c = [], []
    for it in range(iters + 3):
        flush.fill_(it & 0xff)
        ev[0].record(stream)
        g_rp.replay()
        ev[1].record(stream)
        flush.fill_(it & 0xff)
        ev[2].record(stream)
        g_cb.replay()
        ev[3].record(stream)
        torch.cuda.synchronize()
        if it >= 3:
            t_rp.append(ev[0].elapsed_time(ev[1]))
            t_c.append(ev[2].elapsed_time(ev[3]))
    sb = stage_bytes(cfg)
    med = lambda v: sorted(v)[len(v) // 2]
    rp_bytes = sb["route"] + sb["maps"] + sb["permute"]
    return {"route_permute": {"gbs": rp_bytes / (med(t_rp) * 1e-3) / 1e9, "bytes": rp_bytes, "ms": med(t_rp),
                              "calls": "moe_route + moe_permute, stand-alone (CUDA-graph replay), cold L2, median of %d" % iters},
            "combine": {"gbs": sb["combine"] / (med(t_c) * 1e-3) / 1e9, "bytes": sb["combine"], "ms": med(t_c),
                        "calls": "moe_unpermute_combine, stand-alone (CUDA-graph replay), cold L2, median of %d" % iters}}


def run_cuda(args, cfg):
    import torch
    import torch.distributed as dist
    import paper_2605_31463_b200 as moe
    from paper_2605_31463_b200.buffers import LayerBuffers, act_dtype, to_device
    moe.lib()
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    peaks = load_peaks()
    dt = act_dtype(cfg)
    cfg_r = replica_seed(cfg, rank)
    lb = LayerBuffers(cfg)
    lb.load(X=wl.gen_X(cfg_r), dY=wl.gen_dY(cfg_r), Wr=wl.gen_Wr(cfg), bias=wl.gen_bias(cfg))
    g = torch.Generator(device="cuda").manual_seed(1234)
    std = cfg.w_std if cfg.w_std > 0 else None
    for w, fan_in in ((lb.Wg, cfg.H), (lb.Wu, cfg.H), (lb.Wd, cfg.F), (lb.Wg_s, cfg.H), (lb.Wu_s, cfg.H), (lb.Wd_s, cfg.F_shared)):
        if w is None:
            continue
        for e in range(w.shape[0] if w.dim() == 3 else 1):   # expert by expert: bounded fp32 temporaries
            dst = w[e] if w.dim() == 3 else w
            dst.copy_(torch.randn(dst.shape, generator=g, device="cuda", dtype=torch.float32) * (std or fan_in ** -0.5))
    stream = torch.cuda.current_stream()

    def sync_all():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    cached = bool(args.fp8_weight_cache) and cfg.dtype == wl.DTYPE_FP8
    if cached:     # PAPER.md:116 FP8 weight cache: quantise once (outside the timed region), reuse for every micro-batch
        moe.moe_fp8_quantize_weights(lb.ccfg, lb.Wg, lb.Wu, lb.Wd, lb.Wg_s, lb.Wu_s, lb.Wd_s, lb.ctx, stream)

    def fwd(st=None):
        if cached:
            moe.moe_layer_fwd(lb.ccfg, lb.X, lb.Wr, lb.bias, None, None, None, None, None, None, lb.Y, lb.topk_idx,
                              lb.topk_w, lb.ctx, lb.ws, st)
        else:
            lb.forward(st)

    def step():
        fwd(stream)
        lb.backward(stream)

    for _ in range(max(3, args.warmup)):
        step()
    sync_all()
    # ---- eager pass with the library's stage events on (stage table, launch count) ----
    moe.moe_profile_enable(True)
    n0 = moe.moe_launch_count()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    sync_all()
    ev0.record(stream)
    for _ in range(args.steps):
        step()
    ev1.record(stream)
    sync_all()
    launches = moe.moe_launch_count() - n0
    ms_eager = ev0.elapsed_time(ev1)
    stages = {}
    for name in moe.STAGES:
        t, n = moe.moe_profile_stage_ms(name)
        if n:
            stages[name] = {"ms_per_step": t / args.steps, "segments_per_step": n / args.steps}
    moe.moe_profile_enable(False)
    # ---- timed region: the same step captured once into a CUDA graph (the library never synchronises or allocates,
    # so fwd+bwd is capturable as is) and replayed K times; --no-graph times the eager launches instead ----
    graph = None
    if not args.no_graph:
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph):
            fwd()
            lb.backward()
        for _ in range(3):
            graph.replay()
        sync_all()
    sampler = ClockSampler(local)
    sampler.start()
    sync_all()
    ev0.record(stream)
    for _ in range(args.steps):
        if graph is not None:
            graph.replay()
        else:
            step()
    ev1.record(stream)
    sync_all()
    sampler.stop_flag = True
    ms = ev0.elapsed_time(ev1)
    ms = max_over_ranks(ms, world)
    fl = cfg.flops_fwd_bwd()
    value = world * fl["total"] * args.steps / (ms * 1e-3) / 1e12

    # ---- end to end: host activations in, host results out, copies inside the timed region ----
    # moe_layer_step_host_pipelined: copy-in, compute and copy-out on three streams, two sets of staging buffers, so
    # the PCIe copies of neighbouring steps overlap the compute; every step still moves its own inputs and results.
    n_host = 2
    Xh = [lb.X.cpu().pin_memory() for _ in range(n_host)]
    dYh = [lb.dY.cpu().pin_memory() for _ in range(n_host)]
    Yh = [torch.empty_like(Xh[0]).pin_memory() for _ in range(n_host)]
    dXh = [torch.empty_like(Xh[0]).pin_memory() for _ in range(n_host)]
    lb.make_pipeline()
    s_in, s_comp, s_out = lb.streams
    saved_w = (lb.Wg, lb.Wu, lb.Wd, lb.Wg_s, lb.Wu_s, lb.Wd_s)
    if cached:      # the host steps reuse the cached e4m3 weight codes too (NULL weights = "use the codes in ctx")
        lb.Wg = lb.Wu = lb.Wd = lb.Wg_s = lb.Wu_s = lb.Wd_s = None

    def host_steps(n, first=0):
        for i in range(first, first + n):
            lb.step_host_pipelined(i, Xh[i % n_host], dYh[i % n_host], Yh[i % n_host], dXh[i % n_host])

    host_steps(4)
    sync_all()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(s_in)
    host_steps(args.steps)
    s_out.wait_stream(s_comp)
    s_out.wait_stream(s_in)
    e1.record(s_out)
    sync_all()
    ms_e2e = max_over_ranks(e0.elapsed_time(e1), world)
    # serial variant (one stream: copy in, compute, copy out), for comparison
    for _ in range(2):
        lb.step_host(Xh[0], dYh[0], Yh[0], dXh[0], stream)
    sync_all()
    e0.record(stream)
    for _ in range(args.steps):
        lb.step_host(Xh[0], dYh[0], Yh[0], dXh[0], stream)
    e1.record(stream)
    sync_all()
    ms_serial = max_over_ranks(e0.elapsed_time(e1), world)
    lb.close_pipeline()
    lb.Wg, lb.Wu, lb.Wd, lb.Wg_s, lb.Wu_s, lb.Wd_s = saved_w
    act_bytes = cfg.T * cfg.H * (4 if cfg.dtype == wl.DTYPE_FP32 else 2)
    e2e = {"value": world * fl["total"] * args.steps / (ms_e2e * 1e-3) / 1e12, "unit": UNIT,
           "h2d_bytes_per_step": 2 * act_bytes, "d2h_bytes_per_step": 2 * act_bytes, "ms_per_step": ms_e2e / args.steps,
           "api": "moe_layer_step_host_pipelined (3 streams, 2 staging slots, pinned host buffers, caller-owned pipeline object)",
           "serial_value": world * fl["total"] * args.steps / (ms_serial * 1e-3) / 1e12,
           "serial_ms_per_step": ms_serial / args.steps}

    standalone = time_standalone_movers(moe, lb, cfg, stream) if rank == 0 else None
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    # ---- stage table: TFLOP/s for the GEMMs, GB/s for the HBM-bound movers ----
    # Which bf16 peak applies is decided from the evidence of THIS run (B200_PROFILING.md: burst for a kernel timed
    # alone or in a short region at full clock, sustained for seconds-long loops under the power cap): a timed region
    # shorter than 1 s, or a sampled median SM clock above 0.9 x max, is the burst regime.  Both fractions are printed.
    clocks = sampler.result()
    burst = (ms * 1e-3 < 1.0) or bool(clocks["sm_mhz"] and clocks["sm_max_mhz"] and clocks["sm_mhz"] > 0.9 * clocks["sm_max_mhz"])
    regime = "burst" if burst else "sustained"
    bf16_peak = peaks["bf16_burst"] if burst else peaks["bf16_sustained"]
    sf, sb = stage_flops(cfg), stage_bytes(cfg)
    if lb.rows_fused == 1:     # the combine-bwd slot holds a plain gather of dY (+ the dw reduction): permute's bytes
        sb["combine_bwd"] = sb["permute"]
    elif lb.rows_fused == 2:   # no permute / combine-bwd pass inside the layer: the slots hold only the dw reduction
        sb.pop("permute"); sb.pop("combine_bwd")
    traffic, traffic_src = load_traffic(cfg.name)
    gemm_names = ("gemm1_swiglu", "gemm2", "dgrad_down_swiglu", "dgrad_gateup", "wgrad")

    def stage_peak(name):          # fprop and dgrad of an fp8 config run on e4m3 codes, its wgrad on bf16
        fp8_stage = cfg.dtype == wl.DTYPE_FP8 and name in gemm_names and name != "wgrad"
        return bf16_peak * (NOMINAL_FP8_OVER_BF16 if fp8_stage else 1.0)

    for name, st in stages.items():
        sec = st["ms_per_step"] * 1e-3
        if name in sf and sf[name] and sec > 0:
            st["tflops"] = sf[name] / sec / 1e12
            mult = stage_peak(name) / bf16_peak
            st["frac_measured_burst"] = st["tflops"] / (peaks["bf16_burst"] * mult)
            st["frac_measured_sustained"] = st["tflops"] / (peaks["bf16_sustained"] * mult)
            st["frac_nominal"] = st["tflops"] / (NOMINAL["bf16_tflops"] * mult)
        if name in sb and sec > 0:
            st["gbs"] = sb[name] / sec / 1e9
            st["frac_measured_hbm"] = st["gbs"] / peaks["hbm_gbs"]
            st["frac_nominal_hbm"] = st["gbs"] / NOMINAL["hbm_gbs"]
        if name in sf and name in sb and sf[name] and sec > 0:
            st["bound"], st["frac_of_binding_roof"] = roof(sf[name], sb[name], sec, stage_peak(name), peaks["hbm_gbs"])
    gemm_stages = [n for n in gemm_names if n in stages]
    roofline = gemm_all = None
    if gemm_stages:
        # the dominant kernel = the GEMM stage with the most time; its roof is whichever of tensor / hbm binds (SURVEY.md
        # §8d: configs[2], [3] stream 22.5 / 11.3 GB of weights per pass and are HBM-bound; configs[1], [4] tensor-bound)
        dom = max(gemm_stages, key=lambda n: stages[n]["ms_per_step"])
        st = stages[dom]
        nl = 3 if dom == "wgrad" else 1
        sec = st["ms_per_step"] * 1e-3
        if cfg.dtype == wl.DTYPE_FP32:
            roofline = {"bound": "alu", "kernel": dom, "achieved": st.get("tflops"), "peak": None, "unit": "TFLOP/s", "frac": None,
                        "traffic": None, "note": "configs[0] runs the fp32 CUDA-core path (parity case, not a bench workload)"}
        else:
            bound, frac = roof(sf[dom], sb[dom], sec, stage_peak(dom), peaks["hbm_gbs"])
            tensor = bound == "tensor"
            roofline = {"bound": bound, "kernel": dom,
                        "achieved": st["tflops"] if tensor else st["gbs"],
                        "peak": stage_peak(dom) if tensor else peaks["hbm_gbs"], "unit": "TFLOP/s" if tensor else "GB/s",
                        "frac": frac, "traffic": traffic.get(dom), "traffic_unit": "bytes per launch (ncu dram read+write)",
                        "traffic_source": traffic_src,
                        "algorithmic_flops_per_launch": sf[dom] / nl, "algorithmic_bytes_per_launch": sb[dom] / nl,
                        "launches_per_step": nl, "ms_per_launch": st["ms_per_step"] / nl,
                        "peak_regime": regime, "peak_source": peaks["source"] + f", {regime} bf16"
                        + (" x 2 (assumed fp8:bf16 ratio, not measured)" if stage_peak(dom) != bf16_peak else ""),
                        "frac_tensor_burst": st["frac_measured_burst"], "frac_tensor_sustained": st["frac_measured_sustained"],
                        "frac_tensor_nominal": st["frac_nominal"], "frac_hbm_measured": st["frac_measured_hbm"]}
            if dom == "wgrad":   # dWg and dWu are two launches that each read Xp: bytes as launched, beside the algorithmic minimum
                b_ = 2
                roofline["bytes_per_launch_as_launched"] = (sb[dom] + cfg.T * cfg.K * cfg.H * b_) / nl
        # the aggregate the north_star's ">= 60 % of dense bf16 peak for the grouped GEMMs" is quoted on
        tsec = sum(stages[n]["ms_per_step"] for n in gemm_stages) * 1e-3
        tfl = sum(sf[n] for n in gemm_stages)
        if tsec > 0:
            gemm_all = {"flops": tfl, "ms": tsec * 1e3, "tflops": tfl / tsec / 1e12,
                        "frac_measured_burst": tfl / tsec / 1e12 / peaks["bf16_burst"],
                        "frac_measured_sustained": tfl / tsec / 1e12 / peaks["bf16_sustained"],
                        "frac_nominal_2250": tfl / tsec / 1e12 / NOMINAL["bf16_tflops"], "stages": gemm_stages,
                        "note": "bf16 denominators; an fp8 config's fprop/dgrad stages have twice that peak"}
    for k in ("route_permute", "combine"):
        standalone[k]["frac_measured"] = standalone[k]["gbs"] / peaks["hbm_gbs"]
        standalone[k]["frac_nominal_8000"] = standalone[k]["gbs"] / NOMINAL["hbm_gbs"]
    if roofline is not None:
        # BASELINE.json's metric has two halves (fwd+bwd TFLOP/s; route+permute GB/s) and north_star's 60 % target is quoted
        # on the GEMMs together: all of it sits INSIDE the roofline object, which is the part of the line the driver keeps
        roofline["gemm_all"] = gemm_all
        roofline["movers"] = {"route_permute": standalone["route_permute"], "combine": standalone["combine"]}
    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        f, t, desc = oracle_sample(cfg)
        cpu = {"value": f / t / 1e12, "unit": UNIT, "cores": blas_threads(), "kind": "oracle", "sample": desc,
               "seconds": t}
    from paper_2605_31463_b200 import build as _b
    build_id = _b.build_id()
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(3, args.warmup),
            "ms_per_step": ms / args.steps, "ms_per_step_eager": ms_eager / args.steps,
            "launch": "eager" if args.no_graph else "cuda_graph replay of fwd+bwd", "fp8_weight_cache": cached, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": {0: "f32", 1: "bf16", 2: "fp8_e4m3"}[cfg.dtype], "data": "synthetic",
            "config": {"workload": cfg.name, "T": cfg.T, "H": cfg.H, "E": cfg.E, "K": cfg.K, "F": cfg.F,
                       "F_shared": cfg.F_shared, "row_align": cfg.row_align, "parallelism": f"replicas x{world}",
                       "l2": "not flushed: each step streams > 1 GB of weights and activations, larger than the 126 MB L2",
                       "inputs": "X, dY, Wr, bias from workloads (Philox, seed 0); expert weights torch.randn on device"},
            "flops_per_step": fl, "frac_of_measured_bf16_burst": value / world / peaks["bf16_burst"],
            "frac_of_measured_bf16_sustained": value / world / peaks["bf16_sustained"],
            "frac_of_nominal_bf16_2250": value / world / NOMINAL["bf16_tflops"],
            "clocks": clocks, "e2e": e2e, "gpu_launches": launches, "roofline": roofline,
            "rows_fused": int(lb.rows_fused), "build": build_id, "stages": stages, "cpu_baseline": cpu, "peaks": peaks}
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--config", default="qwen3_30b_a3b_like")
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--fp8-weight-cache", action="store_true",
                    help="fp8 configs: quantise the weights once before the timed region and reuse the codes")
    ap.add_argument("--no-graph", action="store_true", help="time eager launches instead of CUDA-graph replays")
    args = ap.parse_args()
    cfg = pick_config(args.config)
    if args.impl == "reference":
        run_reference(args, cfg)
    else:
        run_cuda(args, cfg)


if __name__ == "__main__":
    main()
