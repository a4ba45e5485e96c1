"""`-m gpu` parity of moe_layer_fwd / moe_layer_bwd (through the C ABI) against the fp64 oracle, element
by element, on configs[0] and on scaled-down copies of configs[1..4] that still span several 128-row
tiles, ragged tails and empty experts; plus the host-buffer step.  Tolerances: BASELINE.json:north_star
(fp32 1e-5 router / tiny, bf16 1e-2, fp8 3e-2 relative Frobenius, S19)."""
import numpy as np
import pytest

import gpu_common as gc
import workloads as wl
from oracle import moe_oracle as orc

pytestmark = pytest.mark.gpu

LAYER_CASES = [
    wl.TINY,
    wl.TINY.replace(name="tiny_align128", row_align=128),
    wl.QWEN3_SMALL,
    wl.QWEN3_SMALL.replace(name="qwen3_small_align128", row_align=128),
    wl.DSV3_SMALL.replace(name="dsv3_small_align128", row_align=128),
    wl.GPTOSS_SMALL.replace(name="gptoss_small_align128", row_align=128),
    wl.TINY.replace(name="tiny_bf16_align128", dtype=wl.DTYPE_BF16, row_align=128),
    wl.QWEN3_SMALL.replace(name="one_token", T=1, row_align=128),
    # degenerate routings: a single expert (every token, weight 1), top-1 of two, and K = E (every expert for every token)
    wl.TINY.replace(name="tiny_one_expert", E=1, K=1),
    wl.QWEN3_SMALL.replace(name="top1_of_two", E=2, K=1, row_align=128),
    wl.QWEN3_SMALL.replace(name="all_experts", T=300, E=4, K=4, row_align=128),
]


@pytest.mark.parametrize("cfg", LAYER_CASES, ids=lambda c: c.name)
def test_layer_fwd_bwd_matches_oracle(cfg):
    inp = gc.gen_inputs(cfg)
    lb = gc.run_gpu_layer(cfg, inp)
    errs = gc.compare_layer(cfg, inp, lb)
    print(cfg.name, {k: (f"{v:.2e}" if isinstance(v, float) else v) for k, v in errs.items()})


def test_layer_is_deterministic():
    import torch
    cfg = wl.QWEN3_SMALL.replace(row_align=128)
    inp = gc.gen_inputs(cfg)
    a = gc.run_gpu_layer(cfg, inp)
    b = gc.run_gpu_layer(cfg, inp)
    for name in ("Y", "dX", "dWr", "dWg", "dWu", "dWd"):
        assert torch.equal(getattr(a, name), getattr(b, name)), name


def test_wgrad_can_be_skipped():
    """dgrad-only backward (the layer-level half of a delayed wgrad): dX unchanged."""
    import torch
    from paper_2605_31463_b200.buffers import LayerBuffers
    cfg = wl.QWEN3_SMALL.replace(row_align=128)
    inp = gc.gen_inputs(cfg)
    full = gc.run_gpu_layer(cfg, inp)
    lb = LayerBuffers(cfg, with_grads=False)
    lb.load(**inp)
    lb.forward(); lb.backward()
    torch.cuda.synchronize()
    assert torch.equal(lb.dX, full.dX)


def test_host_step_matches_device_step():
    import torch
    cfg = wl.QWEN3_SMALL.replace(row_align=128)
    inp = gc.gen_inputs(cfg)
    ref = gc.run_gpu_layer(cfg, inp)
    from paper_2605_31463_b200.buffers import LayerBuffers, act_dtype
    lb = LayerBuffers(cfg)
    lb.load(Wr=inp["Wr"], bias=inp["bias"], W=inp["W"], shared=inp["shared"])
    dt = act_dtype(cfg)
    Xh = torch.from_numpy(inp["X"]).to(dt).pin_memory()
    dYh = torch.from_numpy(inp["dY"]).to(dt).pin_memory()
    Yh = torch.empty_like(Xh).pin_memory()
    dXh = torch.empty_like(Xh).pin_memory()
    lb.step_host(Xh, dYh, Yh, dXh)
    torch.cuda.synchronize()
    assert torch.equal(Yh, ref.Y.cpu()) and torch.equal(dXh, ref.dX.cpu())


def test_cuda_graph_replay_matches_eager():
    """The library neither synchronises nor allocates, so fwd+bwd can be captured into a CUDA graph (what bench.py
    times); a replay on fresh inputs must reproduce the eager result bit for bit."""
    import torch
    cfg = wl.QWEN3_SMALL.replace(row_align=128)
    inp = gc.gen_inputs(cfg)
    ref = gc.run_gpu_layer(cfg, inp)
    from paper_2605_31463_b200.buffers import LayerBuffers
    lb = LayerBuffers(cfg)
    lb.load(**inp)
    lb.forward(); lb.backward()                      # warm-up: lazy function attributes are set outside the capture
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        lb.forward()
        lb.backward()
    for t in (lb.Y, lb.dX, lb.dWg, lb.dWd, lb.dWr):
        t.zero_()
    g.replay()
    torch.cuda.synchronize()
    for name in ("Y", "dX", "dWr", "dWg", "dWu", "dWd"):
        assert torch.equal(getattr(lb, name), getattr(ref, name)), name


WGRAD_CASES = [wl.QWEN3_SMALL.replace(name="qwen3_small_align128", row_align=128),
               wl.DSV3_SMALL.replace(name="dsv3_small_align128", row_align=128),
               wl.GPTOSS_SMALL.replace(name="gptoss_small_align128", row_align=128),
               wl.DSV3_FP8_SMALL.replace(name="dsv3_fp8_small_align128", row_align=128)]


@pytest.mark.parametrize("cfg", WGRAD_CASES, ids=lambda c: c.name)
def test_delayed_wgrad_overwrite_and_fp32_accumulate(cfg):
    """moe_layer_wgrad after a dgrad-only backward (PAPER.md:116 wgrad delay): (a) bf16 overwrite equals the fused
    backward bit for bit AND the oracle (the fused backward's gradients are oracle-checked in
    test_layer_fwd_bwd_matches_oracle; here dX and the delayed gradients are compared with the oracle again);
    (b) fp32 accumulation adds the gradient to what the buffers held: two calls add it twice, the sum is compared
    with the fp64 oracle at a tighter tolerance than bf16 outputs allow, an empty expert's slice is untouched."""
    import torch
    import paper_2605_31463_b200 as moe
    from paper_2605_31463_b200.buffers import LayerBuffers, to_numpy
    inp = gc.gen_inputs(cfg)
    full = gc.run_gpu_layer(cfg, inp)
    lb = LayerBuffers(cfg, with_grads=False)
    lb.load(**inp)
    lb.forward(); lb.backward()
    names = ["dWg", "dWu", "dWd"] + (["dWg_s", "dWu_s", "dWd_s"] if cfg.F_shared else [])
    out = {n: torch.full_like(getattr(full, n), 7.0) for n in names}
    args = [out.get(n) for n in ("dWg", "dWu", "dWd", "dWg_s", "dWu_s", "dWd_s")]
    moe.moe_layer_wgrad(lb.ccfg, lb.X, lb.dY, lb.ctx, lb.ws, *args, 0)
    torch.cuda.synchronize()
    assert torch.equal(lb.dX, full.dX)
    for n in names:
        assert torch.equal(out[n], getattr(full, n)), n
    gc.compare_layer(cfg, inp, full)                                       # ... and the fused backward equals the oracle
    # (b) fp32 main gradients: compared with the ORACLE.  fp32 accumulation removes the bf16 rounding of the output, what is
    # left is the rounding of the bf16 operands (dy, a, dg, du: 2^-9/sqrt(3) ~ 1e-3 relative each, not averaged away
    # by a random-sign contraction), so the bound is 4e-3 (measured 3.1e-3 on dWg: dg carries the roundings of dy, g, u and its own; bf16 outputs: 1e-2); FP8 keeps its own tolerance because the
    # dgrad feeding dg, du is quantised.
    tol32 = 4e-3 if cfg.dtype == wl.DTYPE_BF16 else gc.TOL[cfg.dtype]
    idx_gpu = to_numpy(lb.topk_idx)
    fwd_o = orc.layer_fwd(cfg, inp["X"], inp["Wr"], inp["bias"], inp["W"], inp["shared"], forced_idx=idx_gpu)
    bwd_o = orc.layer_bwd(cfg, inp["dY"], inp["X"], inp["Wr"], inp["W"], fwd_o, inp["shared"])
    g0 = {n: torch.randn(getattr(full, n).shape, device="cuda", dtype=torch.float32) for n in names}
    acc = {n: g0[n].clone() for n in names}
    args = [acc.get(n) for n in ("dWg", "dWu", "dWd", "dWg_s", "dWu_s", "dWd_s")]
    moe.moe_layer_wgrad(lb.ccfg, lb.X, lb.dY, lb.ctx, lb.ws, *args, 1)
    moe.moe_layer_wgrad(lb.ccfg, lb.X, lb.dY, lb.ctx, lb.ws, *args, 1)
    torch.cuda.synchronize()
    counts = to_numpy(lb.ctx_view("counts"))
    worst = 0.0
    for n in names:
        added = (acc[n].double() - g0[n].double()).cpu().numpy()
        ref = 2.0 * bwd_o[n]                                               # two micro-batches of the same gradient
        if added.ndim == 3:
            for e in range(cfg.E):
                if counts[e] == 0:
                    assert torch.equal(acc[n][e], g0[n][e]), (n, e)
                else:
                    err = orc.rel_fro(added[e], ref[e]); worst = max(worst, err)
                    assert err <= tol32, (n, e, err)
        else:
            err = orc.rel_fro(added, ref); worst = max(worst, err)
            assert err <= tol32, (n, err)
    print(cfg.name, f"fp32-accumulated wgrad vs oracle: worst {worst:.2e} (tol {tol32})")


def test_pipelined_host_step_matches_device_step():
    """Six overlapping steps through moe_layer_step_host_pipelined on alternating inputs: every step's host outputs
    equal the plain device step on the same inputs (no buffer of a slot is reused before its consumer has finished)."""
    import torch
    from paper_2605_31463_b200.buffers import LayerBuffers, act_dtype
    cfg = wl.QWEN3_SMALL.replace(row_align=128)
    inp = gc.gen_inputs(cfg)
    inp2 = dict(inp, X=wl.gen_X(cfg.replace(seed=5)), dY=wl.gen_dY(cfg.replace(seed=5)))
    refs = [gc.run_gpu_layer(cfg, inp), gc.run_gpu_layer(cfg, inp2)]
    lb = LayerBuffers(cfg)
    lb.load(Wr=inp["Wr"], bias=inp["bias"], W=inp["W"], shared=inp["shared"])
    lb.make_pipeline()
    dt = act_dtype(cfg)
    Xh = [torch.from_numpy(i["X"]).to(dt).pin_memory() for i in (inp, inp2)]
    dYh = [torch.from_numpy(i["dY"]).to(dt).pin_memory() for i in (inp, inp2)]
    n = 6
    Yh = [torch.empty_like(Xh[0]).pin_memory() for _ in range(n)]
    dXh = [torch.empty_like(Xh[0]).pin_memory() for _ in range(n)]
    for i in range(n):
        lb.step_host_pipelined(i, Xh[i % 2], dYh[i % 2], Yh[i], dXh[i])
    torch.cuda.synchronize()
    for i in range(n):
        assert torch.equal(Yh[i], refs[i % 2].Y.cpu()) and torch.equal(dXh[i], refs[i % 2].dX.cpu()), i


FUSED_CASES = [wl.QWEN3_SMALL.replace(name="qwen3_small_align128", row_align=128),
               wl.DSV3_SMALL.replace(name="dsv3_small_align128", row_align=128),
               wl.GPTOSS_SMALL.replace(name="gptoss_small_align128", row_align=128)]


@pytest.mark.parametrize("level", [0, 2])
@pytest.mark.parametrize("cfg", FUSED_CASES, ids=lambda c: c.name)
def test_other_fusion_levels_match_oracle(cfg, level):
    """bf16 layers default to moe_layer_rows_fused = 1 (routing weight in the GEMM-1 / dgrad-down epilogues, dw from the
    dgrad-down epilogue; covered by test_layer_fwd_bwd_matches_oracle).  cfg.opt_rows_fused = 1 (level 0) keeps w in the combine and
    the combine-backward pass, = 3 (level 2) also gathers the rows of X / dY inside the GEMMs (TMA tile::gather4) with Xp / dy as
    by-product copies: same oracle, same tolerance, and all three agree on the routing bit for bit."""
    import torch
    inp = gc.gen_inputs(cfg)
    dflt = gc.run_gpu_layer(cfg, inp)
    assert dflt.rows_fused == 1
    cfg = cfg.replace(opt_rows_fused=level + 1)
    lb = gc.run_gpu_layer(cfg, inp)
    assert lb.rows_fused == level
    errs = gc.compare_layer(cfg, inp, lb)
    assert torch.equal(lb.topk_idx, dflt.topk_idx) and torch.equal(lb.topk_w, dflt.topk_w)
    print(cfg.name, "fusion level", level, {k: (f"{v:.2e}" if isinstance(v, float) else v) for k, v in errs.items()})


def test_fused_rows_query():
    import paper_2605_31463_b200 as moe
    assert moe.moe_layer_rows_fused(wl.QWEN3_SMALL.replace(row_align=128)) == 1
    # fp32, unaligned groups and FP8 keep w in the combine and the combine-backward pass
    assert moe.moe_layer_rows_fused(wl.TINY) == 0
    assert moe.moe_layer_rows_fused(wl.QWEN3_SMALL) == 0
    assert moe.moe_layer_rows_fused(wl.DSV3_FP8_SMALL.replace(row_align=128)) == 0


@pytest.mark.parametrize("pair", [0, 2])
@pytest.mark.parametrize("cfg", [wl.QWEN3_SMALL.replace(name="qwen3_small_align128", row_align=128),
                                 wl.QWEN3_SMALL.replace(name="qwen3_small_align256", row_align=256),
                                 wl.GPTOSS_SMALL.replace(name="gptoss_small_align128", row_align=128)], ids=lambda c: c.name)
def test_cta_pair_kernel_levels_match_oracle(cfg, pair):
    """moe_config_t::opt_pair (level + 1): level 1 (default, the other tests) runs the weight gradients and single-group GEMMs on the cta_group::2 pair
    kernel; 0 keeps every GEMM on the 1-CTA kernel; 2 also runs the ragged expert GEMMs as M-tile pairs (device-built
    pair / unpaired tile lists) followed by the 1-CTA kernel over the unpaired last tiles.  With row_align = 256 every
    tile is paired.  Same oracle, same tolerance."""
    cfg = cfg.replace(opt_pair=pair + 1)
    inp = gc.gen_inputs(cfg)
    lb = gc.run_gpu_layer(cfg, inp)
    errs = gc.compare_layer(cfg, inp, lb)
    print(cfg.name, "pair level", pair, {k: (f"{v:.2e}" if isinstance(v, float) else v) for k, v in errs.items()})
