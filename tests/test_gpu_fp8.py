"""`-m gpu` parity of the FP8 e4m3 block-scaled path against the oracle:
quantisers bit-exact (codes and scales) on identical bf16 input, the stand-alone fp8 grouped GEMM and the whole
layer forward + backward against the fake-quant oracle (tolerance 3e-2, BASELINE.json:north_star)."""
import numpy as np
import pytest

import gpu_common as gc
import workloads as wl
from oracle import moe_oracle as orc

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def env():
    import torch
    import paper_2605_31463_b200 as moe
    from paper_2605_31463_b200 import buffers
    moe.lib()
    return torch, moe, buffers


def _dev(torch, x, dtype):
    return torch.from_numpy(np.ascontiguousarray(x)).cuda().to(dtype).contiguous()


def _act_input(rows, cols, seed):
    """bf16-grid values with a wide dynamic range, an all-zero block, an all-zero row and exact powers of two."""
    v = wl.normal(seed, "aux", (rows, cols), 1.0, wl.DTYPE_BF16)
    scale = np.exp2(np.random.default_rng(seed).integers(-12, 12, size=(rows, 1))).astype(np.float32)
    v = orc.bf16_round(v * scale)
    if rows > 2:
        v[1, :min(128, cols)] = 0.0
        v[2, :] = 0.0
    if rows > 3:
        v[3, :] = 448.0
        v[3, 0] = 0.5
    return v


@pytest.mark.parametrize("rows,cols", [(1, 128), (5, 8), (37, 320), (300, 512), (1024, 7168)])
@pytest.mark.parametrize("mode", [0, 1])
def test_quantize_act_bit_exact(env, rows, cols, mode):
    torch, moe, _ = env
    v = _act_input(rows, cols, 11 + rows)
    codes_o, scale_o = orc.quantize_1x128(v, mode)
    vd = _dev(torch, v, torch.bfloat16)
    codes = torch.full((rows, cols), 0x55, dtype=torch.uint8, device="cuda")
    scales = torch.full((rows, (cols + 127) // 128), -1.0, dtype=torch.float32, device="cuda")
    moe.moe_quantize_act(vd, rows, cols, mode, codes, scales)
    torch.cuda.synchronize()
    assert np.array_equal(scales.cpu().numpy(), scale_o), "scales must be bit-exact"
    assert np.array_equal(codes.cpu().numpy(), codes_o), "codes must be bit-exact"


@pytest.mark.parametrize("batch,rows,cols", [(1, 128, 128), (3, 200, 320), (4, 384, 512), (2, 8, 8)])
@pytest.mark.parametrize("mode", [0, 1])
def test_quantize_weight_bit_exact(env, batch, rows, cols, mode):
    torch, moe, _ = env
    w = wl.normal(7, "aux", (batch, rows, cols), 0.02, wl.DTYPE_BF16)
    w[0, :min(128, rows), :min(128, cols)] = 0.0                     # an all-zero block -> scale 1, codes 0
    codes_o, scale_o = orc.quantize_128x128(w, mode)
    wd = _dev(torch, w, torch.bfloat16)
    codes = torch.full((batch, rows, cols), 0x55, dtype=torch.uint8, device="cuda")
    scales = torch.full(scale_o.shape, -1.0, dtype=torch.float32, device="cuda")
    moe.moe_quantize_weight(wd, batch, rows, cols, mode, codes, scales)
    torch.cuda.synchronize()
    assert np.array_equal(scales.cpu().numpy(), scale_o)
    assert np.array_equal(codes.cpu().numpy(), codes_o)


F8_GEMM_CASES = [
    ("qwen3_small", wl.QWEN3_SMALL.replace(dtype=wl.DTYPE_FP8, row_align=128), 384, 512),
    ("dsv3_small", wl.DSV3_SMALL.replace(dtype=wl.DTYPE_FP8, row_align=128), 256, 512),
    ("skew_empty", wl.GPTOSS_SMALL.replace(dtype=wl.DTYPE_FP8, row_align=128, H=384, F=384), 384, 384),
    ("deep_k", wl.QWEN3_SMALL.replace(dtype=wl.DTYPE_FP8, row_align=128, T=300), 128, 7168),
]


@pytest.mark.parametrize("name,cfg,N,Kd", F8_GEMM_CASES, ids=[c[0] for c in F8_GEMM_CASES])
@pytest.mark.parametrize("mode", [0, 1])
def test_fp8_grouped_gemm_fwd(env, name, cfg, N, Kd, mode):
    """C = dequant(A) dequant(B[e])^T on the GPU's own codes: tolerance is fp32 summation only (1e-2 covers bf16 out)."""
    torch, moe, _ = env
    cfg = cfg.replace(fp8_scale_mode=mode)
    z = wl.gen_logits(cfg)
    idx_o, _ = orc.route(z, wl.gen_bias(cfg), cfg, key_dtype=np.float32)
    counts, off, p2f, _ = orc.permute_maps(idx_o, cfg.E, cfg.row_align)
    R = moe.moe_padded_rows(cfg)
    n = int(off[-1])
    A = np.zeros((R, Kd), np.float32)
    A[:n] = wl.normal(3, "aux", (n, Kd), 1.0, wl.DTYPE_BF16) * (p2f >= 0)[:, None]
    B = wl.normal(5, "aux", (cfg.E, N, Kd), 0.05, wl.DTYPE_BF16)
    Aq, As = orc.quantize_1x128(A, mode)
    Bq, Bs = orc.quantize_128x128(B, mode)
    ws_b, _ = moe.moe_workspace_bytes(cfg)
    ws = torch.empty(ws_b, dtype=torch.uint8, device="cuda")
    Cd = torch.zeros((R, N), dtype=torch.bfloat16, device="cuda")
    moe.moe_grouped_gemm_fwd(cfg, N, Kd, _dev(torch, Aq, torch.uint8), _dev(torch, Bq, torch.uint8),
                             _dev(torch, off, torch.int32), Cd, _dev(torch, As, torch.float32),
                             _dev(torch, Bs, torch.float32), ws)
    torch.cuda.synchronize()
    Cg = Cd.float().cpu().numpy()
    Adq = orc.dequantize_1x128(Aq, As)
    for e in range(cfg.E):
        r0, r1 = int(off[e]), int(off[e]) + int(counts[e])
        if r1 == r0:
            continue
        Cr = Adq[r0:r1] @ orc.dequantize_128x128(Bq[e], Bs[e]).T
        err = orc.rel_fro(Cg[r0:r1], Cr)
        assert err <= 1e-2, (e, err)


FP8_LAYER_CASES = [
    wl.DSV3_FP8_SMALL.replace(name="dsv3_fp8_small_align128", row_align=128),
    wl.DSV3_FP8_SMALL.replace(name="dsv3_fp8_small_pow2", row_align=128, fp8_scale_mode=1),
    wl.QWEN3_SMALL.replace(name="qwen3_fp8_small", dtype=wl.DTYPE_FP8, row_align=128),
    wl.GPTOSS_SMALL.replace(name="gptoss_fp8_small", dtype=wl.DTYPE_FP8, row_align=128, H=384, F=384),
]


@pytest.mark.parametrize("cfg", FP8_LAYER_CASES, ids=lambda c: c.name)
def test_fp8_layer_fwd_bwd_matches_fake_quant_oracle(cfg):
    inp = gc.gen_inputs(cfg)
    lb = gc.run_gpu_layer(cfg, inp)
    errs = gc.compare_layer(cfg, inp, lb)
    print(cfg.name, {k: (f"{v:.2e}" if isinstance(v, float) else v) for k, v in errs.items()})


@pytest.mark.parametrize("fused", [0, 1])
@pytest.mark.parametrize("mode", [0, 1])
def test_fused_epilogue_quantisers_are_bit_exact(env, mode, fused):
    """PAPER.md:116 fused FP8 quantisation: the codes and 1x128 scales that the GEMM-1 epilogue emits for `a` (Q-a) and
    the dgrad-down epilogue for [dg|du] (Q-dgu) are the SAME BITS the oracle's quantiser gives on the bf16 tensors those
    kernels wrote (rows of real tokens and padding rows; the shared expert's single-group path included)."""
    torch, moe, buffers = env
    # opt_fp8_fused_quant = 2: quantise in the epilogues; = 1: stand-alone passes
    cfg = wl.DSV3_FP8_SMALL.replace(row_align=128, fp8_scale_mode=mode, opt_fp8_fused_quant=fused + 1)
    inp = gc.gen_inputs(cfg)
    lb = gc.run_gpu_layer(cfg, inp)
    gc.compare_layer(cfg, inp, lb)                              # ... and the layer still matches the fake-quant oracle
    R = int(buffers.to_numpy(lb.ctx_view("offsets"))[-1])
    a = buffers.to_numpy(lb.ctx_view("a"))[:R]
    codes, sc = orc.quantize_1x128(a, mode)
    assert np.array_equal(buffers.to_numpy(lb.ctx_view("aq"))[:R], codes)
    assert np.array_equal(buffers.to_numpy(lb.ctx_view("aq_s"))[:R], sc)
    dgu = buffers.to_numpy(lb.ws_view("dgu"))[:R]
    codes, sc = orc.quantize_1x128(dgu, mode)
    assert np.array_equal(buffers.to_numpy(lb.ws_view("dguq"))[:R], codes)
    assert np.array_equal(buffers.to_numpy(lb.ws_view("dguq_s"))[:R], sc)


@pytest.mark.parametrize("wide", [0, 2])
def test_fp8_tile_width_levels(env, wide):
    """The FP8 GEMMs run 128 x 256 tiles for the plain-epilogue modes by default (moe_config_t::opt_fp8_wide level 1; the other tests).
    Level 0 keeps every GEMM on 128 x 128 tiles, level 2 puts the fused-SwiGLU modes on the wide kernel too: same oracle, same
    tolerance, and the fused quantisers' codes and scales stay bit-exact."""
    torch, moe, buffers = env
    for mode in (0, 1):
        cfg = wl.DSV3_FP8_SMALL.replace(row_align=128, fp8_scale_mode=mode, opt_fp8_wide=wide + 1, opt_fp8_fused_quant=2)
        inp = gc.gen_inputs(cfg)
        lb = gc.run_gpu_layer(cfg, inp)
        gc.compare_layer(cfg, inp, lb)
        R = int(buffers.to_numpy(lb.ctx_view("offsets"))[-1])
        codes, sc = orc.quantize_1x128(buffers.to_numpy(lb.ctx_view("a"))[:R], mode)
        assert np.array_equal(buffers.to_numpy(lb.ctx_view("aq"))[:R], codes)
        assert np.array_equal(buffers.to_numpy(lb.ctx_view("aq_s"))[:R], sc)
        codes, sc = orc.quantize_1x128(buffers.to_numpy(lb.ws_view("dgu"))[:R], mode)
        assert np.array_equal(buffers.to_numpy(lb.ws_view("dguq"))[:R], codes)
        assert np.array_equal(buffers.to_numpy(lb.ws_view("dguq_s"))[:R], sc)


def test_fp8_weight_cache_matches_oracle(env):
    """FP8 weight cache: quantise the weights once with moe_fp8_quantize_weights, then run a NEW
    micro-batch through moe_layer_fwd with NULL weights (the bf16 weights overwritten with garbage first, so nothing
    can read them) and moe_layer_bwd; every output is compared with the fake-quant ORACLE on that micro-batch."""
    torch, moe, buffers = env
    cfg = wl.DSV3_FP8_SMALL.replace(row_align=128)
    inp = gc.gen_inputs(cfg)
    lb = buffers.LayerBuffers(cfg)
    lb.load(**inp)
    moe.moe_fp8_quantize_weights(lb.ccfg, lb.Wg, lb.Wu, lb.Wd, lb.Wg_s, lb.Wu_s, lb.Wd_s, lb.ctx)
    inp2 = dict(inp, X=wl.gen_X(cfg.replace(seed=9)), dY=wl.gen_dY(cfg.replace(seed=9)))
    lb.load(X=inp2["X"], dY=inp2["dY"])
    for w in (lb.Wg, lb.Wu, lb.Wd, lb.Wg_s, lb.Wu_s, lb.Wd_s):
        w.fill_(float("nan"))
    moe.moe_layer_fwd(lb.ccfg, lb.X, lb.Wr, lb.bias, None, None, None, None, None, None, lb.Y, lb.topk_idx, lb.topk_w,
                      lb.ctx, lb.ws)
    moe.moe_layer_bwd(lb.ccfg, lb.dY, lb.X, lb.Wr, None, None, None, None, None, None, lb.ctx, lb.dX, lb.dWr, lb.dWg,
                      lb.dWu, lb.dWd, lb.dWg_s, lb.dWu_s, lb.dWd_s, lb.ws)
    torch.cuda.synchronize()
    errs = gc.compare_layer(cfg, inp2, lb)
    print(cfg.name, {k: (f"{v:.2e}" if isinstance(v, float) else v) for k, v in errs.items()})


def test_fp8_rejects_unaligned():
    import paper_2605_31463_b200 as moe
    cfg = wl.QWEN3_SMALL.replace(dtype=wl.DTYPE_FP8, H=320, row_align=128)
    with pytest.raises(moe.MoEError):
        moe.moe_workspace_bytes(cfg)
