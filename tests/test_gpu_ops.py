"""`-m gpu` parity of the stand-alone C-ABI ops against the fp64 oracle on the same seeded inputs:
moe_route (bit-exact indices, ties -> lower index), moe_permute (bit-exact maps and row copies),
moe_unpermute_combine, moe_swiglu(+bwd), moe_grouped_gemm_fwd/bwd.  SURVEY.md §8(c)."""
import numpy as np
import pytest

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


ROUTE_CASES = [
    wl.TINY, wl.QWEN3_SMALL, wl.DSV3_SMALL, wl.GPTOSS_SMALL,
    wl.DSV3_SMALL.replace(name="dsv3_groupmax", group_score=wl.GROUP_SCORE_MAX),
    wl.DSV3_SMALL.replace(name="dsv3_norenorm", renorm=0),
    wl.QWEN3_SMALL.replace(name="qwen3_norenorm", renorm=0),
    wl.TINY.replace(name="k_eq_e", K=8), wl.TINY.replace(name="k1", K=1), wl.TINY.replace(name="t1", T=1),
    wl.QWEN3.replace(name="qwen3_full_route"), wl.DSV3.replace(name="dsv3_full_route"),
    wl.GPTOSS.replace(name="gptoss_full_route"),
    wl.QWEN3_SMALL.replace(name="e1000", E=1000, K=32, T=77),
]


@pytest.mark.parametrize("cfg", ROUTE_CASES, ids=lambda c: c.name)
@pytest.mark.parametrize("ties", [0, 3])
def test_route_bit_exact(env, cfg, ties):
    torch, moe, _ = env
    z = wl.gen_logits(cfg, ties=ties)
    bias = wl.gen_bias(cfg)
    zd = _dev(torch, z, torch.float32)
    bd = _dev(torch, bias, torch.float32) if bias is not None else None
    idx = torch.full((cfg.T, cfg.K), -7, dtype=torch.int32, device="cuda")
    w = torch.empty((cfg.T, cfg.K), dtype=torch.float32, device="cuda")
    moe.moe_route(cfg, zd, bd, idx, w)
    torch.cuda.synchronize()
    # both sides take the fp32 selection decision on identical key bits (replay mode, S3)
    idx_o, w_o = orc.route(z, bias, cfg, key_dtype=np.float32)
    assert np.array_equal(idx.cpu().numpy(), idx_o)
    assert orc.rel_fro(w.cpu().numpy(), w_o) <= 1e-5
    assert np.abs(w.cpu().numpy() - w_o).max() <= 1e-5 * max(1.0, cfg.routed_scale)


def test_route_hand_made_ties(env):
    torch, moe, _ = env
    cfg = wl.TINY.replace(T=4, E=8, K=3)
    z = np.zeros((4, 8), np.float32)            # all equal -> experts 0,1,2
    z[1, [5, 2, 7]] = 1.0                       # three-way tie at the top -> 2,5,7
    z[2, 7] = 2.0; z[2, [3, 4]] = 1.0           # 7, then tie 3,4
    z[3] = np.arange(8, dtype=np.float32)       # 7,6,5
    idx = torch.empty((4, 3), dtype=torch.int32, device="cuda")
    w = torch.empty((4, 3), dtype=torch.float32, device="cuda")
    moe.moe_route(cfg, _dev(torch, z, torch.float32), None, idx, w)
    assert idx.cpu().tolist() == [[0, 1, 2], [2, 5, 7], [7, 3, 4], [7, 6, 5]]
    assert np.allclose(w.cpu().numpy().sum(1), 1.0, atol=1e-6)


PERM_CASES = [wl.TINY, wl.QWEN3_SMALL, wl.GPTOSS_SMALL, wl.DSV3_SMALL, wl.TINY.replace(name="t1", T=1),
              wl.TINY.replace(name="t1025", T=1025, K=3), wl.QWEN3.replace(name="qwen3_full_perm"),
              wl.GPTOSS.replace(name="gptoss_full_perm"),
              # > 256 chunks of 1024 positions: the chunk histograms are prefix-summed by their own launch (permute.cu)
              wl.QWEN3.replace(name="many_chunks", T=40001, H=64, F=64)]


@pytest.mark.parametrize("cfg", PERM_CASES, ids=lambda c: c.name)
@pytest.mark.parametrize("align", [1, 128])
def test_permute_maps_and_rows_bit_exact(env, cfg, align):
    torch, moe, buffers = env
    cfg = cfg.replace(row_align=align)
    dt = buffers.act_dtype(cfg)
    z = wl.gen_logits(cfg)
    idx_o, w_o = orc.route(z, wl.gen_bias(cfg), cfg, key_dtype=np.float32)
    X = wl.gen_X(cfg)
    R = moe.moe_padded_rows(cfg)
    ws_b, _ = moe.moe_workspace_bytes(cfg)
    ws = torch.empty(ws_b, dtype=torch.uint8, device="cuda")
    idx = _dev(torch, idx_o, torch.int32)
    counts = torch.empty(cfg.E, dtype=torch.int32, device="cuda")
    offsets = torch.empty(cfg.E + 1, dtype=torch.int32, device="cuda")
    p2f = torch.empty(R, dtype=torch.int32, device="cuda")
    f2p = torch.empty(cfg.TK, dtype=torch.int32, device="cuda")
    Xd = _dev(torch, X, dt)
    Xp = torch.full((R, cfg.H), 7.0, dtype=dt, device="cuda")
    moe.moe_permute(cfg, Xd, idx, counts, offsets, p2f, f2p, Xp, ws)
    torch.cuda.synchronize()
    c_o, off_o, p2f_o, f2p_o = orc.permute_maps(idx_o, cfg.E, align)
    n = int(off_o[-1])
    assert np.array_equal(counts.cpu().numpy(), c_o)
    assert np.array_equal(offsets.cpu().numpy(), off_o)
    assert np.array_equal(f2p.cpu().numpy(), f2p_o)
    assert np.array_equal(p2f.cpu().numpy()[:n], p2f_o)
    assert (p2f.cpu().numpy()[n:] == -1).all()
    Xp_o = orc.permute_rows(X, p2f_o, cfg.K)
    assert np.array_equal(Xp[:n].float().cpu().numpy(), Xp_o.astype(np.float32))
    # property pins at any size: each token appears exactly K times; bijection
    live = p2f.cpu().numpy()[:n]
    live = live[live >= 0]
    assert np.array_equal(np.sort(live), np.arange(cfg.TK))
    assert (np.bincount(live // cfg.K, minlength=cfg.T) == cfg.K).all()
    # permute -> combine with w = 1/K is the identity, bit-exactly (K is a power of two)
    if cfg.K in (1, 2, 4, 8):
        w = torch.full((cfg.T, cfg.K), 1.0 / cfg.K, dtype=torch.float32, device="cuda")
        Y = torch.empty_like(Xd)
        moe.moe_unpermute_combine(cfg, Xp, w, f2p, None, Y)
        torch.cuda.synchronize()
        assert torch.equal(Y, Xd)


@pytest.mark.parametrize("cfg", [wl.TINY, wl.QWEN3_SMALL, wl.DSV3_SMALL], ids=lambda c: c.name)
def test_unpermute_combine(env, cfg):
    torch, moe, buffers = env
    dt = buffers.act_dtype(cfg)
    z = wl.gen_logits(cfg)
    idx_o, w_o = orc.route(z, wl.gen_bias(cfg), cfg, key_dtype=np.float32)
    _, off_o, p2f_o, f2p_o = orc.permute_maps(idx_o, cfg.E, 1)
    y = wl.normal(cfg.seed, "aux", (cfg.TK, cfg.H), 1.0, wl.DTYPE_FP32 if cfg.dtype == 0 else wl.DTYPE_BF16)
    sh = wl.gen_dY(cfg)
    w32 = w_o.astype(np.float32)
    Y = torch.empty((cfg.T, cfg.H), dtype=dt, device="cuda")
    for shared in (None, sh):
        moe.moe_unpermute_combine(cfg, _dev(torch, y, dt), _dev(torch, w32, torch.float32),
                                  _dev(torch, f2p_o, torch.int32), _dev(torch, shared, dt) if shared is not None else None, Y)
        torch.cuda.synchronize()
        ref = orc.unpermute_combine(y, w32, f2p_o, shared)
        tol = 1e-6 if cfg.dtype == 0 else 4e-3       # one bf16 rounding of the output: 2^-9 relative
        assert orc.rel_fro(Y.float().cpu().numpy(), ref) <= tol


@pytest.mark.parametrize("dtype", [wl.DTYPE_FP32, wl.DTYPE_BF16])
@pytest.mark.parametrize("rows,F", [(1, 8), (333, 264), (2048, 768)])
def test_swiglu_fwd_bwd(env, dtype, rows, F):
    torch, moe, buffers = env
    cfg = wl.TINY.replace(dtype=dtype, F=F)
    dt = buffers.act_dtype(cfg)
    gu = wl.normal(0, "aux", (rows, 2 * F), 1.5, dtype)
    da = wl.normal(1, "aux", (rows, F), 1.0, dtype)
    gud, dad = _dev(torch, gu, dt), _dev(torch, da, dt)
    a = torch.empty((rows, F), dtype=dt, device="cuda")
    dgu = torch.empty((rows, 2 * F), dtype=dt, device="cuda")
    moe.moe_swiglu(cfg, gud, a, rows)
    moe.moe_swiglu_bwd(cfg, gud, dad, dgu, rows)
    torch.cuda.synchronize()
    tol = 1e-6 if dtype == 0 else 4e-3
    assert orc.rel_fro(a.float().cpu().numpy(), orc.swiglu(gu[:, :F], gu[:, F:])) <= tol
    dg, du = orc.swiglu_bwd(da, gu[:, :F], gu[:, F:])
    assert orc.rel_fro(dgu.float().cpu().numpy(), np.concatenate([dg, du], 1)) <= tol


GEMM_CASES = [
    # (name, base cfg, N, Kdim)
    ("tiny_fp32", wl.TINY, 256, 128),
    ("tiny_fp32_ragged", wl.TINY.replace(T=77, K=3), 72, 36),
    ("bf16_small", wl.QWEN3_SMALL.replace(row_align=128), 384, 512),
    ("bf16_n_tail", wl.QWEN3_SMALL.replace(row_align=128), 200, 320),
    ("bf16_skew_empty", wl.GPTOSS_SMALL.replace(row_align=128), 320, 320),
    ("bf16_k2880", wl.GPTOSS_SMALL.replace(row_align=128, T=300), 2880 // 4, 2880),
    ("bf16_packed_rows", wl.QWEN3_SMALL, 384, 512),
]


@pytest.mark.parametrize("name,cfg,N,Kd", GEMM_CASES, ids=[c[0] for c in GEMM_CASES])
def test_grouped_gemm_fwd_bwd(env, name, cfg, N, Kd):
    torch, moe, buffers = env
    dt = buffers.act_dtype(cfg)
    sd = wl.DTYPE_FP32 if cfg.dtype == 0 else wl.DTYPE_BF16
    z = wl.gen_logits(cfg)
    idx_o, _ = orc.route(z, wl.gen_bias(cfg), cfg, key_dtype=np.float32)
    counts, off, p2f, _ = orc.permute_maps(idx_o, cfg.E, cfg.row_align)
    R = moe.moe_padded_rows(cfg)
    n = int(off[-1])
    live = (p2f >= 0)[:, None]
    A = np.zeros((R, Kd), np.float32); A[:n] = wl.normal(3, "aux", (n, Kd), 1.0, sd) * live
    dC = np.zeros((R, N), np.float32); dC[:n] = wl.normal(4, "aux", (n, N), 1.0, sd) * live
    B = wl.normal(5, "aux", (cfg.E, N, Kd), 0.05, sd)
    ws_b, _ = moe.moe_workspace_bytes(cfg)
    ws = torch.empty(ws_b, dtype=torch.uint8, device="cuda")
    offd = _dev(torch, off, torch.int32)
    Ad, Bd, dCd = _dev(torch, A, dt), _dev(torch, B, dt), _dev(torch, dC, dt)
    Cd = torch.zeros((R, N), dtype=dt, device="cuda")
    dAd = torch.zeros((R, Kd), dtype=dt, device="cuda")
    dBd = torch.full((cfg.E, N, Kd), 3.0, dtype=dt, device="cuda")
    moe.moe_grouped_gemm_fwd(cfg, N, Kd, Ad, Bd, offd, Cd, None, None, ws)
    moe.moe_grouped_gemm_bwd(cfg, N, Kd, dCd, Ad, Bd, offd, dAd, dBd, ws)
    torch.cuda.synchronize()
    tol = 1e-5 if cfg.dtype == 0 else 1e-2
    Cg, dAg, dBg = (t.float().cpu().numpy() for t in (Cd, dAd, dBd))
    A64, B64, dC64 = A.astype(np.float64), B.astype(np.float64), dC.astype(np.float64)
    for e in range(cfg.E):
        r0, r1 = int(off[e]), int(off[e]) + int(counts[e])
        Cr = A64[r0:r1] @ B64[e].T
        dAr = dC64[r0:r1] @ B64[e]
        dBr = dC64[r0:r1].T @ A64[r0:r1]
        assert orc.rel_fro(Cg[r0:r1], Cr) <= tol, (e, "C")
        assert orc.rel_fro(dAg[r0:r1], dAr) <= tol, (e, "dA")
        assert orc.rel_fro(dBg[e], dBr) <= tol, (e, "dB")
        if r1 == r0:
            assert not dBg[e].any(), "empty expert must get exact zero dW"
    # dgrad-only / wgrad-only calls (the split a delayed wgrad needs)
    dA2 = torch.zeros_like(dAd)
    moe.moe_grouped_gemm_bwd(cfg, N, Kd, dCd, None, Bd, offd, dA2, None, ws)
    dB2 = torch.zeros_like(dBd)
    moe.moe_grouped_gemm_bwd(cfg, N, Kd, dCd, Ad, None, offd, None, dB2, ws)
    torch.cuda.synchronize()
    assert torch.equal(dA2[:n], dAd[:n]) and torch.equal(dB2, dBd)
