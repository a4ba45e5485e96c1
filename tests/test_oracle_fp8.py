"""Pins for the oracle's FP8 e4m3 block quantisers ("FP8 quantiser" pin)."""
import os

import numpy as np
import pytest
import torch

import workloads as wl
from oracle import moe_oracle as O

GOLD = os.path.join(os.path.dirname(__file__), "golden", "e4m3_spot_values.txt")


def test_e4m3_spot_values_from_format_definition():
    rows = [l.split() for l in open(GOLD) if l.strip() and not l.startswith("#")]
    assert len(rows) >= 10
    for x, want, code in rows:
        c = O.e4m3_encode(np.array([float(x)], np.float32))
        assert int(c[0]) == int(code, 16), (x, hex(int(c[0])), code)
        assert O.e4m3_decode(c)[0] == float(want)


def test_e4m3_table_and_encode_against_torch_float8():
    """Library cross-check: torch.float8_e4m3fn casts (RNE) agree on every finite fp8 value, on all
    midpoints between neighbours, and on random in-range values."""
    codes = np.arange(256, dtype=np.uint8)
    tv = torch.from_numpy(codes).view(torch.float8_e4m3fn).float().numpy().astype(np.float64)
    ok = ~np.isnan(tv)
    assert np.array_equal(np.isnan(O.E4M3_TABLE), ~ok)
    assert np.array_equal(O.E4M3_TABLE[ok], tv[ok])
    pos = np.sort(tv[ok & (tv >= 0)])
    mids = ((pos[:-1] + pos[1:]) / 2).astype(np.float32)
    rnd = (np.random.default_rng(0).standard_normal(20000) * 100).astype(np.float32)
    rnd = rnd[np.abs(rnd) <= 448]
    for v in (pos.astype(np.float32), mids, -mids, rnd, rnd * 1e-3):
        mine = O.e4m3_decode(O.e4m3_encode(v))
        ref = torch.from_numpy(v).to(torch.float8_e4m3fn).float().numpy()
        assert np.array_equal(mine, ref.astype(np.float64))


@pytest.mark.parametrize("mode", [0, 1])
def test_quantiser_properties(mode):
    c = wl.DSV3_FP8_SMALL
    X = wl.gen_X(c)
    X[3, 128:256] = 0                                                     # an all-zero block
    codes, sc = O.quantize_1x128(X, mode)
    assert codes.shape == X.shape and sc.shape == (c.T, c.H // 128)
    assert sc[3, 1] == 1.0 and not codes[3, 128:256].any()                 # amax = 0 => scale 1, codes 0
    amax = np.abs(X.reshape(c.T, -1, 128)).max(axis=2)
    if mode == 1:
        m, _ = np.frexp(sc)
        assert (m == 0.5).all()                                            # powers of two
        assert (sc.astype(np.float64) * 448 >= amax).all()
        assert (sc.astype(np.float64) * 448 < 2 * np.maximum(amax, 1e-30))[amax > 0].all()
    else:
        assert (np.abs(sc.astype(np.float64) * 448 - amax) <= amax * 2.0 ** -23)[amax > 0].all()   # 1 ulp of fp32
    d = O.dequantize_1x128(codes, sc)
    # each block's largest element maps to +-448 (mode 0) and error is bounded by half a quantum
    assert np.abs(d - X).max() <= np.abs(X).max() / 16 + 1e-9
    # idempotent on its own output (power-of-two scales; mode 0 re-derives the same amax)
    if mode == 1:
        c2, s2 = O.quantize_1x128(d.astype(np.float32), mode)
        assert np.array_equal(O.dequantize_1x128(c2, s2), d)


def test_weight_quantiser_blocks_and_transpose_symmetry():
    """128x128 blocks are square: quantising W^T gives the transposed codes and scales (so the same
    codes serve fprop and the transposed dgrad)."""
    W = wl.normal(0, "Wg", (256, 384), 0.02, wl.DTYPE_BF16)
    c, s = O.quantize_128x128(W, 0)
    ct, st = O.quantize_128x128(np.ascontiguousarray(W.T), 0)
    assert s.shape == (2, 3) and np.array_equal(ct, c.T) and np.array_equal(st, s.T)
    blk = np.abs(W[128:256, 256:384]).max()
    assert s[1, 2] == np.float32(blk) / np.float32(448)
    # ragged: 200 x 130 pads with zeros, scales shape (2, 2)
    c2, s2 = O.quantize_128x128(W[:200, :130], 0)
    assert c2.shape == (200, 130) and s2.shape == (2, 2)


def test_fp8_layer_close_to_unquantised_and_runs_backward():
    """Information + sanity: fake-quant forward stays within a few % of the fp64 layer (S18 measured
    3.7% for one K=7168 GEMM); backward runs and empty experts keep zero grads."""
    c = wl.DSV3_FP8_SMALL.replace(T=128, H=256, F=128, F_shared=128)
    X = wl.gen_X(c); Wr = wl.gen_Wr(c); b = wl.gen_bias(c)
    W = wl.gen_all_expert_weights(c, threads=4); sh = wl.gen_shared_weights(c); dY = wl.gen_dY(c)
    f8 = O.layer_fwd(c, X, Wr, b, W, sh)
    f = O.layer_fwd(c.replace(dtype=1), X, Wr, b, W, sh)
    assert np.array_equal(f8["idx"], f["idx"])
    e = O.rel_fro(f8["Y"], f["Y"])
    assert 1e-3 < e < 0.08, e
    b8 = O.layer_bwd(c, dY, X, Wr, W, f8, sh)
    bb = O.layer_bwd(c.replace(dtype=1), dY, X, Wr, W, f, sh)
    for k in ("dX", "dWg", "dWd", "dWr", "dWg_s"):
        assert O.rel_fro(b8[k], bb[k]) < 0.1, k


# ---------------------------------------------------------------------------------------------
# bf16_round and the FP8 quantisation-point composition (R9): pins that do not retype the oracle
# ---------------------------------------------------------------------------------------------


def test_bf16_round_ties_to_even_and_matches_torch():
    """bf16 keeps 8 significant bits: 1 + 2^-8 lies halfway between 1 and 1 + 2^-7 (even mantissa: 1);
    1 + 3*2^-8 lies halfway between 1 + 2^-7 and 1 + 2^-6 (even mantissa: 1 + 2^-6).  Truncation or
    round-half-up fails one of the two.  Library cross-check: torch's fp32 -> bfloat16 cast."""
    x = np.array([1 + 2.0 ** -8, 1 + 3 * 2.0 ** -8, -(1 + 2.0 ** -8), 1 + 2.0 ** -8 + 2.0 ** -20, 1 + 2.0 ** -9], np.float32)
    want = np.array([1.0, 1 + 2.0 ** -6, -1.0, 1 + 2.0 ** -7, 1.0], np.float32)
    assert np.array_equal(O.bf16_round(x), want)
    g = np.random.default_rng(7)
    v = np.concatenate([g.standard_normal(100000).astype(np.float32) * np.float32(s) for s in (1.0, 1e-3, 300.0)])
    ref = torch.from_numpy(v).to(torch.bfloat16).float().numpy()
    assert np.array_equal(O.bf16_round(v), ref)
    assert np.array_equal(O.bf16_round(v.astype(np.float64)), ref)      # fp64 input is first narrowed to fp32


def _on_grid(rng, shape, block, lo_exp=-6, hi_exp=2):
    """Random values that a mode-1 (power-of-two scale) e4m3 block quantiser reproduces exactly: per block a
    scale 2^k and finite e4m3 values, one of them with magnitude in (224, 448] so the quantiser picks 2^k again.
    `block` = (rows, cols) of a scale block.  Built from torch's float8 decode, not from the oracle."""
    R, C = shape
    br, bc = block
    codes = rng.integers(0, 0x7F, size=shape).astype(np.uint8)           # 0x00..0x7E: finite, non-negative
    codes |= (rng.integers(0, 2, size=shape).astype(np.uint8) << 7)       # random sign
    val = torch.from_numpy(codes).view(torch.float8_e4m3fn).float().numpy().astype(np.float64)
    out = np.empty(shape, np.float64)
    for r0 in range(0, R, br):
        for c0 in range(0, C, bc):
            blk = val[r0:r0 + br, c0:c0 + bc]
            blk[rng.integers(0, blk.shape[0]), rng.integers(0, blk.shape[1])] = rng.choice([240.0, 288.0, 448.0, -320.0])
            out[r0:r0 + br, c0:c0 + bc] = blk * 2.0 ** int(rng.integers(lo_exp, hi_exp))
    return out.astype(np.float32)


def _torch_fq_1x128_pow2(v):
    """Independent restatement of Q-act (mode 1) with library casts: bf16 cast, per 1x128 block amax,
    scale 2^ceil(log2(amax/448)), torch.float8_e4m3fn cast (RNE, values are in range), dequantise."""
    t = torch.from_numpy(np.asarray(v, np.float32)).to(torch.bfloat16).float()
    R, C = t.shape
    b = t.reshape(R, C // 128, 128)
    amax = b.abs().amax(dim=2, keepdim=True)
    scale = torch.where(amax > 0, torch.exp2(torch.ceil(torch.log2(amax / 448.0))), torch.ones_like(amax))
    q = (b / scale).to(torch.float8_e4m3fn).float() * scale
    return q.reshape(R, C).double().numpy()


def test_fp8_composition_identity_grid_forward():
    """With power-of-two scales and X, W already on the e4m3 x 2^k grid of their blocks, Q-X and Q-W are the
    identity: the FP8 forward's g, u must equal the unquantised forward's, and y differs from it ONLY by Q-a
    (1x128 along F, on the bf16-rounded a, before the down projection)."""
    rng = np.random.default_rng(11)
    n, H, F = 24, 256, 256
    X = _on_grid(rng, (n, H), (1, 128), -9, -6)
    Wg, Wu = _on_grid(rng, (F, H), (128, 128), -9, -5), _on_grid(rng, (F, H), (128, 128), -9, -5)
    Wd = _on_grid(rng, (H, F), (128, 128), -9, -5)
    assert np.array_equal(O.fq_act(X, 1), X.astype(np.float64))
    for W in (Wg, Wu, Wd):
        assert np.array_equal(O.fq_weight(W, 1), W.astype(np.float64))
    g8, u8, a8, y8 = O.expert_ffn_fwd_fp8(X.astype(np.float64), Wg, Wu, Wd, 1)
    g, u, a, y = O.expert_ffn_fwd(X, Wg, Wu, Wd)
    assert np.abs(g8 - g).max() <= 1e-13 * np.abs(g).max() and np.abs(u8 - u).max() <= 1e-13 * np.abs(u).max()
    assert np.abs(a8 - a).max() <= 1e-13 * np.abs(a).max()
    y_ref = _torch_fq_1x128_pow2(a) @ Wd.astype(np.float64).T
    assert np.abs(y8 - y_ref).max() <= 1e-12 * np.abs(y_ref).max()
    assert 1e-3 < O.rel_fro(y8, y) < 0.06          # Q-a is really there (dropping it gives exactly 0)


def test_fp8_composition_identity_grid_backward():
    """Same construction for the dgrad: dY on the grid => Q-dY is the identity, and because the gating weight
    is applied AFTER the GEMM, dg/du equal the unquantised backward of dy = w*dY (quantising w*dY instead
    would move them by ~3 %).  dX differs only by Q-dgu; the wgrad reads the bf16-rounded tensors."""
    rng = np.random.default_rng(12)
    n, H, F = 24, 256, 256
    X = _on_grid(rng, (n, H), (1, 128), -9, -6)
    dY = _on_grid(rng, (n, H), (1, 128))
    Wg, Wu = _on_grid(rng, (F, H), (128, 128), -9, -5), _on_grid(rng, (F, H), (128, 128), -9, -5)
    Wd = _on_grid(rng, (H, F), (128, 128), -9, -5)
    wr = rng.uniform(0.05, 0.6, n)                                          # generic weights: w*dY is OFF the grid
    dy = wr[:, None] * dY.astype(np.float64)
    assert O.rel_fro(O.fq_act(dy, 1), dy) > 1e-3
    g, u, a, y = O.expert_ffn_fwd(X, Wg, Wu, Wd)
    dX8, dWg8, dWu8, dWd8, dg8, du8 = O.expert_ffn_bwd_fp8(dY.astype(np.float64), wr, dy, X.astype(np.float64),
                                                            g, u, a, Wg, Wu, Wd, 1)
    dX, dWg, dWu, dWd, dg, du = O.expert_ffn_bwd(dy, X, g, u, a, Wg, Wu, Wd)
    assert np.abs(dg8 - dg).max() <= 1e-12 * np.abs(dg).max() and np.abs(du8 - du).max() <= 1e-12 * np.abs(du).max()
    dX_ref = _torch_fq_1x128_pow2(dg) @ Wg.astype(np.float64) + _torch_fq_1x128_pow2(du) @ Wu.astype(np.float64)
    assert np.abs(dX8 - dX_ref).max() <= 1e-12 * np.abs(dX_ref).max()
    assert 1e-3 < O.rel_fro(dX8, dX) < 0.06

    def b(v):
        return torch.from_numpy(np.asarray(v, np.float32)).to(torch.bfloat16).double().numpy()

    assert np.abs(dWd8 - b(dy).T @ b(a)).max() <= 1e-12 * np.abs(dWd).max()
    assert np.abs(dWg8 - b(dg).T @ X.astype(np.float64)).max() <= 1e-12 * np.abs(dWg).max()
    assert np.abs(dWu8 - b(du).T @ X.astype(np.float64)).max() <= 1e-12 * np.abs(dWu).max()


def test_fp8_layer_quantises_x_once_per_token_and_dy_unweighted():
    """Layer-level composition: on grid inputs the FP8 layer's saved g, u equal the bf16-oracle layer's, for the
    routed AND the shared expert, and the backward's dg match (Q-X / Q-dY sit on the un-permuted [T,H] tensors)."""
    rng = np.random.default_rng(13)
    c = wl.DSV3_FP8_SMALL.replace(T=64, H=256, F=128, F_shared=128, E=8, K=2, n_group=1, topk_group=1, fp8_scale_mode=1)
    X = _on_grid(rng, (c.T, c.H), (1, 128), -9, -6); dY = _on_grid(rng, (c.T, c.H), (1, 128))
    Wr = wl.gen_Wr(c); b = wl.gen_bias(c)
    W = tuple(np.stack([_on_grid(rng, s, (128, 128), -9, -5) for _ in range(c.E)])
              for s in ((c.F, c.H), (c.F, c.H), (c.H, c.F)))
    sh = (_on_grid(rng, (c.F_shared, c.H), (128, 128), -9, -5), _on_grid(rng, (c.F_shared, c.H), (128, 128), -9, -5),
          _on_grid(rng, (c.H, c.F_shared), (128, 128), -9, -5))
    f8 = O.layer_fwd(c, X, Wr, b, W, sh)
    f = O.layer_fwd(c.replace(dtype=1), X, Wr, b, W, sh)
    for k in ("g", "u", "a"):
        assert np.abs(f8[k] - f[k]).max() <= 1e-12 * np.abs(f[k]).max(), k
        assert np.abs(f8["shared"][k] - f["shared"][k]).max() <= 1e-12 * np.abs(f["shared"][k]).max(), k
    assert 1e-3 < O.rel_fro(f8["y"], f["y"]) < 0.06
    b8 = O.layer_bwd(c, dY, X, Wr, W, f8, sh)
    # the unquantised backward evaluated at the FP8 forward's saved g, u, a (only y differs between the two)
    bb = O.layer_bwd(c.replace(dtype=1), dY, X, Wr, W, dict(f8), sh)
    for k in ("dg", "du"):
        assert np.abs(b8[k] - bb[k]).max() <= 1e-12 * np.abs(bb[k]).max(), k
    assert 1e-3 < O.rel_fro(b8["dX"], bb["dX"]) < 0.06
