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
