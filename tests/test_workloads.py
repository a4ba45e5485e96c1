"""Input recipe checks: determinism, storage-dtype exactness, skew statistics."""
import numpy as np

import workloads as wl


def test_streams_are_deterministic_and_independent():
    a = wl.gen_X(wl.TINY); b = wl.gen_X(wl.TINY)
    assert np.array_equal(a, b)
    assert not np.array_equal(wl.gen_X(wl.TINY.replace(seed=1)), a)
    g0, u0, _ = wl.gen_expert_weights(wl.TINY, 0)
    g1, _, _ = wl.gen_expert_weights(wl.TINY, 1)
    assert not np.array_equal(g0, g1) and not np.array_equal(g0, u0)


def test_parallel_generation_is_thread_count_invariant():
    c = wl.QWEN3_SMALL
    a = wl.gen_all_expert_weights(c, threads=1)
    b = wl.gen_all_expert_weights(c, threads=4)
    for x, y in zip(a, b):
        assert np.array_equal(x, y)


def test_bf16_round_trip_and_rne():
    x = np.array([1.0, 1.00390625, 1.01171875, -3.1415927, 65504.0, 1e-3], np.float32)
    # 1 + 2^-8 is a tie between 1.0 and 1+2^-7 -> even (1.0); 1 + 3*2^-8 ties -> 1+2^-6
    r = wl.bf16_bits_to_f32(wl.f32_to_bf16_bits(x))
    assert r[0] == 1.0 and r[1] == 1.0 and r[2] == np.float32(1.015625)
    assert np.array_equal(wl.bf16_bits_to_f32(wl.f32_to_bf16_bits(r)), r)
    X = wl.gen_X(wl.QWEN3_SMALL)
    assert np.array_equal(wl.round_to_storage(X, wl.DTYPE_BF16), X)      # already on the bf16 grid
    assert abs(X.std() - 1.0) < 0.02 and abs(X.mean()) < 0.02


def test_tiny_config_stds():
    c = wl.TINY
    Wg, Wu, Wd = wl.gen_expert_weights(c, 3)
    assert abs(Wg.std() * np.sqrt(c.H) - 1) < 0.05 and abs(Wd.std() * np.sqrt(c.F) - 1) < 0.05
    assert abs(wl.gen_Wr(c).std() - 0.02) < 0.003


def test_zipf_skew_statistics_configs4():
    """SURVEY.md §8d configs[5]: top-6 experts ~41% of rows, 8 experts empty (-30 offset)."""
    c = wl.GPTOSS
    o = wl.zipf_offsets(c)
    assert (o == -30).sum() == 8 and o.max() == 0.0
    rng = np.random.default_rng(0)
    z = rng.standard_normal((4096, c.E)).astype(np.float32) * 0.91 + o[None, :]
    idx = np.argsort(-z, axis=1)[:, :c.K]
    cnt = np.bincount(idx.reshape(-1), minlength=c.E)
    share = np.sort(cnt)[::-1][:6].sum() / cnt.sum()
    assert 0.33 < share < 0.5
    assert (cnt == 0).sum() >= 8


def test_flop_counts():
    f = wl.QWEN3.flops_fwd_bwd()
    assert abs(f["routed"] / 1e12 - 1.855) < 0.001 and f["shared"] == 0
    assert abs(wl.DSV3.flops_fwd_bwd()["routed"] / 1e12 - 8.66) < 0.01
