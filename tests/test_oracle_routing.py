"""Pins for the oracle's routing and permutation (SURVEY.md §8c "What pins each part").
None of these re-type the oracle's own formula: they use brute force, invariants the paper states
(PAPER.md:436), closed forms, and reductions to simpler cases."""
import itertools

import numpy as np
import pytest

import workloads as wl
from oracle import moe_oracle as O


def brute_topk(keys, K):
    """Full sort with the (key desc, index asc) comparator, pure Python."""
    out = []
    for row in keys:
        order = sorted(range(len(row)), key=lambda e: (-float(row[e]), e))
        out.append(order[:K])
    return np.array(out, np.int32)


def test_topk_bruteforce_with_handmade_ties():
    keys = np.array([[1.0, 3.0, 3.0, 2.0, 3.0, -1.0],
                     [0.0, 0.0, 0.0, 0.0, 0.0, 0.0],
                     [5.0, 4.0, 3.0, 2.0, 1.0, 0.0],
                     [-2.0, -1.0, -1.0, -3.0, -1.0, -1.0]])
    got = O.topk_select(keys, 3)
    assert np.array_equal(got, brute_topk(keys, 3))
    assert got[0].tolist() == [1, 2, 4] and got[1].tolist() == [0, 1, 2] and got[3].tolist() == [1, 2, 4]


@pytest.mark.parametrize("seed", [0, 1, 2])
def test_topk_bruteforce_random_with_ties(seed):
    c = wl.MoEConfig("t", T=64, H=8, E=24, K=5, F=8, seed=seed)
    z = wl.gen_logits(c, ties=3)
    idx, w = O.route(z, None, c)
    assert np.array_equal(idx, brute_topk(z, c.K))


def test_routing_validity_paper_b22():
    """IDs in [0, num_experts); weights non-negative and sum to 1 over the top-k."""
    for c in (wl.TINY, wl.QWEN3_SMALL, wl.GPTOSS_SMALL, wl.DSV3_SMALL):
        z = wl.gen_logits(c)
        idx, w = O.route(z, wl.gen_bias(c), c)
        assert idx.min() >= 0 and idx.max() < c.E
        assert all(len(set(r)) == c.K for r in idx.tolist())                # distinct per token
        assert (w >= 0).all()
        assert np.abs(w.sum(axis=1) - c.routed_scale).max() < 1e-12


def test_softmax_order_closed_form():
    """softmax-over-all -> top-k -> renormalise (Qwen3 style) == top-k -> softmax-over-k (GPT-OSS style)."""
    c = wl.QWEN3_SMALL
    z = wl.gen_logits(c).astype(np.float64)
    idx, w = O.route(z, None, c)
    p = np.exp(z) / np.exp(z).sum(axis=1, keepdims=True)                    # softmax over all experts
    top = np.argsort(-p, axis=1, kind="stable")[:, :c.K]
    ps = np.take_along_axis(p, top, axis=1)
    assert np.array_equal(top, idx)
    assert np.abs(ps / ps.sum(axis=1, keepdims=True) - w).max() < 1e-14


def test_no_renorm_softmax_is_full_softmax():
    c = wl.QWEN3_SMALL.replace(renorm=0)
    z = wl.gen_logits(c).astype(np.float64)
    idx, w = O.route(z, None, c)
    p = np.exp(z) / np.exp(z).sum(axis=1, keepdims=True)
    assert np.abs(np.take_along_axis(p, idx.astype(np.int64), axis=1) - w).max() < 1e-15


def test_sigmoid_path_special_case():
    """b = 0, c = 1  =>  w = s / sum(s) and selection == plain top-k on z (sigmoid is monotone)."""
    c = wl.DSV3_SMALL.replace(n_group=1, topk_group=1, routed_scale=1.0, has_bias=0)
    z = wl.gen_logits(c).astype(np.float64)
    idx, w = O.route(z, None, c)
    assert np.array_equal(idx, brute_topk(z, c.K))
    s = 1 / (1 + np.exp(-np.take_along_axis(z, idx.astype(np.int64), axis=1)))
    assert np.abs(s / s.sum(axis=1, keepdims=True) - w).max() < 1e-15


def test_bias_is_selection_only():
    c = wl.DSV3_SMALL
    z = wl.gen_logits(c).astype(np.float64)
    b = np.zeros(c.E, np.float32); b[5] = 10.0                              # expert 5 always selected first
    idx, w = O.route(z, b, c)
    assert (idx[:, 0] == 5).all()
    s5 = 1 / (1 + np.exp(-z[:, 5]))
    ssum = (1 / (1 + np.exp(-np.take_along_axis(z, idx.astype(np.int64), axis=1)))).sum(axis=1)
    assert np.abs(w[:, 0] - c.routed_scale * s5 / ssum).max() < 1e-14       # the bias is not in w


def test_zipf_offset_is_a_selection_offset_on_the_softmax_path():
    """configs[4] reading (S21): the Zipf per-expert offset o[e] skews WHICH experts are chosen
    (key = z + o) while the gating weights are the softmax over the chosen experts' UNBIASED logits.
    Selection is pinned by brute force on z + o, the weights by torch.softmax on the gathered z, and the
    load skew (top 5 % of experts ~ 40 % of the rows, empty experts exist) by counting."""
    import torch
    c = wl.GPTOSS_SMALL
    z = wl.gen_logits(c).astype(np.float64)
    o = wl.gen_bias(c)
    idx, w = O.route(z, o, c)
    assert np.array_equal(idx, brute_topk(z + o.astype(np.float64)[None, :], c.K))
    zs = torch.from_numpy(np.take_along_axis(z, idx.astype(np.int64), axis=1))
    assert np.abs(w - torch.softmax(zs, dim=1).numpy()).max() < 1e-15
    w_biased = torch.softmax(zs + torch.from_numpy(o.astype(np.float64))[torch.from_numpy(idx.astype(np.int64))], dim=1).numpy()
    assert np.abs(w - w_biased).max() > 1e-2                                # the two readings really differ
    cfull = wl.GPTOSS
    counts = np.bincount(O.route(wl.gen_logits(cfull).astype(np.float64), wl.gen_bias(cfull), cfull)[0].reshape(-1),
                         minlength=cfull.E)
    top = np.sort(counts)[::-1]
    assert 0.35 < top[:6].sum() / counts.sum() < 0.55 and (counts == 0).sum() >= 4


def test_group_limit_reductions_and_membership():
    c = wl.DSV3_SMALL
    z = wl.gen_logits(c).astype(np.float64)
    b = wl.gen_bias(c)
    plain, _ = O.route(z, b, c.replace(n_group=1, topk_group=1))
    allg, _ = O.route(z, b, c.replace(topk_group=c.n_group))
    assert np.array_equal(plain, allg)                                      # Kg = G reduces to plain top-k
    idx, _ = O.route(z, b, c)
    per = c.E // c.n_group
    grp = idx // per
    assert max(len(set(r)) for r in grp.tolist()) <= c.topk_group           # <= Kg distinct groups
    # every selected expert lies in a kept group, recomputed by brute force
    key = (1 / (1 + np.exp(-z))) + b[None, :].astype(np.float64)
    for t in range(0, c.T, 37):
        sc = []
        for g in range(c.n_group):
            v = sorted(key[t, g * per:(g + 1) * per], reverse=True)
            sc.append(v[0] + v[1])
        kept = sorted(range(c.n_group), key=lambda g: (-sc[g], g))[:c.topk_group]
        assert set(grp[t].tolist()) <= set(kept)
        cand = [e for e in range(c.E) if e // per in kept]
        want = sorted(cand, key=lambda e: (-key[t, e], e))[:c.K]
        assert idx[t].tolist() == want


def test_group_score_max_variant():
    c = wl.DSV3_SMALL.replace(group_score=0)
    z = wl.gen_logits(c).astype(np.float64)
    idx, _ = O.route(z, None, c.replace(has_bias=0))
    per = c.E // c.n_group
    key = 1 / (1 + np.exp(-z))
    for t in range(0, c.T, 61):
        sc = [key[t, g * per:(g + 1) * per].max() for g in range(c.n_group)]
        kept = sorted(range(c.n_group), key=lambda g: (-sc[g], g))[:c.topk_group]
        assert set((idx[t] // per).tolist()) <= set(kept)


def test_fp32_key_mode_matches_fp64_away_from_ties():
    c = wl.DSV3_SMALL
    z = wl.gen_logits(c)
    b = wl.gen_bias(c)
    i64, _ = O.route(z, b, c)
    i32, _ = O.route(z, b, c, key_dtype=np.float32)
    assert (i64 != i32).any(axis=1).mean() < 0.01                           # only near-ties may differ


# ------------------------------------------------------------------ permutation (R6)

@pytest.mark.parametrize("row_align", [1, 16, 128])
def test_permutation_invariants(row_align):
    for c in (wl.TINY, wl.GPTOSS_SMALL):
        z = wl.gen_logits(c)
        idx, w = O.route(z, wl.gen_bias(c), c)
        counts, off, p2f, f2p = O.permute_maps(idx, c.E, row_align)
        TK = c.T * c.K
        assert counts.sum() == TK and len(off) == c.E + 1 and off[0] == 0
        assert (off % row_align == 0).all() and p2f.size == off[-1]
        valid = p2f[p2f >= 0]
        assert np.array_equal(np.sort(valid), np.arange(TK))                # bijection on [0, TK)
        assert np.array_equal(p2f[f2p], np.arange(TK))                      # p2f o f2p = id
        tok = valid // c.K
        assert (np.bincount(tok, minlength=c.T) == c.K).all()               # each token exactly K times
        for e in range(c.E):
            seg = p2f[off[e]:off[e + 1]]
            n = counts[e]
            assert (seg[:n] >= 0).all() and (seg[n:] == -1).all()
            assert (np.diff(seg[:n]) > 0).all()                             # ascending flat position
            assert (idx.reshape(-1)[seg[:n]] == e).all()
            assert off[e + 1] - off[e] == -(-n // row_align) * row_align
        if c is wl.GPTOSS_SMALL:
            assert (counts == 0).sum() >= 1                                 # empty experts exist


def test_permutation_bruteforce_tiny():
    idx = np.array([[2, 0], [1, 2], [0, 1], [2, 1]], np.int32)
    counts, off, p2f, f2p = O.permute_maps(idx, 4, 1)
    assert counts.tolist() == [2, 3, 3, 0] and off.tolist() == [0, 2, 5, 8, 8]
    assert p2f.tolist() == [1, 4, 2, 5, 7, 0, 3, 6]
    assert f2p.tolist() == [5, 0, 2, 6, 1, 3, 7, 4]
    counts, off, p2f, f2p = O.permute_maps(idx, 4, 4)
    assert off.tolist() == [0, 4, 8, 12, 12]
    assert p2f.tolist() == [1, 4, -1, -1, 2, 5, 7, -1, 0, 3, 6, -1]


@pytest.mark.parametrize("K", [2, 4, 8])
def test_permute_combine_identity_bit_exact(K):
    """w == 1/K (a power of two): combine(permute(X)) == X bit-exactly, even on bf16-grid values."""
    c = wl.QWEN3_SMALL.replace(K=K, T=300)
    X = wl.gen_X(c)
    idx, _ = O.route(wl.gen_logits(c), None, c)
    _, _, p2f, f2p = O.permute_maps(idx, c.E, 16)
    Xp = O.permute_rows(X, p2f, K)
    Y = O.unpermute_combine(Xp, np.full((c.T, K), 1.0 / K), f2p)
    assert np.array_equal(Y, X.astype(np.float64))
    assert (Xp[p2f < 0] == 0).all()
