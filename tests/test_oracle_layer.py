"""Pins for the oracle's expert FFN, combine and backward: special cases that reduce to
library routines (numpy.matmul / einsum, torch.nn.functional.silu, torch.autograd on an independent
dense-masked formulation), invariances, and central finite differences on configs[0]."""
import numpy as np
import pytest
import torch

import workloads as wl
from oracle import moe_oracle as O


def _inputs(c):
    X = wl.gen_X(c); Wr = wl.gen_Wr(c); b = wl.gen_bias(c)
    W = wl.gen_all_expert_weights(c, threads=4)
    sh = wl.gen_shared_weights(c)
    dY = wl.gen_dY(c)
    return X, Wr, b, W, sh, dY


def test_single_expert_is_dense_swiglu_ffn():
    """E = 1, K = 1  =>  textbook dense SwiGLU FFN, gate weight exactly 1."""
    c = wl.MoEConfig("dense", T=40, H=32, E=1, K=1, F=48, dtype=0, w_std=-1.0)
    X, Wr, b, W, sh, dY = _inputs(c)
    f = O.layer_fwd(c, X, Wr, b, W)
    assert np.array_equal(f["w"], np.ones((c.T, 1)))
    Xt = torch.from_numpy(X).double()
    g = Xt @ torch.from_numpy(W[0][0]).double().T
    u = Xt @ torch.from_numpy(W[1][0]).double().T
    ref = (torch.nn.functional.silu(g) * u) @ torch.from_numpy(W[2][0]).double().T
    assert np.abs(f["Y"] - ref.numpy()).max() < 1e-12


def test_equal_counts_is_batched_matmul():
    """Round-robin routing with equal counts  =>  einsum over [E, n, H]."""
    c = wl.MoEConfig("rr", T=48, H=16, E=4, K=1, F=24, dtype=0, w_std=-1.0)
    X, Wr, b, W, sh, dY = _inputs(c)
    forced = (np.arange(c.T) % c.E).astype(np.int32)[:, None]
    f = O.layer_fwd(c, X, Wr, b, W, forced_idx=forced)
    Xe = X.astype(np.float64).reshape(c.T // c.E, c.E, c.H).transpose(1, 0, 2)          # [E, n, H]
    g = np.einsum("enh,efh->enf", Xe, W[0].astype(np.float64))
    u = np.einsum("enh,efh->enf", Xe, W[1].astype(np.float64))
    a = g / (1 + np.exp(-g)) * u
    y = np.einsum("enf,ehf->enh", a, W[2].astype(np.float64))
    ref = y.transpose(1, 0, 2).reshape(c.T, c.H)                                        # w == 1 (K = 1)
    assert np.abs(f["Y"] - ref).max() < 1e-12


def test_shared_weight_set_invariance():
    """All experts share one weight set  =>  Y = FFN(X) whatever the routing (sum_j w_j = 1)."""
    c = wl.QWEN3_SMALL.replace(T=64, H=64, F=32, E=8, K=4)
    X, Wr, b, W, sh, dY = _inputs(c)
    W1 = tuple(np.repeat(w[:1], c.E, axis=0) for w in W)
    f = O.layer_fwd(c, X, Wr, b, W1)
    _, _, _, y = O.expert_ffn_fwd(X, W1[0][0], W1[1][0], W1[2][0])
    assert np.abs(f["Y"] - y).max() < 1e-13


def _torch_dense_layer(c, X, Wr, b, W, sh, idx):
    """Independent formulation for autograd: dense gating matrix, every expert applied to every token,
    selection (an integer decision, no gradient) taken from idx."""
    dd = torch.float64
    Xt = torch.tensor(X, dtype=dd, requires_grad=True)
    Wrt = torch.tensor(Wr, dtype=dd, requires_grad=True)
    Wt = [torch.tensor(w, dtype=dd, requires_grad=True) for w in W]
    z = Xt @ Wrt.T
    sel = torch.zeros(c.T, c.E, dtype=torch.bool)
    sel[torch.arange(c.T)[:, None], torch.tensor(idx, dtype=torch.long)] = True
    if c.score_fn == 0:
        if c.renorm:
            gate = torch.softmax(z.masked_fill(~sel, float("-inf")), dim=1)
        else:
            gate = torch.softmax(z, dim=1) * sel
    else:
        s = torch.sigmoid(z) * sel
        gate = s / (s.sum(dim=1, keepdim=True) + 1e-20) if c.renorm else s
    gate = gate * c.routed_scale
    Y = torch.zeros(c.T, c.H, dtype=dd)
    for e in range(c.E):
        h = torch.nn.functional.silu(Xt @ Wt[0][e].T) * (Xt @ Wt[1][e].T)
        Y = Y + gate[:, e:e + 1] * (h @ Wt[2][e].T)
    sht = None
    if sh is not None:
        sht = [torch.tensor(w, dtype=dd, requires_grad=True) for w in sh]
        Y = Y + (torch.nn.functional.silu(Xt @ sht[0].T) * (Xt @ sht[1].T)) @ sht[2].T
    return Y, Xt, Wrt, Wt, sht


@pytest.mark.parametrize("variant", ["softmax", "softmax_norenorm", "sigmoid_group_shared", "sigmoid_norenorm"])
def test_backward_matches_autograd_of_dense_formulation(variant):
    base = wl.MoEConfig("g", T=96, H=48, E=8, K=3, F=40, dtype=0, w_std=-1.0)
    c = {"softmax": base,
         "softmax_norenorm": base.replace(renorm=0),
         "sigmoid_group_shared": base.replace(score_fn=1, n_group=4, topk_group=2, K=3, routed_scale=2.5,
                                              has_bias=1, bias_kind="normal", F_shared=24),
         "sigmoid_norenorm": base.replace(score_fn=1, renorm=0, routed_scale=2.5)}[variant]
    X, Wr, b, W, sh, dY = _inputs(c)
    Wr = Wr * 20                                             # make the gate far from uniform
    f = O.layer_fwd(c, X, Wr, b, W, sh)
    bw = O.layer_bwd(c, dY, X, Wr, W, f, sh)
    Y, Xt, Wrt, Wt, sht = _torch_dense_layer(c, X, Wr, b, W, sh, f["idx"])
    assert np.abs(Y.detach().numpy() - f["Y"]).max() < 1e-11
    (Y * torch.tensor(dY, dtype=torch.float64)).sum().backward()
    tol = 1e-10
    assert O.rel_fro(bw["dX"], Xt.grad.numpy()) < tol
    assert O.rel_fro(bw["dWr"], Wrt.grad.numpy()) < tol
    assert O.rel_fro(bw["dWg"], Wt[0].grad.numpy()) < tol
    assert O.rel_fro(bw["dWu"], Wt[1].grad.numpy()) < tol
    assert O.rel_fro(bw["dWd"], Wt[2].grad.numpy()) < tol
    if sh is not None:
        for k, t in zip(("dWg_s", "dWu_s", "dWd_s"), sht):
            assert O.rel_fro(bw[k], t.grad.numpy()) < tol
    # structural invariants of dz (SURVEY.md §8c "gradients" pin)
    dzs = np.take_along_axis(bw["dz"], f["idx"].astype(np.int64), axis=1)
    if c.score_fn == 0 and c.renorm:
        assert np.abs(dzs.sum(axis=1)).max() < 1e-12        # sum over selected dz_j = 0
    assert np.count_nonzero(bw["dz"]) <= c.T * c.K or not c.renorm or c.score_fn == 1
    if c.score_fn == 1 and c.renorm:
        zs = np.take_along_axis(f["z"], f["idx"].astype(np.int64), axis=1)
        s = 1 / (1 + np.exp(-zs))
        ds = dzs / (s * (1 - s))
        assert np.abs((s * ds).sum(axis=1)).max() < 1e-10   # degree-0 homogeneity: sum_i s_i ds_i = 0


def test_finite_differences_tiny_config():
    """north_star: finite-difference gradients on the tiny config (central, h = 1e-6, rel err <= 1e-6)."""
    c = wl.TINY
    X, Wr, b, W, sh, dY = _inputs(c)
    X = X.astype(np.float64); Wr = Wr.astype(np.float64)
    W = tuple(w.astype(np.float64) for w in W)
    f = O.layer_fwd(c, X, Wr, b, W)
    bw = O.layer_bwd(c, dY, X, Wr, W, f)

    def loss(X_, Wr_, W_):
        ff = O.layer_fwd(c, X_, Wr_, b, W_)
        return (ff["Y"] * dY).sum(), ff["idx"]

    rng = np.random.default_rng(0)
    h = 1e-6
    checked = 0
    tensors = {"X": (X, bw["dX"]), "Wr": (Wr, bw["dWr"]), "Wg": (W[0], bw["dWg"]),
               "Wu": (W[1], bw["dWu"]), "Wd": (W[2], bw["dWd"])}
    for name, (A, dA) in tensors.items():
        for _ in range(6):
            pos = tuple(rng.integers(0, s) for s in A.shape)
            old = A[pos]
            A[pos] = old + h; lp, ip = loss(X, Wr, W)
            A[pos] = old - h; lm, im = loss(X, Wr, W)
            A[pos] = old
            if not (np.array_equal(ip, f["idx"]) and np.array_equal(im, f["idx"])):
                continue                                     # a top-k flip: not differentiable there
            fd = (lp - lm) / (2 * h)
            an = dA[pos]
            assert abs(fd - an) <= 1e-6 * max(1.0, abs(an)) + 1e-7, (name, pos, fd, an)
            checked += 1
    assert checked >= 25


def test_empty_expert_has_zero_weight_grads():
    c = wl.GPTOSS_SMALL.replace(T=200, H=64, F=64)
    X, Wr, b, W, sh, dY = _inputs(c)
    f = O.layer_fwd(c, X, Wr, b, W)
    bw = O.layer_bwd(c, dY, X, Wr, W, f)
    empty = np.where(f["counts"] == 0)[0]
    assert len(empty) >= 1
    for e in empty:
        assert not bw["dWg"][e].any() and not bw["dWu"][e].any() and not bw["dWd"][e].any()
    assert (f["g"][f["perm_to_flat"] < 0] == 0).all()


def test_row_align_does_not_change_results():
    c = wl.QWEN3_SMALL.replace(T=128, H=64, F=32)
    X, Wr, b, W, sh, dY = _inputs(c)
    f1 = O.layer_fwd(c, X, Wr, b, W)
    f2 = O.layer_fwd(c.replace(row_align=128), X, Wr, b, W)
    assert np.abs(f1["Y"] - f2["Y"]).max() < 1e-14
    b1 = O.layer_bwd(c, dY, X, Wr, W, f1)
    b2 = O.layer_bwd(c.replace(row_align=128), dY, X, Wr, W, f2)
    for k in ("dX", "dWr", "dWg", "dWu", "dWd"):
        assert np.abs(b1[k] - b2[k]).max() < 1e-12
