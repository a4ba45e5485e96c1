"""Pins for the oracle's widened rows (readings A1..A3, V1, V2): the auxiliary global-level
load-balancing loss, the threshold-gated variable-k router and the
zero-computation experts.  None re-types the oracle: closed forms, brute force in pure Python,
special cases with a known answer, and torch.autograd on an independent dense formulation."""
import numpy as np
import pytest
import torch

import workloads as wl
from oracle import moe_oracle as O

DD = torch.float64


def _inputs(c):
    X = wl.gen_X(c); Wr = wl.gen_Wr(c); b = wl.gen_bias(c)
    W = wl.gen_all_expert_weights(c, threads=4)
    sh = wl.gen_shared_weights(c)
    dY = wl.gen_dY(c)
    return X, Wr, b, W, sh, dY


# ------------------------------------------------------------------------------------------------------------
# A1..A3  auxiliary load-balancing loss
# ------------------------------------------------------------------------------------------------------------

def test_aux_loss_closed_forms():
    """Perfect balance: f_e = 1/E and p uniform => L = coef * E * E * (1/E)(1/E) = coef exactly.  Total collapse onto one
    expert with p -> one-hot => L -> coef * E (the maximum); the loss is what [30] calls E * sum f P scaled by the coefficient."""
    c = wl.MoEConfig("aux", T=64, H=8, E=8, K=2, F=8, dtype=0, aux_coef=1e-3)
    z = np.zeros((c.T, c.E))
    idx = np.stack([np.arange(c.T) % c.E, (np.arange(c.T) + 4) % c.E], axis=1).astype(np.int32)   # 16 assignments per expert
    L, f, P = O.aux_loss(c, z, idx)
    assert np.allclose(f, 1 / c.E, atol=0, rtol=1e-15) and np.allclose(P, 1 / c.E, rtol=1e-15)
    assert abs(L - c.aux_coef) < 1e-18
    z2 = np.full((c.T, c.E), -40.0); z2[:, 3] = 40.0
    idx2 = np.full((c.T, 1), 3, np.int32)
    L2, f2, P2 = O.aux_loss(c.replace(K=1), z2, idx2)
    assert f2[3] == 1.0 and abs(L2 - c.aux_coef * c.E) < 1e-12
    # a caller-supplied global fraction vector replaces the batch's own counts (global-level balance)
    fg = np.arange(1, c.E + 1, dtype=np.float64); fg /= fg.sum()
    L3, f3, _ = O.aux_loss(c, z, idx, f_global=fg)
    assert np.array_equal(f3, fg) and abs(L3 - c.aux_coef * c.E * (fg / c.E).sum()) < 1e-18
    # variable-k: f divides by the number of assignments actually made
    idx4 = idx.copy(); idx4[::2, 1] = -1
    _, f4, _ = O.aux_loss(c, z, idx4)
    assert abs(f4.sum() - 1.0) < 1e-15 and np.bincount(idx4[idx4 >= 0], minlength=c.E)[0] / (idx4 >= 0).sum() == f4[0]


@pytest.mark.parametrize("score_fn", [0, 1])
def test_aux_gradient_matches_autograd_and_finite_differences(score_fn):
    c = wl.MoEConfig("aux", T=24, H=8, E=10, K=3, F=8, dtype=0, score_fn=score_fn, aux_coef=0.37,
                     n_zero=1, n_copy=1, aux_zc_weight=0.25)
    rng = np.random.default_rng(3)
    z = rng.standard_normal((c.T, c.E)) * 1.5
    f = rng.random(c.E); f /= f.sum()
    dz = O.aux_dz(c, z, f)
    zt = torch.tensor(z, dtype=DD, requires_grad=True)
    p = torch.softmax(zt, dim=1) if score_fn == 0 else torch.sigmoid(zt) / torch.sigmoid(zt).sum(dim=1, keepdim=True)
    eta = torch.ones(c.E, dtype=DD); eta[-2:] = c.aux_zc_weight
    L = c.aux_coef * c.E * (eta * torch.tensor(f, dtype=DD) * p.mean(dim=0)).sum()
    L.backward()
    assert np.abs(dz - zt.grad.numpy()).max() < 1e-15
    assert abs(float(L.detach()) - O.aux_loss(c, z, None, f_global=f)[0]) < 1e-15
    if score_fn == 0:
        assert np.abs(dz.sum(axis=1)).max() < 1e-16           # softmax: the gradient is orthogonal to the all-ones direction
    h = 1e-6
    for t, j in ((0, 0), (5, 9), (23, 4)):
        zp = z.copy(); zp[t, j] += h
        zm = z.copy(); zm[t, j] -= h
        fd = (O.aux_loss(c, zp, None, f_global=f)[0] - O.aux_loss(c, zm, None, f_global=f)[0]) / (2 * h)
        assert abs(fd - dz[t, j]) < 1e-8


# ------------------------------------------------------------------------------------------------------------
# V1  threshold-gated variable-k routing
# ------------------------------------------------------------------------------------------------------------

def _brute_threshold(s, thr, K):
    out = []
    for row in s:
        act = [e for e in range(len(row)) if row[e] > thr[e]]
        act.sort(key=lambda e: (-float(row[e]), e))
        if not act:
            act = [min(range(len(row)), key=lambda e: (-float(row[e]), e))]
        out.append((act[:K] + [-1] * K)[:K])
    return np.array(out, np.int32)


def test_threshold_router_bruteforce_and_validity():
    c = wl.MoEConfig("dyn", T=400, H=16, E=16, K=4, F=8, dtype=0, score_fn=1, route_mode=1)
    z = wl.gen_logits(c).astype(np.float64)
    thr = wl.gen_threshold(c)
    idx, w = O.route(z, None, c, threshold=thr)
    s = 1 / (1 + np.exp(-z))
    assert np.array_equal(idx, _brute_threshold(s, thr.astype(np.float64), c.K))
    k = (idx >= 0).sum(axis=1)
    assert k.min() >= 1 and k.max() == c.K and len(set(k.tolist())) >= 3          # the count really varies per token
    assert ((s > thr[None, :]).sum(axis=1) == 0).any()                            # ... and the top-1 fallback is exercised
    assert ((s > thr[None, :]).sum(axis=1) > c.K).any()                           # ... and so is the K-slot cap
    # PAPER.md:436 carries over: ids in range or empty, weights >= 0, sum to 1 over the selected experts, 0 on empty slots
    assert ((idx >= -1) & (idx < c.E)).all() and (w >= 0).all()
    assert np.abs(w.sum(axis=1) - 1.0).max() < 1e-12 and (w[idx < 0] == 0).all()
    for t in range(c.T):
        sel = idx[t][idx[t] >= 0]
        assert len(set(sel.tolist())) == len(sel)
    # hand-made ties: equal gates -> lower index first; threshold is strict (s == thr is NOT active)
    z2 = np.zeros((2, 4)); thr2 = np.array([0.4, 0.4, 0.5, 0.6], np.float32)
    i2, w2 = O.route(z2, None, c.replace(T=2, E=4, K=3), threshold=thr2)
    assert i2.tolist() == [[0, 1, -1], [0, 1, -1]] and np.allclose(w2[:, :2], 0.5)
    # fixed top-k is the special case "threshold below every gate, K slots": same experts as R4 on the sigmoid keys
    i3, _ = O.route(z, None, c, threshold=np.full(c.E, -1.0, np.float32))
    assert np.array_equal(i3, O.topk_select(s, c.K))


def test_permutation_with_empty_slots():
    c = wl.MoEConfig("dyn", T=300, H=16, E=12, K=4, F=8, dtype=0, score_fn=1, route_mode=1)
    idx, _ = O.route(wl.gen_logits(c).astype(np.float64), None, c, threshold=wl.gen_threshold(c))
    for align in (1, 128):
        counts, offsets, p2f, f2p = O.permute_maps(idx, c.E, align)
        n = int((idx >= 0).sum())
        assert counts.sum() == n and (p2f >= 0).sum() == n
        flat = idx.reshape(-1)
        assert ((f2p >= 0) == (flat >= 0)).all()                                   # an empty slot owns no row
        ok = np.nonzero(flat >= 0)[0]
        assert np.array_equal(p2f[f2p[ok]], ok)                                    # bijection on the occupied slots
        for e in range(c.E):
            rows = p2f[offsets[e]:offsets[e] + counts[e]]
            assert (flat[rows] == e).all() and (np.diff(rows) > 0).all()           # stable: ascending flat position
        assert (p2f[offsets[-1]:] < 0).all() if p2f.size > offsets[-1] else True


# ------------------------------------------------------------------------------------------------------------
# V2  zero-computation experts
# ------------------------------------------------------------------------------------------------------------

def test_zero_computation_experts_special_cases():
    """K = 1 and every token forced onto one zero-computation expert: Y = 0 (zero), Y = X (copy), Y = v (constant);
    the FFN experts then see no token and get exactly zero gradients."""
    c = wl.MoEConfig("zc", T=40, H=16, E=7, K=1, F=8, dtype=0, w_std=-1.0, n_zero=1, n_copy=1, n_const=2)
    assert c.E_ffn == 3
    X, Wr, b, W, sh, dY = _inputs(c)
    assert W[0].shape[0] == 3
    v = wl.gen_zc_const(c)
    for e, want in ((3, np.zeros_like(X)), (4, X), (5, np.repeat(v[0:1], c.T, 0)), (6, np.repeat(v[1:2], c.T, 0))):
        f = O.layer_fwd(c, X, Wr, b, W, forced_idx=np.full((c.T, 1), e, np.int32), extras=dict(zc_const=v))
        assert np.array_equal(f["w"], np.ones((c.T, 1))) and np.abs(f["Y"] - want).max() < 1e-15, e
        bw = O.layer_bwd(c, dY, X, Wr, W, f, extras=dict(zc_const=v))
        assert not bw["dWg"].any() and not bw["dWd"].any()
        if e == 4:
            assert np.abs(bw["dXp"][:c.T] - dY[f["perm_to_flat"][:c.T]]).max() < 1e-15
        if e == 6:
            assert np.abs(bw["dzc_const"][1] - dY.astype(np.float64).sum(axis=0)).max() < 1e-12 and not bw["dzc_const"][0].any()


def _torch_dense_variant(c, X, Wr, W, v, idx, f_const):
    """Independent dense formulation: every FFN expert on every token, zero / copy / constant experts written out,
    gate = (sigmoid or softmax over the selected set) from idx; L_aux from P = mean_t p with f held constant."""
    Xt = torch.tensor(X, dtype=DD, requires_grad=True)
    Wrt = torch.tensor(Wr, dtype=DD, requires_grad=True)
    Wt = [torch.tensor(w, dtype=DD, requires_grad=True) for w in W]
    vt = torch.tensor(v, dtype=DD, requires_grad=True) if v is not None else None
    z = Xt @ Wrt.T
    sel = torch.zeros(c.T, c.E, dtype=torch.bool)
    for t in range(c.T):
        for e in idx[t]:
            if e >= 0:
                sel[t, e] = True
    if c.score_fn == 0 and c.route_mode == 0:
        gate = torch.softmax(z.masked_fill(~sel, float("-inf")), dim=1)
        p = torch.softmax(z, dim=1)
    else:
        s = torch.sigmoid(z)
        gate = s * sel / ((s * sel).sum(dim=1, keepdim=True) + 1e-20)
        p = s / s.sum(dim=1, keepdim=True)
    gate = gate * c.routed_scale
    Y = torch.zeros(c.T, c.H, dtype=DD)
    for e in range(c.E):
        kind = O.zc_kind(c, e)           # only the index arithmetic of the pool layout is shared
        if kind is None:
            out = (torch.nn.functional.silu(Xt @ Wt[0][e].T) * (Xt @ Wt[1][e].T)) @ Wt[2][e].T
        elif kind[0] == "zero":
            continue
        elif kind[0] == "copy":
            out = Xt
        else:
            out = vt[kind[1]][None, :].expand(c.T, c.H)
        Y = Y + gate[:, e:e + 1] * out
    eta = torch.ones(c.E, dtype=DD)
    nz = c.n_zero + c.n_copy + c.n_const
    if nz:
        eta[c.E - nz:] = c.aux_zc_weight
    Laux = c.aux_coef * c.E * (eta * torch.tensor(f_const, dtype=DD) * p.mean(dim=0)).sum()
    return Y, Laux, Xt, Wrt, Wt, vt


@pytest.mark.parametrize("variant", ["softmax_zc_aux", "threshold_zc_aux", "threshold_plain"])
def test_variant_backward_matches_autograd(variant):
    base = wl.MoEConfig("v", T=80, H=24, E=9, K=3, F=20, dtype=0, w_std=-1.0)
    c = {"softmax_zc_aux": base.replace(n_zero=1, n_copy=1, n_const=1, aux_coef=0.2, aux_zc_weight=0.5),
         "threshold_zc_aux": base.replace(score_fn=1, route_mode=1, n_zero=1, n_copy=1, n_const=1, aux_coef=0.2,
                                          routed_scale=1.5),
         "threshold_plain": base.replace(score_fn=1, route_mode=1)}[variant]
    X, Wr, b, W, sh, dY = _inputs(c)
    Wr = Wr * 12
    v = wl.gen_zc_const(c)
    ex = dict(zc_const=v, threshold=wl.gen_threshold(c))
    f = O.layer_fwd(c, X, Wr, b, W, extras=ex)
    if c.route_mode == 1:
        assert len(set((f["idx"] >= 0).sum(axis=1).tolist())) >= 2
    bw = O.layer_bwd(c, dY, X, Wr, W, f, extras=ex)
    f_const = f["aux_f"] if c.aux_coef else np.zeros(c.E)
    Y, Laux, Xt, Wrt, Wt, vt = _torch_dense_variant(c, X, Wr, W, v, f["idx"], f_const)
    assert np.abs(Y.detach().numpy() - f["Y"]).max() < 1e-11
    if c.aux_coef:
        assert abs(float(Laux.detach()) - f["aux_loss"]) < 1e-14
    ((Y * torch.tensor(dY, dtype=DD)).sum() + Laux).backward()
    tol = 1e-10
    assert O.rel_fro(bw["dX"], Xt.grad.numpy()) < tol
    assert O.rel_fro(bw["dWr"], Wrt.grad.numpy()) < tol
    for k, t in zip(("dWg", "dWu", "dWd"), Wt):
        assert O.rel_fro(bw[k], t.grad.numpy()) < tol, k
    if vt is not None:
        assert O.rel_fro(bw["dzc_const"], vt.grad.numpy()) < tol
