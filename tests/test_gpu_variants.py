"""`-m gpu` parity of the widened rows against the fp64 oracle, through the C ABI:
auxiliary load-balancing loss and its dense router backward (A1..A3), softmax gating without
renormalisation (dense dz), threshold-gated variable-k routing (V1) and zero-computation experts
(V2).  Same comparison as the plain layer (tests/gpu_common.py): integer outputs bit-exact in replay
mode, every activation and gradient element-, tile- and tensor-wise within the north_star tolerance."""
import numpy as np
import pytest

import gpu_common as gc
import workloads as wl
from oracle import moe_oracle as orc

pytestmark = pytest.mark.gpu

Q = wl.QWEN3_SMALL
VARIANT_CASES = [
    Q.replace(name="aux_softmax_align128", row_align=128, aux_coef=0.05),
    Q.replace(name="aux_softmax_packed_fp32", dtype=wl.DTYPE_FP32, T=300, H=128, F=64, aux_coef=0.05),
    Q.replace(name="softmax_norenorm_align128", row_align=128, renorm=0),
    wl.DSV3_SMALL.replace(name="aux_sigmoid_groups_shared", row_align=128, aux_coef=0.05),
    Q.replace(name="threshold_align128", row_align=128, score_fn=1, route_mode=1, K=6),
    Q.replace(name="threshold_aux_fp32", dtype=wl.DTYPE_FP32, T=300, H=128, F=64, score_fn=1, route_mode=1, K=5,
              aux_coef=0.05, routed_scale=1.5),
    Q.replace(name="zc_align128", row_align=128, n_zero=1, n_copy=1, n_const=2, aux_coef=0.05, aux_zc_weight=0.3),
    Q.replace(name="zc_threshold_e64", row_align=128, E=64, K=8, score_fn=1, route_mode=1, n_zero=2, n_copy=2, n_const=1,
              aux_coef=0.02),
    Q.replace(name="zc_fp32_packed", dtype=wl.DTYPE_FP32, T=300, H=128, F=64, n_zero=1, n_copy=2, n_const=1),
    wl.DSV3_FP8_SMALL.replace(name="fp8_zc_aux", row_align=128, n_group=1, topk_group=1, n_copy=1, n_const=1, aux_coef=0.05),
]


@pytest.mark.parametrize("cfg", VARIANT_CASES, ids=lambda c: c.name)
def test_variant_layer_fwd_bwd_matches_oracle(cfg):
    inp = gc.gen_inputs(cfg)
    lb = gc.run_gpu_layer(cfg, inp)
    errs = gc.compare_layer(cfg, inp, lb)
    if cfg.route_mode == 1:
        from paper_2605_31463_b200.buffers import to_numpy
        k = (to_numpy(lb.topk_idx) >= 0).sum(axis=1)
        assert k.min() >= 1 and len(set(k.tolist())) >= 3            # the number of active experts really varies
    print(cfg.name, {k: (f"{v:.2e}" if isinstance(v, float) else v) for k, v in errs.items()})


def test_aux_loss_with_global_fractions():
    """Global-level balance: the caller supplies f of the global batch; loss and gradient follow it."""
    import torch
    from paper_2605_31463_b200.buffers import LayerBuffers
    cfg = Q.replace(row_align=128, aux_coef=0.05)
    inp = gc.gen_inputs(cfg)
    fg = np.random.default_rng(5).random(cfg.E).astype(np.float32)
    fg /= fg.sum()
    lb = LayerBuffers(cfg)
    lb.load(**inp)
    lb.aux_f_global = torch.from_numpy(fg).cuda()
    lb.forward(); lb.backward()
    torch.cuda.synchronize()
    gc.compare_layer(cfg, dict(inp, f_global=fg), lb)


THR_CASES = [Q.replace(name="thr_e128", T=4096, E=128, K=8, score_fn=1, route_mode=1),
             Q.replace(name="thr_e1000_k32", T=512, E=1000, K=32, score_fn=1, route_mode=1, renorm=0, routed_scale=2.0),
             Q.replace(name="thr_e8_k2", T=777, E=8, K=2, score_fn=1, route_mode=1)]


@pytest.mark.parametrize("cfg", THR_CASES, ids=lambda c: c.name)
def test_route_threshold_bit_exact(cfg):
    """moe_route_threshold vs the oracle on identical fp32 logits: slots (incl. the -1 fill) bit-exact, weights 1e-5;
    planted exact ties between gates and a gate planted exactly ON its threshold (strict >: not active)."""
    import torch
    import paper_2605_31463_b200 as moe
    z = wl.gen_logits(cfg, ties=2)
    thr = wl.gen_threshold(cfg)
    z[0, :] = -20.0                                                    # no expert admits token 0: top-1 fallback
    s3 = np.float32(1.0 / (1.0 + np.exp(-np.float64(z[3, 1]))))
    thr[1] = s3                                                        # gate == threshold for (token 3, expert 1)
    zd, td = torch.from_numpy(z).cuda(), torch.from_numpy(thr).cuda()
    idx = torch.empty(cfg.T, cfg.K, dtype=torch.int32, device="cuda")
    w = torch.empty(cfg.T, cfg.K, dtype=torch.float32, device="cuda")
    moe.moe_route_threshold(cfg, zd, td, idx, w)
    torch.cuda.synchronize()
    idx_o, w_o = orc.route(z, None, cfg, key_dtype=np.float32, threshold=thr)
    assert np.array_equal(idx.cpu().numpy(), idx_o)
    assert orc.rel_fro(w.cpu().numpy(), w_o) <= gc.TOL_ROUTER
    assert (idx_o[0, 1:] == -1).all() and idx_o[0, 0] >= 0
    assert 1 not in idx_o[3].tolist() or (idx_o[3] >= 0).sum() == 1     # not active; at most the top-1 fallback


def test_permute_and_combine_accept_empty_slots():
    """moe_permute / moe_unpermute_combine on a variable-k selection: maps bit-exact vs the oracle, -1 slots own no row,
    and with w = 1/k_t on the filled slots combine(permute(X)) == X up to one bf16 rounding."""
    import torch
    import paper_2605_31463_b200 as moe
    from paper_2605_31463_b200.buffers import to_numpy
    cfg = Q.replace(row_align=128, score_fn=1, route_mode=1, K=4, E=16, T=900)
    idx_o, _ = orc.route(wl.gen_logits(cfg).astype(np.float64), None, cfg, threshold=wl.gen_threshold(cfg))
    X = wl.gen_X(cfg)
    R = moe.moe_padded_rows(cfg)
    ws_b, _ = moe.moe_workspace_bytes(cfg)
    dev = "cuda"
    idx = torch.from_numpy(idx_o).to(dev)
    Xd = torch.from_numpy(X).to(dev, torch.bfloat16)
    counts = torch.empty(cfg.E, dtype=torch.int32, device=dev); offsets = torch.empty(cfg.E + 1, dtype=torch.int32, device=dev)
    p2f = torch.empty(R, dtype=torch.int32, device=dev); f2p = torch.empty(cfg.TK, dtype=torch.int32, device=dev)
    Xp = torch.empty(R, cfg.H, dtype=torch.bfloat16, device=dev); ws = torch.empty(ws_b, dtype=torch.uint8, device=dev)
    moe.moe_permute(cfg, Xd, idx, counts, offsets, p2f, f2p, Xp, ws)
    c_o, o_o, p2f_o, f2p_o = orc.permute_maps(idx_o, cfg.E, cfg.row_align)
    assert np.array_equal(to_numpy(counts), c_o) and np.array_equal(to_numpy(offsets), o_o)
    assert np.array_equal(to_numpy(f2p), f2p_o) and np.array_equal(to_numpy(p2f)[:p2f_o.size], p2f_o)
    assert np.array_equal(to_numpy(Xp)[:p2f_o.size], orc.permute_rows(X, p2f_o, cfg.K))
    k = (idx_o >= 0).sum(axis=1, keepdims=True)
    w = np.where(idx_o >= 0, 1.0 / k, 0.0).astype(np.float32)
    Y = torch.empty_like(Xd)
    moe.moe_unpermute_combine(cfg, Xp, torch.from_numpy(w).to(dev), f2p, None, Y)
    torch.cuda.synchronize()
    ref = orc.unpermute_combine(orc.permute_rows(X, p2f_o, cfg.K), w.astype(np.float64), f2p_o)
    assert orc.rel_fro(to_numpy(Y), ref) <= 4e-3
