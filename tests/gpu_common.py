"""Shared helpers of the `-m gpu` parity tests: run the CUDA path through the C ABI and the fp64 oracle on
the same seeded inputs and compare (routing in replay mode, S19 error metric)."""
from __future__ import annotations

import numpy as np

import workloads as wl
from oracle import moe_oracle as orc

TOL = {wl.DTYPE_FP32: 1e-5, wl.DTYPE_BF16: 1e-2, wl.DTYPE_FP8: 3e-2}   # BASELINE.json:north_star
TOL_ROUTER = 1e-5


def gen_inputs(cfg):
    X, dY, Wr, bias = wl.gen_X(cfg), wl.gen_dY(cfg), wl.gen_Wr(cfg), wl.gen_bias(cfg)
    W = wl.gen_all_expert_weights(cfg)
    shared = wl.gen_shared_weights(cfg)
    return dict(X=X, dY=dY, Wr=Wr, bias=bias, W=W, shared=shared)


def run_gpu_layer(cfg, inp, backward=True):
    import torch
    from paper_2605_31463_b200.buffers import LayerBuffers
    lb = LayerBuffers(cfg)
    lb.load(**inp)
    lb.forward()
    if backward:
        lb.backward()
    torch.cuda.synchronize()
    return lb


def check_routing_replay(cfg, z_gpu, bias, idx_gpu, w_gpu, z_truth=None):
    """Bit-exact indices given identical logits (replay mode), fp32 weights within 1e-5; in truth mode a
    mismatch is tolerated only at a verified near-tie of the fp64 keys (gap < 1e-5)."""
    idx_o, w_o = orc.route(z_gpu, bias, cfg, key_dtype=np.float32)
    assert np.array_equal(idx_o, idx_gpu), f"routing indices differ on {(idx_o != idx_gpu).any(axis=1).sum()} tokens"
    assert orc.rel_fro(w_gpu, w_o) <= TOL_ROUTER
    if z_truth is not None:
        idx_t, _ = orc.route(z_truth, bias, cfg)
        bad = np.nonzero((idx_t != idx_gpu).any(axis=1))[0]
        if bad.size:
            key = orc.group_limit(orc.selection_keys(z_truth[bad], bias, cfg), cfg)
            srt = -np.sort(-key, axis=1)
            gaps = np.abs(np.diff(srt[:, :cfg.K + 1], axis=1)).min(axis=1)
            assert (gaps < 1e-5).all(), f"truth-mode mismatch at a non-tie: min gaps {gaps}"
        return bad.size
    return 0


def compare_layer(cfg, inp, lb, backward=True, tol=None):
    """Oracle on the same inputs with the GPU's (replay-verified) selection; returns the error table."""
    from paper_2605_31463_b200.buffers import to_numpy
    tol = TOL[cfg.dtype] if tol is None else tol
    z_gpu = to_numpy(lb.ctx_view("z"))
    idx_gpu = to_numpy(lb.topk_idx)
    w_gpu = to_numpy(lb.topk_w)
    z_o = orc.router_logits(inp["X"], inp["Wr"])
    assert orc.rel_fro(z_gpu, z_o) <= TOL_ROUTER, f"router logits {orc.rel_fro(z_gpu, z_o)}"
    n_near = check_routing_replay(cfg, z_gpu, inp["bias"], idx_gpu, w_gpu, z_truth=z_o)
    fwd = orc.layer_fwd(cfg, inp["X"], inp["Wr"], inp["bias"], inp["W"], inp["shared"], forced_idx=idx_gpu)
    errs = {"near_ties": n_near}
    # integer maps: bit-exact
    for name, ref in (("counts", fwd["counts"]), ("offsets", fwd["offsets"]), ("flat_to_perm", fwd["flat_to_perm"])):
        got = to_numpy(lb.ctx_view(name))
        assert np.array_equal(got, ref), name
    R = int(fwd["offsets"][-1])
    assert np.array_equal(to_numpy(lb.ctx_view("perm_to_flat"))[:R], fwd["perm_to_flat"])
    assert orc.rel_fro(w_gpu, fwd["w"]) <= TOL_ROUTER
    if cfg.dtype != wl.DTYPE_FP8:
        assert np.array_equal(to_numpy(lb.ctx_view("Xp"))[:R], fwd["Xp"].astype(np.float32)), "Xp must be a bit-exact copy"
    gu = to_numpy(lb.ctx_view("gu"))[:R]
    errs["g"] = orc.rel_fro(gu[:, :cfg.F], fwd["g"])
    errs["u"] = orc.rel_fro(gu[:, cfg.F:], fwd["u"])
    errs["a"] = orc.rel_fro(to_numpy(lb.ctx_view("a"))[:R], fwd["a"])
    errs["y"] = orc.rel_fro(to_numpy(lb.ctx_view("y"))[:R], fwd["y"])
    errs["Y"] = orc.rel_fro(to_numpy(lb.Y), fwd["Y"])
    if backward:
        bwd = orc.layer_bwd(cfg, inp["dY"], inp["X"], inp["Wr"], inp["W"], fwd, inp["shared"])
        errs["dw"] = orc.rel_fro(to_numpy(lb.ws_view("dw")), bwd["dw"])
        errs["dX"] = orc.rel_fro(to_numpy(lb.dX), bwd["dX"])
        errs["dWr"] = orc.rel_fro(to_numpy(lb.dWr), bwd["dWr"])
        for name, got in (("dWg", lb.dWg), ("dWu", lb.dWu), ("dWd", lb.dWd)):
            g = to_numpy(got)
            per = [orc.rel_fro(g[e], bwd[name][e]) for e in range(cfg.E)]
            errs[name] = float(np.max(per))                      # S19: max over experts; empty expert -> exact 0
        if inp["shared"] is not None:
            for name, got in (("dWg_s", lb.dWg_s), ("dWu_s", lb.dWu_s), ("dWd_s", lb.dWd_s)):
                errs[name] = orc.rel_fro(to_numpy(got), bwd[name])
    bad = {k: v for k, v in errs.items() if k != "near_ties" and not (v <= tol)}
    assert not bad, f"{cfg.name}: over tolerance {tol}: {bad}; all: {errs}"
    return errs
