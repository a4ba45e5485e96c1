"""Shared helpers of the `-m gpu` parity tests: run the CUDA path through the C ABI and the fp64 oracle on
the same seeded inputs and compare (routing in replay mode, S19 error metric)."""
from __future__ import annotations

import numpy as np

import workloads as wl
from oracle import moe_oracle as orc

TOL = {wl.DTYPE_FP32: 1e-5, wl.DTYPE_BF16: 1e-2, wl.DTYPE_FP8: 3e-2}   # BASELINE.json:north_star
TOL_ROUTER = 1e-5
TILE_ROWS, TILE_COLS = 128, 64     # the GEMM kernels' store granularity: one 128-row tile x one 64-column TMA box


def tile_gate(name, G, R, tol):
    """Tile-local parity gate beside the whole-tensor S19 norm (which a stale 128 x 32 chunk of one tile would pass:
    1/32768 of configs[1]'s y moves the norm by 5e-3).  Two bounds, both derived from the tolerance:
      (1) every (128-row x 64-column) block:  ||G - R||_blk <= 4 tol * max(||R||_blk, 0.05 rms(R) sqrt(n_blk));
          an all-zero reference block (padding rows) requires an all-zero result;
      (2) every element:  |G - R| <= 6 tol max(rms(R), rms(R[row])) + tol |R|   (catches a single stale or garbage
          element; the row term is there because every row is its own GEMM row whose error scales with ITS magnitude --
          gating weights and FP8 block scales make row norms differ by an order of magnitude).
    Returns the worst block ratio (in units of tol)."""
    G = np.asarray(G, np.float64); R = np.asarray(R, np.float64)
    assert G.shape == R.shape, (name, G.shape, R.shape)
    if R.size == 0:
        return 0.0
    rms = float(np.sqrt(np.mean(R * R)))
    D = G - R
    row_rms = np.sqrt(np.mean(R * R, axis=1, keepdims=True)) if R.ndim == 2 else rms
    bad = np.abs(D) > 6 * tol * np.maximum(rms, row_rms) + tol * np.abs(R)
    if bad.any():
        where = np.argwhere(bad)[:6]
        detail = [(tuple(int(v) for v in ix), float(G[tuple(ix)]), float(R[tuple(ix)]),
                   float(row_rms[ix[0], 0]) if R.ndim == 2 else rms) for ix in where]
        raise AssertionError(f"{name}: {int(bad.sum())} elements outside 6*tol*max(rms, row rms) + tol*|R| "
                             f"(tol {tol}, rms {rms:.3e}; (index, got, want, row rms): {detail})")
    nr, nc = -(-R.shape[0] // TILE_ROWS), -(-R.shape[1] // TILE_COLS)
    D2 = np.zeros((nr * TILE_ROWS, nc * TILE_COLS)); R2 = np.zeros_like(D2)
    D2[:R.shape[0], :R.shape[1]] = D * D; R2[:R.shape[0], :R.shape[1]] = R * R
    dn = np.sqrt(D2.reshape(nr, TILE_ROWS, nc, TILE_COLS).sum(axis=(1, 3)))
    rn = np.sqrt(R2.reshape(nr, TILE_ROWS, nc, TILE_COLS).sum(axis=(1, 3)))
    zero = rn == 0
    assert not (dn[zero] != 0).any(), f"{name}: non-zero output where the reference block is exactly zero"
    floor = 0.05 * rms * np.sqrt(TILE_ROWS * TILE_COLS)
    ratio = dn / np.maximum(rn, floor)
    worst = float(ratio.max())
    assert worst <= 4 * tol, (f"{name}: block {tuple(int(v) for v in np.unravel_index(ratio.argmax(), ratio.shape))} "
                              f"rel err {worst:.3e} > 4*tol ({tol})")
    return worst / tol


def tile_gate_torch(name, G, R, tol):
    """tile_gate for big tensors, evaluated on the device in torch fp64 (G: device tensor, R: the oracle's NumPy fp64 array):
    the same two bounds, ~100x faster than NumPy on a 15 M-element weight gradient.  Returns (worst block ratio in units
    of tol, ||G - R||_F / ||R||_F)."""
    import torch
    G = G.to(torch.float64)
    R = torch.as_tensor(np.ascontiguousarray(R), dtype=torch.float64).to(G.device)
    assert tuple(G.shape) == tuple(R.shape) and R.dim() == 2, (name, tuple(G.shape), tuple(R.shape))
    if R.numel() == 0:
        return 0.0, 0.0
    rms = float(R.pow(2).mean().sqrt())
    D = G - R
    row_rms = R.pow(2).mean(dim=1, keepdim=True).sqrt()
    bad = D.abs() > 6 * tol * torch.clamp(row_rms, min=rms) + tol * R.abs()
    nbad = int(bad.sum())
    if nbad:
        ix = torch.nonzero(bad)[:6].tolist()
        detail = [((i, j), float(G[i, j]), float(R[i, j]), float(row_rms[i, 0])) for i, j in ix]
        raise AssertionError(f"{name}: {nbad} elements outside 6*tol*max(rms, row rms) + tol*|R| "
                             f"(tol {tol}, rms {rms:.3e}; (index, got, want, row rms): {detail})")
    nr, nc = -(-R.shape[0] // TILE_ROWS), -(-R.shape[1] // TILE_COLS)
    pad = (0, nc * TILE_COLS - R.shape[1], 0, nr * TILE_ROWS - R.shape[0])
    D2 = torch.nn.functional.pad(D * D, pad); R2 = torch.nn.functional.pad(R * R, pad)
    dn = D2.reshape(nr, TILE_ROWS, nc, TILE_COLS).sum(dim=(1, 3)).sqrt()
    rn = R2.reshape(nr, TILE_ROWS, nc, TILE_COLS).sum(dim=(1, 3)).sqrt()
    assert not bool((dn[rn == 0] != 0).any()), f"{name}: non-zero output where the reference block is exactly zero"
    floor = 0.05 * rms * np.sqrt(TILE_ROWS * TILE_COLS)
    ratio = dn / torch.clamp(rn, min=floor)
    worst = float(ratio.max())
    assert worst <= 4 * tol, f"{name}: block rel err {worst:.3e} > 4*tol ({tol})"
    nR = float(R.norm())
    fro = float(D.norm()) / nR if nR > 0 else (0.0 if float(D.norm()) == 0 else float("inf"))
    return worst / tol, fro


def gen_inputs(cfg):
    X, dY, Wr, bias = wl.gen_X(cfg), wl.gen_dY(cfg), wl.gen_Wr(cfg), wl.gen_bias(cfg)
    W = wl.gen_all_expert_weights(cfg)
    shared = wl.gen_shared_weights(cfg)
    inp = dict(X=X, dY=dY, Wr=Wr, bias=bias, W=W, shared=shared)
    if cfg.route_mode == 1:
        inp["threshold"] = wl.gen_threshold(cfg)
    if cfg.n_const:
        inp["zc_const"] = wl.gen_zc_const(cfg)
    return inp


def oracle_extras(inp):
    return {k: inp[k] for k in ("threshold", "zc_const", "f_global") if k in inp}


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


def check_routing_replay(cfg, z_gpu, bias, idx_gpu, w_gpu, z_truth=None, threshold=None):
    """Bit-exact indices given identical logits (replay mode), fp32 weights within 1e-5; in truth mode a
    mismatch is tolerated only at a verified near-tie of the fp64 keys (gap < 1e-5; threshold routing: also a gate
    within 1e-5 of its threshold)."""
    idx_o, w_o = orc.route(z_gpu, bias, cfg, key_dtype=np.float32, threshold=threshold)
    assert np.array_equal(idx_o, idx_gpu), f"routing indices differ on {(idx_o != idx_gpu).any(axis=1).sum()} tokens"
    assert orc.rel_fro(w_gpu, w_o) <= TOL_ROUTER
    if z_truth is not None:
        idx_t, _ = orc.route(z_truth, bias, cfg, threshold=threshold)
        bad = np.nonzero((idx_t != idx_gpu).any(axis=1))[0]
        if bad.size and cfg.route_mode == 1:
            s = orc.sigmoid(z_truth[bad])
            srt = -np.sort(-s, axis=1)
            gaps = np.minimum(np.abs(np.diff(srt, axis=1)).min(axis=1), np.abs(s - threshold[None, :].astype(np.float64)).min(axis=1))
            assert (gaps < 1e-5).all(), f"truth-mode mismatch at a non-tie: min gaps {gaps}"
        elif bad.size:
            key = orc.group_limit(orc.selection_keys(z_truth[bad], bias, cfg), cfg)
            srt = -np.sort(-key, axis=1)
            gaps = np.abs(np.diff(srt[:, :cfg.K + 1], axis=1)).min(axis=1)
            assert (gaps < 1e-5).all(), f"truth-mode mismatch at a non-tie: min gaps {gaps}"
        return bad.size
    return 0


def row_weights(p2f, w):
    """Routing weight of every permuted row (0 for padding rows): w.reshape(-1)[perm_to_flat]."""
    p2f = np.asarray(p2f, np.int64)
    return np.where(p2f >= 0, np.asarray(w, np.float64).reshape(-1)[np.maximum(p2f, 0)], 0.0)


def compare_layer(cfg, inp, lb, backward=True, tol=None):
    """Oracle on the same inputs with the GPU's (replay-verified) selection; returns the error table."""
    from paper_2605_31463_b200.buffers import to_numpy
    tol = TOL[cfg.dtype] if tol is None else tol
    z_gpu = to_numpy(lb.ctx_view("z"))
    idx_gpu = to_numpy(lb.topk_idx)
    w_gpu = to_numpy(lb.topk_w)
    z_o = orc.router_logits(inp["X"], inp["Wr"])
    assert orc.rel_fro(z_gpu, z_o) <= TOL_ROUTER, f"router logits {orc.rel_fro(z_gpu, z_o)}"
    n_near = check_routing_replay(cfg, z_gpu, inp["bias"], idx_gpu, w_gpu, z_truth=z_o, threshold=inp.get("threshold"))
    ex = oracle_extras(inp)
    fwd = orc.layer_fwd(cfg, inp["X"], inp["Wr"], inp["bias"], inp["W"], inp["shared"], forced_idx=idx_gpu, extras=ex)
    errs = {"near_ties": n_near}
    # integer maps: bit-exact
    for name, ref in (("counts", fwd["counts"]), ("offsets", fwd["offsets"]), ("flat_to_perm", fwd["flat_to_perm"])):
        got = to_numpy(lb.ctx_view(name))
        assert np.array_equal(got, ref), name
    R = int(fwd["offsets"][-1])
    assert np.array_equal(to_numpy(lb.ctx_view("perm_to_flat"))[:R], fwd["perm_to_flat"])
    assert orc.rel_fro(w_gpu, fwd["w"]) <= TOL_ROUTER
    if cfg.dtype != wl.DTYPE_FP8:      # fused rows: Xp is GEMM-1's by-product copy of its gathered tiles
        assert np.array_equal(to_numpy(lb.ctx_view("Xp"))[:R], fwd["Xp"].astype(np.float32)), "Xp must be a bit-exact copy"
    # fused rows (moe_layer_rows_fused): the saved a and y carry the row's routing weight, padding rows stay zero
    wrow = row_weights(fwd["perm_to_flat"], fwd["w"]) if lb.rows_fused else np.ones(R)
    gu = to_numpy(lb.ctx_view("gu"))[:R]
    acts = [("g", gu[:, :cfg.F], fwd["g"]), ("u", gu[:, cfg.F:], fwd["u"]),
            ("a", to_numpy(lb.ctx_view("a"))[:R], fwd["a"] * wrow[:, None]),
            ("y", to_numpy(lb.ctx_view("y"))[:R], fwd["y"] * wrow[:, None]), ("Y", to_numpy(lb.Y), fwd["Y"])]
    if cfg.aux_coef:                                             # A1..A2: loss value, f, P (fp32 router-side quantities)
        errs["aux_loss"] = abs(float(to_numpy(lb.aux_loss)[0]) - fwd["aux_loss"]) / abs(fwd["aux_loss"])
        assert errs["aux_loss"] <= TOL_ROUTER, errs["aux_loss"]
        assert float(to_numpy(lb.ctx_view("aux_loss"))[0]) == float(to_numpy(lb.aux_loss)[0])
        assert orc.rel_fro(to_numpy(lb.ctx_view("aux_f")), fwd["aux_f"]) <= TOL_ROUTER
        assert orc.rel_fro(to_numpy(lb.ctx_view("aux_P")), fwd["aux_P"]) <= TOL_ROUTER
        del errs["aux_loss"]
    if backward:
        bwd = orc.layer_bwd(cfg, inp["dY"], inp["X"], inp["Wr"], inp["W"], fwd, inp["shared"], extras=ex)
        if lb.rows_fused:              # ws "dy": dgrad-down's by-product copy of the gathered dY rows, unweighted, zero padding
            p2f = np.asarray(fwd["perm_to_flat"], np.int64)
            dyp = np.where((p2f >= 0)[:, None], inp["dY"].astype(np.float32)[np.maximum(p2f, 0) // cfg.K], 0.0)
            assert np.array_equal(to_numpy(lb.ws_view("dy"))[:R], dyp), "gathered dY must be a bit-exact copy"
        errs["dw"] = orc.rel_fro(to_numpy(lb.ws_view("dw")), bwd["dw"])
        errs["dWr"] = orc.rel_fro(to_numpy(lb.dWr), bwd["dWr"])
        dgu = to_numpy(lb.ws_view("dgu"))[:R]
        acts += [("dg", dgu[:, :cfg.F], bwd["dg"]), ("du", dgu[:, cfg.F:], bwd["du"]),
                 ("dXp", to_numpy(lb.ws_view("dXp"))[:R], bwd["dXp"]), ("dX", to_numpy(lb.dX), bwd["dX"])]
        dz_sel = np.where(idx_gpu >= 0, np.take_along_axis(bwd["dz"], np.maximum(idx_gpu, 0).astype(np.int64), axis=1), 0.0)
        errs["dz"] = orc.rel_fro(to_numpy(lb.ws_view("dz")), dz_sel)
        if cfg.aux_coef or cfg.n_zero + cfg.n_copy + cfg.n_const or (cfg.score_fn == 0 and not cfg.renorm and cfg.route_mode == 0):
            errs["dz_dense"] = orc.rel_fro(to_numpy(lb.ws_view("dz_dense")), bwd["dz"])   # dense router backward (A3)
        if cfg.n_const:
            errs["dzc_const"] = orc.rel_fro(to_numpy(lb.d_zc_const), bwd["dzc_const"])
        for name, got in (("dWg", lb.dWg), ("dWu", lb.dWu), ("dWd", lb.dWd)):
            g = to_numpy(got)
            per = [orc.rel_fro(g[e], bwd[name][e]) for e in range(cfg.E_ffn)]
            errs[name] = float(np.max(per))                      # S19: max over experts; empty expert -> exact 0
        if inp["shared"] is not None:
            for name, got in (("dWg_s", lb.dWg_s), ("dWu_s", lb.dWu_s), ("dWd_s", lb.dWd_s)):
                errs[name] = orc.rel_fro(to_numpy(got), bwd[name])
    worst_tile = 0.0
    for name, got, ref in acts:
        errs[name] = orc.rel_fro(got, ref)                       # S19 whole-tensor norm
        worst_tile = max(worst_tile, tile_gate(f"{cfg.name}:{name}", got, ref, tol))
    bad = {k: v for k, v in errs.items() if k != "near_ties" and not (v <= tol)}
    assert not bad, f"{cfg.name}: over tolerance {tol}: {bad}; all: {errs}"
    errs["worst_tile_over_tol"] = worst_tile
    return errs
