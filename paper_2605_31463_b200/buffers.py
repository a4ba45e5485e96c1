"""Device-memory plumbing for the MoE layer: allocates every buffer the C ABI needs with torch and
exposes the saved-for-backward fields of `ctx` / `ws` as typed tensor views.  No arithmetic here."""
from __future__ import annotations

import numpy as np
import torch

from . import (make_config, make_extras, moe_ctx_field, moe_layer_rows_fused, moe_layer_bwd, moe_layer_bwd_ex, moe_layer_fwd, moe_layer_fwd_ex,
               moe_layer_step_host,
               moe_layer_step_host_pipelined, moe_padded_rows, moe_pipeline_create, moe_pipeline_destroy,
               moe_workspace_bytes, moe_ws_field)


def act_dtype(cfg) -> torch.dtype:
    return torch.float32 if cfg.dtype == 0 else torch.bfloat16


def to_device(x: np.ndarray | None, dtype: torch.dtype, device="cuda"):
    """numpy fp32 array whose values are exactly representable in `dtype` -> device tensor (lossless)."""
    if x is None:
        return None
    return torch.from_numpy(np.ascontiguousarray(x)).to(device=device, dtype=dtype).contiguous()


def to_numpy(t: torch.Tensor) -> np.ndarray:
    if t.dtype in (torch.bfloat16, torch.float16):
        t = t.float()
    return t.detach().cpu().numpy()


class LayerBuffers:
    """All device buffers of one MoE layer (weights, gradients, ctx, ws, outputs)."""

    def __init__(self, cfg, device="cuda", with_grads=True):
        self.cfg = cfg
        self.ccfg = make_config(cfg)
        self.device = device
        dt = act_dtype(cfg)
        T, H, E, K, F, Fs = cfg.T, cfg.H, cfg.E, cfg.K, cfg.F, cfg.F_shared
        self.R = moe_padded_rows(cfg)
        self.rows_fused = moe_layer_rows_fused(cfg)     # >= 1: ctx "a" / "y" carry the routing weight, ws "dy" is unweighted
        ws_b, ctx_b = moe_workspace_bytes(cfg)
        e = lambda *shape, dtype=dt: torch.empty(*shape, dtype=dtype, device=device)
        self.ws = e(ws_b, dtype=torch.uint8)
        self.ctx = e(ctx_b, dtype=torch.uint8)
        self.X, self.dY, self.Y, self.dX = e(T, H), e(T, H), e(T, H), e(T, H)
        self.Wr = e(E, H)
        self.bias = e(E, dtype=torch.float32) if cfg.has_bias else None
        Ef = E - getattr(cfg, "n_zero", 0) - getattr(cfg, "n_copy", 0) - getattr(cfg, "n_const", 0)   # experts with FFN weights
        self.Wg, self.Wu, self.Wd = e(Ef, F, H), e(Ef, F, H), e(Ef, H, F)
        self.Wg_s = self.Wu_s = self.Wd_s = None
        if Fs:
            self.Wg_s, self.Wu_s, self.Wd_s = e(Fs, H), e(Fs, H), e(H, Fs)
        self.topk_idx = e(T, K, dtype=torch.int32)
        self.topk_w = e(T, K, dtype=torch.float32)
        self.dWr = self.dWg = self.dWu = self.dWd = self.dWg_s = self.dWu_s = self.dWd_s = None
        if with_grads:
            self.dWr, self.dWg, self.dWu, self.dWd = e(E, H), e(Ef, F, H), e(Ef, F, H), e(Ef, H, F)
            if Fs:
                self.dWg_s, self.dWu_s, self.dWd_s = e(Fs, H), e(Fs, H), e(H, Fs)
        # extras of the widened rows (moe_extras_t): thresholds, constant experts, balance loss
        self.threshold = e(E, dtype=torch.float32) if getattr(cfg, "route_mode", 0) == 1 else None
        nc = getattr(cfg, "n_const", 0)
        self.zc_const = e(nc, H) if nc else None
        self.d_zc_const = e(nc, H) if (nc and with_grads) else None
        self.aux_loss = e(1, dtype=torch.float32) if getattr(cfg, "aux_coef", 0.0) else None
        self.aux_f_global = None
        self.use_ex = any(t is not None for t in (self.threshold, self.zc_const, self.aux_loss))

    # ---- loading inputs (numpy fp32 on the storage grid) ----
    def extras(self):
        return make_extras(self.threshold, self.zc_const, self.d_zc_const, self.aux_f_global, self.aux_loss)

    def load(self, X=None, dY=None, Wr=None, bias=None, W=None, shared=None, threshold=None, zc_const=None):
        dt = act_dtype(self.cfg)
        if threshold is not None: self.threshold.copy_(to_device(threshold, torch.float32, self.device))
        if zc_const is not None: self.zc_const.copy_(to_device(zc_const, dt, self.device))
        if X is not None: self.X.copy_(to_device(X, dt, self.device))
        if dY is not None: self.dY.copy_(to_device(dY, dt, self.device))
        if Wr is not None: self.Wr.copy_(to_device(Wr, dt, self.device))
        if bias is not None: self.bias.copy_(to_device(bias, torch.float32, self.device))
        if W is not None:
            for dst, src in zip((self.Wg, self.Wu, self.Wd), W):
                dst.copy_(to_device(src, dt, self.device))
        if shared is not None:
            for dst, src in zip((self.Wg_s, self.Wu_s, self.Wd_s), shared):
                dst.copy_(to_device(src, dt, self.device))

    # ---- the two calls ----
    def forward(self, stream=None):
        if self.use_ex:
            return moe_layer_fwd_ex(self.ccfg, self.X, self.Wr, self.bias, self.Wg, self.Wu, self.Wd, self.Wg_s, self.Wu_s,
                                    self.Wd_s, self.Y, self.topk_idx, self.topk_w, self.ctx, self.ws, self.extras(), stream)
        moe_layer_fwd(self.ccfg, self.X, self.Wr, self.bias, self.Wg, self.Wu, self.Wd, self.Wg_s, self.Wu_s,
                      self.Wd_s, self.Y, self.topk_idx, self.topk_w, self.ctx, self.ws, stream)

    def backward(self, stream=None):
        if self.use_ex:
            return moe_layer_bwd_ex(self.ccfg, self.dY, self.X, self.Wr, self.Wg, self.Wu, self.Wd, self.Wg_s, self.Wu_s,
                                    self.Wd_s, self.ctx, self.dX, self.dWr, self.dWg, self.dWu, self.dWd, self.dWg_s,
                                    self.dWu_s, self.dWd_s, self.ws, self.extras(), stream)
        moe_layer_bwd(self.ccfg, self.dY, self.X, self.Wr, self.Wg, self.Wu, self.Wd, self.Wg_s, self.Wu_s,
                      self.Wd_s, self.ctx, self.dX, self.dWr, self.dWg, self.dWu, self.dWd, self.dWg_s, self.dWu_s,
                      self.dWd_s, self.ws, stream)

    def step_host(self, X_host, dY_host, Y_host, dX_host, stream=None):
        moe_layer_step_host(self.ccfg, X_host, dY_host, Y_host, dX_host, self.X, self.dY, self.Y, self.dX, self.Wr,
                            self.bias, self.Wg, self.Wu, self.Wd, self.Wg_s, self.Wu_s, self.Wd_s, self.dWr, self.dWg,
                            self.dWu, self.dWd, self.dWg_s, self.dWu_s, self.dWd_s, self.topk_idx, self.topk_w,
                            self.ctx, self.ws, stream)

    def make_pipeline(self):
        """Second set of staging buffers and the three streams of moe_layer_step_host_pipelined."""
        self.stage = [(self.X, self.dY, self.Y, self.dX),
                      tuple(torch.empty_like(self.X) for _ in range(4))]
        self.streams = tuple(torch.cuda.Stream() for _ in range(3))
        self.pipeline = moe_pipeline_create()

    def close_pipeline(self):
        if getattr(self, "pipeline", None) is not None:
            torch.cuda.synchronize()
            moe_pipeline_destroy(self.pipeline)
            self.pipeline = None

    def step_host_pipelined(self, i, X_host, dY_host, Y_host, dX_host):
        Xd, dYd, Yd, dXd = self.stage[i & 1]
        moe_layer_step_host_pipelined(self.pipeline, self.ccfg, i & 1, X_host, dY_host, Y_host, dX_host, Xd, dYd, Yd, dXd, self.Wr,
                                      self.bias, self.Wg, self.Wu, self.Wd, self.Wg_s, self.Wu_s, self.Wd_s, self.dWr,
                                      self.dWg, self.dWu, self.dWd, self.dWg_s, self.dWu_s, self.dWd_s, self.topk_idx,
                                      self.topk_w, self.ctx, self.ws, *self.streams)

    # ---- typed views into ctx / ws ----
    _CTX = {"z": ("f32", lambda c, R: (c.T, c.E)), "counts": ("i32", lambda c, R: (c.E,)),
            "offsets": ("i32", lambda c, R: (c.E + 1,)), "perm_to_flat": ("i32", lambda c, R: (R,)),
            "flat_to_perm": ("i32", lambda c, R: (c.T * c.K,)), "Xp": ("act", lambda c, R: (R, c.H)),
            "gu": ("act", lambda c, R: (R, 2 * c.F)), "a": ("act", lambda c, R: (R, c.F)),
            "y": ("act", lambda c, R: (R, c.H)), "gu_s": ("act", lambda c, R: (c.T, 2 * c.F_shared)),
            "a_s": ("act", lambda c, R: (c.T, c.F_shared)), "y_s": ("act", lambda c, R: (c.T, c.H)),
            "aux_f": ("f32", lambda c, R: (c.E,)), "aux_P": ("f32", lambda c, R: (c.E,)),
            "aux_loss": ("f32", lambda c, R: (1,)),
            "aq": ("u8", lambda c, R: (R, c.F)), "aq_s": ("f32", lambda c, R: (R, c.F // 128))}
    _WS = {"dw": ("f32", lambda c, R: (c.T, c.K)), "dz": ("f32", lambda c, R: (c.T, c.K)),
           "dy": ("act", lambda c, R: (R, c.H)), "dgu": ("act", lambda c, R: (R, 2 * c.F)),
           "dXp": ("act", lambda c, R: (R, c.H)), "dz_dense": ("f32", lambda c, R: (c.T, c.E)),
           "dguq": ("u8", lambda c, R: (R, 2 * c.F)), "dguq_s": ("f32", lambda c, R: (R, 2 * c.F // 128))}

    def _view(self, buf, field_fn, table, name):
        kind, shape_fn = table[name]
        off, ln = field_fn(self.ccfg, name)
        dt = {"f32": torch.float32, "i32": torch.int32, "u8": torch.uint8, "act": act_dtype(self.cfg)}[kind]
        return buf[off:off + ln].view(dt).view(*shape_fn(self.cfg, self.R))

    def ctx_view(self, name):
        return self._view(self.ctx, moe_ctx_field, self._CTX, name)

    def ws_view(self, name):
        return self._view(self.ws, moe_ws_field, self._WS, name)
