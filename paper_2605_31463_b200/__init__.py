"""Python binding of libmoe_b200.so (include/moe_b200.h): argument marshalling only.

Every step of the MoE hot path runs in the CUDA kernels behind the C ABI; this module turns torch
tensors into device pointers, checks shapes/dtypes, and raises on a non-zero status.  There is no CPU
fallback: if the shared library is missing the import of `lib()` fails loudly.
PyTorch is used for device memory and streams only.
"""
from __future__ import annotations

import ctypes as C
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libmoe_b200.so")

MOE_OK, MOE_ERR_INVALID_ARG, MOE_ERR_UNSUPPORTED, MOE_ERR_WORKSPACE, MOE_ERR_CUDA = 0, -1, -2, -3, -4
MOE_ERR_TOO_LARGE = -5
MOE_PERMUTE_STATIC_WS_BYTES = 1 << 20   # include/moe_b200.h


class moe_config_t(C.Structure):
    _fields_ = [("T", C.c_int32), ("H", C.c_int32), ("E", C.c_int32), ("K", C.c_int32), ("F", C.c_int32),
                ("n_group", C.c_int32), ("topk_group", C.c_int32), ("score_fn", C.c_int32),
                ("group_score", C.c_int32), ("renorm", C.c_int32), ("routed_scale", C.c_float),
                ("has_bias", C.c_int32), ("F_shared", C.c_int32), ("dtype", C.c_int32),
                ("fp8_scale_mode", C.c_int32), ("row_align", C.c_int32),
                ("route_mode", C.c_int32), ("n_zero", C.c_int32), ("n_copy", C.c_int32), ("n_const", C.c_int32),
                ("aux_coef", C.c_float), ("aux_zc_weight", C.c_float),
                ("opt_rows_fused", C.c_int32), ("opt_pair", C.c_int32), ("opt_fp8_wide", C.c_int32),
                ("opt_fp8_fused_quant", C.c_int32)]


class moe_extras_t(C.Structure):
    _fields_ = [("threshold", C.c_void_p), ("zc_const", C.c_void_p), ("d_zc_const", C.c_void_p),
                ("aux_f_global", C.c_void_p), ("aux_loss", C.c_void_p)]


CONFIG_FIELDS = [f for f, _ in moe_config_t._fields_]


def make_config(cfg) -> moe_config_t:
    """Build the C struct from any object carrying the moe_config_t field names (e.g. workloads.MoEConfig)."""
    if isinstance(cfg, moe_config_t):
        return cfg
    return moe_config_t(**{f: getattr(cfg, f, 0) if f.startswith("opt_") else getattr(cfg, f) for f in CONFIG_FIELDS})


class MoEError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        super().__init__(f"{where}: {status_string(status)} ({status})")


_lib = None

_P, _I32, _I64, _SZP = C.c_void_p, C.c_int32, C.c_int64, C.POINTER(C.c_size_t)
_CFG = C.POINTER(moe_config_t)
_SIGNATURES = {
    "moe_status_string": (C.c_char_p, [_I32]),
    "moe_version": (_I32, []),
    "moe_launch_count": (_I64, []),
    "moe_padded_rows": (_I64, [_CFG]),
    "moe_layer_rows_fused": (_I32, [_CFG]),
    "moe_workspace_bytes": (_I32, [_CFG, _SZP, _SZP]),
    "moe_route": (_I32, [_CFG, _P, _P, _P, _P, _P]),
    "moe_route_threshold": (_I32, [_CFG, _P, _P, _P, _P, _P]),
    "moe_layer_fwd_ex": (_I32, [_CFG] + [_P] * 14 + [C.POINTER(moe_extras_t), _P]),
    "moe_layer_bwd_ex": (_I32, [_CFG] + [_P] * 19 + [C.POINTER(moe_extras_t), _P]),
    "moe_permute": (_I32, [_CFG] + [_P] * 9),
    "moe_permute_static_ws": (_I32, [_CFG] + [_P] * 8),
    "moe_grouped_gemm_fwd": (_I32, [_CFG, _I32, _I32] + [_P] * 8),
    "moe_grouped_gemm_bwd": (_I32, [_CFG, _I32, _I32] + [_P] * 8),
    "moe_swiglu": (_I32, [_CFG, _P, _P, _I64, _P]),
    "moe_swiglu_bwd": (_I32, [_CFG, _P, _P, _P, _I64, _P]),
    "moe_unpermute_combine": (_I32, [_CFG] + [_P] * 6),
    "moe_quantize_act": (_I32, [_P, _I64, _I32, _I32, _P, _P, _P]),
    "moe_quantize_weight": (_I32, [_P, _I32, _I32, _I32, _I32, _P, _P, _P]),
    "moe_fp8_quantize_weights": (_I32, [_CFG] + [_P] * 8),
    "moe_layer_fwd": (_I32, [_CFG] + [_P] * 15),
    "moe_layer_bwd": (_I32, [_CFG] + [_P] * 20),
    "moe_layer_wgrad": (_I32, [_CFG] + [_P] * 10 + [_I32, _P]),
    "moe_layer_step_host": (_I32, [_CFG] + [_P] * 28),
    "moe_pipeline_create": (_I32, [C.POINTER(C.c_void_p)]),
    "moe_pipeline_destroy": (_I32, [_P]),
    "moe_layer_step_host_pipelined": (_I32, [_P, _CFG, _I32] + [_P] * 30),
    "moe_ctx_field": (_I32, [_CFG, C.c_char_p, _SZP, _SZP]),
    "moe_ws_field": (_I32, [_CFG, C.c_char_p, _SZP, _SZP]),
    "moe_profile_enable": (_I32, [_I32]),
    "moe_profile_stage_ms": (_I32, [C.c_char_p, C.POINTER(C.c_double), C.POINTER(C.c_int64)]),
}
EXPORTS = sorted(_SIGNATURES)


def lib() -> C.CDLL:
    """Load libmoe_b200.so (built by paper_2605_31463_b200/build.py or __graft_entry__.build())."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_2605_31463_b200.build` "
                              "(there is no CPU fallback)")
        l = C.CDLL(LIB_PATH)
        for name, (res, args) in _SIGNATURES.items():
            fn = getattr(l, name)
            fn.restype, fn.argtypes = res, args
        _lib = l
    return _lib


def status_string(status: int) -> str:
    return lib().moe_status_string(status).decode()


def _check(status: int, where: str):
    if status != MOE_OK:
        raise MoEError(status, where)


def _ptr(t):
    """Device (or pinned host) pointer of a torch tensor, or NULL."""
    if t is None:
        return None
    if not t.is_contiguous():
        raise ValueError("tensor must be contiguous")
    return C.c_void_p(t.data_ptr())


def _stream(stream=None):
    import torch
    s = stream if stream is not None else torch.cuda.current_stream()
    return C.c_void_p(s.cuda_stream)


# ------------------------------------------------------------------------------------------------
# queries
# ------------------------------------------------------------------------------------------------

def moe_version() -> int:
    return lib().moe_version()


def moe_launch_count() -> int:
    return lib().moe_launch_count()


STAGES = ["router_gemm", "route", "maps", "permute", "gemm1_swiglu", "gemm2", "combine", "combine_bwd",
          "dgrad_down_swiglu", "dgrad_gateup", "wgrad", "router_bwd", "dx_combine", "shared_fwd", "shared_bwd", "quant"]


def moe_profile_enable(on: bool):
    _check(lib().moe_profile_enable(1 if on else 0), "moe_profile_enable")


def moe_profile_stage_ms(stage: str):
    ms, n = C.c_double(0), C.c_int64(0)
    _check(lib().moe_profile_stage_ms(stage.encode(), C.byref(ms), C.byref(n)), "moe_profile_stage_ms")
    return ms.value, n.value


def moe_padded_rows(cfg) -> int:
    r = lib().moe_padded_rows(C.byref(make_config(cfg)))
    if r < 0:
        raise MoEError(MOE_ERR_INVALID_ARG, "moe_padded_rows")
    return r


def moe_layer_rows_fused(cfg) -> int:
    r = lib().moe_layer_rows_fused(C.byref(make_config(cfg)))
    if r < 0:
        raise MoEError(r, "moe_layer_rows_fused")
    return r


def moe_workspace_bytes(cfg):
    ws, ctx = C.c_size_t(0), C.c_size_t(0)
    _check(lib().moe_workspace_bytes(C.byref(make_config(cfg)), C.byref(ws), C.byref(ctx)), "moe_workspace_bytes")
    return ws.value, ctx.value


def _field(fn, cfg, name):
    off, ln = C.c_size_t(0), C.c_size_t(0)
    _check(fn(C.byref(make_config(cfg)), name.encode(), C.byref(off), C.byref(ln)), f"field {name}")
    return off.value, ln.value


def moe_ctx_field(cfg, name):
    return _field(lib().moe_ctx_field, cfg, name)


def moe_ws_field(cfg, name):
    return _field(lib().moe_ws_field, cfg, name)


# ------------------------------------------------------------------------------------------------
# ops (same names as the C ABI; tensors in, status checked)
# ------------------------------------------------------------------------------------------------

def moe_route(cfg, logits, bias, topk_idx, topk_w, stream=None):
    _check(lib().moe_route(C.byref(make_config(cfg)), _ptr(logits), _ptr(bias), _ptr(topk_idx), _ptr(topk_w),
                           _stream(stream)), "moe_route")


def moe_route_threshold(cfg, logits, threshold, topk_idx, topk_w, stream=None):
    _check(lib().moe_route_threshold(C.byref(make_config(cfg)), _ptr(logits), _ptr(threshold), _ptr(topk_idx),
                                     _ptr(topk_w), _stream(stream)), "moe_route_threshold")


def make_extras(threshold=None, zc_const=None, d_zc_const=None, aux_f_global=None, aux_loss=None) -> moe_extras_t:
    """moe_extras_t from torch tensors (None = NULL)."""
    def a(t):
        return None if t is None else _ptr(t).value
    return moe_extras_t(a(threshold), a(zc_const), a(d_zc_const), a(aux_f_global), a(aux_loss))


def moe_layer_fwd_ex(cfg, X, Wr, bias, Wg, Wu, Wd, Wg_s, Wu_s, Wd_s, Y, topk_idx, topk_w, ctx, ws, extras, stream=None):
    _check(lib().moe_layer_fwd_ex(C.byref(make_config(cfg)), _ptr(X), _ptr(Wr), _ptr(bias), _ptr(Wg), _ptr(Wu), _ptr(Wd),
                                  _ptr(Wg_s), _ptr(Wu_s), _ptr(Wd_s), _ptr(Y), _ptr(topk_idx), _ptr(topk_w), _ptr(ctx),
                                  _ptr(ws), C.byref(extras) if extras is not None else None, _stream(stream)),
           "moe_layer_fwd_ex")


def moe_layer_bwd_ex(cfg, dY, X, Wr, Wg, Wu, Wd, Wg_s, Wu_s, Wd_s, ctx, dX, dWr, dWg, dWu, dWd, dWg_s, dWu_s, dWd_s, ws,
                     extras, stream=None):
    _check(lib().moe_layer_bwd_ex(C.byref(make_config(cfg)), _ptr(dY), _ptr(X), _ptr(Wr), _ptr(Wg), _ptr(Wu), _ptr(Wd),
                                  _ptr(Wg_s), _ptr(Wu_s), _ptr(Wd_s), _ptr(ctx), _ptr(dX), _ptr(dWr), _ptr(dWg),
                                  _ptr(dWu), _ptr(dWd), _ptr(dWg_s), _ptr(dWu_s), _ptr(dWd_s), _ptr(ws),
                                  C.byref(extras) if extras is not None else None, _stream(stream)), "moe_layer_bwd_ex")


def moe_permute(cfg, X, topk_idx, counts, offsets, perm_to_flat, flat_to_perm, Xp, ws, stream=None):
    _check(lib().moe_permute(C.byref(make_config(cfg)), _ptr(X), _ptr(topk_idx), _ptr(counts), _ptr(offsets),
                             _ptr(perm_to_flat), _ptr(flat_to_perm), _ptr(Xp), _ptr(ws), _stream(stream)),
           "moe_permute")


def moe_permute_static_ws(cfg, X, topk_idx, counts, offsets, perm_to_flat, flat_to_perm, Xp, stream=None):
    """moe_permute without the `ws` argument, for callers that have no way to allocate one (they are handed only input
    and output tensors by a runtime that owns the device memory, or must not call cudaMalloc).  The scratch is a fixed
    1 MiB array inside the library; ceil(T*K/1024)*E*4 bytes must fit in it (MoEError MOE_ERR_TOO_LARGE otherwise).
    All calls on a GPU share that array: do not let two of them run at the same time.  Make the first call on a
    device outside any stream capture (it looks up the array's address).  See include/moe_b200.h."""
    _check(lib().moe_permute_static_ws(C.byref(make_config(cfg)), _ptr(X), _ptr(topk_idx), _ptr(counts), _ptr(offsets),
                                       _ptr(perm_to_flat), _ptr(flat_to_perm), _ptr(Xp), _stream(stream)),
           "moe_permute_static_ws")


def moe_grouped_gemm_fwd(cfg, N, Kdim, A, B, offsets, Cout, a_scales, b_scales, ws, stream=None):
    _check(lib().moe_grouped_gemm_fwd(C.byref(make_config(cfg)), N, Kdim, _ptr(A), _ptr(B), _ptr(offsets),
                                      _ptr(Cout), _ptr(a_scales), _ptr(b_scales), _ptr(ws), _stream(stream)),
           "moe_grouped_gemm_fwd")


def moe_grouped_gemm_bwd(cfg, N, Kdim, dC, A, B, offsets, dA, dB, ws, stream=None):
    _check(lib().moe_grouped_gemm_bwd(C.byref(make_config(cfg)), N, Kdim, _ptr(dC), _ptr(A), _ptr(B),
                                      _ptr(offsets), _ptr(dA), _ptr(dB), _ptr(ws), _stream(stream)),
           "moe_grouped_gemm_bwd")


def moe_swiglu(cfg, gu, a, rows, stream=None):
    _check(lib().moe_swiglu(C.byref(make_config(cfg)), _ptr(gu), _ptr(a), rows, _stream(stream)), "moe_swiglu")


def moe_swiglu_bwd(cfg, gu, da, dgu, rows, stream=None):
    _check(lib().moe_swiglu_bwd(C.byref(make_config(cfg)), _ptr(gu), _ptr(da), _ptr(dgu), rows, _stream(stream)),
           "moe_swiglu_bwd")


def moe_unpermute_combine(cfg, y, topk_w, flat_to_perm, shared_out, Y, stream=None):
    _check(lib().moe_unpermute_combine(C.byref(make_config(cfg)), _ptr(y), _ptr(topk_w), _ptr(flat_to_perm),
                                       _ptr(shared_out), _ptr(Y), _stream(stream)), "moe_unpermute_combine")


def moe_quantize_act(v, rows, cols, scale_mode, codes, scales, stream=None):
    _check(lib().moe_quantize_act(_ptr(v), rows, cols, scale_mode, _ptr(codes), _ptr(scales), _stream(stream)),
           "moe_quantize_act")


def moe_quantize_weight(w, batch, rows, cols, scale_mode, codes, scales, stream=None):
    _check(lib().moe_quantize_weight(_ptr(w), batch, rows, cols, scale_mode, _ptr(codes), _ptr(scales),
                                     _stream(stream)), "moe_quantize_weight")


def moe_fp8_quantize_weights(cfg, Wg, Wu, Wd, Wg_s, Wu_s, Wd_s, ctx, stream=None):
    _check(lib().moe_fp8_quantize_weights(C.byref(make_config(cfg)), _ptr(Wg), _ptr(Wu), _ptr(Wd), _ptr(Wg_s),
                                          _ptr(Wu_s), _ptr(Wd_s), _ptr(ctx), _stream(stream)),
           "moe_fp8_quantize_weights")


def moe_layer_fwd(cfg, X, Wr, bias, Wg, Wu, Wd, Wg_s, Wu_s, Wd_s, Y, topk_idx, topk_w, ctx, ws, stream=None):
    _check(lib().moe_layer_fwd(C.byref(make_config(cfg)), _ptr(X), _ptr(Wr), _ptr(bias), _ptr(Wg), _ptr(Wu), _ptr(Wd),
                               _ptr(Wg_s), _ptr(Wu_s), _ptr(Wd_s), _ptr(Y), _ptr(topk_idx), _ptr(topk_w), _ptr(ctx),
                               _ptr(ws), _stream(stream)), "moe_layer_fwd")


def moe_layer_bwd(cfg, dY, X, Wr, Wg, Wu, Wd, Wg_s, Wu_s, Wd_s, ctx, dX, dWr, dWg, dWu, dWd, dWg_s, dWu_s, dWd_s, ws,
                  stream=None):
    _check(lib().moe_layer_bwd(C.byref(make_config(cfg)), _ptr(dY), _ptr(X), _ptr(Wr), _ptr(Wg), _ptr(Wu), _ptr(Wd),
                               _ptr(Wg_s), _ptr(Wu_s), _ptr(Wd_s), _ptr(ctx), _ptr(dX), _ptr(dWr), _ptr(dWg),
                               _ptr(dWu), _ptr(dWd), _ptr(dWg_s), _ptr(dWu_s), _ptr(dWd_s), _ptr(ws),
                               _stream(stream)), "moe_layer_bwd")


def moe_layer_wgrad(cfg, X, dY, ctx, ws, dWg, dWu, dWd, dWg_s, dWu_s, dWd_s, accumulate_fp32, stream=None):
    _check(lib().moe_layer_wgrad(C.byref(make_config(cfg)), _ptr(X), _ptr(dY), _ptr(ctx), _ptr(ws), _ptr(dWg), _ptr(dWu),
                                 _ptr(dWd), _ptr(dWg_s), _ptr(dWu_s), _ptr(dWd_s), int(accumulate_fp32), _stream(stream)),
           "moe_layer_wgrad")


def moe_layer_step_host(cfg, X_host, dY_host, Y_host, dX_host, X_dev, dY_dev, Y_dev, dX_dev, Wr, bias, Wg, Wu, Wd,
                        Wg_s, Wu_s, Wd_s, dWr, dWg, dWu, dWd, dWg_s, dWu_s, dWd_s, topk_idx, topk_w, ctx, ws,
                        stream=None):
    args = [X_host, dY_host, Y_host, dX_host, X_dev, dY_dev, Y_dev, dX_dev, Wr, bias, Wg, Wu, Wd, Wg_s, Wu_s, Wd_s,
            dWr, dWg, dWu, dWd, dWg_s, dWu_s, dWd_s, topk_idx, topk_w, ctx, ws]
    _check(lib().moe_layer_step_host(C.byref(make_config(cfg)), *[_ptr(a) for a in args], _stream(stream)),
           "moe_layer_step_host")


def moe_pipeline_create():
    h = C.c_void_p(None)
    _check(lib().moe_pipeline_create(C.byref(h)), "moe_pipeline_create")
    return h


def moe_pipeline_destroy(pipeline):
    _check(lib().moe_pipeline_destroy(pipeline), "moe_pipeline_destroy")


def moe_layer_step_host_pipelined(pipeline, cfg, slot, X_host, dY_host, Y_host, dX_host, X_dev, dY_dev, Y_dev, dX_dev, Wr, bias, Wg,
                                  Wu, Wd, Wg_s, Wu_s, Wd_s, dWr, dWg, dWu, dWd, dWg_s, dWu_s, dWd_s, topk_idx, topk_w, ctx,
                                  ws, stream_in, stream_compute, stream_out):
    args = [X_host, dY_host, Y_host, dX_host, X_dev, dY_dev, Y_dev, dX_dev, Wr, bias, Wg, Wu, Wd, Wg_s, Wu_s, Wd_s,
            dWr, dWg, dWu, dWd, dWg_s, dWu_s, dWd_s, topk_idx, topk_w, ctx, ws]
    _check(lib().moe_layer_step_host_pipelined(pipeline, C.byref(make_config(cfg)), int(slot), *[_ptr(a) for a in args],
                                               _stream(stream_in), _stream(stream_compute), _stream(stream_out)),
           "moe_layer_step_host_pipelined")
