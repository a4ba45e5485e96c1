"""CPU checks of the boundary: the C-ABI library loads and exports every symbol include/moe_b200.h declares,
and the host-only entry points (status strings, size queries, argument validation) behave as documented.
No compute call is made (no GPU here)."""
import ctypes as C
import os
import re

import pytest

import workloads as wl

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "moe_b200.h")


@pytest.fixture(scope="module")
def moe():
    import __graft_entry__ as ge
    ge.build()
    import paper_2605_31463_b200 as m
    return m


def declared_symbols():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(moe_[a-z0-9_]+)\s*\(", src)))


def test_header_declares_north_star_calls():
    names = declared_symbols()
    for need in ("moe_route", "moe_permute", "moe_grouped_gemm_fwd", "moe_grouped_gemm_bwd", "moe_swiglu",
                 "moe_unpermute_combine", "moe_layer_fwd", "moe_layer_bwd"):
        assert need in names


def test_library_exports_every_declared_symbol(moe):
    lib = C.CDLL(moe.LIB_PATH)
    for name in declared_symbols():
        assert hasattr(lib, name), f"{name} declared in moe_b200.h but not exported"
    assert set(declared_symbols()) == set(moe.EXPORTS)


def test_status_strings_and_version(moe):
    assert moe.moe_version() >= 100
    seen = {moe.status_string(s) for s in (0, -1, -2, -3, -4)}
    assert len(seen) == 5


@pytest.mark.parametrize("cfg", list(wl.CONFIGS.values()) + list(wl.SMALL_CONFIGS.values()), ids=lambda c: c.name)
def test_size_queries(moe, cfg):
    for align in (1, 128):
        c = cfg.replace(row_align=align)
        assert moe.moe_padded_rows(c) == c.TK_pad
        ws, ctx = moe.moe_workspace_bytes(c)
        assert ws > 0 and ctx > 0 and ws % 256 == 0 and ctx % 256 == 0
        off, ln = moe.moe_ctx_field(c, "flat_to_perm")
        assert ln == c.TK * 4 and off + ln <= ctx


def test_invalid_configs_are_rejected_on_the_host(moe):
    bad = [wl.TINY.replace(K=9), wl.TINY.replace(T=0), wl.TINY.replace(n_group=3),
           wl.DSV3_SMALL.replace(topk_group=1, K=16), wl.TINY.replace(score_fn=7)]
    for c in bad:
        with pytest.raises(moe.MoEError):
            moe.moe_workspace_bytes(c)
    # NULL pointers: INVALID_ARG before anything is enqueued (no CUDA call happens)
    st = moe.lib().moe_route(C.byref(moe.make_config(wl.TINY)), None, None, None, None, None)
    assert st == moe.MOE_ERR_INVALID_ARG


def test_pipeline_object_is_validated_on_the_host(moe):
    """moe_layer_step_host_pipelined keeps its ordering events in a caller-owned object: a NULL / dead handle is
    INVALID_ARG before anything is enqueued; creating one needs a CUDA device (MOE_ERR_CUDA here)."""
    l = moe.lib()
    assert l.moe_pipeline_destroy(None) == moe.MOE_ERR_INVALID_ARG
    args = [None] * 30
    st = l.moe_layer_step_host_pipelined(None, C.byref(moe.make_config(wl.TINY)), 0, *args)
    assert st == moe.MOE_ERR_INVALID_ARG
    import torch
    if not torch.cuda.is_available():
        h = C.c_void_p(None)
        assert l.moe_pipeline_create(C.byref(h)) == moe.MOE_ERR_CUDA and not h.value


def test_layer_calls_reject_unsupported_configs_before_any_launch(moe):
    """UNSUPPORTED is decided by the pre-flight, not by the stage that would hit the limit: with dummy non-NULL
    pointers and no GPU the call must return UNSUPPORTED (a launch attempt would return MOE_ERR_CUDA instead)."""
    l = moe.lib()
    bad = wl.QWEN3_SMALL.replace(E=2048, K=4)                      # moe_route holds at most 1024 experts per warp
    dummy = C.c_void_p(256)
    st = l.moe_layer_fwd(C.byref(moe.make_config(bad)), *([dummy] * 14), None)
    assert st == moe.MOE_ERR_UNSUPPORTED
    st = l.moe_layer_bwd(C.byref(moe.make_config(bad)), *([dummy] * 19), None)
    assert st == moe.MOE_ERR_UNSUPPORTED
    fp8_unaligned = wl.DSV3_FP8_SMALL.replace(row_align=1)
    st = l.moe_layer_fwd(C.byref(moe.make_config(fp8_unaligned)), *([dummy] * 14), None)
    assert st == moe.MOE_ERR_UNSUPPORTED


def test_ws_layout_does_not_depend_on_the_fusion_selector(moe):
    """The workspace size and every offset inside it are fixed by the shape of the problem alone: opt_rows_fused may
    differ between the sizing query, moe_layer_bwd and a delayed moe_layer_wgrad without moving `dgu` / `dXp` (ADVICE r2,
    layout.cu).  Also: the library reads no environment variable any more."""
    base = wl.QWEN3_SMALL.replace(row_align=128)
    seen = set()
    for sel in (0, 1, 2, 3):
        cfg = base.replace(opt_rows_fused=sel)
        assert moe.moe_layer_rows_fused(cfg) == (1 if sel == 0 else sel - 1)
        seen.add((moe.moe_workspace_bytes(cfg), moe.moe_ws_field(cfg, "dy"), moe.moe_ws_field(cfg, "dgu"),
                  moe.moe_ws_field(cfg, "dXp")))
    assert len(seen) == 1
    with pytest.raises(moe.MoEError):
        moe.moe_workspace_bytes(base.replace(opt_pair=4))
    # (the static CUDA runtime inside the .so imports getenv for its own use, so the sources are what is checked)
    csrc = os.path.join(ROOT, "paper_2605_31463_b200", "csrc")
    for f in os.listdir(csrc):
        assert "getenv" not in open(os.path.join(csrc, f)).read(), f


def test_host_step_rejects_configs_that_need_extras_before_any_copy(moe):
    """moe_layer_step_host takes no moe_extras_t; a threshold-routing or constant-expert config must come back as
    INVALID_ARG from the preflight.  Without a GPU any enqueued copy would fail with MOE_ERR_CUDA instead, so the status
    also proves that nothing was enqueued (api.cu)."""
    l = moe.lib()
    dummy = (C.c_int32 * 4)()
    p = C.cast(dummy, C.c_void_p)
    args = [p] * 27 + [None]                                      # 27 non-NULL pointers + stream
    for cfg in (wl.TINY.replace(score_fn=1, route_mode=1), wl.TINY.replace(n_const=1)):
        st = l.moe_layer_step_host(C.byref(moe.make_config(cfg)), *args)
        assert st == moe.MOE_ERR_INVALID_ARG, moe.status_string(st)
    # a missing weight pointer is caught there as well (Wg is the 11th pointer)
    bad = list(args)
    bad[10] = None
    assert l.moe_layer_step_host(C.byref(moe.make_config(wl.TINY)), *bad) == moe.MOE_ERR_INVALID_ARG
