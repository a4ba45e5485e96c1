"""moe_permute_static_ws: the permutation step for callers that cannot allocate device memory.

moe_permute wants a scratch buffer `ws` from its caller.  A caller that lives inside somebody else's runtime (an operator
plug-in that is given its input and output tensors and nothing else), or in a process that forbids cudaMalloc once it is
up (cudaMalloc stalls the whole device and may fail when the GPU is nearly full), has no such buffer to give.
moe_permute_static_ws keeps the scratch in a fixed 1 MiB array inside libmoe_b200.so instead and takes no `ws`.

The check here is against the existing path, not the oracle (moe_permute itself is compared with the oracle bit by bit
in test_gpu_ops.py): same inputs through both entry points, every output must be identical -- maps and copied rows are
integer / byte work, so the tolerance is zero, as in the other permutation tests.  It is done on several calls in a row
with different shapes, because all calls share the one array and the later ones see what the earlier ones left in it.

This file is named test_zz_* so that pytest collects it last: with `-x` a failure here hides no other test.  It must pass
alone in a fresh process (first use of the array on the device) and after the whole suite.
"""
import ctypes as C

import pytest

import workloads as wl


def _lib():
    import __graft_entry__ as ge
    ge.build()
    import paper_2605_31463_b200 as moe
    moe.lib()
    return moe


def test_static_ws_rejects_what_does_not_fit():
    """Host-side only (no GPU needed): a problem whose chunk histograms exceed the built-in array is refused with
    MOE_ERR_TOO_LARGE before anything is launched; NULL outputs are INVALID_ARG."""
    moe = _lib()
    l = moe.lib()
    dummy = (C.c_int32 * 4)()                     # never dereferenced: the call must fail before any launch
    p = C.cast(dummy, C.c_void_p)
    fits = wl.QWEN3.replace(T=131072, E=256, K=8)           # 1024 chunks * 256 experts * 4 B = exactly 1 MiB
    assert (fits.T * fits.K // 1024) * fits.E * 4 == moe.MOE_PERMUTE_STATIC_WS_BYTES
    big = fits.replace(T=fits.T + 1)                        # one more chunk
    st = l.moe_permute_static_ws(C.byref(moe.make_config(big)), None, p, p, p, p, p, None, None)
    assert st == moe.MOE_ERR_TOO_LARGE
    assert "MOE_PERMUTE_STATIC_WS_BYTES" in moe.status_string(st)
    st = l.moe_permute_static_ws(C.byref(moe.make_config(wl.TINY)), None, p, None, p, p, p, None, None)
    assert st == moe.MOE_ERR_INVALID_ARG


def _both_paths(torch, moe, buffers, cfg, seed_shift):
    """Run moe_permute (caller's ws) and moe_permute_static_ws on the same routing and the same X; return both
    result sets (device tensors) and how much the device's free memory shrank across the new call."""
    dt = buffers.act_dtype(cfg)
    g = torch.Generator(device="cpu").manual_seed(1234 + seed_shift)
    # any valid routing will do: K distinct experts per token
    idx = torch.rand((cfg.T, cfg.E), generator=g).argsort(1)[:, :cfg.K].contiguous().to(torch.int32).cuda()
    X = torch.randn((cfg.T, cfg.H), generator=g).to(dt).cuda()
    R = moe.moe_padded_rows(cfg)
    ws_b, _ = moe.moe_workspace_bytes(cfg)
    ws = torch.empty(ws_b, dtype=torch.uint8, device="cuda")

    def outputs():
        return (torch.full((cfg.E,), -7, dtype=torch.int32, device="cuda"),
                torch.full((cfg.E + 1,), -7, dtype=torch.int32, device="cuda"),
                torch.full((R,), -7, dtype=torch.int32, device="cuda"),
                torch.full((cfg.TK,), -7, dtype=torch.int32, device="cuda"),
                torch.full((R, cfg.H), 7.0, dtype=dt, device="cuda"))

    ref = outputs()
    moe.moe_permute(cfg, X, idx, ref[0], ref[1], ref[2], ref[3], ref[4], ws)
    new = outputs()
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    moe.moe_permute_static_ws(cfg, X, idx, new[0], new[1], new[2], new[3], new[4])
    torch.cuda.synchronize()
    free1 = torch.cuda.mem_get_info()[0]
    return ref, new, free0 - free1


@pytest.mark.gpu
def test_static_ws_matches_moe_permute_on_calls_in_a_row():
    import torch
    moe = _lib()
    from paper_2605_31463_b200 import buffers
    # a large problem first, then smaller ones with other E / K / alignment: the later calls find the earlier calls'
    # histograms still in the shared array and must not be disturbed by them
    cases = [wl.QWEN3.replace(row_align=128), wl.QWEN3_SMALL.replace(row_align=1), wl.DSV3_SMALL.replace(row_align=128),
             wl.TINY.replace(T=1025, K=3, row_align=1), wl.QWEN3_SMALL.replace(row_align=1)]
    names = ("counts", "offsets", "perm_to_flat", "flat_to_perm", "Xp")
    grew = None
    for i, cfg in enumerate(cases):
        ref, new, grew = _both_paths(torch, moe, buffers, cfg, i)
        n = int(ref[1][-1])                                   # rows below offsets[E] are defined
        for name, a, b in zip(names, ref, new):
            if name == "Xp":
                a, b = a[:n].view(torch.uint8), b[:n].view(torch.uint8)
            assert torch.equal(a, b), f"call {i} ({cfg.name}): {name} differs from moe_permute"
        assert int(new[0].sum()) == cfg.TK
    # the last call repeated a shape whose kernels were already loaded: the device's free memory must not have moved
    assert grew == 0, f"moe_permute_static_ws changed free device memory by {grew} bytes"
