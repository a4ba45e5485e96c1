"""Routing-trace dump in the schema of PAPER.md:424 (App. B.2.1 "Collect Routing Trace"): one
`step-<step_id:08d>.npz` per step, holding for every MoE layer the top-k expert IDs and gating weights of every token
of the batch.  Host-side file IO only; the arrays are the `topk_idx` / `topk_w` outputs of moe_route / moe_layer_fwd."""
from __future__ import annotations

import os

import numpy as np


def _to_host(a):
    if hasattr(a, "detach"):                       # torch tensor (device or host)
        a = a.detach().cpu().numpy()
    return np.ascontiguousarray(a)


def dump_routing_trace(out_dir: str, step_id: int, layers) -> str:
    """layers: iterable of (topk_idx [T,K] int32, topk_w [T,K] fp32), one pair per MoE layer in model order.
    Writes out_dir/step-<step_id:08d>.npz with arrays layer<i>.expert_ids and layer<i>.gating_weights."""
    os.makedirs(out_dir, exist_ok=True)
    arrays = {}
    for i, (idx, w) in enumerate(layers):
        idx, w = _to_host(idx), _to_host(w)
        if idx.shape != w.shape or idx.ndim != 2:
            raise ValueError(f"layer {i}: expert IDs {idx.shape} and gating weights {w.shape} must both be [tokens, top_k]")
        arrays[f"layer{i}.expert_ids"] = idx.astype(np.int32, copy=False)
        arrays[f"layer{i}.gating_weights"] = w.astype(np.float32, copy=False)
    path = os.path.join(out_dir, f"step-{step_id:08d}.npz")
    np.savez(path, **arrays)
    return path


def check_routing_trace(path: str, num_experts: int, weight_sum: float = 1.0, atol: float = 1e-4,
                        variable_k: bool = False) -> int:
    """The programmatic check of PAPER.md:436 (App. B.2.2): IDs in [0, num_experts), gating weights non-negative and
    summing to `weight_sum` (1, or the routed scaling factor) over the top-k of every token.  `variable_k` (a
    threshold-gated router): unused slots hold ID -1 with weight 0 and every token keeps >= 1 expert.
    Returns the layer count."""
    z = np.load(path)
    n = 0
    while f"layer{n}.expert_ids" in z:
        idx, w = z[f"layer{n}.expert_ids"], z[f"layer{n}.gating_weights"]
        if idx.shape != w.shape:
            raise ValueError(f"layer {n}: shape mismatch")
        if idx.min() < (-1 if variable_k else 0) or idx.max() >= num_experts:
            raise ValueError(f"layer {n}: expert ID out of range")
        if variable_k and ((w[idx < 0] != 0).any() or (idx[:, 0] < 0).any()):
            raise ValueError(f"layer {n}: an empty slot must have weight 0 and slot 0 must be filled")
        if (w < 0).any() or not np.allclose(w.sum(axis=1), weight_sum, atol=atol):
            raise ValueError(f"layer {n}: gating weights must be non-negative and sum to {weight_sum}")
        n += 1
    if n == 0:
        raise ValueError("no layers in trace")
    return n
