"""fp64 CPU oracle for the routed-expert MoE layer, forward and backward.

TEST INFRASTRUCTURE ONLY.  Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s cpu_baseline /
`--impl reference` leg may import this package.  It shares no code with the CUDA path
(`paper_2605_31463_b200/`), imports nothing from it, and never receives a value computed by it.

What it is: the plain definition of a top-k-gated SwiGLU MoE layer, evaluated expert by expert in
NumPy fp64, in the order and notation of SURVEY.md §8(c) R1..R9.  The paper itself
 states no equation for the layer; it fixes only
  * the routing outputs: "the top-k expert IDs and their gating weights"      (App. B.2.1)
  * their validity: IDs in [0, num_experts), weights non-negative and summing
    to 1 over the top-k selected experts                                       (App. B.2.2)
  * per-expert shapes are data-dependent (dropless)                            (§3.2)
  * SwiGLU [34] expert FFN with fused fwd/bwd kernels, FP8 (e4m3 [22]) training (§3.2)
Every other choice is a reading listed in DESIGN.md ("Readings of the paper"), taken from
SURVEY.md §8(c) S1..S20 and BASELINE.json:north_star / configs.

Widened rows (readings A1..A3, V1, V2 of DESIGN.md section 2): the auxiliary global-level
load-balancing loss, the threshold-gated variable-k router and the
zero-computation experts.  They are off unless the config enables them
(aux_coef != 0, route_mode == 1, n_zero + n_copy + n_const > 0).

Pins (tests/test_oracle_*.py, all `-m "not gpu"`): brute-force top-k with hand-made ties; weight
sum / sign; softmax->top-k->renorm == top-k->softmax closed form; group-limit
reductions; permutation bijection / stability; permute->combine identity with w = 1/K; E=1,K=1 ==
dense SwiGLU FFN; shared-weights invariance; central finite differences of every gradient; e4m3
spot values from the format definition [22].  End-to-end numeric values: PARITY UNPINNED BY THE
PAPER (it prints no worked example of the layer) -- see DESIGN.md.
"""
from __future__ import annotations

import numpy as np

F64 = np.float64
NEG_INF = -np.inf

# =====================================================================================
# R1  router logits                                   (PAPER.md:424 names only the outputs)
# =====================================================================================


def router_logits(X, Wr):
    """z[t,e] = sum_h X[t,h] * Wr[e,h], fp64."""
    return np.asarray(X, F64) @ np.asarray(Wr, F64).T


# =====================================================================================
# R2-R5  routing: scores, group limiting, top-k, gating weights
# =====================================================================================


def sigmoid(z):
    return 1.0 / (1.0 + np.exp(-np.asarray(z, F64)))


def selection_keys(z, bias, cfg, key_dtype=F64):
    """R2.  softmax: key = z (+ b);  sigmoid: key = s + b with s = 1/(1+exp(-z)).

    key_dtype = float32 reproduces the precision in which the kernel takes the (integer) top-k
    decision: s is evaluated in fp64 and rounded once to fp32, the bias add is one IEEE fp32 add.
    """
    z = np.asarray(z)
    if cfg.score_fn == 0:
        key = z.astype(key_dtype)
    else:
        key = sigmoid(z).astype(key_dtype)
    if cfg.has_bias and bias is not None:
        key = key + np.asarray(bias).astype(key_dtype)[None, :]
    return key


def group_limit(key, cfg):
    """R3.  Keep the `topk_group` groups (contiguous blocks of E/n_group experts) with the largest
    group score; score = sum of the two largest keys in the group (group_score=1, DeepSeek-V3 style)
    or their max (group_score=0).  Ties -> lower group index.  Keys outside kept groups -> -inf."""
    G, Kg = cfg.n_group, cfg.topk_group
    if G <= 1 or Kg >= G:
        return key
    T, E = key.shape
    per = E // G
    kg = key.reshape(T, G, per)
    srt = -np.sort(-kg, axis=2)                      # descending within each group
    score = srt[:, :, 0] + srt[:, :, 1] if (cfg.group_score == 1 and per > 1) else srt[:, :, 0]
    keep = np.zeros((T, G), bool)
    sc = score.copy()
    rows = np.arange(T)
    for _ in range(Kg):                              # Kg rounds of arg-max, first (= lowest) index wins ties
        gsel = np.argmax(sc, axis=1)
        keep[rows, gsel] = True
        sc[rows, gsel] = NEG_INF
    out = np.where(np.repeat(keep, per, axis=1), key, np.asarray(NEG_INF, key.dtype))
    return out


def topk_select(key, K):
    """R4.  K rounds of arg-max; ties -> lower expert index; slot j holds the j-th largest key."""
    key = np.array(key, copy=True)
    T = key.shape[0]
    rows = np.arange(T)
    idx = np.empty((T, K), np.int32)
    for j in range(K):
        sel = np.argmax(key, axis=1)                 # numpy returns the first maximal index
        idx[:, j] = sel
        key[rows, sel] = NEG_INF
    return idx


def gate_weights(z, idx, cfg):
    """R5.  fp64 gating weights of the selected experts (the selection bias is never in w).
    softmax, renorm: w_j = exp(z_j - m) / sum_{i in sel} exp(z_i - m);  no renorm: softmax over all E.
    sigmoid, renorm: w_j = c * s_j / (sum_{i in sel} s_i + 1e-20);      no renorm: c * s_j."""
    z = np.asarray(z, F64)
    zs = np.take_along_axis(z, idx.astype(np.int64), axis=1)
    c = float(cfg.routed_scale)
    if cfg.score_fn == 0:
        if cfg.renorm:
            m = zs.max(axis=1, keepdims=True)
            p = np.exp(zs - m)
            w = p / p.sum(axis=1, keepdims=True)
        else:
            m = z.max(axis=1, keepdims=True)
            w = np.exp(zs - m) / np.exp(z - m).sum(axis=1, keepdims=True)
        return c * w
    s = sigmoid(zs)
    if cfg.renorm:
        return c * s / (s.sum(axis=1, keepdims=True) + 1e-20)
    return c * s


def threshold_select(key, thr, K):
    """V1: an expert is active for a token iff its gate s = sigmoid(z) exceeds the expert's
    threshold thr[e]; the number of active experts varies per token.  Active experts fill the K slots in
    (s desc, index asc) order (more than K active: the K largest stay); unused slots hold -1; a token no expert
    admits keeps its single best expert (top-1 fallback), so every token is computed (dropless)."""
    key = np.asarray(key)
    T, E = key.shape
    act = key > np.asarray(thr).astype(key.dtype)[None, :]
    masked = np.where(act, key, np.asarray(NEG_INF, key.dtype))
    idx = topk_select(masked, K)                               # inactive experts have key -inf
    n_act = act.sum(axis=1)
    idx = np.where(np.arange(K)[None, :] < n_act[:, None], idx, -1).astype(np.int32)   # slot j is filled iff j < #active
    none = n_act == 0
    idx[none, 0] = np.argmax(key[none], axis=1)               # first maximal index: ties -> lower expert
    return idx


def gate_weights_masked(z, idx, cfg):
    """R5 over a variable-size selection (slots with idx = -1 are empty: weight 0).  Sigmoid scores only (V1)."""
    z = np.asarray(z, F64)
    ok = idx >= 0
    s = np.where(ok, sigmoid(np.take_along_axis(z, np.where(ok, idx, 0).astype(np.int64), axis=1)), 0.0)
    c = float(cfg.routed_scale)
    if cfg.renorm:
        return c * s / (s.sum(axis=1, keepdims=True) + 1e-20)
    return c * s


def route(z, bias, cfg, key_dtype=F64, forced_idx=None, threshold=None):
    """R2..R5: (topk_idx int32 [T,K], topk_w fp64 [T,K]).  `forced_idx` overrides the selection
    (used by parity tests only for tokens whose k/(k+1) key gap is a verified near-tie).
    route_mode 1 (V1): threshold-gated variable-k selection on the sigmoid gates; `threshold` is thr[E]."""
    if getattr(cfg, "route_mode", 0) == 1:
        if forced_idx is None:
            idx = threshold_select(sigmoid(z).astype(key_dtype), threshold, cfg.K)
        else:
            idx = np.asarray(forced_idx, np.int32)
        return idx, gate_weights_masked(z, idx, cfg)
    if forced_idx is None:
        key = group_limit(selection_keys(z, bias, cfg, key_dtype), cfg)
        idx = topk_select(key, cfg.K)
    else:
        idx = np.asarray(forced_idx, np.int32)
    return idx, gate_weights(z, idx, cfg)


# =====================================================================================
# A1..A3  auxiliary global-level load-balancing loss          ([30])
# =====================================================================================


def router_probs(z, cfg):
    """A2: the differentiable per-token distribution over ALL experts that the balance term averages:
    softmax configs p = softmax(z); sigmoid configs p = s / sum_e s (normalised gate scores)."""
    z = np.asarray(z, F64)
    if cfg.score_fn == 0 and getattr(cfg, "route_mode", 0) == 0:
        m = z.max(axis=1, keepdims=True)
        p = np.exp(z - m)
    else:
        p = sigmoid(z)
    return p / p.sum(axis=1, keepdims=True)


def aux_expert_weights(cfg):
    """V2 (PAPER.md:488 R3): zero-computation experts enter the balance term with weight aux_zc_weight, FFN experts 1."""
    eta = np.ones(cfg.E, F64)
    nz = cfg.n_zero + cfg.n_copy + cfg.n_const
    if nz:
        eta[cfg.E - nz:] = float(cfg.aux_zc_weight)
    return eta


def aux_loss(cfg, z, idx, f_global=None):
    """A1: L_aux = aux_coef * E * sum_e eta_e f_e P_e with f_e = the fraction of the batch's routed assignments that
    went to expert e (counted over the GLOBAL batch: `f_global` when the caller has all-reduced the counts over its
    data-parallel ranks, else this batch's own counts; variable-k routing divides by the number of assignments made,
    PAPER.md:456) and P_e = mean over tokens of p[t, e].  f carries no gradient.  Returns (loss, f, P)."""
    E = cfg.E
    if f_global is None:
        flat = np.asarray(idx).reshape(-1)
        flat = flat[flat >= 0]
        f = np.bincount(flat, minlength=E).astype(F64) / max(flat.size, 1)
    else:
        f = np.asarray(f_global, F64)
    P = router_probs(z, cfg).mean(axis=0)
    return float(cfg.aux_coef) * E * float((aux_expert_weights(cfg) * f * P).sum()), f, P


def aux_dz(cfg, z, f):
    """A3: d L_aux / d z[t, j] (dense [T,E]).  softmax: (c/T) p_j (g_j - sum_e g_e p_e); normalised sigmoid:
    (c/T) s_j (1 - s_j) / S (g_j - sum_e g_e p_e); c = aux_coef * E, g = eta * f."""
    z = np.asarray(z, F64)
    T = z.shape[0]
    p = router_probs(z, cfg)
    g = aux_expert_weights(cfg) * np.asarray(f, F64)
    inner = (p * g[None, :]).sum(axis=1, keepdims=True)
    c = float(cfg.aux_coef) * cfg.E / T
    if cfg.score_fn == 0 and getattr(cfg, "route_mode", 0) == 0:
        return c * p * (g[None, :] - inner)
    s = sigmoid(z)
    return c * s * (1.0 - s) / s.sum(axis=1, keepdims=True) * (g[None, :] - inner)


# =====================================================================================
# R6  permutation into expert-contiguous order (stable counting sort)
# =====================================================================================


def permute_maps(idx, E, row_align=1):
    """counts[E], offsets[E+1], perm_to_flat[offsets[E]], flat_to_perm[T*K].
    Flat position p = t*K + j.  Within an expert rows are in ascending p.  Each group starts at a
    multiple of row_align; padding rows map to -1."""
    flat = np.asarray(idx, np.int64).reshape(-1)
    counts = np.bincount(flat[flat >= 0], minlength=E).astype(np.int32)   # -1 = empty slot (variable-k routing, V1)
    a = max(int(row_align), 1)
    padded = (counts.astype(np.int64) + a - 1) // a * a
    offsets = np.zeros(E + 1, np.int64)
    offsets[1:] = np.cumsum(padded)
    perm_to_flat = np.full(int(offsets[E]), -1, np.int32)
    flat_to_perm = np.full(flat.size, -1, np.int32)
    order = np.argsort(flat, kind="stable")          # ascending expert, then ascending p
    start = int((flat < 0).sum())                    # empty slots sort first and are skipped
    for e in range(E):
        c = int(counts[e])
        p = order[start:start + c]
        r = offsets[e] + np.arange(c)
        perm_to_flat[r] = p
        flat_to_perm[p] = r
        start += c
    return counts, offsets.astype(np.int32), perm_to_flat, flat_to_perm


def permute_rows(X, perm_to_flat, K):
    """Xp[r] = X[perm_to_flat[r] div K]; padding rows are zero."""
    X = np.asarray(X)
    Xp = np.zeros((perm_to_flat.size, X.shape[1]), X.dtype)
    ok = perm_to_flat >= 0
    Xp[ok] = X[perm_to_flat[ok] // K]
    return Xp


def unpermute_combine(y, w, flat_to_perm, shared_out=None):
    """R7 combine.  Y[t] = sum_{j=0..K-1} w[t,j] * y[flat_to_perm[t*K+j]]  (+ shared_out[t])."""
    T, K = w.shape
    y = np.asarray(y, F64)
    Y = np.zeros((T, y.shape[1]), F64)
    f2p = flat_to_perm.reshape(T, K)
    for j in range(K):
        ok = f2p[:, j] >= 0                          # empty slot: no row, no contribution
        Y[ok] += np.asarray(w, F64)[ok, j:j + 1] * y[f2p[ok, j]]
    if shared_out is not None:
        Y += np.asarray(shared_out, F64)
    return Y


# =====================================================================================
# R7  SwiGLU expert FFN, forward                                    ([34])
# =====================================================================================


def swiglu(g, u):
    """a = silu(g) * u = g * sigma(g) * u."""
    g = np.asarray(g, F64)
    return g * sigmoid(g) * np.asarray(u, F64)


def swiglu_bwd(da, g, u):
    """dg = da*u*sigma(g)*(1 + g*(1 - sigma(g))),  du = da*g*sigma(g)."""
    g = np.asarray(g, F64); u = np.asarray(u, F64); da = np.asarray(da, F64)
    s = sigmoid(g)
    return da * u * s * (1.0 + g * (1.0 - s)), da * g * s


def expert_ffn_fwd(Xe, Wg, Wu, Wd):
    """One expert (or the shared expert) on its rows: g = Xe Wg^T, u = Xe Wu^T, a = silu(g)*u,
    y = a Wd^T.  Wg,Wu: [F,H]; Wd: [H,F]."""
    Xe = np.asarray(Xe, F64)
    g = Xe @ np.asarray(Wg, F64).T
    u = Xe @ np.asarray(Wu, F64).T
    a = swiglu(g, u)
    y = a @ np.asarray(Wd, F64).T
    return g, u, a, y


def expert_ffn_bwd(dy, Xe, g, u, a, Wg, Wu, Wd):
    """R8 for one expert: returns dXe, dWg, dWu, dWd (and dg, du)."""
    dy = np.asarray(dy, F64); Xe = np.asarray(Xe, F64)
    da = dy @ np.asarray(Wd, F64)
    dWd = dy.T @ np.asarray(a, F64)
    dg, du = swiglu_bwd(da, g, u)
    dXe = dg @ np.asarray(Wg, F64) + du @ np.asarray(Wu, F64)
    dWg = dg.T @ Xe
    dWu = du.T @ Xe
    return dXe, dWg, dWu, dWd, dg, du


# =====================================================================================
# R9  FP8 e4m3 block quantisers                                  ([22])
# =====================================================================================

E4M3_MAX = 448.0


def _e4m3_table():
    """All 256 e4m3fn values from the format definition: 1 sign, 4 exponent (bias 7), 3 mantissa;
    exponent 0 = subnormal m*2^-9; no infinities; S.1111.111 = NaN."""
    t = np.empty(256, F64)
    for c in range(256):
        s = -1.0 if c & 0x80 else 1.0
        e = (c >> 3) & 0xF
        m = c & 0x7
        if e == 0xF and m == 0x7:
            t[c] = np.nan
        elif e == 0:
            t[c] = s * m * 2.0 ** -9
        else:
            t[c] = s * (1.0 + m / 8.0) * 2.0 ** (e - 7)
    return t


E4M3_TABLE = _e4m3_table()


def e4m3_encode(v):
    """fp32 -> e4m3fn code (uint8): round to nearest, ties to even; |v| > 448 saturates to +-448."""
    v = np.asarray(v, np.float32)
    a = np.minimum(np.abs(v).astype(F64), E4M3_MAX)          # saturate
    mant, ex = np.frexp(a)                                    # a = mant * 2^ex, mant in [0.5,1)
    e = ex - 1                                                # floor(log2 a) for a > 0
    sub = a < 2.0 ** -6
    quantum = np.where(sub, 2.0 ** -9, np.exp2((e - 3).astype(F64)))
    q = np.rint(a / quantum)                                  # exact scaling, RNE
    code_sub = q.astype(np.int64)                             # 0..8 (8 == smallest normal, code 0x08)
    carry = q >= 16
    e2 = np.where(carry, e + 1, e)
    q2 = np.where(carry, 8, q).astype(np.int64)
    code_norm = ((e2 + 7).astype(np.int64) << 3) | (q2 - 8)
    code = np.where(sub, code_sub, code_norm)
    code = np.where(a == 0, 0, code)
    sign = np.signbit(v).astype(np.int64) << 7
    return (code | sign).astype(np.uint8)


def e4m3_decode(code):
    return E4M3_TABLE[np.asarray(code, np.uint8)]


def _block_scale(amax, mode):
    """scale (fp32) from a block's amax (fp32): mode 0 = amax/448; mode 1 = 2^ceil(log2(amax/448));
    amax == 0 -> 1."""
    amax = np.asarray(amax, np.float32)
    r = amax / np.float32(E4M3_MAX)                           # fp32 division
    if mode == 1:
        m, ex = np.frexp(r)                                   # r = m*2^ex, m in [0.5,1)
        r = np.where(m == np.float32(0.5), np.ldexp(np.float32(1), ex - 1),
                     np.ldexp(np.float32(1), ex)).astype(np.float32)
    return np.where(amax == 0, np.float32(1), r).astype(np.float32)


def quantize_1x128(v, mode=0):
    """Activation quantiser: blocks of 128 along the last axis.  Input: values on the bf16 grid
    (held in fp32).  Returns (codes uint8 [R,C], scales fp32 [R, ceil(C/128)])."""
    v = np.asarray(v, np.float32)
    R, C = v.shape
    nb = (C + 127) // 128
    pad = np.zeros((R, nb * 128), np.float32)
    pad[:, :C] = v
    blk = pad.reshape(R, nb, 128)
    scale = _block_scale(np.abs(blk).max(axis=2), mode)
    codes = e4m3_encode(blk / scale[:, :, None])              # fp32 division, then RNE to e4m3
    return codes.reshape(R, nb * 128)[:, :C], scale


def quantize_128x128(w, mode=0):
    """Weight quantiser: 128x128 blocks over the last two axes.  Returns (codes, scales
    [..., ceil(R/128), ceil(C/128)])."""
    w = np.asarray(w, np.float32)
    lead = w.shape[:-2]
    R, C = w.shape[-2:]
    rb, cb = (R + 127) // 128, (C + 127) // 128
    pad = np.zeros(lead + (rb * 128, cb * 128), np.float32)
    pad[..., :R, :C] = w
    blk = pad.reshape(lead + (rb, 128, cb, 128))
    scale = _block_scale(np.abs(blk).max(axis=(-3, -1)), mode)
    codes = e4m3_encode(blk / scale[..., :, None, :, None])
    return codes.reshape(lead + (rb * 128, cb * 128))[..., :R, :C], scale


def dequantize_1x128(codes, scale):
    R, C = codes.shape
    s = np.repeat(scale.astype(F64), 128, axis=1)[:, :C]
    return e4m3_decode(codes) * s


def dequantize_128x128(codes, scale):
    R, C = codes.shape[-2:]
    s = np.repeat(np.repeat(scale.astype(F64), 128, axis=-2), 128, axis=-1)[..., :R, :C]
    return e4m3_decode(codes) * s


def bf16_round(x):
    """Round fp64/fp32 values to the bf16 grid (RNE), returned as fp32.  Used only where R9 says a
    quantiser's input is the bf16 tensor."""
    u = np.asarray(x, np.float32).view(np.uint32)
    r = ((u >> np.uint32(16)) & np.uint32(1)) + np.uint32(0x7FFF)
    return (((u + r) >> np.uint32(16)) << np.uint32(16)).astype(np.uint32).view(np.float32)


def fq_act(v, mode):
    """fake-quant of an activation tensor: bf16-round, Q 1x128, dequantise (fp64)."""
    c, s = quantize_1x128(bf16_round(v), mode)
    return dequantize_1x128(c, s)


def fq_weight(w, mode):
    c, s = quantize_128x128(np.asarray(w, np.float32), mode)
    return dequantize_128x128(c, s)


def expert_ffn_fwd_fp8(Xq, Wg, Wu, Wd, mode):
    """R9 forward of one expert: Xq = dequantised Q-X rows (fp64); weights bf16-grid, fake-quantised 128x128 here;
    a is bf16-rounded and fake-quantised 1x128 before the down projection (Q-a)."""
    Wgq, Wuq, Wdq = fq_weight(Wg, mode), fq_weight(Wu, mode), fq_weight(Wd, mode)
    g = Xq @ Wgq.T
    u = Xq @ Wuq.T
    a = swiglu(g, u)
    y = fq_act(a, mode) @ Wdq.T
    return g, u, a, y


def expert_ffn_bwd_fp8(dYq, wr, dy, Xb, g, u, a, Wg, Wu, Wd, mode):
    """R9 backward of one expert.  dYq = dequantised Q-dY rows of the expert's tokens, wr = their gating weights
    (applied after the GEMM), dy = wr*dY (bf16 tensor of the wgrad), Xb = the bf16 input rows.  dgrad on
    fake-quantised operands (Q-dY, Q-dgu, Q-W); wgrad on the bf16-rounded tensors."""
    Wgq, Wuq, Wdq = fq_weight(Wg, mode), fq_weight(Wu, mode), fq_weight(Wd, mode)
    da = np.asarray(wr, F64)[:, None] * (dYq @ Wdq)
    dg, du = swiglu_bwd(da, g, u)
    dX = fq_act(dg, mode) @ Wgq + fq_act(du, mode) @ Wuq
    dWd = np.asarray(bf16_round(dy), F64).T @ np.asarray(bf16_round(a), F64)
    dWg = np.asarray(bf16_round(dg), F64).T @ Xb
    dWu = np.asarray(bf16_round(du), F64).T @ Xb
    return dX, dWg, dWu, dWd, dg, du


# =====================================================================================
# whole layer, forward and backward (R1..R9)
# =====================================================================================


def _expert_weights(W, e):
    """W is a tuple of stacked arrays (Wg[E,F,H], Wu[E,F,H], Wd[E,H,F]) or a callable e -> triple."""
    if callable(W):
        return W(e)
    return W[0][e], W[1][e], W[2][e]


def zc_kind(cfg, e):
    """V2: the last n_zero + n_copy + n_const router outputs are zero-computation experts, in that order.
    Returns None for an FFN expert, else ("zero" | "copy" | "const", index within its kind)."""
    nz = cfg.n_zero + cfg.n_copy + cfg.n_const
    j = e - (cfg.E - nz)
    if j < 0:
        return None
    if j < cfg.n_zero:
        return "zero", j
    if j < cfg.n_zero + cfg.n_copy:
        return "copy", j - cfg.n_zero
    return "const", j - cfg.n_zero - cfg.n_copy


def layer_fwd(cfg, X, Wr, bias, W, shared=None, forced_idx=None, key_dtype=F64, extras=None):
    """Forward of the routed-expert layer.  Returns a dict with every intermediate in fp64
    (permuted-row tensors use the R6 layout for cfg.row_align).  `extras` (widened rows): threshold [E] (V1),
    zc_const [n_const, H] (V2), f_global [E] (A1).  W holds the E - n_zc FFN experts."""
    extras = extras or {}
    fp8 = cfg.dtype == 2
    mode = cfg.fp8_scale_mode
    z = router_logits(X, Wr)
    idx, w = route(z, bias, cfg, key_dtype, forced_idx, threshold=extras.get("threshold"))
    counts, offsets, p2f, f2p = permute_maps(idx, cfg.E, cfg.row_align)
    Xin = fq_act(X, mode) if fp8 else np.asarray(X, F64)      # Q-X: once per token, then permuted
    Xp = permute_rows(Xin, p2f, cfg.K)
    R = p2f.size
    g = np.zeros((R, cfg.F), F64); u = np.zeros((R, cfg.F), F64)
    a = np.zeros((R, cfg.F), F64); y = np.zeros((R, cfg.H), F64)
    for e in range(cfg.E):
        lo, c = int(offsets[e]), int(counts[e])
        if c == 0:
            continue
        kind = zc_kind(cfg, e)
        if kind is not None:                                   # V2: no FFN; y = 0 | the token's own (bf16) row | the constant vector
            if kind[0] == "copy":
                y[lo:lo + c] = permute_rows(np.asarray(X, F64), p2f, cfg.K)[lo:lo + c]
            elif kind[0] == "const":
                y[lo:lo + c] = np.asarray(extras["zc_const"], F64)[kind[1]][None, :]
            continue
        Wg, Wu, Wd = _expert_weights(W, e)
        if fp8:
            ge, ue, ae, ye = expert_ffn_fwd_fp8(Xp[lo:lo + c], Wg, Wu, Wd, mode)
        else:
            ge, ue, ae, ye = expert_ffn_fwd(Xp[lo:lo + c], Wg, Wu, Wd)
        g[lo:lo + c], u[lo:lo + c], a[lo:lo + c], y[lo:lo + c] = ge, ue, ae, ye
    sh = None
    if shared is not None:
        if fp8:
            sg, su, sa, sy = expert_ffn_fwd_fp8(Xin, *shared, mode)
        else:
            sg, su, sa, sy = expert_ffn_fwd(X, *shared)
        sh = dict(g=sg, u=su, a=sa, y=sy)
    Y = unpermute_combine(y, w, f2p, None if sh is None else sh["y"])
    out = dict(z=z, idx=idx, w=w, counts=counts, offsets=offsets, perm_to_flat=p2f, flat_to_perm=f2p,
               Xp=Xp, g=g, u=u, a=a, y=y, shared=sh, Y=Y)
    if getattr(cfg, "aux_coef", 0.0):
        out["aux_loss"], out["aux_f"], out["aux_P"] = aux_loss(cfg, z, idx, extras.get("f_global"))
    return out


def router_bwd(cfg, z, idx, w, dw, aux_f=None):
    """R8 router part: dz[T,E] (dense, zero outside the selection unless stated) from dw[T,K].
    softmax+renorm: dz_j = w_j (dw_j - sum_i w_i dw_i) over the selected set (w here includes the
    constant routed_scale c, which the closed form carries through unchanged).
    softmax, no renorm: w_j = c*softmax_all(z)_j  =>  dz_e = p_e (c*[e in sel] dw_e - sum_i w_i dw_i)   (dense).
    sigmoid+renorm (S = sum s_i + 1e-20): ds_j = c (dw_j/S - sum_i dw_i s_i / S^2), dz_j = ds_j s_j (1-s_j).
    sigmoid, no renorm: dz_j = c dw_j s_j (1-s_j).  top-k, group mask, bias and thresholds carry no gradient.
    Empty slots (idx = -1, V1) contribute nothing.  aux_f != None adds the dense gradient of the balance loss (A3)."""
    T, E = z.shape
    ok = np.asarray(idx) >= 0
    idx64 = np.where(ok, idx, 0).astype(np.int64)
    dz = np.zeros((T, E), F64)
    c = float(cfg.routed_scale)
    dw = np.where(ok, np.asarray(dw, F64), 0.0)
    w = np.where(ok, np.asarray(w, F64), 0.0)
    rows = np.nonzero(ok)

    def put(vals):
        dz[rows[0], idx64[ok]] += vals[ok]

    if cfg.score_fn == 0 and getattr(cfg, "route_mode", 0) == 0:
        if cfg.renorm:
            put(w * (dw - (w * dw).sum(axis=1, keepdims=True) / c) if c != 0 else np.zeros_like(w))
        else:
            m = z.max(axis=1, keepdims=True)
            p = np.exp(z - m); p /= p.sum(axis=1, keepdims=True)
            dz = -p * (w * dw).sum(axis=1, keepdims=True)        # sum_i c p_i dw_i over selected
            put(w * dw)
    else:
        s = np.where(ok, sigmoid(np.take_along_axis(np.asarray(z, F64), idx64, axis=1)), 0.0)
        if cfg.renorm:
            S = s.sum(axis=1, keepdims=True) + 1e-20
            ds = c * (dw / S - (dw * s).sum(axis=1, keepdims=True) / S ** 2)
        else:
            ds = c * dw
        put(ds * s * (1.0 - s))
    if aux_f is not None and getattr(cfg, "aux_coef", 0.0):
        dz = dz + aux_dz(cfg, z, aux_f)
    return dz


def layer_bwd(cfg, dY, X, Wr, W, fwd, shared=None, extras=None):
    """Backward for L = sum(Y * dY) (+ L_aux when aux_coef != 0).  Returns dX, dWr, per-expert dWg/dWu/dWd
    (stacked over the FFN experts), shared grads, dzc_const (V2) and the intermediates dw, dz, dy, dg, du, dXp."""
    extras = extras or {}
    fp8 = cfg.dtype == 2
    mode = cfg.fp8_scale_mode
    dY = np.asarray(dY, F64); X64 = np.asarray(X, F64)
    T, K, E = cfg.T, cfg.K, cfg.E
    idx, w, f2p, p2f = fwd["idx"], fwd["w"], fwd["flat_to_perm"], fwd["perm_to_flat"]
    offsets, counts = fwd["offsets"], fwd["counts"]
    R = p2f.size
    ok = p2f >= 0
    tok = np.where(ok, p2f // K, 0)
    wr = np.zeros(R, F64)
    wr[ok] = w.reshape(-1)[p2f[ok]]
    # combine-bwd
    dy = np.zeros((R, cfg.H), F64)
    dy[ok] = wr[ok, None] * dY[tok[ok]]
    f2p2 = f2p.reshape(T, K)
    dw = np.stack([np.where(f2p2[:, j] >= 0, (dY * fwd["y"][np.maximum(f2p2[:, j], 0)]).sum(axis=1), 0.0)
                   for j in range(K)], axis=1)                                           # <dY[t], y_r>; empty slot: 0
    dYq = fq_act(dY, mode) if fp8 else None                                    # Q-dY (w applied after the GEMM)
    Xb = np.asarray(X, F64)                                                    # wgrad uses the bf16 tensors
    Xpb = permute_rows(Xb, p2f, K)
    dXp = np.zeros((R, cfg.H), F64)
    dgs = np.zeros((R, cfg.F), F64); dus = np.zeros((R, cfg.F), F64)
    nzc = cfg.n_zero + cfg.n_copy + cfg.n_const
    Ef = E - nzc                                                               # FFN experts (V2: the rest compute nothing)
    dWg = np.zeros((Ef, cfg.F, cfg.H), F64); dWu = np.zeros((Ef, cfg.F, cfg.H), F64)
    dWd = np.zeros((Ef, cfg.H, cfg.F), F64)
    dzc = np.zeros((cfg.n_const, cfg.H), F64)
    for e in range(E):
        lo, c = int(offsets[e]), int(counts[e])
        if c == 0:
            continue                                                           # empty expert: dW == 0 exactly
        sl = slice(lo, lo + c)
        kind = zc_kind(cfg, e)
        if kind is not None:                                                   # y = 0 | x | v  =>  dXp = 0 | dy | 0, dv = sum dy
            if kind[0] == "copy":
                dXp[sl] = dy[sl]
            elif kind[0] == "const":
                dzc[kind[1]] = dy[sl].sum(axis=0)
            continue
        Wg, Wu, Wd = _expert_weights(W, e)
        if fp8:
            dXp[sl], dWg[e], dWu[e], dWd[e], dg, du = expert_ffn_bwd_fp8(
                dYq[tok[sl]], wr[sl], dy[sl], Xpb[sl], fwd["g"][sl], fwd["u"][sl], fwd["a"][sl], Wg, Wu, Wd, mode)
        else:
            dXp[sl], dWg[e], dWu[e], dWd[e], dg, du = expert_ffn_bwd(
                dy[sl], Xpb[sl], fwd["g"][sl], fwd["u"][sl], fwd["a"][sl], Wg, Wu, Wd)
        dgs[sl], dus[sl] = dg, du
    dz = router_bwd(cfg, fwd["z"], idx, w, dw, aux_f=fwd.get("aux_f"))
    dWr = dz.T @ X64
    dX = dz @ np.asarray(Wr, F64)
    for j in range(K):                                                         # fixed j order; empty slots skipped
        okj = f2p2[:, j] >= 0
        dX[okj] = dX[okj] + dXp[f2p2[okj, j]]
    out = dict(dX=dX, dWr=dWr, dWg=dWg, dWu=dWu, dWd=dWd, dw=dw, dz=dz, dy=dy, dg=dgs, du=dus, dXp=dXp, dzc_const=dzc)
    if shared is not None:
        sh = fwd["shared"]
        if fp8:
            dXs, out["dWg_s"], out["dWu_s"], out["dWd_s"], _, _ = expert_ffn_bwd_fp8(
                dYq, np.ones(T, F64), dY, X64, sh["g"], sh["u"], sh["a"], *shared, mode)
        else:
            dXs, out["dWg_s"], out["dWu_s"], out["dWd_s"], _, _ = expert_ffn_bwd(
                dY, X64, sh["g"], sh["u"], sh["a"], *shared)
        out["dX"] = out["dX"] + dXs
    return out


def rel_fro(G, R):
    """S19 error metric: ||G - R||_F / ||R||_F  (||R|| = 0 requires G == 0 -> returns 0 or inf)."""
    G = np.asarray(G, F64); R = np.asarray(R, F64)
    n = np.linalg.norm(R)
    d = np.linalg.norm(G - R)
    if n == 0:
        return 0.0 if d == 0 else np.inf
    return d / n
