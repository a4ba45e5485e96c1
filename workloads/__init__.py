"""Seeded synthetic MoE-layer workloads (BASELINE.json:configs).

This module serves BOTH the fp64 oracle (tests, cpu_baseline) and the CUDA path (tests, bench).
It holds only configuration records, a counter-based random number source and dtype
representation helpers (fp32 <-> bf16 bit patterns).  It contains none of the method's
arithmetic (no routing, no GEMM, no quantiser) and imports neither `oracle/` nor the CUDA package.

Recipe: one Philox4x64 stream per (seed, tensor id, expert id); values are
drawn in fp32 as N(0, std) and rounded ONCE to the config's storage dtype (bf16 for every config
except the tiny fp32 one), so both sides read identical bits.
"""
from __future__ import annotations

import dataclasses
import math
from concurrent.futures import ThreadPoolExecutor

import numpy as np

# --------------------------------------------------------------------------------------
# configuration record (mirrors moe_config_t in include/moe_b200.h field by field)
# --------------------------------------------------------------------------------------

SCORE_SOFTMAX, SCORE_SIGMOID = 0, 1
GROUP_SCORE_MAX, GROUP_SCORE_TOP2SUM = 0, 1
DTYPE_FP32, DTYPE_BF16, DTYPE_FP8 = 0, 1, 2


@dataclasses.dataclass(frozen=True)
class MoEConfig:
    name: str
    T: int
    H: int
    E: int
    K: int
    F: int
    n_group: int = 1
    topk_group: int = 1
    score_fn: int = SCORE_SOFTMAX
    group_score: int = GROUP_SCORE_TOP2SUM
    renorm: int = 1
    routed_scale: float = 1.0
    has_bias: int = 0
    F_shared: int = 0
    dtype: int = DTYPE_BF16
    fp8_scale_mode: int = 0
    row_align: int = 1
    # widened rows; all off by default
    route_mode: int = 0            # 0 = top-k (R2..R5), 1 = threshold-gated variable-k on sigmoid gates
    n_zero: int = 0                # zero-computation experts: the LAST n_zero + n_copy + n_const of the E
    n_copy: int = 0                #   router outputs, in this order; weights are held for the first E - n_zc experts
    n_const: int = 0
    aux_coef: float = 0.0          # auxiliary load-balancing loss coefficient; 0 = off
    aux_zc_weight: float = 1.0     # weight of the zero-computation experts in the balance term
    # kernel-variant selectors of moe_config_t (0 = the library default; v > 0 forces level v - 1; include/moe_b200.h)
    opt_rows_fused: int = 0
    opt_pair: int = 0
    opt_fp8_wide: int = 0
    opt_fp8_fused_quant: int = 0
    # input recipe only (not part of moe_config_t)
    w_std: float = 0.02            # expert weight std; <0 means 1/sqrt(fan_in) (configs[0])
    bias_kind: str = "none"        # "none" | "normal" (b~N(0,0.05)) | "zipf" (configs[4] skew offset)
    seed: int = 0

    def replace(self, **kw) -> "MoEConfig":
        return dataclasses.replace(self, **kw)

    @property
    def TK(self) -> int:
        return self.T * self.K

    @property
    def E_ffn(self) -> int:
        """Experts that own FFN weights (all of them unless zero-computation experts are configured)."""
        return self.E - self.n_zero - self.n_copy - self.n_const

    @property
    def TK_pad(self) -> int:
        """Upper bound on permuted rows when every expert group is rounded up to row_align."""
        a = self.row_align
        if a <= 1:
            return self.TK
        return ((self.TK + self.E * (a - 1)) + a - 1) // a * a

    def flops_fwd_bwd(self) -> dict:
        """Algorithmic flop counts."""
        routed = 18 * self.T * self.K * self.H * self.F
        shared = 18 * self.T * self.H * self.F_shared
        router = 6 * self.T * self.H * self.E
        return {"routed": routed, "shared": shared, "router": router, "total": routed + shared + router}


# BASELINE.json:configs[0..4]  (SURVEY.md numbers them 1..5)
TINY = MoEConfig("tiny_fp32", T=256, H=128, E=8, K=2, F=256, dtype=DTYPE_FP32, w_std=-1.0)
QWEN3 = MoEConfig("qwen3_30b_a3b_like", T=8192, H=2048, E=128, K=8, F=768)
DSV3 = MoEConfig("deepseek_v3_like", T=4096, H=7168, E=256, K=8, F=2048, n_group=8, topk_group=4,
                 score_fn=SCORE_SIGMOID, routed_scale=2.5, has_bias=1, F_shared=2048, bias_kind="normal")
DSV3_FP8 = DSV3.replace(name="deepseek_v3_like_fp8", dtype=DTYPE_FP8)
GPTOSS = MoEConfig("gpt_oss_like_skew", T=16384, H=2880, E=128, K=4, F=2880, has_bias=1, bias_kind="zipf")

CONFIGS = {c.name: c for c in (TINY, QWEN3, DSV3, DSV3_FP8, GPTOSS)}

# Scaled-down cases with the same structure, sized so the fp64 oracle finishes in seconds while the
# CUDA path still spans several 128-row tiles, ragged tails, partial N tiles and empty experts.
QWEN3_SMALL = QWEN3.replace(name="qwen3_small", T=1000, H=512, E=16, K=4, F=384)
DSV3_SMALL = DSV3.replace(name="dsv3_small", T=600, H=512, E=32, K=4, F=256, n_group=4, topk_group=2,
                          F_shared=384)
DSV3_FP8_SMALL = DSV3_SMALL.replace(name="dsv3_fp8_small", dtype=DTYPE_FP8)
GPTOSS_SMALL = GPTOSS.replace(name="gptoss_small", T=1500, H=320, E=32, K=4, F=320)
SMALL_CONFIGS = {c.name: c for c in (QWEN3_SMALL, DSV3_SMALL, DSV3_FP8_SMALL, GPTOSS_SMALL)}

# --------------------------------------------------------------------------------------
# dtype representation helpers (no method arithmetic)
# --------------------------------------------------------------------------------------


def f32_to_bf16_bits(x: np.ndarray) -> np.ndarray:
    """Round-to-nearest-even fp32 -> bf16, returned as uint16 bit patterns (finite inputs)."""
    u = np.ascontiguousarray(x, dtype=np.float32).view(np.uint32)
    r = ((u >> np.uint32(16)) & np.uint32(1)) + np.uint32(0x7FFF)
    return ((u + r) >> np.uint32(16)).astype(np.uint16)


def bf16_bits_to_f32(b: np.ndarray) -> np.ndarray:
    return (np.ascontiguousarray(b, dtype=np.uint16).astype(np.uint32) << np.uint32(16)).view(np.float32)


def round_to_storage(x: np.ndarray, dtype: int) -> np.ndarray:
    """fp32 array holding values exactly representable in the config's storage dtype."""
    if dtype == DTYPE_FP32:
        return np.ascontiguousarray(x, dtype=np.float32)
    return bf16_bits_to_f32(f32_to_bf16_bits(x))


# --------------------------------------------------------------------------------------
# counter-based random source
# --------------------------------------------------------------------------------------

# fixed tensor ids: one independent Philox stream per (seed, tensor id, expert id)
TENSOR_IDS = {"X": 1, "Wr": 2, "bias": 3, "Wg": 4, "Wu": 5, "Wd": 6, "Wg_s": 7, "Wu_s": 8, "Wd_s": 9,
              "dY": 10, "perm": 11, "logits": 12, "aux": 13}


def _rng(seed: int, tensor: str, sub: int = 0) -> np.random.Generator:
    return np.random.Generator(np.random.Philox(key=[int(seed), TENSOR_IDS[tensor] * (1 << 32) + int(sub)]))


def normal(seed: int, tensor: str, shape, std: float, dtype: int, sub: int = 0) -> np.ndarray:
    g = _rng(seed, tensor, sub)
    x = g.standard_normal(shape, dtype=np.float32)
    x *= np.float32(std)
    return round_to_storage(x, dtype)


def _act_dtype(cfg: MoEConfig) -> int:
    return DTYPE_FP32 if cfg.dtype == DTYPE_FP32 else DTYPE_BF16


def _w_std(cfg: MoEConfig, fan_in: int) -> float:
    return cfg.w_std if cfg.w_std > 0 else 1.0 / math.sqrt(fan_in)


def gen_X(cfg: MoEConfig) -> np.ndarray:
    return normal(cfg.seed, "X", (cfg.T, cfg.H), 1.0, _act_dtype(cfg))


def gen_dY(cfg: MoEConfig) -> np.ndarray:
    return normal(cfg.seed, "dY", (cfg.T, cfg.H), 1.0, _act_dtype(cfg))


def gen_Wr(cfg: MoEConfig) -> np.ndarray:
    return normal(cfg.seed, "Wr", (cfg.E, cfg.H), 0.02, _act_dtype(cfg))


def zipf_offsets(cfg: MoEConfig) -> np.ndarray:
    """configs[4] skew: rank rho(e) from a seeded permutation of experts;
    o = 0.5*ln(rho^-1.2) for the first 15/16 of the ranks, -30 for the rest (those experts get no tokens)."""
    rho = _rng(cfg.seed, "perm").permutation(cfg.E) + 1          # ranks 1..E
    live = (cfg.E * 15) // 16                                    # 120 of 128
    o = np.where(rho <= live, 0.5 * np.log(rho.astype(np.float64) ** -1.2), -30.0)
    return o.astype(np.float32)


def gen_bias(cfg: MoEConfig):
    """Selection-only per-expert bias b[E] (fp32), or None."""
    if not cfg.has_bias:
        return None
    if cfg.bias_kind == "zipf":
        return zipf_offsets(cfg)
    return normal(cfg.seed, "bias", (cfg.E,), 0.05, DTYPE_FP32)


def gen_expert_weights(cfg: MoEConfig, e: int):
    """(Wg[F,H], Wu[F,H], Wd[H,F]) of routed expert e; logical layout [out, in]."""
    dt = _act_dtype(cfg)
    Wg = normal(cfg.seed, "Wg", (cfg.F, cfg.H), _w_std(cfg, cfg.H), dt, e)
    Wu = normal(cfg.seed, "Wu", (cfg.F, cfg.H), _w_std(cfg, cfg.H), dt, e)
    Wd = normal(cfg.seed, "Wd", (cfg.H, cfg.F), _w_std(cfg, cfg.F), dt, e)
    return Wg, Wu, Wd


def gen_shared_weights(cfg: MoEConfig):
    if cfg.F_shared == 0:
        return None
    dt = _act_dtype(cfg)
    Fs = cfg.F_shared
    return (normal(cfg.seed, "Wg_s", (Fs, cfg.H), _w_std(cfg, cfg.H), dt),
            normal(cfg.seed, "Wu_s", (Fs, cfg.H), _w_std(cfg, cfg.H), dt),
            normal(cfg.seed, "Wd_s", (cfg.H, Fs), _w_std(cfg, Fs), dt))


def gen_all_expert_weights(cfg: MoEConfig, threads: int = 8):
    """Stacked (Wg[E,F,H], Wu[E,F,H], Wd[E,H,F]) fp32 arrays; experts generated in parallel
    (each from its own stream, so the result does not depend on the thread count)."""
    Wg = np.empty((cfg.E_ffn, cfg.F, cfg.H), np.float32)
    Wu = np.empty((cfg.E_ffn, cfg.F, cfg.H), np.float32)
    Wd = np.empty((cfg.E_ffn, cfg.H, cfg.F), np.float32)

    def one(e):
        Wg[e], Wu[e], Wd[e] = gen_expert_weights(cfg, e)

    with ThreadPoolExecutor(max_workers=threads) as ex:
        list(ex.map(one, range(cfg.E_ffn)))
    return Wg, Wu, Wd


def gen_threshold(cfg: MoEConfig) -> np.ndarray:
    """Per-expert gate thresholds of the variable-k router (route_mode 1), fp32 in (0, 1): N(0.62, 0.03) so that with
    logits of std 0.91 a token activates a handful of experts, some tokens none (top-1 fallback) and some more than K."""
    t = 0.62 + normal(cfg.seed, "aux", (cfg.E,), 0.03, DTYPE_FP32, 1)
    return np.clip(t, 0.05, 0.95).astype(np.float32)


def gen_zc_const(cfg: MoEConfig):
    """Constant experts' vectors [n_const, H] (activation dtype grid), or None."""
    if cfg.n_const == 0:
        return None
    return normal(cfg.seed, "aux", (cfg.n_const, cfg.H), 1.0, _act_dtype(cfg), 2)


def gen_logits(cfg: MoEConfig, std: float = 0.91, ties: int = 0) -> np.ndarray:
    """Stand-alone fp32 router logits for moe_route tests (std 0.91 = what X·Wr^T gives on
    configs[1]).  `ties` > 0 plants that many exact duplicates per row."""
    z = normal(cfg.seed, "logits", (cfg.T, cfg.E), std, DTYPE_FP32)
    if ties:
        g = _rng(cfg.seed, "aux")
        for _ in range(ties):
            src = g.integers(0, cfg.E, cfg.T)
            dst = g.integers(0, cfg.E, cfg.T)
            z[np.arange(cfg.T), dst] = z[np.arange(cfg.T), src]
    return z
