"""Seeded synthetic input generators for the five BASELINE.json configs.

This module holds *inputs only* (shapes, seeds, value distributions) and none of
the method's arithmetic: no decoder math, no paging, no sampler, no advantages.
Both the CUDA path (through the binding) and the CPU oracle (through the tests /
bench) consume the arrays produced here; neither side imports the other.

Recipe (shapes from BASELINE.json `configs`):
  weights   bf16(RNE) of 0.02*N(0,1), numpy default_rng(0), one stream in the fixed
            tensor order embed, then per layer wq wk wv wo wg wu wd, then lm_head;
            norm gains are 1.0.
  prompts   uniform ints in [0, V), seed 3000+cfg.
  lengths   seed 1000+cfg (cfg4: [1000+cfg, step]); lognormal / Pareto as listed.
  rewards   seed 2000+cfg, Bernoulli.
  philox    seed 4000+cfg (+step for cfg4).
The synthetic workloads stand in for the paper's public math prompts and
Qwen2.5-3B / Llama-3.2-3B weights: same decoder family shapes, G
completions per prompt, heavy-tailed completion lengths.  Nothing of that
dataset is reproduced here.
"""
from __future__ import annotations

from dataclasses import dataclass, field, asdict
from typing import Dict, Iterator, List, Optional, Tuple

import numpy as np


@dataclass(frozen=True)
class ModelConfig:
    n_layers: int
    d_model: int
    n_q_heads: int
    n_kv_heads: int
    head_dim: int
    d_ff: int
    vocab: int
    rope_theta: float
    rms_eps: float = 1e-6
    page_tokens: int = 64

    @property
    def q_dim(self) -> int:
        return self.n_q_heads * self.head_dim

    @property
    def kv_dim(self) -> int:
        return self.n_kv_heads * self.head_dim

    def kv_bytes_per_token(self) -> int:
        """bf16 K and V over all layers (SURVEY.md section 8 'KVB')."""
        return 2 * self.n_layers * self.kv_dim * 2

    def decode_weight_bytes(self) -> int:
        """bf16 weight bytes streamed once per decode step (SURVEY.md section 8 'W')."""
        d, q, kv, f = self.d_model, self.q_dim, self.kv_dim, self.d_ff
        per_layer = d * q + 2 * d * kv + q * d + 3 * d * f
        return 2 * (self.n_layers * per_layer + self.vocab * d)

    def n_params(self) -> int:
        return self.decode_weight_bytes() // 2 + self.vocab * self.d_model


@dataclass(frozen=True)
class Workload:
    cfg: int
    model: ModelConfig
    n_prompts: int
    prompt_len: int
    G: int
    max_new: int
    length_kind: str          # "lognormal" | "pareto"
    length_scale: float       # median (lognormal) or x_min (pareto)
    length_shape: float       # sigma (lognormal) or alpha (pareto)
    sampling: str             # "greedy" | "gumbel"
    temperature: float
    reward_p: Optional[float]  # None => p_prompt ~ U(0,1) per prompt
    adv_mode: str             # "GRPO" | "DAPO"
    g_choices: Tuple[int, ...] = ()
    n_rollout_steps: int = 1

    @property
    def philox_seed(self) -> int:
        return 4000 + self.cfg


WORKLOADS: Dict[int, Workload] = {
    1: Workload(1, ModelConfig(2, 128, 4, 4, 32, 512, 1024, 1e4, 1e-6, 16),
                1, 32, 4, 128, "lognormal", 48.0, 0.5, "greedy", 1.0, 0.5, "GRPO"),
    2: Workload(2, ModelConfig(24, 896, 14, 2, 64, 4864, 151936, 1e6, 1e-6, 64),
                8, 256, 8, 4096, "lognormal", 1024.0, 0.8, "gumbel", 1.0, 0.4, "GRPO"),
    3: Workload(3, ModelConfig(28, 1536, 12, 2, 128, 8960, 151936, 1e6, 1e-6, 64),
                16, 512, 16, 8192, "lognormal", 2048.0, 1.0, "gumbel", 1.0, None, "DAPO"),
    4: Workload(4, ModelConfig(28, 3584, 28, 4, 128, 18944, 152064, 1e6, 1e-6, 64),
                16, 512, 32, 8192, "lognormal", 2048.0, 1.0, "gumbel", 1.0, 0.5, "GRPO",
                g_choices=(4, 8, 16, 32), n_rollout_steps=10),
    5: Workload(5, ModelConfig(28, 3584, 28, 4, 128, 18944, 152064, 1e6, 1e-6, 64),
                8, 1024, 32, 16384, "pareto", 512.0, 1.5, "gumbel", 1.0, 0.5, "DAPO"),
}


# ---------------------------------------------------------------------------
# bf16 bit helpers (input encoding only)
# ---------------------------------------------------------------------------
def f32_to_bf16_bits(x: np.ndarray) -> np.ndarray:
    """float32 -> bf16 bit pattern (uint16), round to nearest even."""
    u = np.ascontiguousarray(x, dtype=np.float32).view(np.uint32)
    r = (u + np.uint32(0x7FFF) + ((u >> np.uint32(16)) & np.uint32(1))) >> np.uint32(16)
    return r.astype(np.uint16)


def bf16_bits_to_f32(b: np.ndarray) -> np.ndarray:
    return (np.ascontiguousarray(b, dtype=np.uint16).astype(np.uint32) << np.uint32(16)).view(np.float32)


WEIGHT_ORDER = ("wq", "wk", "wv", "wo", "wg", "wu", "wd")


def weight_shapes(m: ModelConfig) -> Dict[str, Tuple[int, int]]:
    """[out][in] row-major shapes of every weight matrix."""
    return {
        "embed": (m.vocab, m.d_model),
        "wq": (m.q_dim, m.d_model), "wk": (m.kv_dim, m.d_model), "wv": (m.kv_dim, m.d_model),
        "wo": (m.d_model, m.q_dim),
        "wg": (m.d_ff, m.d_model), "wu": (m.d_ff, m.d_model), "wd": (m.d_model, m.d_ff),
        "lm_head": (m.vocab, m.d_model),
    }


def iter_weights(m: ModelConfig, seed: int = 0, chunk_rows: int = 1 << 14
                 ) -> Iterator[Tuple[str, int, np.ndarray]]:
    """Yield (name, layer or -1, bf16 bits [out][in]) in the fixed stream order."""
    rng = np.random.default_rng(seed)
    shapes = weight_shapes(m)

    def draw(shape):
        out = np.empty(shape, dtype=np.uint16)
        for r0 in range(0, shape[0], chunk_rows):
            r1 = min(shape[0], r0 + chunk_rows)
            z = rng.standard_normal((r1 - r0, shape[1]), dtype=np.float32)
            z *= np.float32(0.02)
            out[r0:r1] = f32_to_bf16_bits(z)
        return out

    yield "embed", -1, draw(shapes["embed"])
    for l in range(m.n_layers):
        for name in WEIGHT_ORDER:
            yield name, l, draw(shapes[name])
    yield "lm_head", -1, draw(shapes["lm_head"])


def make_weights(m: ModelConfig, seed: int = 0) -> Dict[str, object]:
    """All weights in memory: {'embed','lm_head': u16[...], 'wq'..'wd': [per-layer u16],
    'norm1','norm2': [per-layer u16 ones], 'final_norm': u16 ones}."""
    w: Dict[str, object] = {name: [None] * m.n_layers for name in WEIGHT_ORDER}
    for name, l, arr in iter_weights(m, seed):
        if l < 0:
            w[name] = arr
        else:
            w[name][l] = arr
    one = f32_to_bf16_bits(np.ones(m.d_model, dtype=np.float32))
    w["norm1"] = [one.copy() for _ in range(m.n_layers)]
    w["norm2"] = [one.copy() for _ in range(m.n_layers)]
    w["final_norm"] = one.copy()
    return w


def make_prompts(wl: Workload, n_prompts: Optional[int] = None, prompt_len: Optional[int] = None
                 ) -> Tuple[np.ndarray, np.ndarray]:
    """(concatenated tokens int32, offsets int32 [n_prompts+1])."""
    n = wl.n_prompts if n_prompts is None else n_prompts
    P = wl.prompt_len if prompt_len is None else prompt_len
    rng = np.random.default_rng(3000 + wl.cfg)
    toks = rng.integers(0, wl.model.vocab, size=n * P, dtype=np.int64).astype(np.int32)
    offs = (np.arange(n + 1, dtype=np.int64) * P).astype(np.int32)
    return toks, offs


def make_forced_lengths(wl: Workload, G: Optional[int] = None, step: int = 0,
                        n_prompts: Optional[int] = None) -> np.ndarray:
    """Forced completion lengths int32 [n_prompts*G], prompt-major (sid = p*G+g)."""
    G = wl.G if G is None else G
    n = (wl.n_prompts if n_prompts is None else n_prompts) * G
    seed = [1000 + wl.cfg, step] if wl.n_rollout_steps > 1 else 1000 + wl.cfg
    rng = np.random.default_rng(seed)
    if wl.length_kind == "lognormal":
        z = rng.standard_normal(n)
        ell = np.rint(wl.length_scale * np.exp(wl.length_shape * z))
    elif wl.length_kind == "pareto":
        u = 1.0 - rng.random(n)            # (0, 1]
        ell = np.floor(wl.length_scale * u ** (-1.0 / wl.length_shape))
    else:
        raise ValueError(wl.length_kind)
    return np.clip(ell, 1, wl.max_new).astype(np.int32)


def make_rewards(wl: Workload, G: Optional[int] = None, step: int = 0,
                 n_prompts: Optional[int] = None) -> Tuple[np.ndarray, np.ndarray]:
    """(rewards float32 [n_prompts*G] in {0,1}, CSR offsets int32 [n_prompts+1])."""
    G = wl.G if G is None else G
    npmt = wl.n_prompts if n_prompts is None else n_prompts
    seed = [2000 + wl.cfg, step] if wl.n_rollout_steps > 1 else 2000 + wl.cfg
    rng = np.random.default_rng(seed)
    if wl.reward_p is None:
        p = np.repeat(rng.random(npmt), G)
    else:
        p = np.full(npmt * G, wl.reward_p)
    r = (rng.random(npmt * G) < p).astype(np.float32)
    offs = (np.arange(npmt + 1, dtype=np.int64) * G).astype(np.int32)
    return r, offs


def g_schedule(wl: Workload) -> List[int]:
    """cfg4: seeded neighbour-move random walk over g_choices (stand-in for the SAGC
    controller's trajectory, Alg.1 l.16-17: only neighbour moves)."""
    if not wl.g_choices:
        return [wl.G] * wl.n_rollout_steps
    rng = np.random.default_rng(5000 + wl.cfg)
    idx = int(rng.integers(0, len(wl.g_choices)))
    out = []
    for _ in range(wl.n_rollout_steps):
        out.append(wl.g_choices[idx])
        idx = int(np.clip(idx + int(rng.integers(-1, 2)), 0, len(wl.g_choices) - 1))
    return out


def tiny_variant(cfg: int = 1, **overrides) -> Workload:
    """A Workload with fields overridden (used by tests for ragged / GQA cases)."""
    base = asdict(WORKLOADS[cfg])
    model = base.pop("model")
    mo = {k[len("model_"):]: v for k, v in overrides.items() if k.startswith("model_")}
    model.update(mo)
    base.update({k: v for k, v in overrides.items() if not k.startswith("model_")})
    base["g_choices"] = tuple(base["g_choices"])
    return Workload(model=ModelConfig(**model), **base)
