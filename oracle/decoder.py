"""ORACLE (test infrastructure, never on the product path) -- float32 reference decoder.

Plain, slow CPU statement of the policy forward pass that "synchronous group rollout
generation" (sec 3.1, Alg.1 l.7) runs once per generated token.
The paper names the model family only (Qwen2.5-3B-Instruct / Llama-3.2-3B-Instruct,
PAPER.md l.167) and is otherwise silent on the decoder; BASELINE.json north_star fixes
"a float32 reference decoder" with "RMSNorm, RoPE theta, SwiGLU FFN, q/kv heads, bf16
weights".  Readings (C1):

  per token at position p, x = E[token]; for each layer
     h  = x * rsqrt(mean(x^2) + eps) * w1                       (pre-norm, eps inside sqrt)
     q  = Wq h, k = Wk h, v = Wv h          (y = W x, W row-major [out][in], no biases)
     RoPE rotate-half on every q and k head: pairs (i, i+hd/2), theta_i = base^(-2i/hd),
          (a, b) -> (a cos - b sin, b cos + a sin), angle p*theta_i and cos/sin in float64
     k, v rounded to bf16 (RNE) when stored  -- the ONLY rounding point
     q-head j uses kv-head j // (Hq/Hkv);  s_i = q.k_i / sqrt(hd), i <= p
     a = softmax(s) (max-subtracted);  o = sum a_i v_i;  x += Wo o
     h2 = rmsnorm(x; w2);  x += Wd( silu(Wg h2) * (Wu h2) ),  silu(z) = z / (1 + exp(-z))
  logits = Wlm rmsnorm(x; wf)

Arithmetic is float32 (weights are bf16 values widened exactly); matmuls are numpy
float32 library calls (a library primitive used as one step), no blocking or fusion.
`kv_round=False` gives the pure-fp32 model used by the transformers pin.

Pins (tests/test_oracle_decoder.py): brute-force no-cache recompute == cached decode;
position-0 RoPE identity; single-entry context o = v; L=0 closed form; RoPE
relative-position invariance; GQA == MHA with repeated KV weights; a transformers
LlamaForCausalLM (independent library implementation) on the same weights.
RoPE pairing, eps and norm placement are not fixed by the paper ("parity unpinned by the
paper"); they are pinned to the library model the paper names (Llama/Qwen family).
"""
from __future__ import annotations

from typing import Dict, List, Optional, Sequence

import numpy as np


def _bf16_bits_to_f32(b: np.ndarray) -> np.ndarray:
    return (np.ascontiguousarray(b, dtype=np.uint16).astype(np.uint32) << np.uint32(16)).view(np.float32)


def round_to_bf16(x: np.ndarray) -> np.ndarray:
    """float32 -> nearest bf16 value (ties to even), returned as float32."""
    u = np.ascontiguousarray(x, dtype=np.float32).view(np.uint32)
    r = (u + np.uint32(0x7FFF) + ((u >> np.uint32(16)) & np.uint32(1))) & np.uint32(0xFFFF0000)
    return r.view(np.float32)


def rmsnorm(x: np.ndarray, w: np.ndarray, eps: float) -> np.ndarray:
    x = x.astype(np.float32)
    ms = np.mean(x * x, axis=-1, keepdims=True, dtype=np.float32)
    return (x * (np.float32(1.0) / np.sqrt(ms + np.float32(eps)))).astype(np.float32) * w


def silu(z: np.ndarray) -> np.ndarray:
    z = z.astype(np.float32)
    return (z / (np.float32(1.0) + np.exp(-z))).astype(np.float32)


def rope_tables(positions: np.ndarray, head_dim: int, theta: float):
    """cos/sin [n][hd/2] float32; angles evaluated in float64."""
    half = head_dim // 2
    inv = np.float64(theta) ** (-(2.0 * np.arange(half, dtype=np.float64)) / head_dim)
    ang = np.asarray(positions, dtype=np.float64)[:, None] * inv[None, :]
    return np.cos(ang).astype(np.float32), np.sin(ang).astype(np.float32)


def apply_rope(x: np.ndarray, cos: np.ndarray, sin: np.ndarray) -> np.ndarray:
    """x [n][H][hd] float32, cos/sin [n][hd/2]."""
    half = x.shape[-1] // 2
    a, b = x[..., :half], x[..., half:]
    c, s = cos[:, None, :], sin[:, None, :]
    return np.concatenate([a * c - b * s, b * c + a * s], axis=-1).astype(np.float32)


class RefDecoder:
    """cfg needs: n_layers d_model n_q_heads n_kv_heads head_dim d_ff vocab rope_theta rms_eps.
    weights: dict of bf16 bit patterns (uint16), layout [out][in]:
      embed, lm_head, final_norm, and per-layer lists wq wk wv wo wg wu wd norm1 norm2."""

    def __init__(self, cfg, weights: Dict[str, object], kv_round: bool = True,
                 cache_f32: bool = True):
        self.cfg = cfg
        self.w = weights
        self.kv_round = kv_round
        self._cache: Dict = {} if cache_f32 else None

    # -- weights ----------------------------------------------------------------
    def W(self, name: str, layer: int = -1) -> np.ndarray:
        key = (name, layer)
        if self._cache is not None and key in self._cache:
            return self._cache[key]
        raw = self.w[name] if layer < 0 else self.w[name][layer]
        f = _bf16_bits_to_f32(raw)
        if self._cache is not None:
            self._cache[key] = f
        return f

    # -- one layer over n rows with explicit K/V context ------------------------------
    def _qkv(self, l: int, x: np.ndarray, positions: np.ndarray):
        c = self.cfg
        n = x.shape[0]
        h = rmsnorm(x, self.W("norm1", l), c.rms_eps)
        q = (h @ self.W("wq", l).T).reshape(n, c.n_q_heads, c.head_dim)
        k = (h @ self.W("wk", l).T).reshape(n, c.n_kv_heads, c.head_dim)
        v = (h @ self.W("wv", l).T).reshape(n, c.n_kv_heads, c.head_dim)
        cos, sin = rope_tables(positions, c.head_dim, c.rope_theta)
        q = apply_rope(q, cos, sin)
        k = apply_rope(k, cos, sin)
        if self.kv_round:
            k = round_to_bf16(k)
            v = round_to_bf16(v)
        return q, k, v

    def _attend(self, q: np.ndarray, K: np.ndarray, V: np.ndarray) -> np.ndarray:
        """q [Hq][hd]; K, V [ctx][Hkv][hd] -> o [Hq*hd]."""
        c = self.cfg
        r = c.n_q_heads // c.n_kv_heads
        o = np.empty((c.n_q_heads, c.head_dim), dtype=np.float32)
        scale = np.float32(1.0 / np.sqrt(np.float64(c.head_dim)))
        for j in range(c.n_q_heads):
            kj = K[:, j // r, :]
            s = (kj @ q[j]) * scale
            s = s - np.max(s)
            e = np.exp(s).astype(np.float32)
            a = e / np.sum(e, dtype=np.float32)
            o[j] = a @ V[:, j // r, :]
        return o.reshape(-1)

    def _mlp_residual(self, l: int, x: np.ndarray, o: np.ndarray) -> np.ndarray:
        c = self.cfg
        x = x + o @ self.W("wo", l).T
        h2 = rmsnorm(x, self.W("norm2", l), c.rms_eps)
        a = silu(h2 @ self.W("wg", l).T) * (h2 @ self.W("wu", l).T)
        return (x + a @ self.W("wd", l).T).astype(np.float32)

    def logits_from_hidden(self, x: np.ndarray) -> np.ndarray:
        hf = rmsnorm(x, self.W("final_norm"), self.cfg.rms_eps)
        return (hf @ self.W("lm_head").T).astype(np.float32)

    # -- full-sequence causal pass (no KV cache; the brute-force definition) --------------
    def forward_full(self, tokens: Sequence[int], logits_at: Optional[Sequence[int]] = None,
                     pos0: int = 0, return_kv: bool = False):
        """All positions at once with a causal mask.  Returns logits [len(logits_at)][V]
        (default: every position).  K and V are rounded before use exactly as the cached
        path stores them."""
        c = self.cfg
        toks = np.asarray(tokens, dtype=np.int64)
        T = toks.shape[0]
        pos = np.arange(pos0, pos0 + T)
        x = self.W("embed")[toks].astype(np.float32)
        kvs = []
        for l in range(c.n_layers):
            q, k, v = self._qkv(l, x, pos)
            o = np.empty((T, c.n_q_heads * c.head_dim), dtype=np.float32)
            for i in range(T):
                o[i] = self._attend(q[i], k[: i + 1], v[: i + 1])
            x = self._mlp_residual(l, x, o)
            if return_kv:
                kvs.append((k, v))
        idx = np.arange(T) if logits_at is None else np.asarray(logits_at, dtype=np.int64)
        lg = self.logits_from_hidden(x[idx])
        return (lg, kvs) if return_kv else lg

    # -- cached decode ------------------------------------------------------------
    def new_cache(self) -> List[List[np.ndarray]]:
        """Per layer: [K list, V list]; entries are [Hkv][hd] float32 (bf16-valued)."""
        return [[[], []] for _ in range(self.cfg.n_layers)]

    def fork_cache(self, cache):
        return [[list(K), list(V)] for K, V in cache]

    def step(self, token: int, position: int, cache) -> np.ndarray:
        """Consume one token at `position`, append its K,V to `cache`, return logits [V]."""
        c = self.cfg
        x = self.W("embed")[int(token)][None, :].astype(np.float32)
        pos = np.asarray([position])
        for l in range(c.n_layers):
            q, k, v = self._qkv(l, x, pos)
            cache[l][0].append(k[0])
            cache[l][1].append(v[0])
            K = np.stack(cache[l][0])
            V = np.stack(cache[l][1])
            o = self._attend(q[0], K, V)[None, :]
            x = self._mlp_residual(l, x, o)
        return self.logits_from_hidden(x)[0]

    def prefill(self, tokens: Sequence[int]):
        """Prompt pass: returns (last-row logits [V], cache holding the prompt's K,V)."""
        lg, kvs = self.forward_full(tokens, logits_at=[len(tokens) - 1], return_kv=True)
        cache = [[list(k), list(v)] for k, v in kvs]
        return lg[0], cache
