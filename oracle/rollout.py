"""ORACLE (test infrastructure, never on the product path) -- synchronous group rollout.

Sequential statement of what `sagc_rollout_group` computes (sec 3.1:
"generate G completions {y_i}"; l.76: l_i = "generated token length ... under a fixed
maximum L_max"; Alg.1 l.7 "Run rollout generation with group size G"; l.153: "the GPU
computes per-sequence token counts l_i. For each group we compute summary statistics
l_max, l_median").  Composition of oracle.decoder (forward pass), oracle.philox (sampler),
oracle.paging (page bookkeeping) and oracle.groupstats (length summaries).

Position / step numbering (reading C1): prompt tokens at 0..P-1; generated
token j (1-based) sits at position P+j-1; token 1 is sampled from the prefill's last-row
logits (the G completions draw G Gumbel vectors keyed by sid, so greedy completions of a
prompt are identical while they last); decode step t >= 2 consumes token t-1 at position
P+t-2 and samples token t.  A sequence retires at the end of step t when
l == forced length, or token == stop_token, or l == max_new; the stop token is counted.
The KV of a sequence's final token is never computed.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import List, Optional, Sequence

import numpy as np

from . import groupstats, paging, philox
from .decoder import RefDecoder


@dataclass
class RolloutResult:
    tokens: np.ndarray            # int32 [nseq][max_new], pad -1
    lengths: np.ndarray           # int32 [nseq]
    len_stats: np.ndarray         # int32 [n_prompts][3] = max, sum, median_x2
    ratio_max_mean: np.ndarray    # float32 [n_prompts]
    paging: Optional[paging.PagedKVState] = None
    logits: dict = field(default_factory=dict)     # (sid, t) -> float32 [V] when requested


def rollout_group(dec: RefDecoder, prompt_tokens: Sequence[int], prompt_offsets: Sequence[int],
                  G: int, mode: int, temperature: float, seed: int, max_new: int,
                  forced_lengths: Optional[Sequence[int]] = None, stop_token: int = -1,
                  n_pages: Optional[int] = None, page_tokens: int = 16,
                  keep_logits: bool = False, forced_tokens: Optional[np.ndarray] = None
                  ) -> RolloutResult:
    """Free-running (or, with `forced_tokens` [nseq][max_new], teacher-forced) rollout."""
    offs = [int(o) for o in prompt_offsets]
    n_prompts = len(offs) - 1
    nseq = n_prompts * G
    prompt_lens = [offs[p + 1] - offs[p] for p in range(n_prompts)]
    toks = -np.ones((nseq, max_new), dtype=np.int32)
    ell = np.zeros(nseq, dtype=np.int32)
    res_logits = {}

    st = None
    if n_pages is not None:
        max_blocks = (max(prompt_lens) + max_new + page_tokens - 1) // page_tokens
        st = paging.PagedKVState(n_pages, page_tokens, prompt_lens, G, max_blocks)
        st.prefill()

    def pick(lg, sid, t):
        if keep_logits:
            res_logits[(sid, t)] = lg.copy()
        if forced_tokens is not None:
            return int(forced_tokens[sid, t - 1])
        return philox.sample_token(lg, mode, temperature, seed, sid, t)

    def done(sid, t, tok):
        if forced_lengths is not None and int(forced_lengths[sid]) == t:
            return True
        return (stop_token >= 0 and tok == stop_token) or t == max_new

    # prefill once per prompt; the G completions fork the prompt's cache
    caches = [None] * nseq
    live: List[int] = []
    fin = []
    for p in range(n_prompts):
        lg, cache = dec.prefill(prompt_tokens[offs[p]:offs[p + 1]])
        for g in range(G):
            sid = p * G + g
            caches[sid] = dec.fork_cache(cache)
            tok = pick(lg, sid, 1)
            toks[sid, 0] = tok
            ell[sid] = 1
            live.append(sid)
            fin.append(done(sid, 1, tok))
    if st is not None:
        st.end_step(1, fin)
    live = [s for s, f in zip(live, fin) if not f]

    t = 2
    while live:
        if st is not None:
            st.begin_step(t)
        fin = []
        for sid in live:
            P = prompt_lens[sid // G]
            lg = dec.step(int(toks[sid, t - 2]), P + t - 2, caches[sid])
            tok = pick(lg, sid, t)
            toks[sid, t - 1] = tok
            ell[sid] = t
            fin.append(done(sid, t, tok))
        if st is not None:
            st.end_step(t, fin)
        for sid, f in zip(live, fin):
            if f:
                caches[sid] = None
        live = [s for s, f in zip(live, fin) if not f]
        t += 1

    goffs = np.arange(n_prompts + 1, dtype=np.int64) * G
    stats, ratio = groupstats.length_stats(ell, goffs)
    return RolloutResult(toks, ell, stats, ratio, st, res_logits)


def teacher_forced_logits(dec: RefDecoder, prompt: Sequence[int], gen_tokens: Sequence[int],
                          steps: Sequence[int]) -> np.ndarray:
    """Logits from which generated tokens `steps` (1-based t) were sampled, given that the
    sequence is prompt + gen_tokens: one causal pass over prompt + gen_tokens[:max(steps)-1];
    the logits for token t are the row at position P + t - 2."""
    P = len(prompt)
    tmax = max(int(s) for s in steps)
    seq = list(int(x) for x in prompt) + [int(x) for x in gen_tokens[: tmax - 1]]
    rows = [P + int(s) - 2 for s in steps]
    return dec.forward_full(seq, logits_at=rows)


def token_logprobs(dec: RefDecoder, prompt: Sequence[int], gen_tokens: Sequence[int]) -> np.ndarray:
    """log pi(y_t | x, y_<t), t = 1..len(gen_tokens): the policy log-probabilities the GRPO / DAPO objective is built
    from ("compute per-completion rewards" / "form group-relative advantages" act on these
    sampled completions).  Definition written out: one teacher-forced causal pass, then
    log-softmax (float64, max-subtracted) of the logits row that predicts token t, read at token t."""
    L = len(gen_tokens)
    lg = teacher_forced_logits(dec, prompt, gen_tokens, list(range(1, L + 1))).astype(np.float64)
    mx = lg.max(axis=1, keepdims=True)
    lse = mx[:, 0] + np.log(np.exp(lg - mx).sum(axis=1))
    return lg[np.arange(L), np.asarray(gen_tokens, dtype=np.int64)] - lse
