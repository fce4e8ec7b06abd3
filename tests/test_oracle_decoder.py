"""Pins for oracle/decoder.py and oracle/rollout.py (no GPU)."""
import numpy as np
import pytest

from oracle import decoder as od
from oracle import philox, rollout
from paper_2606_02218_b200 import workloads as wl


def _tiny(**kw):
    w = wl.tiny_variant(1, **kw)
    return w, wl.make_weights(w.model, seed=0)


def test_round_to_bf16_ties_to_even_and_idempotent():
    x = np.array([1.0, 1.0 + 2 ** -8, 1.0 + 3 * 2 ** -8, 1.0 + 2 ** -9, -3.14159, 0.0], dtype=np.float32)
    r = od.round_to_bf16(x)
    assert r[0] == 1.0 and r[1] == 1.0 and r[2] == np.float32(1.0 + 2 ** -6) and r[3] == 1.0
    assert np.array_equal(od.round_to_bf16(r), r)
    assert np.all(np.abs(r - x) <= np.abs(x) * 2.0 ** -8)
    # the harness' weight encoder is an independent implementation of the same rounding
    z = np.random.default_rng(0).standard_normal(1000).astype(np.float32)
    assert np.array_equal(wl.bf16_bits_to_f32(wl.f32_to_bf16_bits(z)), od.round_to_bf16(z))


def test_cached_decode_equals_no_cache_brute_force():
    w, weights = _tiny()
    dec = od.RefDecoder(w.model, weights)
    toks = np.random.default_rng(1).integers(0, w.model.vocab, size=21)
    full = dec.forward_full(toks)
    lg, cache = dec.prefill(toks[:13])
    assert np.allclose(lg, full[12], atol=2e-5)
    for i in range(13, 21):
        lg = dec.step(int(toks[i]), i, cache)
        assert np.allclose(lg, full[i], atol=2e-5)
    assert len(cache[0][0]) == 21


def test_rope_identity_at_position_zero_and_norm_preserving():
    x = np.random.default_rng(2).standard_normal((3, 2, 32)).astype(np.float32)
    cos, sin = od.rope_tables(np.array([0, 5, 17000]), 32, 1e4)
    y = od.apply_rope(x, cos, sin)
    assert np.array_equal(y[0], x[0])
    assert np.allclose(np.linalg.norm(y, axis=-1), np.linalg.norm(x, axis=-1), rtol=1e-5)
    # pair (i, i+hd/2), angle p*theta_i, theta_0 = 1: position 5, pair 0 is a rotation by 5 rad
    a, b = x[1, 0, 0], x[1, 0, 16]
    assert y[1, 0, 0] == pytest.approx(a * np.cos(5.0) - b * np.sin(5.0), rel=1e-5)
    assert y[1, 0, 16] == pytest.approx(b * np.cos(5.0) + a * np.sin(5.0), rel=1e-5)


def test_rope_relative_position_invariance():
    w, weights = _tiny()
    dec = od.RefDecoder(w.model, weights, kv_round=False)
    toks = np.random.default_rng(3).integers(0, w.model.vocab, size=12)
    a = dec.forward_full(toks, pos0=0)
    b = dec.forward_full(toks, pos0=1000)
    assert np.allclose(a, b, atol=5e-4)          # fp32 cos/sin at large angles


def test_zero_layers_closed_form_and_single_entry_context():
    w, weights = _tiny(model_n_layers=0)
    dec = od.RefDecoder(w.model, weights)
    E = wl.bf16_bits_to_f32(weights["embed"]).astype(np.float64)
    Wlm = wl.bf16_bits_to_f32(weights["lm_head"]).astype(np.float64)
    x = E[7]
    ref = Wlm @ (x / np.sqrt(np.mean(x * x) + 1e-6))
    assert np.allclose(dec.forward_full([7])[0], ref, atol=1e-5)
    # one cached entry: softmax over a single score is 1, so o = v
    w1, weights1 = _tiny()
    d1 = od.RefDecoder(w1.model, weights1)
    K = np.random.default_rng(4).standard_normal((1, 4, 32)).astype(np.float32)
    V = np.random.default_rng(5).standard_normal((1, 4, 32)).astype(np.float32)
    q = np.random.default_rng(6).standard_normal((4, 32)).astype(np.float32)
    assert np.array_equal(d1._attend(q, K, V), V.reshape(-1))
    # q = 0: uniform attention, o = mean(v)
    K5 = np.random.default_rng(7).standard_normal((5, 4, 32)).astype(np.float32)
    V5 = np.random.default_rng(8).standard_normal((5, 4, 32)).astype(np.float32)
    assert np.allclose(d1._attend(np.zeros((4, 32), np.float32), K5, V5), V5.mean(0).reshape(-1), atol=1e-6)


def test_gqa_equals_mha_with_repeated_kv_weights():
    w, weights = _tiny(model_n_kv_heads=2)
    m = w.model
    mha = wl.tiny_variant(1).model
    rep = dict(weights)
    r = m.n_q_heads // m.n_kv_heads
    for name in ("wk", "wv"):
        rep[name] = [np.repeat(a.reshape(m.n_kv_heads, m.head_dim, m.d_model), r, axis=0)
                     .reshape(m.n_q_heads * m.head_dim, m.d_model) for a in weights[name]]
    toks = np.random.default_rng(9).integers(0, m.vocab, size=9)
    a = od.RefDecoder(m, weights).forward_full(toks)
    b = od.RefDecoder(mha, rep).forward_full(toks)
    assert np.allclose(a, b, atol=1e-6)


def test_against_transformers_llama():
    """Independent library implementation: pins rotate-half RoPE, pre-norm, eps placement,
    SwiGLU, GQA grouping, untied LM head (KV rounding off: the library has none)."""
    torch = pytest.importorskip("torch")
    tf = pytest.importorskip("transformers")
    w, weights = _tiny(model_n_kv_heads=2, model_rope_theta=1e4)
    m = w.model
    cfg = tf.LlamaConfig(vocab_size=m.vocab, hidden_size=m.d_model, intermediate_size=m.d_ff,
                         num_hidden_layers=m.n_layers, num_attention_heads=m.n_q_heads,
                         num_key_value_heads=m.n_kv_heads, head_dim=m.head_dim, hidden_act="silu",
                         rms_norm_eps=m.rms_eps, rope_theta=m.rope_theta, attention_bias=False,
                         mlp_bias=False, tie_word_embeddings=False, max_position_embeddings=256,
                         attn_implementation="eager")
    try:
        model = tf.LlamaForCausalLM(cfg).to(torch.float32).eval()
    except Exception as e:                                        # pragma: no cover
        pytest.skip(f"transformers model construction failed: {e}")
    # non-trivial norm gains so that gain placement is pinned too
    rng = np.random.default_rng(12)
    for key in ("norm1", "norm2"):
        weights[key] = [wl.f32_to_bf16_bits((1.0 + 0.1 * rng.standard_normal(m.d_model)).astype(np.float32))
                        for _ in range(m.n_layers)]
    weights["final_norm"] = wl.f32_to_bf16_bits((1.0 + 0.1 * rng.standard_normal(m.d_model)).astype(np.float32))
    f = lambda b: torch.from_numpy(wl.bf16_bits_to_f32(b).copy())
    sd = {"model.embed_tokens.weight": f(weights["embed"]), "lm_head.weight": f(weights["lm_head"]),
          "model.norm.weight": f(weights["final_norm"])}
    names = {"wq": "self_attn.q_proj", "wk": "self_attn.k_proj", "wv": "self_attn.v_proj",
             "wo": "self_attn.o_proj", "wg": "mlp.gate_proj", "wu": "mlp.up_proj", "wd": "mlp.down_proj",
             "norm1": "input_layernorm", "norm2": "post_attention_layernorm"}
    for l in range(m.n_layers):
        for k, v in names.items():
            sd[f"model.layers.{l}.{v}.weight"] = f(weights[k][l])
    missing = model.load_state_dict(sd, strict=False)
    assert not [k for k in missing.missing_keys if "rotary" not in k]
    toks = np.random.default_rng(10).integers(0, m.vocab, size=17)
    with torch.no_grad():
        ref = model(torch.from_numpy(toks)[None, :]).logits[0].numpy()
    got = od.RefDecoder(m, weights, kv_round=False).forward_full(toks)
    assert np.allclose(got, ref, atol=2e-5), float(np.abs(got - ref).max())


def test_rollout_greedy_prefix_property_lengths_and_stop():
    w, weights = _tiny()
    dec = od.RefDecoder(w.model, weights)
    ptoks, poffs = wl.make_prompts(w)
    forced = np.array([5, 12, 1, 9], dtype=np.int32)
    res = rollout.rollout_group(dec, ptoks, poffs, 4, 0, 1.0, 0, 16, forced_lengths=forced,
                                n_pages=64, page_tokens=16)
    assert res.lengths.tolist() == forced.tolist()
    long = res.tokens[1]
    for s in range(4):                                            # greedy: prefixes of one another
        n = forced[s]
        assert np.array_equal(res.tokens[s, :n], long[:n]) and np.all(res.tokens[s, n:] == -1)
    assert res.len_stats[0].tolist() == [12, 27, 14] and res.ratio_max_mean[0] == np.float32(48) / np.float32(27)
    assert sorted(res.paging.free_stack) == list(range(64))
    # stop token = the 4th greedy token: every completion stops there (stop token counted)
    stop = int(long[3])
    first = int(np.argmax(long[:12] == stop)) + 1
    res2 = rollout.rollout_group(dec, ptoks, poffs, 4, 0, 1.0, 0, 16, stop_token=stop)
    assert res2.lengths.tolist() == [first] * 4 and res2.tokens[0, first - 1] == stop
    # max_new caps
    res3 = rollout.rollout_group(dec, ptoks, poffs, 2, 0, 1.0, 0, 6)
    assert res3.lengths.tolist() == [6, 6]


def test_rollout_gumbel_teacher_forced_consistency():
    w, weights = _tiny()
    dec = od.RefDecoder(w.model, weights)
    ptoks, poffs = wl.make_prompts(w)
    res = rollout.rollout_group(dec, ptoks, poffs, 3, 1, 1.0, 4001, 10, forced_lengths=[10, 4, 7],
                                keep_logits=True)
    assert len({tuple(r) for r in res.tokens.tolist()}) == 3      # distinct Gumbel draws per sid
    lg = rollout.teacher_forced_logits(dec, ptoks, res.tokens[0], steps=[1, 5, 10])
    for row, t in zip(lg, (1, 5, 10)):
        assert np.allclose(row, res.logits[(0, t)], atol=2e-5)
        assert philox.sample_token(row, 1, 1.0, 4001, 0, t) == res.tokens[0, t - 1]


def test_token_logprobs_pins():
    """oracle.rollout.token_logprobs: (i) library routine: scipy.special.log_softmax of the same logits; (ii) invariant:
    the log-probs over the whole vocabulary of one position sum to 1 in probability; (iii) brute force: a sequence's
    log-likelihood equals the sum of the step-by-step cached-decode log-softmax values."""
    oro = rollout
    w = wl.WORKLOADS[1]
    weights = wl.make_weights(w.model, 0)
    dec = od.RefDecoder(w.model, weights)
    rng = np.random.default_rng(0)
    prompt = rng.integers(0, w.model.vocab, size=9)
    gen = rng.integers(0, w.model.vocab, size=7)
    lp = oro.token_logprobs(dec, prompt, gen)
    assert lp.shape == (7,) and np.all(lp < 0)
    scipy_special = pytest.importorskip("scipy.special")
    lg = oro.teacher_forced_logits(dec, prompt, gen, list(range(1, 8))).astype(np.float64)
    ref = scipy_special.log_softmax(lg, axis=1)
    assert np.allclose(lp, ref[np.arange(7), gen], atol=1e-12)
    assert np.allclose(np.exp(ref).sum(axis=1), 1.0, atol=1e-12)
    # brute force through the cached decode path
    lg0, cache = dec.prefill(prompt)
    rows = [lg0]
    for t in range(1, 7):
        rows.append(dec.step(int(gen[t - 1]), len(prompt) + t - 1, cache))
    step_lp = [float(scipy_special.log_softmax(r.astype(np.float64))[gen[t]]) for t, r in enumerate(rows)]
    assert np.allclose(lp, step_lp, atol=2e-4)
