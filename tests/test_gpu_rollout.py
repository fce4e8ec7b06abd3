"""GPU parity, path level: sagc_rollout_group through the C ABI vs the CPU oracle.

Bit-exact: page tables, free stack, allocation log, retirement log, lengths, length statistics,
ratio.  Teacher-forced logits: max abs error <= 3e-2.  Tokens: the oracle replays the GPU's
tokens; every position must satisfy gpu_token == oracle_argmax or oracle top-2 margin < 1e-2,
with >= 99.5% plain agreement (BASELINE.json north_star; reading C1).
"""
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from oracle import decoder as odec
from oracle import paging as opg
from oracle import philox as oph
from oracle import rollout as oro
from oracle import groupstats as ogs
from paper_2606_02218_b200 import workloads as wl


@pytest.fixture(scope="module")
def B():
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    from paper_2606_02218_b200 import binding
    binding.lib()
    return binding


def _pool_pages(w, G, n_prompts, P, max_new):
    page = w.model.page_tokens
    return n_prompts * (P // page + G * ((max_new + P % page + page - 1) // page + 1)) + 8


def _structure_model(B, w, n_pages, max_seqs, max_ctx):
    """A handle with a zero-layer stand-in model: structure-only runs never touch the weights."""
    mc = wl.ModelConfig(0, 32, 1, 1, 32, 32, 16, 1e4, 1e-6, w.model.page_tokens)
    one = wl.f32_to_bf16_bits(np.ones(32, np.float32))
    weights = {"embed": np.zeros((16, 32), np.uint16), "lm_head": np.zeros((16, 32), np.uint16), "final_norm": one}
    for k in ("wq", "wk", "wv", "wo", "wg", "wu", "wd", "norm1", "norm2"):
        weights[k] = []
    return B.Model(mc, weights, n_pages, max_seqs, max_ctx)


def _check_structure(B, m, st, out, ell_expected):
    assert np.array_equal(out.lengths.cpu().numpy(), ell_expected)
    nseq = len(ell_expected)
    pt = m.debug_page_table()
    assert pt.shape[0] == nseq
    mb = min(pt.shape[1], st.page_table.shape[1])
    assert np.array_equal(pt[:, :mb], st.page_table[:, :mb])
    assert np.all(pt[:, mb:] == -1) and np.all(st.page_table[:, mb:] == -1)
    assert np.array_equal(m.debug_free_stack(), np.asarray(st.free_stack, dtype=np.int32))
    assert np.array_equal(m.debug_alloc_log(), np.asarray(st.alloc_log, dtype=np.int32).reshape(-1, 3))
    assert np.array_equal(m.debug_retire_log(), np.asarray(st.retire_log, dtype=np.int32).reshape(-1, 2))
    assert m.debug_peak_pages() == st.peak_used


# ---------------------------------------------------------------------------- a1, a4, a13 (all five configs)
@pytest.mark.parametrize("cfg,G", [(1, 4), (2, 8), (3, 16), (4, 4), (4, 32), (5, 32)])
def test_structure_only_bit_exact(B, cfg, G):
    w = wl.WORKLOADS[cfg]
    fl = wl.make_forced_lengths(w, G=G, step=3)
    _, offs = wl.make_prompts(w)
    P, n_prompts, page = w.prompt_len, w.n_prompts, w.model.page_tokens
    st, _ = opg.run_structure_only(10 ** 6, page, [P] * n_prompts, G, fl, w.max_new)
    n_pages = st.peak_used + 5                                   # just above the oracle's peak
    st, _ = opg.run_structure_only(n_pages, page, [P] * n_prompts, G, fl, w.max_new)
    m = _structure_model(B, w, n_pages, n_prompts * G, P + w.max_new)
    out = m.rollout_group(None, offs, G, max_new_tokens=w.max_new, forced_lengths=fl,
                          flags=B.FLAG_STRUCTURE_ONLY | B.FLAG_LOG)
    ell = np.minimum(fl, w.max_new).astype(np.int32)
    _check_structure(B, m, st, out, ell)
    goffs = np.arange(n_prompts + 1) * G
    st_o, ra_o = ogs.length_stats(ell, goffs)
    assert np.array_equal(out.len_stats.cpu().numpy(), st_o)
    assert np.array_equal(out.ratio_max_mean.cpu().numpy().view(np.uint32), ra_o.view(np.uint32))
    assert np.all(out.ratio_max_mean.cpu().numpy() >= 1.0)
    m.close()


def test_structure_ragged_prompts_and_pool_exhaustion(B):
    w = wl.tiny_variant(1)
    plens = [5, 16, 33, 47, 1]
    offs = np.concatenate([[0], np.cumsum(plens)]).astype(np.int32)
    G = 3
    rng = np.random.default_rng(5)
    fl = rng.integers(1, 60, size=len(plens) * G).astype(np.int32)
    fl[0] = 1; fl[4] = 60
    st, _ = opg.run_structure_only(10 ** 5, 16, plens, G, fl, 48)
    n_pages = st.peak_used
    st, _ = opg.run_structure_only(n_pages, 16, plens, G, fl, 48)
    m = _structure_model(B, w, n_pages, len(plens) * G, 47 + 48)
    out = m.rollout_group(None, offs, G, max_new_tokens=48, forced_lengths=fl, flags=B.FLAG_STRUCTURE_ONLY | B.FLAG_LOG)
    _check_structure(B, m, st, out, np.minimum(fl, 48).astype(np.int32))
    m.close()
    m = _structure_model(B, w, n_pages - 1, len(plens) * G, 47 + 48)      # one page short -> SAGC_EPAGES
    with pytest.raises(B.SagcError) as ei:
        m.rollout_group(None, offs, G, max_new_tokens=48, forced_lengths=fl, flags=B.FLAG_STRUCTURE_ONLY)
    assert ei.value.code == B.EPAGES
    with pytest.raises(opg.PagePoolExhausted):
        opg.run_structure_only(n_pages - 1, 16, plens, G, fl, 48)
    m.close()


# ---------------------------------------------------------------------------- full path, tiny configs
def _token_rule(dec, w_mode, temperature, seed, prompts, offs, G, toks, lens, pos_stride=1):
    """Replay the GPU's tokens through the oracle (teacher forcing)."""
    n_bad, n_dis, n_all = 0, 0, 0
    for sid in range(len(lens)):
        p = sid // G
        prompt = prompts[offs[p]:offs[p + 1]]
        L = int(lens[sid])
        steps = list(range(1, L + 1, pos_stride))
        lg = oro.teacher_forced_logits(dec, prompt, toks[sid, :L], steps)
        for i, t in enumerate(steps):
            s = oph.perturbed_scores(lg[i], w_mode, temperature, seed, sid, t)
            n_all += 1
            if int(np.argmax(s)) != int(toks[sid, t - 1]):
                n_dis += 1
                if oph.top2_margin(s) >= 1e-2:
                    n_bad += 1
    return n_bad, n_dis, n_all


def _dump_error(dec, prompts, offs, G, toks, lens, dump, lg):
    """max |gpu - oracle| over the dumped logits rows, the oracle teacher-forced on the GPU's own tokens (so the
    comparison holds whether or not a free-running sequence forked at a near-tie)."""
    worst = 0.0
    for sid in sorted({s for s, _ in dump}):
        p = sid // G
        steps = [t for (s2, t) in dump if s2 == sid]
        ref = oro.teacher_forced_logits(dec, prompts[offs[p]:offs[p + 1]], toks[sid, :lens[sid]], steps)
        for i, t in enumerate(steps):
            worst = max(worst, float(np.max(np.abs(lg[dump.index((sid, t))] - ref[i]))))
    return worst


@pytest.mark.parametrize("path", [0, 1, 2])
def test_config1_end_to_end(B, path):
    w = wl.WORKLOADS[1]
    weights = wl.make_weights(w.model, 0)
    prompts, offs = wl.make_prompts(w)
    fl = wl.make_forced_lengths(w)
    dec = odec.RefDecoder(w.model, weights)
    n_pages = _pool_pages(w, w.G, w.n_prompts, w.prompt_len, w.max_new)
    ref = oro.rollout_group(dec, prompts, offs, w.G, 0, 1.0, w.philox_seed, w.max_new, forced_lengths=fl,
                            n_pages=n_pages, page_tokens=w.model.page_tokens, keep_logits=True)
    m = B.Model(w.model, weights, n_pages, w.n_prompts * w.G, w.prompt_len + w.max_new)
    dump = [(sid, t) for sid in range(w.G) for t in range(1, int(min(fl[sid], w.max_new)) + 1, 5)]
    out = m.rollout_group(prompts, offs, w.G, mode=B.MODE_GREEDY, seed=w.philox_seed, max_new_tokens=w.max_new,
                          forced_lengths=fl, path=path, flags=B.FLAG_LOG, dump=dump, timing=True)
    toks = out.tokens.cpu().numpy()
    assert np.array_equal(out.lengths.cpu().numpy(), ref.lengths)
    _check_structure(B, m, ref.paging, out, ref.lengths)
    # teacher-forced logits (free-running == teacher-forced while the tokens agree)
    lg = out.dump_logits.cpu().numpy()
    assert _dump_error(dec, prompts, offs, w.G, toks, ref.lengths, dump, lg) <= 3e-2
    n_bad, n_dis, n_all = _token_rule(dec, 0, 1.0, w.philox_seed, prompts, offs, w.G, toks, ref.lengths)
    assert n_bad == 0 and n_dis <= 0.005 * n_all, (n_bad, n_dis, n_all)
    assert np.array_equal(toks, ref.tokens)                      # config 1: exact free-running equality
    assert np.all(toks[np.arange(toks.shape[1])[None, :] >= ref.lengths[:, None]] == -1)
    # greedy completions of one prompt are prefixes of one another
    for a in range(w.G):
        for b in range(w.G):
            n = min(ref.lengths[a], ref.lengths[b])
            assert np.array_equal(toks[a, :n], toks[b, :n])
    assert np.array_equal(out.len_stats.cpu().numpy(), ref.len_stats)
    assert np.array_equal(out.ratio_max_mean.cpu().numpy().view(np.uint32), ref.ratio_max_mean.view(np.uint32))
    assert out.timing["kernel_launches"] > 0 and out.timing["total_tokens"] == int(ref.lengths.sum())
    # the same call through host buffers
    outh = m.rollout_group(prompts, offs, w.G, mode=B.MODE_GREEDY, seed=w.philox_seed, max_new_tokens=w.max_new,
                           forced_lengths=fl, path=path, host=True)
    assert np.array_equal(outh.tokens.numpy(), toks) and np.array_equal(outh.lengths.numpy(), ref.lengths)
    m.close()


@pytest.mark.parametrize("mode,step_kernel", [(0, 0), (1, 0), (0, 1), (1, 1)])
def test_tiny_gqa_ragged_prompts(B, monkeypatch, mode, step_kernel):
    """GQA (r = 4), head_dim 64, prompts whose lengths are not page multiples, Gumbel sampling; per-layer kernels and
    the persistent decode-step kernel."""
    monkeypatch.setenv("SAGC_STEP", str(step_kernel))
    w = wl.tiny_variant(1, model_n_q_heads=8, model_n_kv_heads=2, model_head_dim=64, model_d_model=256,
                        model_d_ff=768, model_n_layers=3, model_vocab=2048, model_page_tokens=16)
    weights = wl.make_weights(w.model, 1)
    plens = [7, 16, 41]
    offs = np.concatenate([[0], np.cumsum(plens)]).astype(np.int32)
    prompts = np.random.default_rng(9).integers(0, w.model.vocab, size=offs[-1]).astype(np.int32)
    G, max_new = 3, 40
    fl = np.array([1, 40, 17, 16, 9, 33, 25, 2, 40], dtype=np.int32)
    dec = odec.RefDecoder(w.model, weights)
    n_pages = 200
    seed = 77
    ref = oro.rollout_group(dec, prompts, offs, G, mode, 0.7, seed, max_new, forced_lengths=fl, n_pages=n_pages,
                            page_tokens=16, keep_logits=True)
    m = B.Model(w.model, weights, n_pages, len(plens) * G, 41 + max_new)
    dump = [(sid, t) for sid in range(9) for t in (1, 2, int(fl[sid])) if t <= fl[sid]]
    out = m.rollout_group(prompts, offs, G, mode=mode, temperature=0.7, seed=seed, max_new_tokens=max_new,
                          forced_lengths=fl, flags=B.FLAG_LOG, dump=dump)
    toks = out.tokens.cpu().numpy()
    _check_structure(B, m, ref.paging, out, ref.lengths)
    n_bad, n_dis, n_all = _token_rule(dec, mode, 0.7, seed, prompts, offs, G, toks, ref.lengths)
    assert n_bad == 0 and n_dis <= max(1, 0.005 * n_all), (n_bad, n_dis, n_all)
    assert _dump_error(dec, prompts, offs, G, toks, ref.lengths, dump, out.dump_logits.cpu().numpy()) <= 3e-2
    m.close()


def test_stop_token_mode_config1(B):
    w = wl.WORKLOADS[1]
    weights = wl.make_weights(w.model, 0)
    prompts, offs = wl.make_prompts(w)
    dec = odec.RefDecoder(w.model, weights)
    # pick as stop token the token the greedy completion emits at step 9
    probe = oro.rollout_group(dec, prompts, offs, 1, 0, 1.0, 0, 24)
    stop = int(probe.tokens[0, 8])
    ref = oro.rollout_group(dec, prompts, offs, 2, 0, 1.0, 0, 24, stop_token=stop, n_pages=64, page_tokens=16)
    m = B.Model(w.model, weights, 64, 2, w.prompt_len + 24)
    out = m.rollout_group(prompts, offs, 2, mode=B.MODE_GREEDY, max_new_tokens=24, stop_token=stop, flags=B.FLAG_LOG)
    assert np.array_equal(out.tokens.cpu().numpy(), ref.tokens)
    assert np.array_equal(out.lengths.cpu().numpy(), ref.lengths)
    assert ref.lengths[0] <= 9 and out.tokens.cpu().numpy()[0, ref.lengths[0] - 1] == stop   # stop token is counted
    _check_structure(B, m, ref.paging, out, ref.lengths)
    m.close()


def test_bad_arguments_fail_loudly(B):
    w = wl.WORKLOADS[1]
    weights = wl.make_weights(w.model, 0)
    prompts, offs = wl.make_prompts(w)
    m = B.Model(w.model, weights, 64, 4, 64)
    with pytest.raises(B.SagcError) as ei:
        m.rollout_group(prompts, offs, 8, max_new_tokens=8)              # nseq > max_seqs
    assert ei.value.code == B.EINVAL
    with pytest.raises(B.SagcError):
        m.rollout_group(prompts, offs, 4, max_new_tokens=64)             # P + max_new > max_ctx
    with pytest.raises(B.SagcError):
        m.rollout_group(prompts, offs, 4, mode=B.MODE_GUMBEL, temperature=0.0, max_new_tokens=8)
    m.close()


# ---------------------------------------------------------------------------- configs 2..5: sampled slices
def _sampled_parity(B, cfg, n_prompts, P, G, max_new, fl, path, n_dump_seq=3):
    """Run a truncated instance of a BASELINE config (full-size model, fewer / shorter sequences) and
    compare against the oracle teacher-forced on the GPU's own tokens."""
    w = wl.WORKLOADS[cfg]
    weights = wl.make_weights(w.model, 0)
    prompts, offs = wl.make_prompts(w, n_prompts=n_prompts, prompt_len=P)
    mode = 1 if w.sampling == "gumbel" else 0
    n_pages = _pool_pages(w, G, n_prompts, P, max_new)
    m = B.Model(w.model, weights, n_pages, n_prompts * G, P + max_new)
    sids = list(range(0, n_prompts * G, max(1, (n_prompts * G) // n_dump_seq)))[:n_dump_seq]
    dump = [(sid, t) for sid in sids for t in sorted({1, 2, int(fl[sid]) // 2 + 1, int(fl[sid])}) if 1 <= t <= fl[sid]]
    out = m.rollout_group(prompts, offs, G, mode=mode, temperature=w.temperature, seed=w.philox_seed,
                          max_new_tokens=max_new, forced_lengths=fl, path=path, flags=B.FLAG_LOG, dump=dump)
    toks = out.tokens.cpu().numpy()
    lens = out.lengths.cpu().numpy()
    assert np.array_equal(lens, np.minimum(fl, max_new))
    st, _ = opg.run_structure_only(n_pages, w.model.page_tokens, [P] * n_prompts, G, fl, max_new)
    _check_structure(B, m, st, out, lens)
    dec = odec.RefDecoder(w.model, weights, cache_f32=w.model.n_params() < 1e9)
    lg = out.dump_logits.cpu().numpy()
    worst, n_bad, n_dis, n_all = 0.0, 0, 0, 0
    for sid in sids:
        p = sid // G
        steps = [t for (s, t) in dump if s == sid]
        ref = oro.teacher_forced_logits(dec, prompts[offs[p]:offs[p + 1]], toks[sid, :lens[sid]], steps)
        for i, t in enumerate(steps):
            k = dump.index((sid, t))
            worst = max(worst, float(np.max(np.abs(lg[k] - ref[i]))))
            s = oph.perturbed_scores(ref[i], mode, w.temperature, w.philox_seed, sid, t)
            n_all += 1
            if int(np.argmax(s)) != int(toks[sid, t - 1]):
                n_dis += 1
                n_bad += oph.top2_margin(s) >= 1e-2
    # the product path proper: no logits dump -> LM head and sampler fused, logits never stored.  Same arithmetic, same
    # Philox keys: the tokens must be identical to the run above.
    out2 = m.rollout_group(prompts, offs, G, mode=mode, temperature=w.temperature, seed=w.philox_seed,
                           max_new_tokens=max_new, forced_lengths=fl, path=path)
    assert np.array_equal(out2.tokens.cpu().numpy(), toks)
    m.close()
    assert worst <= 3e-2, worst
    assert n_bad == 0 and n_dis <= 0.005 * n_all, (n_bad, n_dis, n_all)
    return worst


@pytest.mark.parametrize("variant", ["step_kernel", "per_layer_kernels", "register_hmma"])
def test_config2_truncated(B, monkeypatch, variant):
    """0.5B shape: 2 prompts x 256 x G=8 (16 live rows, then fewer) through the three decode paths that exist:
    the per-layer tcgen05 kernels (default), the persistent decode-step kernel (SAGC_STEP=1) and the
    register-HMMA kernels (SAGC_TC=0: the path of shapes that are not multiples of 128)."""
    if variant == "step_kernel":
        monkeypatch.setenv("SAGC_STEP", "1")
    if variant == "register_hmma":
        monkeypatch.setenv("SAGC_TC", "0")
    fl = np.array([3, 14, 14, 2, 14, 9, 5, 14, 14, 1, 14, 7, 14, 14, 4, 14], dtype=np.int32)
    _sampled_parity(B, 2, 2, 256, 8, 14, fl, 0)


@pytest.mark.parametrize("step_kernel,att_tc", [(0, 0), (0, 2), (1, 0)])
def test_config3_truncated(B, monkeypatch, step_kernel, att_tc):
    """1.5B shape (head_dim 128, r = 6, DAPO config): 1 prompt x 96 tokens (ragged vs the 64-token page) x G=16.
    att_tc = 2 forces the tcgen05 attention kernel at these short contexts too (by default it takes the steps with
    >= 32 live rows or >= 2 048 cached tokens), 0 = the register-HMMA unit on every step."""
    monkeypatch.setenv("SAGC_STEP", str(step_kernel))
    monkeypatch.setenv("SAGC_ATT_TC", str(att_tc))
    fl = np.array([10, 3, 10, 10, 1, 10, 7, 10, 10, 10, 5, 10, 10, 2, 10, 10], dtype=np.int32)
    _sampled_parity(B, 3, 1, 96, 16, 10, fl, 0, n_dump_seq=2)


@pytest.mark.parametrize("cfg,G,att_tc", [(4, 32, 1), (4, 32, 2), (4, 32, 0)])
def test_config4_truncated(B, monkeypatch, cfg, G, att_tc):
    """7B shape (configs 4 and 5 share it): 1 prompt x 128 tokens x G=32 -> 32 live rows on the tcgen05 path,
    then the tail path; logits of two sampled sequences against the fp32 oracle.  att_tc: 1 = default policy (tcgen05
    attention while 32 rows are live, register-HMMA below), 2 = tcgen05 attention on every step, 0 = never."""
    monkeypatch.setenv("SAGC_ATT_TC", str(att_tc))
    fl = np.array([6, 4, 6, 3, 6, 2, 6, 1, 6, 4, 6, 3] + [1, 2, 3, 4] * 5, dtype=np.int32)   # 6 live in steps 5-6
    _sampled_parity(B, cfg, 1, 128, G, 6, fl, 0, n_dump_seq=2)


def test_variable_G_per_call_same_handle(B):
    """Config 4's pattern: the controller re-chooses G every rollout step; one handle, a seeded G schedule,
    per-step Philox seed = base + step.  Every call must match the oracle exactly (tiny model)."""
    w = wl.tiny_variant(1, n_prompts=2)
    weights = wl.make_weights(w.model, 0)
    prompts, offs = wl.make_prompts(w, n_prompts=2, prompt_len=24)       # ragged vs the 16-token page
    dec = odec.RefDecoder(w.model, weights)
    m = B.Model(w.model, weights, 400, 2 * 16, 24 + 20)
    rng = np.random.default_rng(4)
    for step, G in enumerate([4, 8, 16, 8, 4]):
        fl = rng.integers(1, 21, size=2 * G).astype(np.int32)
        seed = 4004 + step
        ref = oro.rollout_group(dec, prompts, offs, G, 1, 1.0, seed, 20, forced_lengths=fl, n_pages=400, page_tokens=16)
        out = m.rollout_group(prompts, offs, G, mode=B.MODE_GUMBEL, temperature=1.0, seed=seed, max_new_tokens=20,
                              forced_lengths=fl, flags=B.FLAG_LOG)
        _check_structure(B, m, ref.paging, out, ref.lengths)
        toks = out.tokens.cpu().numpy()
        n_bad, n_dis, n_all = _token_rule(dec, 1, 1.0, seed, prompts, offs, G, toks, ref.lengths)
        assert n_bad == 0 and n_dis <= max(1, 0.005 * n_all), (step, G, n_bad, n_dis, n_all)
        assert np.array_equal(out.len_stats.cpu().numpy(), ref.len_stats)
    m.close()


def test_no_graph_flag_gives_identical_tokens(B):
    """SAGC_FLAG_NO_GRAPH launches the same kernels directly: tokens, lengths and page state must not change."""
    w = wl.tiny_variant(1, model_n_q_heads=4, model_n_kv_heads=2, model_head_dim=64, model_d_model=256,
                        model_d_ff=512, model_n_layers=2, model_vocab=1024, model_page_tokens=16)
    weights = wl.make_weights(w.model, 3)
    prompts, offs = wl.make_prompts(w, n_prompts=2, prompt_len=20)
    fl = np.array([9, 30, 30, 2, 17, 30], dtype=np.int32)
    m = B.Model(w.model, weights, 100, 6, 20 + 30)
    outs = []
    for flags in (B.FLAG_LOG, B.FLAG_LOG | B.FLAG_NO_GRAPH):
        out = m.rollout_group(prompts, offs, 3, mode=B.MODE_GUMBEL, temperature=0.9, seed=11, max_new_tokens=30,
                              forced_lengths=fl, flags=flags)
        outs.append((out.tokens.cpu().numpy(), out.lengths.cpu().numpy(), m.debug_page_table(), m.debug_alloc_log()))
    for a, b in zip(outs[0], outs[1]):
        assert np.array_equal(a, b)
    m.close()


@pytest.mark.parametrize("G,mode,ctas", [(3, "gumbel", 5), (20, "gumbel", 3), (20, "greedy", 148), (9, "gumbel", 148)])
def test_fused_lm_head_sampler_gives_identical_tokens(B, monkeypatch, G, mode, ctas):
    """a11 + a12 fused (persistent tcgen05 LM head with the Gumbel arg-max in its epilogue, logits never stored) against the
    unfused LM head -> k_sample path: the logit arithmetic and the Philox keys are the same, so tokens must be identical.
    SAGC_LM_CTAS forces several vocabulary tiles per CTA (TMEM double buffer, ring wrap-around, ragged tile counts)."""
    w = wl.tiny_variant(1, model_n_q_heads=4, model_n_kv_heads=2, model_head_dim=64, model_d_model=256,
                        model_d_ff=512, model_n_layers=2, model_vocab=8192, model_page_tokens=16)
    weights = wl.make_weights(w.model, 5)
    prompts, offs = wl.make_prompts(w, n_prompts=2, prompt_len=20)
    rng = np.random.default_rng(G)
    fl = rng.integers(1, 25, size=2 * G).astype(np.int32)
    fl[0] = 24
    outs = []
    for fused in ("1", "0"):
        monkeypatch.setenv("SAGC_LM_FUSED", fused)
        monkeypatch.setenv("SAGC_LM_CTAS", str(ctas))
        m = B.Model(w.model, weights, 200, 2 * G, 20 + 24)
        out = m.rollout_group(prompts, offs, G, mode=B.MODE_GUMBEL if mode == "gumbel" else B.MODE_GREEDY, temperature=0.8,
                              seed=23, max_new_tokens=24, forced_lengths=fl, flags=B.FLAG_LOG)
        outs.append((out.tokens.cpu().numpy(), out.lengths.cpu().numpy(), m.debug_page_table()))
        m.close()
    for a, b in zip(outs[0], outs[1]):
        assert np.array_equal(a, b)
    assert (outs[0][0] >= 0).sum() == int(fl.sum())


def test_sagc_controller_closes_the_loop_on_the_gpu(B):
    """f1 + f3 (Alg.1 l.173-210, sec 5.2 l.216-218): the CPU-side controller picks G, every rollout step is one
    sagc_rollout_group call with B_t = 16 / G_t prompts on one handle, and the (max, sum, median_x2) triples that come
    back from the GPU -- the only thing the controller needs (l.153-157) -- equal the oracle's on the same lengths."""
    from paper_2606_02218_b200.controller import SAGCController, run_sagc
    w = wl.tiny_variant(1)
    weights = wl.make_weights(w.model, 0)
    prompts_all, _ = wl.make_prompts(w, n_prompts=4, prompt_len=24)
    m = B.Model(w.model, weights, 600, 16, 24 + 32)
    rng = np.random.default_rng(12)
    seen = []

    def step(t, G, n_prompts):
        offs = (np.arange(n_prompts + 1) * 24).astype(np.int32)
        fl = np.clip(np.rint(12 * np.exp(0.25 * rng.standard_normal(n_prompts * G))), 1, 32).astype(np.int32)
        out = m.rollout_group(prompts_all[: n_prompts * 24], offs, G, mode=B.MODE_GUMBEL, seed=900 + t, max_new_tokens=32,
                              forced_lengths=fl)
        st = out.len_stats.cpu().numpy()
        st_o, _ = ogs.length_stats(fl, np.arange(n_prompts + 1) * G)
        assert np.array_equal(st, st_o)
        seen.append((G, n_prompts))
        return st

    c = SAGCController([2, 4, 8, 16], delta=0.4, eta_lambda=0.5, gamma=0.9, seed=2, g0=4)
    log = run_sagc(step, c, 12, effective_batch=16)
    m.close()
    assert all(g * b == 16 for g, b in seen)
    assert all(abs(c.sizes.index(r["next_G"]) - c.sizes.index(r["G"])) <= 1 for r in log)
    assert all(r["lambda"] >= 0 for r in log)
