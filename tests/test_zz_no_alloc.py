"""sagc_attention_noalloc (include/sagc.h): the split-K paged attention with its scratch in the library's static device
array -- for callers that may not call cudaMalloc.  Checked against the existing path (sagc_debug_attention, which
allocates its scratch per call) on two calls in a row with DIFFERENT shapes, so the second call finds the first one's
partials, counters and live list in the shared array.  Tolerance: the 2e-5 of tests/test_gpu_kernels.py (both
outputs against the fp64 definition) and 1e-5 between the two paths.

Collected last on purpose (the suite runs with pytest -x); runs alone in a fresh process as well.
"""
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from paper_2606_02218_b200 import workloads as wl


@pytest.fixture(scope="module")
def B():
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    from paper_2606_02218_b200 import binding
    binding.lib()
    return binding


def _case(seed, ctxs, Hq, Hkv, hd, page):
    """seeded paged K/V cache with shuffled pages + the fp64 definition of softmax(q K^T / sqrt(hd)) V per row"""
    rng = np.random.default_rng(seed)
    ctxs = np.asarray(ctxs, dtype=np.int32)
    M = len(ctxs)
    nb = (ctxs + page - 1) // page
    n_pages = int(nb.sum()) + 3
    perm = rng.permutation(n_pages)
    pt = -np.ones((M, int(nb.max())), dtype=np.int32)
    k = 0
    for m in range(M):
        pt[m, :nb[m]] = perm[k:k + nb[m]]
        k += int(nb[m])
    kv = wl.f32_to_bf16_bits(rng.standard_normal((n_pages, 2, Hkv, page, hd)).astype(np.float32))
    kvf = wl.bf16_bits_to_f32(kv).astype(np.float64)
    q = rng.standard_normal((M, Hq, hd)).astype(np.float32)
    r = Hq // Hkv
    ref = np.zeros((M, Hq, hd))
    for m in range(M):
        c = int(ctxs[m])
        K = np.concatenate([kvf[pt[m, b], 0] for b in range(nb[m])], axis=1)[:, :c]
        V = np.concatenate([kvf[pt[m, b], 1] for b in range(nb[m])], axis=1)[:, :c]
        for h in range(Hq):
            s = K[h // r] @ q[m, h].astype(np.float64) / np.sqrt(hd)
            p = np.exp(s - s.max())
            ref[m, h] = (p / p.sum()) @ V[h // r]
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    return dev(q), dev(kv.view(np.int16)), dev(pt), dev(ctxs), ref


CALLS = [  # (ctxs, Hq, Hkv, hd, page, n_splits): 7B-like heads then 0.5B-like heads, ragged contexts over several tiles
    ([1, 63, 64, 65, 129, 700, 1500, 2300, 128, 3], 28, 4, 128, 64, 8),
    ([900, 2, 127, 1025, 16, 4100], 14, 2, 64, 64, 16),
]


def test_noalloc_attention_matches_the_allocating_path_twice_in_a_row(B):
    cases = [(_case(40 + i, *c[:5]), c) for i, c in enumerate(CALLS)]
    seen = set()
    for rep in range(2):                     # the pair twice: every call after the first sees stale scratch
        for (q, kv, pt, ctx, ref), (_, Hq, Hkv, hd, page, ns) in cases:
            want = B.debug_attention(q, kv, pt, ctx, Hq, Hkv, hd, page, ns, 0)
            out = torch.full((q.shape[0], Hq, hd), float("nan"), dtype=torch.float32, device=q.device)
            torch.cuda.synchronize()
            free0 = torch.cuda.mem_get_info()[0]
            B.attention_noalloc(q, kv, pt, ctx, out, Hq, Hkv, hd, page, ns)
            torch.cuda.synchronize()
            free1 = torch.cuda.mem_get_info()[0]
            if hd in seen:                   # (a kernel's first launch may load its module: not an allocation of the call)
                assert free1 >= free0, (free0, free1)
            seen.add(hd)
            got, want = out.cpu().numpy(), want.cpu().numpy()
            assert np.isfinite(got).all()
            assert np.max(np.abs(got - want)) <= 1e-5, np.max(np.abs(got - want))
            assert np.max(np.abs(got - ref)) < 2e-5, np.max(np.abs(got - ref))


def test_noalloc_attention_rejects_sizes_beyond_the_static_scratch(B):
    (q, kv, pt, ctx, _), (_, Hq, Hkv, hd, page, _) = _case(40, *CALLS[0][:5]), CALLS[0]
    M = 64                                                        # 64 rows x 28 heads x 16 splits x 130 floats = 14.9 MB > 8 MiB
    qq = q[:1].expand(M, Hq, hd).contiguous()
    ptt = pt[:1].expand(M, pt.shape[1]).contiguous()
    cc = ctx[:1].expand(M).contiguous()
    out = torch.zeros((M, Hq, hd), dtype=torch.float32, device=q.device)
    with pytest.raises(B.SagcError, match="SAGC_NOALLOC_SCRATCH_BYTES"):
        B.attention_noalloc(qq, kv, ptt, cc, out, Hq, Hkv, hd, page, 16)
    assert float(out.abs().max()) == 0.0                          # nothing was launched
    out1 = torch.empty((M, Hq, hd), dtype=torch.float32, device=q.device)
    B.attention_noalloc(qq, kv, ptt, cc, out1, Hq, Hkv, hd, page, 4)      # the same rows fit with 4 splits
    want = B.debug_attention(qq, kv, ptt, cc, Hq, Hkv, hd, page, 4, 0)
    torch.cuda.synchronize()
    assert float((out1 - want).abs().max()) <= 1e-5
