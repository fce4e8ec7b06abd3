"""Pins for oracle/groupstats.py (no GPU): what the paper fixes (R >= 1, S = 1[R > tau]),
north_star invariants (zero sum, unit std, all-equal -> 0, DAPO drops), closed forms from
tests/golden, numpy library routines."""
import numpy as np
import pytest

from conftest import golden_lines
from oracle import groupstats as gs


def _csr(sizes):
    return np.concatenate([[0], np.cumsum(sizes)]).astype(np.int32)


def test_length_worked_examples():
    for ln in golden_lines("length_stats_example.txt"):
        a, b, c, d = [x.split() for x in ln.split("|")]
        ell = [int(x) for x in a]
        stats, ratio = gs.length_stats(ell, [0, len(ell)])
        assert stats[0].tolist() == [int(x) for x in b]
        assert ratio[0] == np.float32(float(c[0]))
        R = gs.straggler_ratio_max_median(stats)
        assert R[0] == pytest.approx(float(c[1]), rel=1e-12)
        assert int(gs.straggler_event(R, 1.25)[0]) == int(d[0])


def test_length_stats_against_numpy_and_ratio_at_least_one():
    rng = np.random.default_rng(3)
    sizes = [1, 2, 3, 4, 7, 8, 16, 32, 5]
    off = _csr(sizes)
    ell = rng.integers(1, 16385, size=off[-1]).astype(np.int32)
    stats, ratio = gs.length_stats(ell, off)
    for g, G in enumerate(sizes):
        seg = ell[off[g]:off[g + 1]].astype(np.float64)
        assert stats[g, 0] == seg.max() and stats[g, 1] == seg.sum()
        assert stats[g, 2] == 2 * np.median(seg)
        assert ratio[g] == pytest.approx(seg.max() / seg.mean(), rel=1e-6)
        assert ratio[g] >= 1.0                                   # max >= mean
    assert np.all(gs.straggler_ratio_max_median(stats) >= 1.0)
    st, ra = gs.length_stats([9, 9, 9, 9], [0, 4])
    assert ra[0] == 1.0 and gs.straggler_ratio_max_median(st)[0] == 1.0   # equality iff all equal


def test_straggler_probability_grows_with_G():
    # larger G => more straggler events (i.i.d. lognormal lengths)
    rng = np.random.default_rng(0)
    rates = []
    for G in (4, 8, 16, 32):
        ell = np.clip(np.rint(1024 * np.exp(0.3 * rng.standard_normal(400 * G))), 1, 1 << 20)
        stats, _ = gs.length_stats(ell, np.arange(401) * G)
        rates.append(gs.straggler_event(gs.straggler_ratio_max_median(stats)).mean())
    assert rates == sorted(rates) and rates[0] < rates[-1]


def test_advantage_invariants():
    rng = np.random.default_rng(5)
    sizes = [4, 8, 16, 32, 3, 2]
    off = _csr(sizes)
    r = rng.standard_normal(off[-1]).astype(np.float32)
    adv, keep = gs.group_advantage(r, off, gs.GRPO)
    assert keep.tolist() == [1] * len(sizes)
    for g in range(len(sizes)):
        a = adv[off[g]:off[g + 1]].astype(np.float64)
        assert abs(a.sum()) < 1e-5 * len(a)
        assert a.std() == pytest.approx(1.0, abs=1e-6)
    # shift / positive-scale invariance
    adv2, _ = gs.group_advantage((3.0 * r + 2.0).astype(np.float32), off, gs.GRPO)
    assert np.allclose(adv, adv2, atol=2e-5)
    # order: larger reward -> larger advantage
    seg = slice(off[1], off[2])
    assert np.array_equal(np.argsort(r[seg], kind="stable"), np.argsort(adv[seg], kind="stable"))


def test_advantage_closed_form_bernoulli():
    for ln in golden_lines("advantage_closed_form.txt"):
        G, k, a1, a0 = ln.split()
        G, k = int(G), int(k)
        r = np.array([1.0] * k + [0.0] * (G - k), dtype=np.float32)
        adv, keep = gs.group_advantage(r, [0, G], gs.DAPO)
        assert keep[0] == 1
        assert np.allclose(adv[:k], float(a1), rtol=1e-6) and np.allclose(adv[k:], float(a0), rtol=1e-6)
        adv1, _ = gs.group_advantage(r, [0, G], gs.GRPO, ddof=1)
        assert np.allclose(adv1, adv * np.sqrt((G - 1) / G), rtol=1e-6)


def test_all_equal_groups_zero_and_dapo_drops():
    third = np.float32(1.0) / np.float32(3.0)          # mean of identical values may be off by an ulp
    r = np.array([third] * 7 + [0.0, 1.0, 1.0, 0.0] + [5.0], dtype=np.float32)
    off = [0, 7, 11, 12]
    adv, keep = gs.group_advantage(r, off, gs.DAPO)
    assert np.all(adv[:7] == 0) and adv[11] == 0
    assert keep.tolist() == [0, 1, 0]
    adv_g, keep_g = gs.group_advantage(r, off, gs.GRPO)
    assert keep_g.tolist() == [1, 1, 1] and np.array_equal(adv, adv_g)


def test_advantage_against_numpy_library_with_eps_and_ddof():
    rng = np.random.default_rng(11)
    r = rng.random(24).astype(np.float32)
    off = [0, 8, 24]
    for ddof in (0, 1):
        adv, _ = gs.group_advantage(r, off, gs.GRPO, ddof=ddof, eps=1e-4)
        for g in range(2):
            seg = r[off[g]:off[g + 1]].astype(np.float64)
            ref = (seg - seg.mean()) / (seg.std(ddof=ddof) + 1e-4)
            assert np.allclose(adv[off[g]:off[g + 1]], ref, rtol=1e-6, atol=1e-7)
