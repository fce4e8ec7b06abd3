"""Pins for oracle/philox.py (no GPU).  KATs from tests/golden (published Random123
vectors), distributional check of Gumbel-max against softmax, T->0 reduction to greedy."""
import numpy as np

from conftest import golden_lines
from oracle import philox


def test_philox_known_answers():
    lines = golden_lines("philox4x32_10_kat.txt")
    assert len(lines) == 3
    for ln in lines:
        h = [int(x, 16) for x in ln.split()]
        assert philox.philox4x32_10(h[0:4], h[4:6]) == tuple(h[6:10])


def test_vectorised_draws_match_scalar():
    seed, sid, t = (0x9ABCDEF0 << 32) | 0x12345678, 37, 911
    d = philox.philox_draws(seed, sid, t, 5, 23)          # ragged start and end
    for i, v in enumerate(range(5, 28)):
        ref = philox.philox4x32_10((v >> 2, t, sid, 0), (seed & 0xFFFFFFFF, seed >> 32))[v & 3]
        assert int(d[i]) == ref


def test_draws_keyed_on_identity_not_slot():
    a = philox.philox_draws(7, 3, 5, 0, 64)
    assert not np.array_equal(a, philox.philox_draws(7, 4, 5, 0, 64))
    assert not np.array_equal(a, philox.philox_draws(7, 3, 6, 0, 64))
    assert not np.array_equal(a, philox.philox_draws(8, 3, 5, 0, 64))
    assert np.array_equal(a[8:24], philox.philox_draws(7, 3, 5, 8, 16))


def test_uniform_strictly_inside_unit_interval_and_fp32_exact():
    x = np.array([0, 511, 512, 0xFFFFFFFF, 0x80000000], dtype=np.uint32)
    u = philox.uniform_from_u32(x)
    assert np.all(u > 0) and np.all(u < 1)
    assert np.array_equal(u.astype(np.float32).astype(np.float64), u)
    assert u[0] == 2.0 ** -24 and u[1] == u[0] and u[2] == 3 * 2.0 ** -24 and u[3] == 1.0 - 2.0 ** -24


def test_gumbel_max_frequencies_follow_softmax():
    # chi-square of empirical token frequencies vs softmax(logits / T), V = 16 toy
    rng = np.random.default_rng(0)
    V, n, T = 16, 20000, 0.7
    logits = rng.standard_normal(V).astype(np.float32)
    p = np.exp(logits.astype(np.float64) / T)
    p /= p.sum()
    counts = np.zeros(V)
    for t in range(1, n + 1):
        counts[philox.sample_token(logits, 1, T, seed=123, sid=t % 7, t=t)] += 1
    chi2 = float(np.sum((counts - n * p) ** 2 / (n * p)))
    assert chi2 < 37.7          # chi-square 15 dof, p = 0.001


def test_gumbel_mean_is_euler_gamma():
    g = philox.gumbel_from_u32(philox.philox_draws(1, 0, 1, 0, 1 << 16)).astype(np.float64)
    assert abs(g.mean() - 0.5772156649) < 0.02
    assert abs(g.var() - np.pi ** 2 / 6) < 0.05


def test_low_temperature_reduces_to_greedy_and_ties_take_lowest_index():
    rng = np.random.default_rng(1)
    logits = rng.standard_normal(64).astype(np.float32)
    assert philox.sample_token(logits, 1, 1e-6, 5, 2, 9) == int(np.argmax(logits))
    tie = np.zeros(8, dtype=np.float32)
    tie[[3, 5]] = 2.0
    assert philox.sample_token(tie, 0, 1.0, 0, 0, 1) == 3


def test_top2_margin():
    assert philox.top2_margin(np.array([0.0, 3.0, 2.5, -1.0])) == 0.5
