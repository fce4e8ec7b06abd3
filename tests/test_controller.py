"""SAGC controller (Alg.1 l.173-210, Eq.1-2 l.78-83, Eq.8 l.137): host logic, CPU only.

Pins: lambda >= 0; only neighbour moves; ties toward the smaller G; gamma = 1 gives the
Beta posterior counts; the Thompson draws follow scipy's Beta; the paper's worked length example; and a closed-loop
simulation on synthetic lengths whose straggler probability grows with G: the long-run straggler rate settles at delta.
"""
import math

import numpy as np
import pytest

from paper_2606_02218_b200.controller import SAGCController, run_sagc, straggler_events, straggler_ratio


def _stats(lengths, G):
    ell = np.asarray(lengths).reshape(-1, G)
    srt = np.sort(ell, axis=1)
    med2 = srt[:, (G - 1) // 2] + srt[:, G // 2]
    return np.stack([ell.max(1), ell.sum(1), med2], axis=1)


def test_worked_example_eq1():
    """tests/golden/length_stats_example.txt: lengths (100, 200, 300, 1000) -> R = 4.0, S(tau = 1.25) = 1."""
    st = _stats([100, 200, 300, 1000], 4)
    assert st.tolist() == [[1000, 1600, 500]]
    assert straggler_ratio(st)[0] == 4.0 and straggler_events(st, 1.25)[0] == 1
    assert straggler_events(_stats([100, 100, 100, 124], 4), 1.25)[0] == 0        # R = 1.24
    assert straggler_events(_stats([100, 100, 100, 125], 4), 1.25)[0] == 0        # R = 1.25 is not > tau
    assert straggler_events(_stats([100, 100, 100, 126], 4), 1.25)[0] == 1


def test_first_update_by_hand():
    c = SAGCController([4, 8, 16], delta=0.25, eta_lambda=0.5, gamma=0.9, seed=1, g0=8)
    nxt = c.update([1, 1, 0, 1])                          # S_bar = 0.75
    assert c.lam == pytest.approx(0.5 * (0.75 - 0.25))
    assert c.alpha[8] == pytest.approx(0.9 * 1 + 0.75) and c.beta[8] == pytest.approx(0.9 * 1 + 0.25)
    assert c.alpha[4] == 1.0 and c.beta[16] == 1.0        # other arms untouched
    assert nxt == 16                                      # lambda = 0.25 < log2(16/8): the utility term wins whatever p~ is
    c2 = SAGCController([4, 8, 16], g0=4)
    c2.update([0])
    assert c2.lam == 0.0                                  # projection onto lambda >= 0 (Eq.8)


def test_invariants_random_walk():
    rng = np.random.default_rng(3)
    c = SAGCController([4, 8, 16, 32], delta=0.3, eta_lambda=0.7, gamma=0.95, seed=5)
    g_prev = c.G
    for _ in range(2000):
        g = c.update(rng.integers(0, 2, size=rng.integers(1, 9)))
        assert c.lam >= 0.0
        assert abs(c.sizes.index(g) - c.sizes.index(g_prev)) <= 1           # Alg.1 l.16: neighbour moves only
        assert all(a > 0 and b > 0 for a, b in zip(c.alpha.values(), c.beta.values()))
        g_prev = g
    assert {h["G"] for h in c.history} == {4, 8, 16, 32}                     # every arm gets explored


def test_gamma_one_gives_beta_counts():
    c = SAGCController([4, 8], gamma=1.0, g0=4, seed=0)
    n = {4: [0, 0], 8: [0, 0]}
    rng = np.random.default_rng(0)
    for _ in range(300):
        s = int(rng.integers(0, 2))
        g = c.G
        c.update([s])
        n[g][0] += s; n[g][1] += 1 - s
    for g in (4, 8):
        assert c.alpha[g] == 1 + n[g][0] and c.beta[g] == 1 + n[g][1]


def test_tie_breaks_toward_smaller_G():
    class Tie(SAGCController):
        pass
    c = Tie([4, 8, 16], g0=8, seed=0)
    c.lam = 0.0
    # make every score equal: u(G) = log2 G differs, so force equality through a patched utility
    import paper_2606_02218_b200.controller as mod
    orig = mod.math.log2
    try:
        mod.math.log2 = lambda g: 1.0
        c.eta_lambda = 1e-12; c.delta = 0.5
        assert c.update([0, 1]) == 4                      # all three neighbours tie -> the smallest
    finally:
        mod.math.log2 = orig


def test_thompson_draws_follow_scipy_beta():
    stats = pytest.importorskip("scipy.stats")
    c = SAGCController([4, 8], g0=4, seed=11, gamma=1.0)
    c.alpha[4], c.beta[4] = 3.5, 1.25
    draws = np.array([c.rng.beta(c.alpha[4], c.beta[4]) for _ in range(4000)])
    assert stats.kstest(draws, stats.beta(3.5, 1.25).cdf).pvalue > 1e-3


def test_closed_loop_rate_settles_at_delta():
    """Synthetic lengths ~ lognormal(sigma): P(R > 1.25 | G) grows with G, so the constraint E[S | G] <= delta binds
    between the smallest and the largest size and the primal-dual loop must hold the long-run straggler rate at delta."""
    sizes, sigma, delta = [4, 8, 16, 32], 0.13, 0.45
    rng = np.random.default_rng(7)

    def p_of(G, n=4000):
        return float(np.mean(straggler_events(_stats(np.rint(1024 * np.exp(sigma * rng.standard_normal(n * G))), G))))
    p = {G: p_of(G) for G in sizes}
    assert p[4] < p[8] < p[16] < p[32] and p[4] < delta < p[32]      # the premise of the test

    def step(t, G, B):
        return _stats(np.rint(1024 * np.exp(sigma * rng.standard_normal(B * G))), G)
    c = SAGCController(sizes, delta=delta, eta_lambda=0.2, gamma=0.97, seed=3, g0=4)
    log = run_sagc(step, c, 6000, effective_batch=64)
    assert all(r["n_prompts"] == 64 // r["G"] for r in log)           # fixed effective batch B_t = 64 / G_t (sec 5.2)
    rate = np.mean([r["S_bar"] for r in log[2000:]])
    assert abs(rate - delta) < 0.05, (rate, p)
    # an unreachable target pins the controller at an end of the range
    c_hi = SAGCController(sizes, delta=0.999, eta_lambda=0.2, gamma=0.97, seed=3, g0=4)
    log_hi = run_sagc(step, c_hi, 600, effective_batch=64)
    assert np.mean([r["G"] == 32 for r in log_hi[200:]]) > 0.9


def test_group_fifo_assembles_groups_across_microbatches():
    """PAPER.md sec C.2-C.3 (l.433-439): completed groups queue up in FIFO order; a group delivered in pieces counts once,
    when its last completion arrives."""
    from paper_2606_02218_b200.controller import GroupFIFO
    q = GroupFIFO()
    ell, offs = q.drain()
    assert ell.shape == (0,) and offs.tolist() == [0]
    assert not q.push("a", [100, 200], 4)
    assert q.push("b", [7, 9, 8, 30], 4)                  # b completes first
    assert q.pending() == 1
    assert q.push("a", [300, 1000], 4)
    ell, offs = q.drain()
    assert offs.tolist() == [0, 4, 8] and ell.tolist() == [7, 9, 8, 30, 100, 200, 300, 1000]
    st = np.concatenate([_stats(ell[offs[g]:offs[g + 1]], 4) for g in range(2)])
    assert st.tolist() == [[30, 54, 17], [1000, 1600, 500]] and straggler_events(st).tolist() == [1, 1]
    assert q.drain()[1].tolist() == [0] and q.pending() == 0
    with pytest.raises(ValueError):
        q.push("c", [1, 2, 3], 2)
