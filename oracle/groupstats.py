"""ORACLE (test infrastructure, never on the product path) -- group statistics.

Plain, slow, sequential CPU statement of what `sagc_group_advantage` and the length
statistics of `sagc_rollout_group` compute.  Shares no code with the CUDA path.

Paper passages:
  * PAPER.md l.74  (sec 3.1): "compute rewards {r_i}, and use group-relative baselines
    (e.g., mean/standardized rewards)" -> advantages A_i = (r_i - mean) / std per group.
  * PAPER.md l.114-116 (sec 4): GRPO / DAPO both "(iii) form group-relative advantages".
  * PAPER.md l.78 Eq.(1): R = max_i l_i / median_i l_i ; l.32 (Fig.1 caption) and
    BASELINE.json north_star use max / mean -> both are returned.
  * PAPER.md l.83 Eq.(2): S = 1[R > tau]; tau = 1.25 in the experiments (l.248).
Readings where the paper is silent are listed in DESIGN.md "Readings" (C4, C5).

Pins (tests/test_oracle_groupstats.py): zero-sum / unit-std invariants, the closed form for
0/1 rewards, shift/scale invariance, numpy mean/std/median as library routines, the
worked length example in tests/golden/length_stats_example.txt.
"""
from __future__ import annotations

import math
from typing import Tuple

import numpy as np

GRPO = 0
DAPO = 1


def group_advantage(rewards, group_offsets, mode: int = GRPO, ddof: int = 0, eps: float = 0.0
                    ) -> Tuple[np.ndarray, np.ndarray]:
    """Per group g = rewards[off[g]:off[g+1]] (CSR, variable G allowed):

      all_equal := (max == min) by exact comparison, or G == 1
      all_equal  -> A = 0;  keep = 0 in DAPO mode, 1 in GRPO mode
      otherwise  -> mean = sum r / G ; std = sqrt(sum (r-mean)^2 / (G - ddof))   (two pass, fp64)
                    A_i = (r_i - mean) / (std + eps) ; keep = 1
    Returns (advantages float32 [n], keep uint8 [n_groups]).
    """
    r = np.asarray(rewards, dtype=np.float32)
    off = np.asarray(group_offsets, dtype=np.int64)
    n_groups = len(off) - 1
    adv = np.zeros(r.shape[0], dtype=np.float32)
    keep = np.ones(n_groups, dtype=np.uint8)
    for g in range(n_groups):
        lo, hi = int(off[g]), int(off[g + 1])
        G = hi - lo
        if G <= 0:
            keep[g] = 0 if mode == DAPO else 1
            continue
        vals = [float(r[i]) for i in range(lo, hi)]          # exact widening to fp64
        all_equal = (max(vals) == min(vals)) or G == 1
        if all_equal or G - ddof <= 0:
            keep[g] = 0 if mode == DAPO else 1
            continue
        mean = math.fsum(vals) / G
        var = math.fsum((v - mean) * (v - mean) for v in vals) / (G - ddof)
        std = math.sqrt(var)
        for i in range(lo, hi):
            adv[i] = np.float32((float(r[i]) - mean) / (std + eps))
    return adv, keep


def length_stats(lengths, group_offsets) -> Tuple[np.ndarray, np.ndarray]:
    """Per group: (max, sum, median_x2) as int32 [n_groups][3] and ratio max/mean as float32.

    median_x2 = sum of the two middle order statistics (2*middle for odd G), so the
    median (average of the two middle values for even G) stays an exact integer.
    ratio_max_mean = float32(max*G) / float32(sum): both integers < 2^24 in every config,
    one correctly rounded fp32 division -> bit-exact on any IEEE machine.
    Empty group -> stats 0, ratio 0.
    """
    ell = np.asarray(lengths, dtype=np.int64)
    off = np.asarray(group_offsets, dtype=np.int64)
    n_groups = len(off) - 1
    stats = np.zeros((n_groups, 3), dtype=np.int32)
    ratio = np.zeros(n_groups, dtype=np.float32)
    for g in range(n_groups):
        lo, hi = int(off[g]), int(off[g + 1])
        G = hi - lo
        if G <= 0:
            continue
        s = sorted(int(v) for v in ell[lo:hi])
        mx = s[-1]
        tot = sum(s)
        med2 = s[(G - 1) // 2] + s[G // 2]
        stats[g] = (mx, tot, med2)
        ratio[g] = np.float32(mx * G) / np.float32(tot)
    return stats, ratio


def straggler_ratio_max_median(stats: np.ndarray) -> np.ndarray:
    """Eq.(1): R = max / median = 2*max / median_x2 (fp64)."""
    st = np.asarray(stats, dtype=np.float64)
    return 2.0 * st[:, 0] / st[:, 2]


def straggler_event(R, tau: float = 1.25) -> np.ndarray:
    """Eq.(2): S = 1[R > tau]."""
    return (np.asarray(R) > tau).astype(np.uint8)
