"""ORACLE (test infrastructure, never on the product path) -- Philox4x32-10 and the
Gumbel-max sampler.

The paper is silent on sampling; BASELINE.json north_star fixes "a greedy or Philox-keyed
Gumbel sampler" and "Philox draws ... must be bit-exact".  Definition (reading C2):

  Philox4x32-10 (Salmon et al., SC'11): multipliers M0 = 0xD2511F53, M1 = 0xCD9E8D57,
  Weyl key increments W0 = 0x9E3779B9, W1 = 0xBB67AE85, 10 rounds, round
     (c0,c1,c2,c3) -> (hi(M1*c2) ^ c1 ^ k0, lo(M1*c2), hi(M0*c0) ^ c3 ^ k1, lo(M0*c0)),
  key bumped by (W0, W1) between rounds.
  key     = (seed & 0xffffffff, seed >> 32)
  counter = (v >> 2, t, sid, 0);  the draw for vocab id v is output word (v & 3)
            t = 1-based index of the generated token, sid = p*G + g (never the batch slot)
  u       = ((x >> 9) + 0.5) * 2^-23          (24 significant bits: exact in fp32, strictly
            inside (0,1); SURVEY's (x>>8, 2^-24) variant needs 25 bits and is NOT fp32-exact)
  g       = -log(-log(u))                     (oracle: float64, then cast to float32)
  token   = argmax_v ( logits[v] / T + g_v ), lowest v on exact ties;  greedy: argmax logits.

Pins (tests/test_oracle_philox.py): the published Random123 known-answer vectors in
tests/golden/philox4x32_10_kat.txt; chi-square of Gumbel-max frequencies against
softmax(logits/T); T->0 reduces to greedy.
"""
from __future__ import annotations

import numpy as np

M0 = 0xD2511F53
M1 = 0xCD9E8D57
W0 = 0x9E3779B9
W1 = 0xBB67AE85
MASK = 0xFFFFFFFF


def philox4x32_10(counter, key):
    """Scalar reference: counter = 4 python ints, key = 2 python ints -> 4 ints."""
    c0, c1, c2, c3 = (int(c) & MASK for c in counter)
    k0, k1 = (int(k) & MASK for k in key)
    for _ in range(10):
        p0 = M0 * c0
        p1 = M1 * c2
        c0, c1, c2, c3 = ((p1 >> 32) ^ c1 ^ k0) & MASK, p1 & MASK, ((p0 >> 32) ^ c3 ^ k1) & MASK, p0 & MASK
        k0 = (k0 + W0) & MASK
        k1 = (k1 + W1) & MASK
    return c0, c1, c2, c3


def philox_draws(seed: int, sid: int, t: int, v0: int, n: int) -> np.ndarray:
    """uint32 draws for vocab ids v0 .. v0+n-1 of (seed, sid, t).  Vectorised over v only."""
    v = np.arange(v0, v0 + n, dtype=np.uint64)
    blk = v >> np.uint64(2)
    ublk, inv = np.unique(blk, return_inverse=True)
    c0 = ublk.astype(np.uint64)
    c1 = np.full_like(c0, np.uint64(t & MASK))
    c2 = np.full_like(c0, np.uint64(sid & MASK))
    c3 = np.zeros_like(c0)
    k0 = np.uint64(seed & MASK)
    k1 = np.uint64((seed >> 32) & MASK)
    m = np.uint64(MASK)
    for _ in range(10):
        p0 = np.uint64(M0) * c0           # < 2^64, exact in uint64
        p1 = np.uint64(M1) * c2
        n0 = ((p1 >> np.uint64(32)) ^ c1 ^ k0) & m
        n1 = p1 & m
        n2 = ((p0 >> np.uint64(32)) ^ c3 ^ k1) & m
        n3 = p0 & m
        c0, c1, c2, c3 = n0, n1, n2, n3
        k0 = (k0 + np.uint64(W0)) & m
        k1 = (k1 + np.uint64(W1)) & m
    words = np.stack([c0, c1, c2, c3], axis=1)          # [nblk][4]
    out = words[inv, (v & np.uint64(3)).astype(np.int64)]
    return out.astype(np.uint32)


def uniform_from_u32(x: np.ndarray) -> np.ndarray:
    """u = ((x >> 9) + 0.5) * 2^-23, float64 (exactly representable in fp32)."""
    return ((np.asarray(x, dtype=np.uint32) >> np.uint32(9)).astype(np.float64) + 0.5) * (2.0 ** -23)


def gumbel_from_u32(x: np.ndarray) -> np.ndarray:
    u = uniform_from_u32(x)
    return (-np.log(-np.log(u))).astype(np.float32)


def perturbed_scores(logits: np.ndarray, mode: int, temperature: float, seed: int, sid: int, t: int
                     ) -> np.ndarray:
    """Scores whose argmax is the sampled token (float32).  mode 0: greedy, 1: Gumbel."""
    lg = np.asarray(logits, dtype=np.float32)
    if mode == 0:
        return lg
    g = gumbel_from_u32(philox_draws(seed, sid, t, 0, lg.shape[0]))
    return (lg / np.float32(temperature) + g).astype(np.float32)


def sample_token(logits: np.ndarray, mode: int, temperature: float, seed: int, sid: int, t: int) -> int:
    s = perturbed_scores(logits, mode, temperature, seed, sid, t)
    return int(np.argmax(s))          # numpy argmax returns the first (lowest) index on ties


def top2_margin(scores: np.ndarray) -> float:
    s = np.asarray(scores, dtype=np.float64)
    if s.shape[0] < 2:
        return float("inf")
    part = np.partition(s, -2)
    return float(part[-1] - part[-2])
