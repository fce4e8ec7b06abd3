"""SAGC -- Straggler-Aware Group-Size Control (Alg.1, l.173-210; Eq.1-2 l.78-83; Eq.6-8 l.126-139; sec 4.3
l.145-147): the CPU-side controller that picks the GRPO/DAPO group size G for the next rollout step from the length
summaries the GPU returns.  A few lines of host code that call the library; every GPU step is `Model.rollout_group`.

Readings (C6; the paper leaves them open, l.443):
  * R = max / median per group with the even-G median = mean of the two middle lengths: R = 2 max / median_x2 from the
    integer triple `rollout_group` returns (Eq.1); S = [R > tau], tau = 1.25 (l.248).
  * Alg.1 l.9-11: ONE pseudo-observation per step, the empirical straggler rate S_bar over the step's groups:
    lambda <- max(0, lambda + eta (S_bar - delta));  alpha_G <- gamma alpha_G + S_bar;  beta_G <- gamma beta_G + (1 - S_bar)
    (with gamma = 1 and S_bar in {0, 1} these are the Beta posterior counts).
  * l.12-17: Thompson sample p~_G ~ Beta(alpha_G, beta_G) for EVERY G, score U~(G) = log2 G - lambda p~_G, move to the
    arg-max over the neighbourhood {prev(G), G, next(G)}, ties toward the smaller G.
  * delta, eta_lambda, gamma are not given by the paper: defaults delta = 0.25, eta_lambda = 0.5, gamma = 0.9.
  * fixed effective batch (sec 5.2 l.216-218, Table 5): B_t = EB / G_t prompts per step, EB = 64.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field
from typing import Callable, List, Optional, Sequence

import numpy as np


def straggler_ratio(len_stats: np.ndarray) -> np.ndarray:
    """R = max / median per group (Eq.1) from the int32 [n_groups][3] = (max, sum, median_x2) triple."""
    st = np.asarray(len_stats, dtype=np.float64)
    return 2.0 * st[:, 0] / st[:, 2]


def straggler_events(len_stats: np.ndarray, tau: float = 1.25) -> np.ndarray:
    """S = [R > tau] per group (Eq.2)."""
    return (straggler_ratio(len_stats) > tau).astype(np.int32)


@dataclass
class SAGCController:
    sizes: Sequence[int]                       # allowed group sizes, sorted ascending (Alg.1 "Require")
    delta: float = 0.25                        # target straggler rate
    tau: float = 1.25                          # straggler threshold on R
    eta_lambda: float = 0.5                    # dual step size
    gamma: float = 0.9                         # forgetting factor in (0, 1]
    seed: int = 0
    g0: Optional[int] = None                   # initial group size (Alg.1: random)
    lam: float = field(default=0.0, init=False)
    history: List[dict] = field(default_factory=list, init=False)

    def __post_init__(self):
        self.sizes = sorted(int(g) for g in self.sizes)
        if len(set(self.sizes)) != len(self.sizes) or not self.sizes:
            raise ValueError("sizes must be distinct and non-empty")
        if not (0.0 < self.gamma <= 1.0) or not (0.0 < self.delta < 1.0) or self.eta_lambda <= 0 or self.tau <= 1.0:
            raise ValueError("need gamma in (0,1], delta in (0,1), eta_lambda > 0, tau > 1")
        self.rng = np.random.default_rng(self.seed)
        self.alpha = {g: 1.0 for g in self.sizes}                # Alg.1 l.2-4
        self.beta = {g: 1.0 for g in self.sizes}
        self.G = int(self.g0) if self.g0 is not None else int(self.rng.choice(self.sizes))
        if self.G not in self.alpha:
            raise ValueError("g0 must be one of sizes")

    def neighbourhood(self, G: int) -> List[int]:
        i = self.sizes.index(G)
        return self.sizes[max(0, i - 1): i + 2]                 # Alg.1 l.16

    def update(self, S: Sequence[int]) -> int:
        """Alg.1 l.9-17 for one finished rollout step run at self.G; S = the straggler event of each completed group.
        Returns the group size of the next step."""
        s_bar = float(np.mean(S))                                                    # l.9
        self.lam = max(0.0, self.lam + self.eta_lambda * (s_bar - self.delta))      # l.10 (Eq.8)
        G = self.G
        self.alpha[G] = self.gamma * self.alpha[G] + s_bar                          # l.11
        self.beta[G] = self.gamma * self.beta[G] + (1.0 - s_bar)
        p = {g: float(self.rng.beta(self.alpha[g], self.beta[g])) for g in self.sizes}   # l.12-13
        score = {g: math.log2(g) - self.lam * p[g] for g in self.sizes}             # l.14 (Eq.6)
        best = None
        for g in self.neighbourhood(G):                                             # l.16-17, ascending: ties -> smaller G
            if best is None or score[g] > score[best]:
                best = g
        self.history.append({"G": G, "S_bar": s_bar, "lambda": self.lam, "next_G": best})
        self.G = best
        return best


def run_sagc(rollout_step: Callable[[int, int, int], np.ndarray], controller: SAGCController, n_steps: int,
             effective_batch: Optional[int] = 64, n_prompts: Optional[int] = None) -> List[dict]:
    """The control loop of Fig.3 / Alg.1 l.6-18.  `rollout_step(step, G, n_prompts)` runs one synchronous group rollout
    (normally `Model.rollout_group`) and returns its `len_stats` as a host int array [n_prompts][3].
    With `effective_batch` the number of prompts per step is B_t = effective_batch // G_t (sec 5.2); otherwise `n_prompts`."""
    log = []
    for t in range(n_steps):
        G = controller.G
        B = max(1, effective_batch // G) if effective_batch else int(n_prompts)
        stats = np.asarray(rollout_step(t, G, B))
        S = straggler_events(stats, controller.tau)
        R = straggler_ratio(stats)
        nxt = controller.update(S)
        log.append({"step": t, "G": G, "n_prompts": B, "R_mean": float(R.mean()), "S_bar": float(S.mean()),
                    "lambda": controller.lam, "next_G": nxt})
    return log


class GroupFIFO:
    """FIFO of completed groups between generation and the controller (PAPER.md sec C.2 l.433-435: "it drains a FIFO
    queue of recently completed groups (token-length vectors)"; sec C.3 l.439: "groups can be assembled across
    microbatches until the expected group size is reached, then emitted as a single observation").
    `push(prompt_id, lengths, expected)` may deliver a group's completions in several pieces (micro-batches); a group
    enters the queue once `expected` lengths have arrived.  `drain()` returns the token-length vectors of the groups
    completed since the last drain, in completion order, as (lengths int32 concatenated, CSR offsets int32) -- the
    input of `sagc_length_stats`; `drain_stats()` runs that kernel and returns the (max, sum, median_x2) triples."""

    def __init__(self):
        self._partial = {}
        self._ready: List[np.ndarray] = []

    def push(self, prompt_id, lengths: Sequence[int], expected: int) -> bool:
        buf = self._partial.setdefault(prompt_id, [])
        buf.extend(int(x) for x in lengths)
        if len(buf) > expected:
            raise ValueError(f"group {prompt_id}: {len(buf)} completions delivered, {expected} expected")
        if len(buf) < expected:
            return False
        self._ready.append(np.asarray(self._partial.pop(prompt_id), dtype=np.int32))
        return True

    def pending(self) -> int:
        return len(self._partial)

    def drain(self):
        groups, self._ready = self._ready, []
        offs = np.concatenate([[0], np.cumsum([g.shape[0] for g in groups])]).astype(np.int32)
        ell = np.concatenate(groups).astype(np.int32) if groups else np.zeros(0, dtype=np.int32)
        return ell, offs

    def drain_stats(self, device: str = "cuda:0") -> np.ndarray:
        """(max, sum, median_x2) per drained group through the library's segmented kernel (step a14)."""
        import torch
        from . import binding
        ell, offs = self.drain()
        if offs.shape[0] == 1:
            return np.zeros((0, 3), dtype=np.int32)
        st, _ = binding.length_stats(torch.from_numpy(ell).to(device), torch.from_numpy(offs).to(device))
        return st.cpu().numpy()
