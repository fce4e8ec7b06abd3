"""ORACLE (test infrastructure, never on the product path) -- paged KV bookkeeping.

Sequential statement of the page-table / free-list / retirement state machine.  The
paper is silent on the KV cache; BASELINE.json north_star requires "a paged KV cache that
stores each prompt's prefix once and shares it across its G completions, with page tables
and a free list" and "sequence retirement and batch compaction that free pages as soon as
a completion ends", bit-exact against this oracle.  Order conventions are DESIGN.md
reading C3 (any fixed order is correct; they are fixed so both sides can be compared):

  * free list = LIFO stack whose pops initially return 0, 1, 2, ...
  * prefill, prompts ascending p: pop floor(P/page) SHARED pages (logical blocks 0..),
    refcount G each; if P mod page != 0, then for g ascending pop one PRIVATE page per
    completion (the partial prompt block is copied into it).
  * decode step t >= 2 writes KV position P + t - 2; a live sequence whose position is
    the first slot of a logical block pops a page at the start of the step, ascending sid.
  * end of step t (t >= 1): every live sequence that finished retires in ascending sid:
    push its private pages in ascending logical order, then decrement the refcount of
    each shared prefix page in ascending logical order and push those that reach 0.
  * live list stays sorted by sid (stable compaction).
  * pool exhaustion -> PagePoolExhausted (no preemption).

Pins (tests/test_oracle_paging.py): conservation invariants at every step, the
closed-form peak, brute force against a naive dict-of-lists allocator.
"""
from __future__ import annotations

from typing import List, Sequence, Tuple

import numpy as np


class PagePoolExhausted(RuntimeError):
    pass


class PagedKVState:
    def __init__(self, n_pages: int, page_tokens: int, prompt_lens: Sequence[int], G: int,
                 max_blocks: int):
        self.n_pages = n_pages
        self.page = page_tokens
        self.G = G
        self.prompt_lens = [int(p) for p in prompt_lens]
        self.n_prompts = len(self.prompt_lens)
        self.nseq = self.n_prompts * G
        self.max_blocks = max_blocks
        self.free_stack = [n_pages - 1 - i for i in range(n_pages)]   # pop() -> 0,1,2,...
        self.refcnt = [0] * n_pages
        self.page_table = -np.ones((self.nseq, max_blocks), dtype=np.int32)
        self.n_blocks = [0] * self.nseq            # logical blocks currently mapped
        self.n_shared = [0] * self.nseq
        self.alloc_log: List[Tuple[int, int, int]] = []   # (step, sid, page); step 0 = prefill
        self.retire_log: List[Tuple[int, int]] = []       # (step, sid)
        self.live: List[int] = []
        self.peak_used = 0

    # -- primitive stack ops -------------------------------------------------
    def _pop(self, step: int, sid: int) -> int:
        if not self.free_stack:
            raise PagePoolExhausted(f"step {step} sid {sid}")
        pg = self.free_stack.pop()
        self.alloc_log.append((step, sid, pg))
        self.peak_used = max(self.peak_used, self.n_pages - len(self.free_stack))
        return pg

    def _push(self, pg: int) -> None:
        self.free_stack.append(pg)

    # -- protocol ------------------------------------------------------------
    def prefill(self) -> None:
        for p, P in enumerate(self.prompt_lens):
            nsh = P // self.page
            shared = []
            for b in range(nsh):
                pg = self._pop(0, p * self.G)          # logged against the group's first sid
                self.refcnt[pg] = self.G
                shared.append(pg)
            for g in range(self.G):
                sid = p * self.G + g
                self.page_table[sid, :nsh] = shared
                self.n_blocks[sid] = nsh
                self.n_shared[sid] = nsh
            if P % self.page != 0:
                for g in range(self.G):
                    sid = p * self.G + g
                    pg = self._pop(0, sid)
                    self.page_table[sid, nsh] = pg
                    self.n_blocks[sid] = nsh + 1
        self.live = list(range(self.nseq))

    def begin_step(self, t: int) -> None:
        """Start of decode step t >= 2: allocate pages for KV position P + t - 2."""
        for sid in self.live:
            pos = self.prompt_lens[sid // self.G] + t - 2
            if pos % self.page == 0:
                b = pos // self.page
                assert b == self.n_blocks[sid]
                pg = self._pop(t, sid)
                self.page_table[sid, b] = pg
                self.n_blocks[sid] = b + 1

    def end_step(self, t: int, finished: Sequence[bool]) -> None:
        """End of step t: `finished[i]` says whether live[i] retires now."""
        new_live = []
        for i, sid in enumerate(self.live):
            if not finished[i]:
                new_live.append(sid)
                continue
            for b in range(self.n_shared[sid], self.n_blocks[sid]):
                self._push(int(self.page_table[sid, b]))
            for b in range(self.n_shared[sid]):
                pg = int(self.page_table[sid, b])
                self.refcnt[pg] -= 1
                if self.refcnt[pg] == 0:
                    self._push(pg)
            self.retire_log.append((t, sid))
        self.live = new_live

    def used_pages(self) -> int:
        return self.n_pages - len(self.free_stack)


def run_structure_only(n_pages: int, page_tokens: int, prompt_lens: Sequence[int], G: int,
                       forced_lengths: Sequence[int], max_new: int, snapshot_steps=()):
    """Run the whole state machine for forced lengths without a model (it does not depend
    on token values).  Returns the final PagedKVState; `snapshots[t]` holds a copy of the
    page table and live list taken right after begin_step(t) for t in snapshot_steps."""
    forced = [int(x) for x in forced_lengths]
    max_len = max(prompt_lens) + max_new
    max_blocks = (max_len + page_tokens - 1) // page_tokens
    st = PagedKVState(n_pages, page_tokens, prompt_lens, G, max_blocks)
    st.prefill()
    snapshots = {}
    t = 1
    while st.live:
        if t >= 2:
            st.begin_step(t)
        if t in snapshot_steps:
            snapshots[t] = (st.page_table.copy(), list(st.live), st.used_pages())
        fin = [(forced[sid] == t) or (t == max_new) for sid in st.live]
        st.end_step(t, fin)
        t += 1
    return st, snapshots
