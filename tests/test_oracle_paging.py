"""Pins for oracle/paging.py (no GPU): conservation invariants at every step, the
closed-form peak, brute force against a naive dict-of-lists allocator, ragged prompts."""
import numpy as np
import pytest

from oracle import paging


def _check_invariants(st: paging.PagedKVState, t: int):
    owned = {}
    for sid in st.live:
        for b in range(st.n_blocks[sid]):
            pg = int(st.page_table[sid, b])
            assert pg >= 0
            shared = b < st.n_shared[sid]
            owned.setdefault(pg, []).append((sid, shared))
    free = set(st.free_stack)
    assert len(free) == len(st.free_stack)                       # no page twice on the stack
    assert not (free & set(owned))                               # free and owned are disjoint
    assert len(free) + len(owned) == st.n_pages                  # conservation
    for pg, users in owned.items():
        if users[0][1]:                                          # shared prefix page
            grp = {sid // st.G for sid, _ in users}
            assert len(grp) == 1 and all(s for _, s in users)
            assert st.refcnt[pg] == len(users)                   # refcount == live seqs of the prompt
        else:
            assert len(users) == 1                               # private page owned once


def _run(n_pages, page, prompt_lens, G, forced, max_new):
    max_blocks = (max(prompt_lens) + max_new + page - 1) // page
    st = paging.PagedKVState(n_pages, page, prompt_lens, G, max_blocks)
    st.prefill()
    _check_invariants(st, 0)
    t, used = 1, []
    while st.live:
        if t >= 2:
            st.begin_step(t)
        _check_invariants(st, t)
        used.append(st.used_pages())
        st.end_step(t, [forced[s] == t or t == max_new for s in st.live])
        assert st.live == sorted(st.live)
        t += 1
    return st, used


@pytest.mark.parametrize("prompt_lens,G,page", [([32], 4, 16), ([37, 5, 16], 3, 16), ([64, 100], 8, 32)])
def test_invariants_and_closed_form_peak(prompt_lens, G, page):
    rng = np.random.default_rng(sum(prompt_lens))
    nseq, max_new = len(prompt_lens) * G, 90
    forced = rng.integers(1, max_new + 20, size=nseq)
    st, used = _run(4096, page, prompt_lens, G, forced, max_new)
    assert sorted(st.free_stack) == list(range(4096))            # everything returned at the end
    ell = np.minimum(forced, max_new)
    # closed form: pages in use during step t (after begin_step, before retirement)
    for t, u in enumerate(used, start=1):
        tot = 0
        for p, P in enumerate(prompt_lens):
            livep = [s for s in range(p * G, (p + 1) * G) if ell[s] >= t]
            if livep:
                tot += P // page
            # private blocks cover KV positions [floor(P/page)*page, P + t - 2]
            npos = (P % page) + (t - 1)
            tot += len(livep) * (-(-npos // page))
        assert u == tot
    assert st.peak_used == max(used)
    assert [s for _, s in st.retire_log] != [] and len(st.retire_log) == nseq
    assert [x[0] for x in st.retire_log] == sorted(x[0] for x in st.retire_log)


def test_brute_force_naive_allocator():
    """Replay with a naive allocator (dict of lists, sorted free list popped by recorded
    LIFO order) and compare every page id handed out."""
    rng = np.random.default_rng(9)
    prompt_lens, G, page, max_new = [20, 33], 4, 8, 40
    forced = rng.integers(1, 45, size=8)
    st, _ = _run(64, page, prompt_lens, G, forced, max_new)
    # naive model: free list as python list used as a stack, ownership as dict sid -> [pages]
    free = list(range(63, -1, -1))
    own, shared, ref, log = {}, {}, {}, []
    for p, P in enumerate(prompt_lens):
        shared[p] = [free.pop() for _ in range(P // page)]
        for pg in shared[p]:
            ref[pg] = G
            log.append((0, p * G, pg))
        for g in range(G):
            own[p * G + g] = []
        if P % page:
            for g in range(G):
                pg = free.pop()
                own[p * G + g].append(pg)
                log.append((0, p * G + g, pg))
    live = list(range(8))
    t = 1
    while live:
        if t >= 2:
            for s in live:
                pos = prompt_lens[s // G] + t - 2
                if pos % page == 0:
                    pg = free.pop()
                    own[s].append(pg)
                    log.append((t, s, pg))
        nxt = []
        for s in live:
            if forced[s] == t or t == max_new:
                free.extend(own.pop(s))
                for pg in shared[s // G]:
                    ref[pg] -= 1
                    if ref[pg] == 0:
                        free.append(pg)
            else:
                nxt.append(s)
        live = nxt
        t += 1
    assert log == st.alloc_log
    assert free == st.free_stack


def test_forced_length_one_and_exhaustion():
    st, _ = _run(16, 16, [32], 4, [1, 1, 1, 1], 8)
    assert st.retire_log == [(1, 0), (1, 1), (1, 2), (1, 3)]
    assert len(st.alloc_log) == 2                                # only the two shared prefix pages
    with pytest.raises(paging.PagePoolExhausted):
        _run(3, 16, [32], 4, [40] * 4, 64)


def test_run_structure_only_matches_manual_loop():
    forced = [3, 17, 9, 30]
    st, snaps = paging.run_structure_only(64, 16, [32], 4, forced, 24, snapshot_steps=(2, 17))
    assert [s for _, s in st.retire_log] == [0, 2, 1, 3]
    assert [t for t, _ in st.retire_log] == [3, 9, 17, 24]       # last one capped by max_new
    table, live, used = snaps[17]
    assert live == [1, 3] and used == 2 + 2 * 1                  # 2 shared + one private page each
    assert table[1, 2] >= 0 and table[0, 2] == st.page_table[0, 2]
