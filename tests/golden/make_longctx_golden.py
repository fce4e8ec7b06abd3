#!/usr/bin/env python
"""Writes tests/golden/longctx_<case>.txt: ORACLE logits of teacher-forced long-context rollouts.

Imports only `oracle/` and the seeded input generators (`paper_2606_02218_b200.workloads`); nothing
here touches the CUDA path.  The GPU test (tests/test_gpu_longctx.py) runs the same teacher-forced
rollout through the C ABI (`forced_tokens`, logits dump) and compares the dumped rows with these.

Why a cache: one oracle pass over a 4 352-token sequence of the 0.5B shape, or a 2 175-token sequence
of the 7B shape, takes minutes of CPU (SURVEY.md section 8(c) "Full-size configs on a CPU": "pick the
sample once and cache oracle outputs on disk keyed by the input hashes").  A full logits row is
152 k floats, so each compared position stores the oracle's values at a fixed seeded sample of
N_IDS vocabulary ids plus its TOP_K largest entries (ids and values) as float32 bit patterns.  The
file is keyed by the SHA-256 of every input array; the test recomputes the key from its own inputs.

    python tests/golden/make_longctx_golden.py [case ...]        (minutes per case, 8 cores)
"""
from __future__ import annotations

import hashlib
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from oracle import decoder as odec            # noqa: E402
from oracle import rollout as oro             # noqa: E402
from paper_2606_02218_b200 import workloads as wl   # noqa: E402

N_IDS, TOP_K = 192, 8
HERE = os.path.dirname(os.path.abspath(__file__))

# case -> (cfg, n_prompts, P, G, max_new, forced lengths, {sid: [t, ...]})
# cfg2 (0.5B shape): 8 live rows at most (the 8-way split-K attention regime of the tail), <= 2 live beyond
# step 1150, sid 0 runs to context 256 + 4096 = 4352 (> 4096); t = 1-based generated-token index, the logits
# row of (sid, t) is computed at context P + t - 1.
CASES = {
    "cfg2": (2, 1, 256, 8, 4096, [4096, 1500, 1150, 900, 600, 300, 1100, 40],
             {0: [1, 2, 3, 64, 65, 257, 600, 1099, 1101, 1151, 1501, 2000, 2817, 3000, 3500, 3841, 3842, 4000, 4095, 4096],
              1: [1, 2, 17, 129, 300, 301, 599, 601, 700, 899, 901, 1000, 1100, 1150, 1151, 1300, 1499, 1500],
              2: [1, 2, 33, 100, 299, 400, 600, 768, 769, 900, 901, 1000, 1099, 1100, 1101, 1149, 1150],
              4: [1, 2, 5, 40, 41, 63, 64, 65, 128, 256, 299, 300, 301, 450, 599, 600]}),
    # 7B shape (configs 4 and 5 share it): one sequence to context 128 + 2048 = 2176
    "cfg5": (5, 1, 128, 2, 2048, [2048, 300],
             {0: [1, 2, 3, 64, 65, 300, 301, 302, 512, 897, 1024, 1500, 1921, 2000, 2047, 2048]}),
}


def case_inputs(name):
    cfg, n_prompts, P, G, max_new, fl, pos = CASES[name]
    w = wl.WORKLOADS[cfg]
    prompts, offs = wl.make_prompts(w, n_prompts=n_prompts, prompt_len=P)
    ftok = np.random.default_rng(7000 + cfg).integers(0, w.model.vocab, size=(n_prompts * G, max_new), dtype=np.int64).astype(np.int32)
    ids = np.sort(np.random.default_rng(7100 + cfg).choice(w.model.vocab, size=N_IDS, replace=False)).astype(np.int64)
    return w, prompts, offs, G, max_new, np.asarray(fl, dtype=np.int32), ftok, ids, pos


def input_key(w, weights_seed, prompts, offs, fl, ftok, ids, pos) -> str:
    h = hashlib.sha256()
    h.update(repr((w.cfg, w.model, weights_seed, sorted((k, tuple(v)) for k, v in pos.items()))).encode())
    for a in (prompts, offs, fl, ftok, ids):
        h.update(np.ascontiguousarray(a).tobytes())
    return h.hexdigest()


def f32_hex(a) -> str:
    return " ".join(f"{int(x):08x}" for x in np.ascontiguousarray(a, dtype=np.float32).view(np.uint32))


def main(names):
    for name in names:
        w, prompts, offs, G, max_new, fl, ftok, ids, pos = case_inputs(name)
        t0 = time.time()
        weights = wl.make_weights(w.model, 0)
        dec = odec.RefDecoder(w.model, weights, cache_f32=w.model.n_params() < 1e9)
        key = input_key(w, 0, prompts, offs, fl, ftok, ids, pos)
        lines = [f"# oracle teacher-forced logits, case {name}: written by tests/golden/make_longctx_golden.py (oracle/ only)",
                 "# reading: DESIGN.md C1; SURVEY.md 8(c) 'Full-size configs on a CPU'; PAPER.md l.74-76 (rollout of G completions)",
                 f"key {key}", "ids " + " ".join(str(int(i)) for i in ids)]
        for sid in sorted(pos):
            p = sid // G
            steps = [t for t in pos[sid] if t <= fl[sid]]
            lg = oro.teacher_forced_logits(dec, prompts[offs[p]:offs[p + 1]], ftok[sid, :fl[sid]], steps)
            for i, t in enumerate(steps):
                row = lg[i]
                top = np.argsort(-row, kind="stable")[:TOP_K]
                lines.append(f"pos {sid} {t}")
                lines.append("val " + f32_hex(row[ids]))
                lines.append("top " + " ".join(str(int(v)) for v in top))
                lines.append("tov " + f32_hex(row[top]))
            print(f"[{name}] sid {sid}: {len(steps)} positions, {time.time() - t0:.0f} s", flush=True)
        with open(os.path.join(HERE, f"longctx_{name}.txt"), "w") as f:
            f.write("\n".join(lines) + "\n")
        print(f"[{name}] done in {time.time() - t0:.0f} s", flush=True)


if __name__ == "__main__":
    main(sys.argv[1:] or list(CASES))
