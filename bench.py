#!/usr/bin/env python
"""bench.py -- rollout decode tokens/s on B200 for BASELINE.json configs[1] (the 0.5B-shaped decoder).

A "step" is one whole synchronous group rollout (prefill once per prompt, then autoregressive
decode of n_prompts*G completions until the longest finishes, then the group statistics and the
group-relative advantages) over one seeded synthetic batch.  `value` = generated tokens / time
with inputs resident in HBM; `e2e` = the same through sagc_rollout_group_host with host buffers.
See DESIGN.md "Measurement".  One JSON line on stdout (rank 0).
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2606_02218_b200 import workloads as wl  # noqa: E402

METRIC = "rollout_decode_tokens_per_s"
UNIT = "tokens/s"


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.proc = None
        self.lines = []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-i", str(self.index), "-lms", "200"], stdout=subprocess.PIPE, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except Exception:
            self.proc = None

    def _read(self):
        for ln in self.proc.stdout:
            self.lines.append(ln.strip())

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except ValueError:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


SLICE_PREFILL, SLICE_CTX, SLICE_ROWS, SLICE_STEPS = 64, 512, 8, 8


def _blas_threads():
    try:
        from threadpoolctl import threadpool_info
        nt = [p["num_threads"] for p in threadpool_info() if p.get("user_api") == "blas"]
        if nt:
            return int(max(nt))
    except Exception:
        pass
    return int(os.cpu_count() or 1)


def oracle_slice(w, weights, single_thread=False):
    """The CPU oracle, as it stands, on the slice BASELINE.md section 4 plans: one 64-token prefill (timed on its
    own), then SLICE_STEPS decode steps of SLICE_ROWS sequences whose context grows to SLICE_CTX.  The cache is set
    up by an (untimed) oracle prefill of SLICE_CTX - SLICE_STEPS tokens forked SLICE_ROWS ways.
    Returns {decode tokens/s, prefill tokens/s, threads}."""
    from oracle import decoder as odec, philox as oph
    from contextlib import nullcontext
    try:
        from threadpoolctl import threadpool_limits
        lim = threadpool_limits(limits=1) if single_thread else nullcontext()
    except Exception:
        lim = nullcontext()
    with lim:
        dec = odec.RefDecoder(w.model, weights)
        P0 = SLICE_CTX - SLICE_STEPS
        prompts, _ = wl.make_prompts(w, n_prompts=1, prompt_len=P0)
        mode = 1 if w.sampling == "gumbel" else 0
        t0 = time.perf_counter()
        dec.prefill(prompts[:SLICE_PREFILL])
        t_pf = time.perf_counter() - t0
        threads = 1 if single_thread else _blas_threads()
        lg, cache = dec.prefill(prompts)                      # untimed: brings the cache to context SLICE_CTX - SLICE_STEPS
        caches = [dec.fork_cache(cache) for _ in range(SLICE_ROWS)]
        toks = [oph.sample_token(lg, mode, w.temperature, w.philox_seed, g, 1) for g in range(SLICE_ROWS)]
        t0 = time.perf_counter()
        for t in range(2, SLICE_STEPS + 2):
            for g in range(SLICE_ROWS):
                lg = dec.step(toks[g], P0 + t - 2, caches[g])
                toks[g] = oph.sample_token(lg, mode, w.temperature, w.philox_seed, g, t)
        dt = time.perf_counter() - t0
    return {"decode_tokens_per_s": SLICE_ROWS * SLICE_STEPS / dt, "prefill_tokens_per_s": SLICE_PREFILL / t_pf, "threads": threads}


SLICE_TEXT = (f"{SLICE_PREFILL}-token prefill (timed on its own), then {SLICE_STEPS} decode steps of {SLICE_ROWS} sequences at "
              f"context {SLICE_CTX - SLICE_STEPS + 1}..{SLICE_CTX} (BASELINE.md section 4); numpy fp32 oracle")


def gpu_slice(B, make_model, w):
    """The GPU on the identical slice: 1 prompt of SLICE_CTX - SLICE_STEPS tokens, G = SLICE_ROWS, SLICE_STEPS decode steps."""
    P0 = SLICE_CTX - SLICE_STEPS
    prompts, offs = wl.make_prompts(w, n_prompts=1, prompt_len=P0)
    m = make_model(64, SLICE_ROWS, SLICE_CTX + 8)
    mode = B.MODE_GUMBEL if w.sampling == "gumbel" else B.MODE_GREEDY
    fl = np.full(SLICE_ROWS, SLICE_STEPS + 1, np.int32)
    for _ in range(3):
        out = m.rollout_group(prompts, offs, SLICE_ROWS, mode=mode, temperature=w.temperature, seed=w.philox_seed,
                              max_new_tokens=SLICE_STEPS + 1, forced_lengths=fl, timing=True)
    m.close()
    return SLICE_ROWS * SLICE_STEPS / (out.timing["decode_ms"] * 1e-3)


def run_reference(args, rank, world):
    """--impl reference: the CPU oracle on a bounded sample of the same workload (rank 0 only)."""
    if rank != 0:
        return
    w = wl.WORKLOADS[args.cfg]
    weights = wl.make_weights(w.model, 0)
    for _ in range(args.warmup and 1):
        oracle_slice(w, weights)
    t0 = time.perf_counter()
    acc = [oracle_slice(w, weights) for _ in range(max(args.steps, 1))]
    dt = time.perf_counter() - t0
    tps = float(np.mean([a["decode_tokens_per_s"] for a in acc]))
    cores, sample = acc[0]["threads"], SLICE_TEXT
    line = {"impl": "reference", "metric": METRIC, "value": tps, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * dt / max(args.steps, 1), "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f32 (bf16 weights widened)", "data": "synthetic",
            "config": {"workload": f"configs[{args.cfg - 1}] ({SHAPE_NAMES.get(args.cfg, '?')}-shaped decoder) -- bounded sample", "sample": sample},
            "cpu_baseline": {"value": tps, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": tps, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


def allreduce_max(values, device, world):
    """Max over ranks of a few scalars (the timed region of the slowest replica is the job's time)."""
    import torch
    import torch.distributed as dist
    t = torch.tensor(list(values), device=device, dtype=torch.float64)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t]


SHAPE_NAMES = {1: "tiny", 2: "0.5B", 3: "1.5B", 4: "7B", 5: "7B"}


def decode_weight_bytes(mc):
    """bf16 weight bytes one decode step reads (W)."""
    q, kv = mc.n_q_heads * mc.head_dim, mc.n_kv_heads * mc.head_dim
    return 2 * (mc.n_layers * (mc.d_model * q + 2 * mc.d_model * kv + q * mc.d_model + 3 * mc.d_model * mc.d_ff) + mc.vocab * mc.d_model)


BF16_SUSTAINED_TFLOPS_FALLBACK = 1400.0


def measured_bf16_sustained():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            return float(json.load(f).get("bf16_tflops_sustained", BF16_SUSTAINED_TFLOPS_FALLBACK))
    return BF16_SUSTAINED_TFLOPS_FALLBACK


def pool_pages(w, fl, max_new):
    """KV pool size: worst case (every completion at the cap) if it fits ~100 GB, else sized for the drawn lengths."""
    mc, page = w.model, w.model.page_tokens
    n_pages = w.n_prompts * (w.prompt_len // page + w.G * ((max_new + page - 1) // page + 1)) + 8
    if n_pages * page * 2 * mc.n_layers * mc.n_kv_heads * mc.head_dim * 2 > 100e9:
        n_pages = int(np.sum((fl + page - 1) // page + 2)) + w.n_prompts * (w.prompt_len // page + 1) + 8
    return n_pages


def phase_table(acc, n_rollouts, peak, mc=None, tf_sustained=None):
    """Per-phase numbers from the accumulated sagc_rollout_timing fields."""
    names = ["full", "mid", "tail"]
    out = {}
    for p in range(3):
        if not acc["ph_steps"][p]:
            continue
        ms_step = acc["ph_ms"][p] / acc["ph_steps"][p]
        gbs = acc["ph_bytes"][p] / acc["ph_ms"][p] / 1e6
        row = {"decode_steps": acc["ph_steps"][p] // n_rollouts, "avg_live_rows": acc["ph_tok"][p] / acc["ph_steps"][p],
               "tokens_per_s": acc["ph_tok"][p] / acc["ph_ms"][p] * 1e3, "ms_per_decode_step": ms_step, "achieved_gbs": gbs,
               "frac_of_measured": gbs / peak, "frac_of_8tbs": gbs / 8000.0}
        if mc is not None and tf_sustained:
            # two-term roofline: the projections are tensor-bound once the hi/lo MMA work (2 passes x 2 flop per
            # weight and row) outweighs streaming the weights; the KV scan is HBM-bound either way
            Wb = decode_weight_bytes(mc)
            bytes_step = acc["ph_bytes"][p] / acc["ph_steps"][p]
            t_w = Wb / (peak * 1e9)
            t_mma = 2.0 * 2.0 * (Wb / 2.0) * row["avg_live_rows"] / (tf_sustained * 1e12)
            t_two = max(t_w, t_mma) + (bytes_step - Wb) / (peak * 1e9)
            row["two_term_roofline_ms"] = t_two * 1e3
            row["frac_of_two_term"] = t_two * 1e3 / ms_step
            row["bound"] = "tensor" if t_mma > t_w else "hbm"
        out[names[p]] = row
    return out


def accumulate(acc, t):
    acc["tokens"] += t["total_tokens"]; acc["launches"] += t["kernel_launches"] + 1
    acc["prefill_ms"] += t["prefill_ms"]; acc["prefill_flops"] += t["prefill_flops"]; acc["decode_ms"] += t["decode_ms"]
    for p in range(3):
        acc["ph_ms"][p] += t["phase_ms"][p]; acc["ph_bytes"][p] += t["phase_bytes"][p]
        acc["ph_tok"][p] += t["phase_tokens"][p]; acc["ph_steps"][p] += t["phase_steps"][p]


def new_acc():
    return {"tokens": 0, "launches": 0, "ph_ms": [0.0] * 3, "ph_bytes": [0.0] * 3, "ph_tok": [0] * 3, "ph_steps": [0] * 3,
            "prefill_ms": 0.0, "prefill_flops": 0.0, "decode_ms": 0.0}


# dram__bytes_read.sum + dram__bytes_write.sum of ONE decode step (the sum over the step's kernels, <= 8 live rows) from the
# `ncu --set full` captures in profiles/r02_ncu_top_kernels.md, by config: within 2 % of the step's algorithmic bytes
NCU_TRAFFIC = {2: 1.045e9, 4: 1.448e10, 5: 1.448e10}


def kernel_parts(model, B, w, d_prompts, offs, fl, max_new, mode, peak):
    """The three parts of a decode step timed alone with CUDA events on the launching stream (SAGC_FLAG_TIME_KERNELS: direct
    launches instead of graphs, four events per step): layer stack (the persistent decode-step kernel while <= 64 rows are
    live), LM head + sampler, advance.  Algorithmic bytes of a part = the weights it streams (+ the KV scan for the layer stack)."""
    mc = w.model
    out = model.rollout_group(d_prompts, offs, w.G, mode=mode, temperature=w.temperature, seed=w.philox_seed,
                              max_new_tokens=max_new, forced_lengths=fl, timing=True, flags=B.FLAG_TIME_KERNELS)
    t = out.timing
    steps = max(t["kernel_steps"], 1)
    W = decode_weight_bytes(mc)
    W_lm = 2 * mc.vocab * mc.d_model
    bytes_all = sum(t["phase_bytes"])
    ms = t["kernel_ms"]
    parts = {}
    for name, k, nbytes in (("layer_stack", 0, bytes_all - steps * W_lm), ("lm_head_sampler", 1, steps * W_lm), ("advance", 2, 0.0)):
        parts[name] = {"ms_per_step": ms[k] / steps, "share_of_step": ms[k] / max(sum(ms), 1e-9), "bytes_per_step": nbytes / steps,
                       "achieved_gbs": nbytes / ms[k] / 1e6 if ms[k] > 0 else None,
                       "frac": nbytes / ms[k] / 1e6 / peak if ms[k] > 0 else None}
    parts["layer_stack"]["kernel"] = ("k_decode_step (persistent, one launch per step) while <= 64 rows are live; per-layer k_linear_tc / k_attention above"
                                      if os.environ.get("SAGC_STEP", "0") not in ("", "0") else
                                      "per layer: k_linear_tc<QKV>, k_attention (RoPE + KV append fused), k_linear_tc<O+resid>, k_linear_tc<gate/up SwiGLU>, k_linear_tc<down+resid>")
    parts["lm_head_sampler"]["kernel"] = "k_lmhead_sample (fused, <= 64 rows) / k_linear_tc + k_sample above"
    parts["advance"]["kernel"] = "k_advance"
    parts["steps_measured"] = steps
    parts["note"] = "direct launches (no CUDA graph) so that events can bracket each part; shares, not absolutes, carry over to the graph run"
    return parts


def side_7b(B, torch, peak, tf_sustained, device):
    """configs[4] (7B shape, 8 prompts x 1024 x G=32, Pareto lengths capped at 16384) once, after one warm-up rollout."""
    w = wl.WORKLOADS[5]
    mc = w.model
    weights = wl.make_weights(mc, 0)
    prompts, offs = wl.make_prompts(w)
    fl = np.minimum(wl.make_forced_lengths(w), w.max_new).astype(np.int32)
    model = B.Model(mc, weights, pool_pages(w, fl, w.max_new), w.n_prompts * w.G, w.prompt_len + w.max_new, device=device)
    del weights
    d_prompts = torch.from_numpy(prompts).cuda()
    mode = B.MODE_GUMBEL
    acc = new_acc()
    for it in range(2):
        out = model.rollout_group(d_prompts, offs, w.G, mode=mode, temperature=w.temperature, seed=w.philox_seed,
                                  max_new_tokens=w.max_new, forced_lengths=fl, timing=True)
    accumulate(acc, out.timing)
    model.close()
    dec_bytes, dec_ms = sum(acc["ph_bytes"]), sum(acc["ph_ms"])
    return {"workload": "configs[4]: 7B-shaped decoder, 8 prompts x 1024 tokens x G=32, forced lengths pareto(512, 1.5) cap 16384, Gumbel T=1 Philox",
            "rollouts": "1 warm-up + 1 timed", "tokens": acc["tokens"], "tokens_per_s": acc["tokens"] / (out.timing["prefill_ms"] + out.timing["decode_ms"]) * 1e3,
            "decode_achieved_gbs": dec_bytes / dec_ms / 1e6, "decode_frac_of_measured": dec_bytes / dec_ms / 1e6 / peak,
            "decode_frac_of_8tbs": dec_bytes / dec_ms / 1e6 / 8000.0,
            "phases": phase_table(acc, 1, peak, mc, tf_sustained),
            "prefill": {"ms": acc["prefill_ms"], "tflops_model": acc["prefill_flops"] / acc["prefill_ms"] / 1e9 if acc["prefill_ms"] else None},
            "targets": {"full_frac_of_8tbs": 0.70, "tail_frac_of_8tbs": 0.60}}


def run_fixed_eb(args, local):
    """--protocol fixed-eb (sec 5.2 l.216-218, Table 5 l.398-405): the paper compares group
    sizes at a FIXED effective generation batch, B_t = EB / G_t prompts per step (EB = 64).  Each static G in {4, 8, 16, 32}
    and the SAGC controller (paper_2606_02218_b200.controller) run `--eb-steps` rollout steps on the configs[1] model with
    fresh seeded lognormal lengths per step (the paper's lengths come from the evolving policy: these stand in for them).
    Reports time per step, tokens/s and the straggler rate P(max / median > 1.25) per arm: the shape of the paper's
    time-vs-G trade-off, context only."""
    import torch
    from paper_2606_02218_b200 import binding as B
    from paper_2606_02218_b200.controller import SAGCController, run_sagc, straggler_events
    torch.cuda.set_device(local)
    w = wl.WORKLOADS[2]
    mc = w.model
    EB, P, max_new, med, sigma = 64, 256, 1024, 256.0, 0.35
    weights = wl.make_weights(mc, 0)
    page = mc.page_tokens
    model = B.Model(mc, weights, EB // 4 * (P // page) + EB * ((max_new + page - 1) // page + 2) + 8, EB, P + max_new, device=f"cuda:{local}")
    del weights
    prompts, _ = wl.make_prompts(w, n_prompts=EB // 4, prompt_len=P)
    d_prompts = torch.from_numpy(prompts).cuda()
    rng = np.random.default_rng(6000)

    def make_step(acc):
        def step(t, G, n_prompts):
            fl = np.clip(np.rint(med * np.exp(sigma * rng.standard_normal(n_prompts * G))), 1, max_new).astype(np.int32)
            offs = (np.arange(n_prompts + 1) * P).astype(np.int32)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            out = model.rollout_group(d_prompts[: n_prompts * P], offs, G, mode=B.MODE_GUMBEL, temperature=1.0, seed=7000 + t,
                                      max_new_tokens=max_new, forced_lengths=fl)
            e1.record()
            torch.cuda.synchronize()
            st = out.len_stats.cpu().numpy()
            acc.append({"G": G, "ms": e0.elapsed_time(e1), "tokens": int(fl.sum()), "S": float(straggler_events(st).mean())})
            return st
        return step

    rows = []
    for G in (4, 8, 16, 32):
        acc = []
        step = make_step(acc)
        for t in range(args.eb_steps + 1):
            step(t, G, EB // G)
        acc = acc[1:]                                    # first step builds the graphs
        rows.append({"arm": f"static G={G}", "prompts_per_step": EB // G, "ms_per_step": float(np.mean([a["ms"] for a in acc])),
                     "tokens_per_s": sum(a["tokens"] for a in acc) / sum(a["ms"] for a in acc) * 1e3,
                     "straggler_rate": float(np.mean([a["S"] for a in acc]))})
    acc = []
    ctrl = SAGCController([4, 8, 16, 32], delta=0.5, eta_lambda=0.5, gamma=0.9, seed=1, g0=8)
    run_sagc(make_step(acc), ctrl, 4 * args.eb_steps, effective_batch=EB)
    rows.append({"arm": "SAGC (delta=0.5, eta=0.5, gamma=0.9)", "ms_per_step": float(np.mean([a["ms"] for a in acc])),
                 "tokens_per_s": sum(a["tokens"] for a in acc) / sum(a["ms"] for a in acc) * 1e3,
                 "straggler_rate": float(np.mean([a["S"] for a in acc])), "G_trajectory": [a["G"] for a in acc],
                 "mean_G": float(np.mean([a["G"] for a in acc]))})
    model.close()
    print(json.dumps({"protocol": "fixed_effective_batch", "effective_batch": EB, "metric": METRIC, "unit": UNIT, "data": "synthetic",
                      "config": {"workload": f"configs[1] model (0.5B shape), {P}-token prompts, B_t = {EB}/G_t prompts per step, lengths "
                                             f"lognormal({med:g}, {sigma:g}) cap {max_new} redrawn every step"}, "arms": rows}), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--cfg", type=int, default=2)
    ap.add_argument("--max-new", type=int, default=0, help="override max_new_tokens (debug; invalidates the number)")
    ap.add_argument("--n-prompts", type=int, default=0, help="override the number of prompts (profiling windows; invalidates the number)")
    ap.add_argument("--g", type=int, default=0, help="override the group size G (profiling windows; invalidates the number)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-side-7b", action="store_true", help="skip the configs[4] (7B shape) side block (~5 minutes)")
    ap.add_argument("--protocol", default="rollout", choices=["rollout", "fixed-eb"],
                    help="fixed-eb: the paper's fixed-effective-batch comparison of group sizes (side mode, own JSON line)")
    ap.add_argument("--eb-steps", type=int, default=6)
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        return run_reference(args, rank, world)
    if args.protocol == "fixed-eb":
        return run_fixed_eb(args, local) if rank == 0 else None

    import torch
    import torch.distributed as dist
    from paper_2606_02218_b200 import binding as B
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the rollout path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    B.lib()

    w = wl.WORKLOADS[args.cfg]
    if args.n_prompts or args.g:
        w = wl.tiny_variant(args.cfg, n_prompts=args.n_prompts or w.n_prompts, G=args.g or w.G)
    mc = w.model
    max_new = args.max_new or w.max_new
    weights = wl.make_weights(mc, 0)
    prompts, offs = wl.make_prompts(w)
    fl = np.minimum(wl.make_forced_lengths(w), max_new).astype(np.int32)
    rewards, goffs = wl.make_rewards(w)
    nseq = w.n_prompts * w.G
    model = B.Model(mc, weights, pool_pages(w, fl, max_new), nseq, w.prompt_len + max_new, device=f"cuda:{local}")
    mode = B.MODE_GUMBEL if w.sampling == "gumbel" else B.MODE_GREEDY
    adv_mode = B.ADV_DAPO if w.adv_mode == "DAPO" else B.ADV_GRPO
    d_prompts = torch.from_numpy(prompts).cuda()
    d_rewards, d_goffs = torch.from_numpy(rewards).cuda(), torch.from_numpy(goffs).cuda()
    stream = torch.cuda.Stream()
    peak, peak_src = measured_peaks()
    tf_sus = measured_bf16_sustained()

    def step(host=False, timing=True):
        out = model.rollout_group(prompts if host else d_prompts, offs, w.G, mode=mode, temperature=w.temperature,
                                  seed=w.philox_seed, max_new_tokens=max_new, forced_lengths=fl, timing=timing, host=host)
        adv, keep = B.group_advantage(d_rewards, d_goffs, adv_mode)
        return out, adv, keep

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    with torch.cuda.stream(stream):
        for _ in range(max(args.warmup, 3)):
            step()
        barrier()
        sampler = ClockSampler(local)
        sampler.start()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        acc = new_acc()
        e0.record()
        for _ in range(args.steps):
            out, adv, keep = step()
            accumulate(acc, out.timing)
        e1.record()
        barrier()
        clocks = sampler.stop()
        ms = e0.elapsed_time(e1)
        # end to end through the host-buffer entry point (H2D prompts, D2H tokens/lengths/stats inside)
        barrier()
        t0 = time.perf_counter()
        e2e_tok = 0
        for _ in range(args.steps):
            out_h, _, _ = step(host=True, timing=False)
            e2e_tok += int(out_h.lengths.sum())
        torch.cuda.synchronize()
        e2e_s = time.perf_counter() - t0
        parts = kernel_parts(model, B, w, d_prompts, offs, fl, max_new, mode, peak) if rank == 0 else None
        gpu_slice_tps = None
        if rank == 0 and not args.no_cpu_baseline:
            gpu_slice_tps = gpu_slice(B, lambda n_pages, max_seqs, max_ctx: B.Model(mc, weights, n_pages, max_seqs, max_ctx, device=f"cuda:{local}"), w)

    ms, e2e_ms = allreduce_max([ms, e2e_s * 1e3], "cuda", world)
    model.close()
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    dec_bytes = sum(acc["ph_bytes"]); dec_ms = sum(acc["ph_ms"])
    achieved = dec_bytes / dec_ms / 1e6
    ls = parts["layer_stack"]
    line = {"metric": METRIC, "value": world * acc["tokens"] / ms * 1e3, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "bf16", "data": "synthetic",
            "config": {"workload": f"configs[{args.cfg - 1}]: {SHAPE_NAMES.get(args.cfg, '?')}-shaped decoder, {w.n_prompts} prompts x {w.prompt_len} tokens x G={w.G}, "
                                   f"forced lengths {w.length_kind}({w.length_scale:g}, {w.length_shape:g}) cap {max_new}, "
                                   f"{'Gumbel T=%g Philox' % w.temperature if w.sampling == 'gumbel' else 'greedy'}",
                       "tokens_per_step": acc["tokens"] // args.steps,
                       "precision": "bf16 weights and KV cache, activations carried as hi+lo bf16 pairs (~16 mantissa bits), fp32 accumulate", "l2": "weights %.2f GB per decode step > 126 MB L2" % (decode_weight_bytes(mc) / 1e9),
                       "replicas": world},
            "clocks": clocks, "gpu_launches": acc["launches"],
            "e2e": {"value": world * e2e_tok / e2e_ms * 1e3, "unit": UNIT, "h2d_bytes_per_step": int(prompts.nbytes + fl.nbytes),
                    "d2h_bytes_per_step": int(nseq * max_new * 4 + nseq * 4 + w.n_prompts * 16)},
            # Headline roofline = EVERY kernel of every decode step of the timed rollouts (CUDA-graph launches of the step's
            # kernel chain), not the best part of it: algorithmic bytes of all decode steps / device time of all decode steps.
            "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                         "traffic": NCU_TRAFFIC.get(args.cfg), "peak_source": peak_src,
                         "kernel": "one decode step = " + ls["kernel"] + "; then LM head + sampler, advance",
                         "what": "all decode steps of the timed rollouts: algorithmic bytes (layer + LM-head weights once per step + prefix KV once "
                                 "per live group + suffix KV + KV written) / device time between the step-boundary events of the rollout stream",
                         "frac_of_8tbs": achieved / 8000.0},
            # the layer stack of the step timed alone (direct launches bracketed by events, SAGC_FLAG_TIME_KERNELS), with its
            # share of the step; in_graph_estimate = the same bytes over the layer stack's share of the graph-run step time
            "roofline_layer_stack": {"achieved": ls["achieved_gbs"], "frac": ls["frac"], "share_of_decode_step": ls["share_of_step"],
                                     "kernel": ls["kernel"], "bytes_per_step": ls["bytes_per_step"],
                                     "in_graph_estimate_gbs": (ls["bytes_per_step"] * parts["steps_measured"]) / max(ls["share_of_step"] * dec_ms / args.steps, 1e-9) / 1e6},
            "phases": phase_table(acc, args.steps, peak, mc, tf_sus), "kernel_roofline": parts,
            "prefill": {"ms": acc["prefill_ms"] / args.steps, "tflops": acc["prefill_flops"] / acc["prefill_ms"] / 1e9 if acc["prefill_ms"] else None}}
    if not args.no_cpu_baseline:
        multi = oracle_slice(w, weights)
        single = oracle_slice(w, weights, single_thread=True)
        line["cpu_baseline"] = {"value": multi["decode_tokens_per_s"], "unit": UNIT, "cores": multi["threads"], "kind": "oracle",
                                "sample": SLICE_TEXT, "single_thread_value": single["decode_tokens_per_s"],
                                "prefill_tokens_per_s": multi["prefill_tokens_per_s"], "gpu_same_slice_tokens_per_s": gpu_slice_tps}
    del weights
    if not args.no_side_7b and args.cfg == 2 and world == 1:
        try:
            line["side_7b"] = side_7b(B, torch, peak, tf_sus, f"cuda:{local}")
        except Exception as e:                                   # the side block must never cost the headline line
            line["side_7b"] = {"error": repr(e)}
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
