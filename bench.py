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


def oracle_sample(w, weights, n_steps=1):
    """The CPU oracle, as it stands, on a bounded slice of the same workload: 1 prompt of 64 tokens,
    G = 8 completions, 8 generated tokens each (64 tokens/step).  Returns (tokens/s, cores, text)."""
    from oracle import decoder as odec, rollout as oro
    import torch
    dec = odec.RefDecoder(w.model, weights)
    prompts, offs = wl.make_prompts(w, n_prompts=1, prompt_len=64)
    G, max_new = 8, 8
    mode = 1 if w.sampling == "gumbel" else 0
    t0 = time.perf_counter()
    n_tok = 0
    for _ in range(n_steps):
        res = oro.rollout_group(dec, prompts, offs, G, mode, w.temperature, w.philox_seed, max_new)
        n_tok += int(res.lengths.sum())
    dt = time.perf_counter() - t0
    cores = torch.get_num_threads() if hasattr(torch, "get_num_threads") else os.cpu_count()
    try:
        from threadpoolctl import threadpool_info
        nt = [p["num_threads"] for p in threadpool_info() if p.get("user_api") == "blas"]
        if nt:
            cores = max(nt)
    except Exception:
        pass
    return n_tok / dt, int(cores), "1 prompt x 64 tokens prefill, G=8, 8 generated tokens each (numpy fp32 oracle)"


def run_reference(args, rank, world):
    """--impl reference: the CPU oracle on a bounded sample of the same workload (rank 0 only)."""
    if rank != 0:
        return
    w = wl.WORKLOADS[args.cfg]
    weights = wl.make_weights(w.model, 0)
    for _ in range(args.warmup and 1):
        oracle_sample(w, weights, 1)
    t0 = time.perf_counter()
    tps, cores, sample = oracle_sample(w, weights, args.steps)
    dt = time.perf_counter() - t0
    line = {"impl": "reference", "metric": METRIC, "value": tps, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * dt / max(args.steps, 1), "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f32 (bf16 weights widened)", "data": "synthetic",
            "config": {"workload": f"configs[{args.cfg - 1}] (0.5B-shaped decoder) -- bounded sample", "sample": sample},
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


def kernel_roofline(B, torch, mc, peak):
    """Time the largest single launch of a decode step alone (LM head, M = 64): CUDA events on the
    launching stream, weights (272 MB) larger than L2 so every iteration streams from HBM."""
    rng = np.random.default_rng(1)
    N, K, M = mc.vocab, mc.d_model, 64
    W = torch.from_numpy(rng.integers(0, 2 ** 15, size=(N, K), dtype=np.int64).astype(np.int16)).cuda()
    x = torch.randn(M, K, device="cuda")
    for _ in range(3):
        B.debug_linear(W, x, B.PATH_GEMM)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    n = 20
    e0.record()
    for _ in range(n):
        B.debug_linear(W, x, B.PATH_GEMM)
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / n
    nbytes = N * K * 2 + M * K * 4 + M * N * 4
    out = {"kernel": "k_linear_tc<128,STORE> (LM head, 64 live rows; + k_split_rows)", "bytes": nbytes, "ms": ms,
           "achieved_gbs": nbytes / ms / 1e6, "frac": nbytes / ms / 1e6 / peak}
    # the launch the decode step actually uses at <= 64 live rows: LM head + Gumbel sampler fused (logits never stored)
    sids = torch.arange(M, dtype=torch.int32, device="cuda")
    for _ in range(3):
        B.debug_lm_sample(W, x, sids, 5, seed=7)
    torch.cuda.synchronize()
    e0.record()
    for _ in range(n):
        B.debug_lm_sample(W, x, sids, 5, seed=7)
    e1.record()
    torch.cuda.synchronize()
    ms2 = e0.elapsed_time(e1) / n
    nb2 = N * K * 2 + M * K * 4
    out["fused"] = {"kernel": "k_lmhead_sample<128> (persistent LM head + Philox Gumbel arg-max, 64 live rows; + k_split_rows, k_pick_candidates)",
                    "bytes": nb2, "ms": ms2, "achieved_gbs": nb2 / ms2 / 1e6, "frac": nb2 / ms2 / 1e6 / peak,
                    # dram__bytes_read.sum of this kernel at this shape, one launch (profiles/r01_ncu_top_kernels.md)
                    "traffic": 272578048 if (N, K) == (151936, 896) else None}
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--cfg", type=int, default=2)
    ap.add_argument("--max-new", type=int, default=0, help="override max_new_tokens (debug; invalidates the number)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        return run_reference(args, rank, world)

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
    mc = w.model
    max_new = args.max_new or w.max_new
    weights = wl.make_weights(mc, 0)
    prompts, offs = wl.make_prompts(w)
    fl = np.minimum(wl.make_forced_lengths(w), max_new).astype(np.int32)
    rewards, goffs = wl.make_rewards(w)
    page = mc.page_tokens
    nseq = w.n_prompts * w.G
    n_pages = w.n_prompts * (w.prompt_len // page + w.G * ((max_new + page - 1) // page + 1)) + 8
    if n_pages * page * 2 * mc.n_layers * mc.n_kv_heads * mc.head_dim * 2 > 100e9:
        # worst case (every completion at the cap) does not fit: size the pool for the forced lengths actually drawn
        # (an upper bound that needs no retirement: every sequence's own blocks + the shared prefix blocks)
        n_pages = int(np.sum((fl + page - 1) // page + 2)) + w.n_prompts * (w.prompt_len // page + 1) + 8
    model = B.Model(mc, weights, n_pages, nseq, w.prompt_len + max_new, device=f"cuda:{local}")
    mode = B.MODE_GUMBEL if w.sampling == "gumbel" else B.MODE_GREEDY
    adv_mode = B.ADV_DAPO if w.adv_mode == "DAPO" else B.ADV_GRPO
    d_prompts = torch.from_numpy(prompts).cuda()
    d_rewards, d_goffs = torch.from_numpy(rewards).cuda(), torch.from_numpy(goffs).cuda()
    stream = torch.cuda.Stream()

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
        acc = {"tokens": 0, "launches": 0, "ph_ms": [0.0] * 3, "ph_bytes": [0.0] * 3, "ph_tok": [0] * 3, "ph_steps": [0] * 3,
               "prefill_ms": 0.0, "prefill_flops": 0.0, "decode_ms": 0.0}
        e0.record()
        for _ in range(args.steps):
            out, adv, keep = step()
            t = out.timing
            acc["tokens"] += t["total_tokens"]; acc["launches"] += t["kernel_launches"] + 1
            acc["prefill_ms"] += t["prefill_ms"]; acc["prefill_flops"] += t["prefill_flops"]; acc["decode_ms"] += t["decode_ms"]
            for p in range(3):
                acc["ph_ms"][p] += t["phase_ms"][p]; acc["ph_bytes"][p] += t["phase_bytes"][p]
                acc["ph_tok"][p] += t["phase_tokens"][p]; acc["ph_steps"][p] += t["phase_steps"][p]
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
        peak, peak_src = measured_peaks()
        kr = kernel_roofline(B, torch, mc, peak) if rank == 0 else None

    ms, e2e_ms = allreduce_max([ms, e2e_s * 1e3], "cuda", world)
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    names = ["full", "mid", "tail"]
    phases = {}
    for p in range(3):
        if acc["ph_steps"][p]:
            gbs = acc["ph_bytes"][p] / acc["ph_ms"][p] / 1e6
            phases[names[p]] = {"decode_steps": acc["ph_steps"][p] // args.steps, "tokens_per_s": acc["ph_tok"][p] / acc["ph_ms"][p] * 1e3,
                                "ms_per_decode_step": acc["ph_ms"][p] / acc["ph_steps"][p], "achieved_gbs": gbs,
                                "frac_of_measured": gbs / peak, "frac_of_8tbs": gbs / 8000.0}
    dec_bytes = sum(acc["ph_bytes"]); dec_ms = sum(acc["ph_ms"])
    achieved = dec_bytes / dec_ms / 1e6
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
            "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                         "traffic": None, "peak_source": peak_src,
                         "what": "all decode steps of the rollout (every kernel of the step graph): algorithmic bytes "
                                 "(weights once + prefix KV once per live group + suffix KV + KV written) / device time",
                         "frac_of_8tbs": achieved / 8000.0},
            "phases": phases, "kernel_roofline": kr,
            "prefill": {"ms": acc["prefill_ms"] / args.steps, "tflops": acc["prefill_flops"] / acc["prefill_ms"] / 1e9 if acc["prefill_ms"] else None}}
    if not args.no_cpu_baseline:
        tps, cores, sample = oracle_sample(w, weights, 1)
        line["cpu_baseline"] = {"value": tps, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample}
    print(json.dumps(line), flush=True)
    model.close()
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
