"""ctypes binding of include/sagc.h -- argument marshalling only.

Every step of the path runs in the CUDA kernels of libsagc.so; torch is used for device
memory and streams.  The call names mirror the C ABI (`rollout_group`, `group_advantage`,
`length_stats`, `debug_*`).  Missing library or missing GPU -> RuntimeError (no fallback).
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass
from typing import Dict, List, Optional, Sequence, Tuple

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("SAGC_LIB", os.path.join(_HERE, "libsagc.so"))   # SAGC_LIB: A/B a differently built library

OK, EINVAL, ENOMEM, EPAGES, ECUDA = 0, -1, -2, -3, -4
MODE_GREEDY, MODE_GUMBEL = 0, 1
ADV_GRPO, ADV_DAPO = 0, 1
PATH_AUTO, PATH_GEMV, PATH_GEMM = 0, 1, 2
FLAG_STRUCTURE_ONLY, FLAG_LOG, FLAG_NO_GRAPH, FLAG_TIME_KERNELS = 1, 2, 4, 8

EXPORTS = [
    "sagc_model_create", "sagc_model_destroy", "sagc_rollout_group", "sagc_rollout_group_host", "sagc_score_tokens",
    "sagc_group_advantage", "sagc_length_stats", "sagc_debug_page_table", "sagc_debug_free_stack",
    "sagc_debug_alloc_log", "sagc_debug_retire_log", "sagc_debug_peak_pages", "sagc_debug_philox",
    "sagc_debug_linear", "sagc_debug_lm_sample", "sagc_debug_attention", "sagc_attention_noalloc", "sagc_debug_step_trace", "sagc_last_error", "sagc_version",
]


class SagcError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"sagc error {code}: {msg}")
        self.code = code


class _ModelConfig(C.Structure):
    _fields_ = [(n, C.c_int32) for n in ("n_layers", "d_model", "n_q_heads", "n_kv_heads", "head_dim", "d_ff", "vocab")] + \
               [("rope_theta", C.c_float), ("rms_eps", C.c_float)] + \
               [(n, C.c_int32) for n in ("page_tokens", "n_pages", "max_seqs", "max_ctx")]


class _Weights(C.Structure):
    _fields_ = [("embed", C.c_void_p), ("lm_head", C.c_void_p), ("final_norm", C.c_void_p)] + \
               [(n, C.POINTER(C.c_void_p)) for n in ("wq", "wk", "wv", "wo", "wg", "wu", "wd", "norm1", "norm2")]


class _RolloutParams(C.Structure):
    _fields_ = [("mode", C.c_int32), ("temperature", C.c_float), ("seed", C.c_uint64), ("stop_token", C.c_int32),
                ("max_new_tokens", C.c_int32), ("forced_lengths", C.c_void_p), ("forced_tokens", C.c_void_p),
                ("path", C.c_int32), ("flags", C.c_int32), ("n_dump", C.c_int32), ("dump_sid_t", C.c_void_p),
                ("dump_logits", C.c_void_p)]


class _Timing(C.Structure):
    _fields_ = [("prefill_ms", C.c_double), ("decode_ms", C.c_double), ("phase_ms", C.c_double * 3),
                ("phase_steps", C.c_int64 * 3), ("phase_tokens", C.c_int64 * 3), ("phase_bytes", C.c_double * 3),
                ("prefill_tokens", C.c_int64), ("prefill_flops", C.c_double), ("total_tokens", C.c_int64),
                ("kernel_launches", C.c_int64), ("kernel_ms", C.c_double * 3), ("kernel_steps", C.c_int64)]


_lib = None


def lib():
    """Load libsagc.so (built in-tree by paper_2606_02218_b200.build).  Fails loudly if absent."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: run `python -m paper_2606_02218_b200.build` "
                               "(the CUDA extension is the only implementation; there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        L.sagc_last_error.restype = C.c_char_p
        L.sagc_version.restype = C.c_char_p
        L.sagc_model_destroy.restype = None
        L.sagc_model_destroy.argtypes = [C.c_void_p]
        L.sagc_model_create.argtypes = [C.POINTER(_ModelConfig), C.POINTER(_Weights), C.POINTER(C.c_void_p)]
        roll = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int32, C.c_int32, C.POINTER(_RolloutParams), C.c_void_p,
                C.c_void_p, C.c_void_p, C.c_void_p, C.POINTER(_Timing), C.c_void_p]
        L.sagc_rollout_group.argtypes = roll
        L.sagc_rollout_group_host.argtypes = roll
        L.sagc_score_tokens.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int32, C.c_int32, C.c_void_p, C.c_void_p, C.c_int32,
                                        C.c_void_p, C.c_void_p]
        L.sagc_group_advantage.argtypes = [C.c_void_p, C.c_void_p, C.c_int32, C.c_int32, C.c_int32, C.c_float,
                                           C.c_void_p, C.c_void_p, C.c_void_p]
        L.sagc_length_stats.argtypes = [C.c_void_p, C.c_void_p, C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p]
        L.sagc_debug_page_table.argtypes = [C.c_void_p, C.c_void_p, C.c_int32, C.POINTER(C.c_int32), C.POINTER(C.c_int32)]
        L.sagc_debug_free_stack.argtypes = [C.c_void_p, C.c_void_p, C.c_int32, C.POINTER(C.c_int32)]
        L.sagc_debug_alloc_log.argtypes = [C.c_void_p, C.c_void_p, C.c_int32, C.POINTER(C.c_int32)]
        L.sagc_debug_retire_log.argtypes = [C.c_void_p, C.c_void_p, C.c_int32, C.POINTER(C.c_int32)]
        L.sagc_debug_peak_pages.argtypes = [C.c_void_p, C.POINTER(C.c_int32)]
        L.sagc_debug_philox.argtypes = [C.c_uint64, C.c_int32, C.c_int32, C.c_int32, C.c_int32, C.c_void_p, C.c_void_p]
        L.sagc_debug_linear.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int32, C.c_int32, C.c_int32, C.c_int32,
                                        C.c_void_p]
        L.sagc_debug_lm_sample.argtypes = [C.c_void_p, C.c_void_p, C.c_int32, C.c_int32, C.c_int32, C.c_int32, C.c_float,
                                           C.c_uint64, C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.sagc_debug_attention.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int32, C.c_int32,
                                           C.c_int32, C.c_int32, C.c_int32, C.c_int32, C.c_int32, C.c_int32, C.c_void_p,
                                           C.c_void_p]
        L.sagc_attention_noalloc.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int32, C.c_int32,
                                             C.c_int32, C.c_int32, C.c_int32, C.c_int32, C.c_int32, C.c_void_p, C.c_void_p]
        L.sagc_debug_step_trace.argtypes = [C.c_void_p, C.c_int64, C.c_void_p, C.c_int32, C.POINTER(C.c_int32)]
        _lib = L
    return _lib


def _check(rc: int) -> None:
    if rc != OK:
        raise SagcError(rc, lib().sagc_last_error().decode())


def _stream() -> int:
    return torch.cuda.current_stream().cuda_stream


def _require_cuda() -> None:
    if not torch.cuda.is_available():
        raise RuntimeError("no CUDA device: the rollout path has no CPU fallback")


def _dev_u16(a: np.ndarray, device) -> torch.Tensor:
    """bf16 bit patterns (uint16 numpy) -> device tensor holding the same bits."""
    return torch.from_numpy(np.ascontiguousarray(a).view(np.int16)).to(device)


@dataclass
class RolloutOutput:
    tokens: torch.Tensor          # int32 [nseq][max_new], pad -1 (device, or host for host=True)
    lengths: torch.Tensor         # int32 [nseq]
    ratio_max_mean: torch.Tensor  # float32 [n_prompts]
    len_stats: torch.Tensor       # int32 [n_prompts][3] = max, sum, median_x2
    timing: Optional[dict] = None
    dump_logits: Optional[torch.Tensor] = None   # float32 [n_dump][V] (device)


class Model:
    """Owns the device copies of the weights and the opaque sagc_model handle."""

    def __init__(self, mc, weights: Dict[str, object], n_pages: int, max_seqs: int, max_ctx: int,
                 device: str = "cuda:0"):
        _require_cuda()
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        self.mc = mc
        L = mc.n_layers
        self._w = {}
        for name in ("embed", "lm_head", "final_norm"):
            self._w[name] = _dev_u16(weights[name], self.device)
        for name in ("wq", "wk", "wv", "wo", "wg", "wu", "wd", "norm1", "norm2"):
            self._w[name] = [_dev_u16(weights[name][l], self.device) for l in range(L)]
        cfg = _ModelConfig(L, mc.d_model, mc.n_q_heads, mc.n_kv_heads, mc.head_dim, mc.d_ff, mc.vocab,
                           float(mc.rope_theta), float(mc.rms_eps), mc.page_tokens, int(n_pages), int(max_seqs),
                           int(max_ctx))
        w = _Weights()
        w.embed = self._w["embed"].data_ptr()
        w.lm_head = self._w["lm_head"].data_ptr()
        w.final_norm = self._w["final_norm"].data_ptr()
        self._arrs = {}
        for name in ("wq", "wk", "wv", "wo", "wg", "wu", "wd", "norm1", "norm2"):
            arr = (C.c_void_p * max(L, 1))(*[t.data_ptr() for t in self._w[name]])
            self._arrs[name] = arr
            setattr(w, name, C.cast(arr, C.POINTER(C.c_void_p)))
        self._h = C.c_void_p()
        _check(lib().sagc_model_create(C.byref(cfg), C.byref(w), C.byref(self._h)))
        self.n_pages, self.max_seqs, self.max_ctx = int(n_pages), int(max_seqs), int(max_ctx)

    def close(self) -> None:
        if getattr(self, "_h", None) and self._h.value:
            lib().sagc_model_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- sagc_rollout_group / sagc_rollout_group_host ------------------------------------
    def rollout_group(self, prompt_tokens, prompt_offsets, G: int, *, mode: int = MODE_GREEDY,
                      temperature: float = 1.0, seed: int = 0, max_new_tokens: int, forced_lengths=None,
                      stop_token: int = -1, forced_tokens: Optional[torch.Tensor] = None, path: int = PATH_AUTO,
                      flags: int = 0, dump: Optional[Sequence[Tuple[int, int]]] = None, timing: bool = False,
                      host: bool = False) -> RolloutOutput:
        offs = np.ascontiguousarray(prompt_offsets, dtype=np.int32)
        n_prompts = offs.shape[0] - 1
        nseq = n_prompts * G
        prm = _RolloutParams()
        prm.mode, prm.temperature, prm.seed = int(mode), float(temperature), int(seed)
        prm.stop_token, prm.max_new_tokens, prm.path, prm.flags = int(stop_token), int(max_new_tokens), int(path), int(flags)
        fl = None
        if forced_lengths is not None:
            fl = np.ascontiguousarray(forced_lengths, dtype=np.int32)
            assert fl.shape[0] == nseq
            prm.forced_lengths = fl.ctypes.data
        if forced_tokens is not None:
            assert forced_tokens.is_cuda and forced_tokens.dtype == torch.int32 and forced_tokens.is_contiguous()
            prm.forced_tokens = forced_tokens.data_ptr()
        dump_arr, dump_out = None, None
        if dump:
            dump_arr = np.ascontiguousarray(np.asarray(dump, dtype=np.int32).reshape(-1, 2))
            dump_out = torch.zeros((dump_arr.shape[0], self.mc.vocab), dtype=torch.float32, device=self.device)
            prm.n_dump, prm.dump_sid_t, prm.dump_logits = dump_arr.shape[0], dump_arr.ctypes.data, dump_out.data_ptr()
        tm = _Timing() if timing else None
        tm_ref = C.byref(tm) if timing else None
        if host:
            pt = None if prompt_tokens is None else np.ascontiguousarray(prompt_tokens, dtype=np.int32)
            toks = torch.empty((nseq, max_new_tokens), dtype=torch.int32).pin_memory()
            lens = torch.empty((nseq,), dtype=torch.int32).pin_memory()
            ratio = torch.empty((n_prompts,), dtype=torch.float32).pin_memory()
            stats = torch.empty((n_prompts, 3), dtype=torch.int32).pin_memory()
            _check(lib().sagc_rollout_group_host(self._h, None if pt is None else pt.ctypes.data, offs.ctypes.data,
                                                 n_prompts, G, C.byref(prm), toks.data_ptr(), lens.data_ptr(),
                                                 ratio.data_ptr(), stats.data_ptr(), tm_ref, _stream()))
        else:
            if prompt_tokens is None:
                pt_ptr = None
            else:
                if not torch.is_tensor(prompt_tokens):
                    prompt_tokens = torch.from_numpy(np.ascontiguousarray(prompt_tokens, dtype=np.int32)).to(self.device)
                assert prompt_tokens.is_cuda and prompt_tokens.dtype == torch.int32
                pt_ptr = prompt_tokens.data_ptr()
            toks = torch.empty((nseq, max_new_tokens), dtype=torch.int32, device=self.device)
            lens = torch.empty((nseq,), dtype=torch.int32, device=self.device)
            ratio = torch.empty((n_prompts,), dtype=torch.float32, device=self.device)
            stats = torch.empty((n_prompts, 3), dtype=torch.int32, device=self.device)
            _check(lib().sagc_rollout_group(self._h, pt_ptr, offs.ctypes.data, n_prompts, G, C.byref(prm),
                                            toks.data_ptr(), lens.data_ptr(), ratio.data_ptr(), stats.data_ptr(),
                                            tm_ref, _stream()))
        td = None
        if timing:
            td = {"prefill_ms": tm.prefill_ms, "decode_ms": tm.decode_ms, "phase_ms": list(tm.phase_ms),
                  "phase_steps": list(tm.phase_steps), "phase_tokens": list(tm.phase_tokens),
                  "phase_bytes": list(tm.phase_bytes), "prefill_tokens": tm.prefill_tokens,
                  "prefill_flops": tm.prefill_flops, "total_tokens": tm.total_tokens,
                  "kernel_launches": tm.kernel_launches, "kernel_ms": list(tm.kernel_ms), "kernel_steps": tm.kernel_steps}
        return RolloutOutput(toks, lens, ratio, stats, td, dump_out)

    # -- sagc_score_tokens ---------------------------------------------------------------
    def score_tokens(self, prompt_tokens, prompt_offsets, G: int, tokens: torch.Tensor, lengths) -> torch.Tensor:
        """log pi(y_t | x, y_<t) of every generated token: float32 [nseq][max_new] (device), 0 beyond each length."""
        offs = np.ascontiguousarray(prompt_offsets, dtype=np.int32)
        n_prompts = offs.shape[0] - 1
        if not torch.is_tensor(prompt_tokens):
            prompt_tokens = torch.from_numpy(np.ascontiguousarray(prompt_tokens, dtype=np.int32)).to(self.device)
        assert tokens.is_cuda and tokens.dtype == torch.int32 and tokens.is_contiguous()
        lens = np.ascontiguousarray(lengths.cpu().numpy() if torch.is_tensor(lengths) else lengths, dtype=np.int32)
        out = torch.empty(tokens.shape, dtype=torch.float32, device=self.device)
        _check(lib().sagc_score_tokens(self._h, prompt_tokens.data_ptr(), offs.ctypes.data, n_prompts, G, tokens.data_ptr(),
                                       lens.ctypes.data, tokens.shape[1], out.data_ptr(), _stream()))
        return out

    # -- debug / parity exports ---------------------------------------------------------
    def debug_page_table(self) -> np.ndarray:
        max_blocks = (self.max_ctx + self.mc.page_tokens - 1) // self.mc.page_tokens
        out = np.empty((self.max_seqs, max_blocks), dtype=np.int32)
        nseq, mb = C.c_int32(), C.c_int32()
        _check(lib().sagc_debug_page_table(self._h, out.ctypes.data, out.size, C.byref(nseq), C.byref(mb)))
        return out.reshape(-1)[: nseq.value * mb.value].reshape(nseq.value, mb.value).copy()

    def debug_free_stack(self) -> np.ndarray:
        out = np.empty(self.n_pages, dtype=np.int32)
        n = C.c_int32()
        _check(lib().sagc_debug_free_stack(self._h, out.ctypes.data, out.size, C.byref(n)))
        return out[: n.value].copy()

    def _log(self, fn, width: int, cap: int) -> np.ndarray:
        out = np.empty((cap, width), dtype=np.int32)
        n = C.c_int32()
        _check(fn(self._h, out.ctypes.data, cap, C.byref(n)))
        return out[: min(n.value, cap)].copy()

    def debug_alloc_log(self) -> np.ndarray:
        return self._log(lib().sagc_debug_alloc_log, 3, self.n_pages * 16 + 65536)

    def debug_retire_log(self) -> np.ndarray:
        return self._log(lib().sagc_debug_retire_log, 2, self.max_seqs)

    def debug_step_trace(self, record_step: int) -> np.ndarray:
        """(tag, ns) pairs recorded by the persistent decode-step kernel so far; arms step `record_step` of the next rollout."""
        out = np.zeros((16000, 2), dtype=np.uint64)
        n = C.c_int32()
        _check(lib().sagc_debug_step_trace(self._h, int(record_step), out.ctypes.data, 16000, C.byref(n)))
        return out[: n.value].copy()

    def debug_peak_pages(self) -> int:
        p = C.c_int32()
        _check(lib().sagc_debug_peak_pages(self._h, C.byref(p)))
        return p.value


# -- sagc_group_advantage / sagc_length_stats ------------------------------------------------
def group_advantage(rewards: torch.Tensor, group_offsets: torch.Tensor, mode: int = ADV_GRPO, ddof: int = 0,
                    eps: float = 0.0) -> Tuple[torch.Tensor, torch.Tensor]:
    _require_cuda()
    assert rewards.is_cuda and rewards.dtype == torch.float32 and rewards.is_contiguous()
    assert group_offsets.is_cuda and group_offsets.dtype == torch.int32
    n_groups = group_offsets.numel() - 1
    adv = torch.empty_like(rewards)
    keep = torch.empty((max(n_groups, 0),), dtype=torch.uint8, device=rewards.device)
    _check(lib().sagc_group_advantage(rewards.data_ptr(), group_offsets.data_ptr(), n_groups, mode, ddof, eps,
                                      adv.data_ptr(), keep.data_ptr(), _stream()))
    return adv, keep


def length_stats(lengths: torch.Tensor, group_offsets: torch.Tensor) -> Tuple[torch.Tensor, torch.Tensor]:
    _require_cuda()
    assert lengths.is_cuda and lengths.dtype == torch.int32 and group_offsets.dtype == torch.int32
    n_groups = group_offsets.numel() - 1
    stats = torch.empty((n_groups, 3), dtype=torch.int32, device=lengths.device)
    ratio = torch.empty((n_groups,), dtype=torch.float32, device=lengths.device)
    _check(lib().sagc_length_stats(lengths.data_ptr(), group_offsets.data_ptr(), n_groups, stats.data_ptr(),
                                   ratio.data_ptr(), _stream()))
    return stats, ratio


def debug_philox(seed: int, sid: int, t: int, v0: int, n: int, device="cuda:0") -> torch.Tensor:
    _require_cuda()
    out = torch.empty((n,), dtype=torch.int32, device=device)
    _check(lib().sagc_debug_philox(seed, sid, t, v0, n, out.data_ptr(), _stream()))
    return out


def debug_linear(W_bits: torch.Tensor, x: torch.Tensor, path: int = PATH_GEMM) -> torch.Tensor:
    """W_bits: int16 [N][K] bf16 bit patterns; x float32 [M][K] -> y float32 [M][N]."""
    _require_cuda()
    N, K = W_bits.shape
    M = x.shape[0]
    y = torch.empty((M, N), dtype=torch.float32, device=x.device)
    _check(lib().sagc_debug_linear(W_bits.data_ptr(), x.data_ptr(), y.data_ptr(), M, N, K, path, _stream()))
    return y


def debug_lm_sample(W_bits: torch.Tensor, x: torch.Tensor, sids: torch.Tensor, t: int, mode: int = MODE_GUMBEL,
                    temperature: float = 1.0, seed: int = 0, want_logits: bool = False):
    """Fused LM head + sampler: W_bits int16 [V][K], x float32 [M][K], sids int32 [M] -> tokens int32 [M] (, logits [M][V])."""
    _require_cuda()
    V, K = W_bits.shape
    M = x.shape[0]
    tok = torch.empty((M,), dtype=torch.int32, device=x.device)
    lg = torch.empty((M, V), dtype=torch.float32, device=x.device) if want_logits else None
    _check(lib().sagc_debug_lm_sample(W_bits.data_ptr(), x.data_ptr(), M, V, K, mode, temperature, seed, t, sids.data_ptr(),
                                      tok.data_ptr(), lg.data_ptr() if want_logits else None, _stream()))
    return (tok, lg) if want_logits else tok


def debug_attention(q: torch.Tensor, kv_bits: torch.Tensor, page_table: torch.Tensor, ctx: torch.Tensor, Hq: int,
                    Hkv: int, hd: int, page_tokens: int, n_splits: int = 4, variant: int = 0) -> torch.Tensor:
    """q float32 [M][Hq][hd]; kv_bits int16 [n_pages][2][Hkv][page][hd]; page_table int32 [M][max_blocks].
    variant 0 = standalone kernel, 1 = the units of the persistent decode-step kernel, 2 = the tcgen05 decode kernel."""
    _require_cuda()
    M = q.shape[0]
    out = torch.empty((M, Hq, hd), dtype=torch.float32, device=q.device)
    _check(lib().sagc_debug_attention(q.data_ptr(), kv_bits.data_ptr(), page_table.data_ptr(), ctx.data_ptr(), M, Hq,
                                      Hkv, hd, page_tokens, page_table.shape[1], n_splits, variant, out.data_ptr(),
                                      _stream()))
    return out


NOALLOC_SCRATCH_BYTES = 8 << 20


def attention_noalloc(q: torch.Tensor, kv_bits: torch.Tensor, page_table: torch.Tensor, ctx: torch.Tensor, out: torch.Tensor,
                      Hq: int, Hkv: int, hd: int, page_tokens: int, n_splits: int = 4) -> torch.Tensor:
    """sagc_attention_noalloc: shapes as `debug_attention`, but `out` (float32 [M][Hq][hd]) is the caller's and the
    split-K scratch is the library's static device array (<= NOALLOC_SCRATCH_BYTES, else SagcError).  Nothing is
    allocated and the stream is not synchronised; calls that overlap on the GPU race on the shared scratch."""
    _require_cuda()
    M = q.shape[0]
    if out.dtype != torch.float32 or out.numel() != M * Hq * hd or not out.is_contiguous():
        raise ValueError("out must be a contiguous float32 [M][Hq][hd] tensor")
    _check(lib().sagc_attention_noalloc(q.data_ptr(), kv_bits.data_ptr(), page_table.data_ptr(), ctx.data_ptr(), M, Hq,
                                        Hkv, hd, page_tokens, page_table.shape[1], n_splits, out.data_ptr(), _stream()))
    return out
