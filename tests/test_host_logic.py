"""CPU-only checks of the boundary and the host logic (no compute calls: there is no GPU here)."""
import ctypes as C
import os
import re
import subprocess
import sys
import tempfile

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "sagc.h")


@pytest.fixture(scope="module")
def lib():
    from paper_2606_02218_b200 import build, binding
    build.build()
    return binding.lib()


def test_library_exports_every_declared_symbol(lib):
    from paper_2606_02218_b200 import binding
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    declared = sorted(set(re.findall(r"\b(sagc_[a-z_]+)\s*\(", src)))
    assert len(declared) >= 16
    for name in declared:
        assert hasattr(lib, name), name
    assert sorted(binding.EXPORTS) == declared
    assert b"sm_100a" in lib.sagc_version()


def test_ctypes_structs_match_the_header():
    """sizeof / offsetof of every boundary struct, compiled from the header with gcc, against ctypes."""
    from paper_2606_02218_b200 import binding as B
    prog = r'''
#include <stdio.h>
#include <stddef.h>
#include "sagc.h"
int main(void) {
  printf("%zu %zu %zu %zu\n", sizeof(sagc_model_config), sizeof(sagc_weights), sizeof(sagc_rollout_params), sizeof(sagc_rollout_timing));
  printf("%zu %zu %zu %zu %zu\n", offsetof(sagc_model_config, rope_theta), offsetof(sagc_model_config, max_ctx),
         offsetof(sagc_rollout_params, seed), offsetof(sagc_rollout_params, forced_lengths), offsetof(sagc_rollout_params, dump_logits));
  printf("%zu %zu %zu\n", offsetof(sagc_rollout_timing, phase_bytes), offsetof(sagc_rollout_timing, kernel_launches), offsetof(sagc_weights, wq));
  return 0; }'''
    with tempfile.TemporaryDirectory() as td:
        cpath = os.path.join(td, "t.c")
        open(cpath, "w").write(prog)
        exe = os.path.join(td, "t")
        subprocess.run(["gcc", "-I", os.path.join(ROOT, "include"), cpath, "-o", exe], check=True)
        out = subprocess.run([exe], capture_output=True, text=True, check=True).stdout.split()
    got = [int(x) for x in out]
    exp = [C.sizeof(B._ModelConfig), C.sizeof(B._Weights), C.sizeof(B._RolloutParams), C.sizeof(B._Timing),
           B._ModelConfig.rope_theta.offset, B._ModelConfig.max_ctx.offset, B._RolloutParams.seed.offset,
           B._RolloutParams.forced_lengths.offset, B._RolloutParams.dump_logits.offset,
           B._Timing.phase_bytes.offset, B._Timing.kernel_launches.offset, B._Weights.wq.offset]
    assert got == exp


def test_no_gpu_means_loud_failure(lib):
    """The product path has no CPU fallback: without a device every compute entry point errors."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    from paper_2606_02218_b200 import binding as B, workloads as wl
    w = wl.WORKLOADS[1]
    with pytest.raises(RuntimeError):
        B.Model(w.model, wl.make_weights(w.model, 0), 16, 4, 64)
    with pytest.raises(RuntimeError):
        B.group_advantage(torch.zeros(4), torch.zeros(2, dtype=torch.int32))
    rc = lib.sagc_group_advantage(None, None, 1, 0, 0, C.c_float(0.0), None, None, None)
    assert rc == B.EINVAL
    cfg = B._ModelConfig(2, 128, 4, 4, 32, 512, 1024, 1e4, 1e-6, 16, 16, 4, 64)
    h = C.c_void_p()
    rc = lib.sagc_model_create(C.byref(cfg), C.byref(B._Weights()), C.byref(h))
    assert rc == B.ECUDA and b"no CUDA device" in lib.sagc_last_error()


def test_workload_generators_are_seeded_and_shaped():
    from paper_2606_02218_b200 import workloads as wl
    w = wl.WORKLOADS[2]
    fl = wl.make_forced_lengths(w)
    assert fl.shape == (64,) and fl.min() >= 1 and fl.max() <= 4096
    assert np.array_equal(fl, wl.make_forced_lengths(w))
    assert int(fl.sum()) == 71773                      # cfg2 schedule, seed 1002
    assert w.model.decode_weight_bytes() == 987_922_432 and w.model.kv_bytes_per_token() == 12288
    r, offs = wl.make_rewards(wl.WORKLOADS[3])
    assert set(np.unique(r)) <= {0.0, 1.0} and offs[-1] == 256
    sched = wl.g_schedule(wl.WORKLOADS[4])
    assert len(sched) == 10 and all(abs(np.log2(a) - np.log2(b)) <= 1 for a, b in zip(sched, sched[1:]))


def _gloo_worker(rank, world, port, q):
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    out = bench.allreduce_max([1.0 + rank, 10.0 - rank], "cpu", world)
    q.put((rank, out))
    dist.destroy_process_group()


def test_replica_timing_is_max_over_ranks_gloo():
    """N > 1 = independent replicas; the only cross-rank step is the max over ranks of the timed region."""
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_gloo_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = dict(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(60)
    assert res[0] == [2.0, 10.0] and res[1] == [2.0, 10.0]


def test_reference_arm_runs_on_rank0_only():
    sys.path.insert(0, ROOT)
    import bench

    class A:
        cfg, steps, warmup, gpus = 1, 1, 0, 2
    assert bench.run_reference(A, rank=1, world=2) is None      # other ranks exit without work
