"""Rank plumbing of bench.py's multi-GPU (replica) path, on CPU with world_size-2 gloo.

The path has no data-path collective: every rank runs its own replica and the only cross-rank operation
is the max over ranks of the elapsed time.  Also: under torchrun the reference arm prints on rank 0 only.
"""
import json
import os
import subprocess
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    sys.path.insert(0, ROOT)
    import bench
    ms = bench.max_over_ranks(10.0 + 5.0 * rank, world, "cpu")   # rank r measured 10 + 5r ms
    per_rank_zones, steps = 1000, 4
    value = world * per_rank_zones * bench.SUBSTEPS_PER_STEP * steps / (ms * 1e-3)
    out[rank] = (ms, value)
    dist.barrier()
    dist.destroy_process_group()


def test_max_over_ranks_and_aggregate_value_world2():
    world, port = 2, 29731
    with mp.Manager() as man:
        out = man.dict()
        mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    assert res[0][0] == res[1][0] == 15.0            # every rank sees the slowest rank's time
    assert abs(res[0][1] - 2 * 1000 * 3 * 4 / 15e-3) < 1e-6   # whole-job zones over the max time


def test_single_rank_needs_no_process_group():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(3.5, 1, "cpu") == 3.5
    assert not dist.is_initialized()


def test_reference_arm_prints_on_rank0_only():
    env = dict(os.environ, WORLD_SIZE="2", LOCAL_RANK="1", RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "1", "--ref-n", "16"], env=env, capture_output=True, text=True)
    assert r.returncode == 0 and r.stdout.strip() == ""
    env["RANK"] = "0"; env["LOCAL_RANK"] = "0"
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "1", "--ref-n", "16"], env=env, capture_output=True, text=True)
    assert r.returncode == 0, r.stderr
    line = json.loads(r.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["n_gpus"] == 2 and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["e2e"]["h2d_bytes_per_step"] == 0


def test_gpus_flag_starts_one_rank_per_gpu(monkeypatch):
    """`python bench.py --gpus N` outside torchrun re-executes itself under torch.distributed.run with N ranks on
    127.0.0.1 (--gpus was ignored by the GPU arm); under torchrun it does not."""
    sys.path.insert(0, ROOT)
    import bench
    calls = []
    monkeypatch.setattr(bench.subprocess, "call", lambda cmd: calls.append(cmd) or 0)
    monkeypatch.delenv("WORLD_SIZE", raising=False)
    assert bench.main(["--gpus", "4", "--steps", "2", "--warmup", "3", "--shard-weak"]) == 0
    (cmd,) = calls
    assert cmd[1:4] == ["-m", "torch.distributed.run", "--nnodes=1"] and "--nproc-per-node=4" in cmd
    assert cmd[cmd.index("--master-addr") + 1] == "127.0.0.1"
    assert cmd[-7:] == ["--gpus", "4", "--steps", "2", "--warmup", "3", "--shard-weak"]
    assert os.path.basename(cmd[cmd.index("--master-port") + 2]) == "bench.py"


def test_launcher_runs_two_ranks_end_to_end_over_gloo():
    """The launcher started for real with world_size 2 on CPU: every rank builds only its own slab of the
    weak-scaling box (PAPER.md:244 shape), the ranks agree on the field scale, rank 0 prints one line."""
    sys.path.insert(0, ROOT)
    import bench
    import workloads as wl
    stub = os.path.join(ROOT, "tests", "helpers", "rank_stub.py")
    cmd = bench.launcher_command(["10"], 2, port=29747, script=stub)
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK")}
    r = subprocess.run(cmd, env=env, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    out = json.loads(lines[0])
    assert out["n_gpus"] == 2 and out["grid"] == [10, 10, 10] and out["zslab"] == [0, 10] and out["nz_global"] == 20
    assert out["ms"] >= 20.0                                  # the slower rank's sleep
    # the global box generated in one piece has the same field maximum as the slabs agreed on
    import numpy as np
    g = wl.kerr_sweep(10, zmult=2)
    assert abs(np.sqrt((g.prim8[5:8] ** 2).sum(axis=0)).max() - out["bmax_euclid"]) <= 1e-12 * out["bmax_euclid"]


def test_roofline_inputs_belong_to_the_kernels_in_the_tree():
    """bench.py's DRAM-traffic and flop inputs (profiles/roofline_inputs.json) are ncu measurements of one build of
    the kernels; the file names that build by a hash of the kernel sources and bench.py flags it stale otherwise
    (the constants were hard-coded from an earlier build).  The committed file must match."""
    sys.path.insert(0, ROOT)
    import bench
    d = bench.roofline_inputs()
    assert not d["stale"], (d["kernel_source_sha"], bench.kernel_source_hash())
    main = d["headline_numerator"]
    for dt in ("f64", "f32", "f32h"):
        assert d["flops_per_zone"][main][dt] > 0 and d["dram_bytes_per_zone"][dt] > 0
    # measured traffic can only exceed the algorithmic byte count (52 words per zone)
    assert d["dram_bytes_per_zone"]["f64"] >= 52 * 8 and d["dram_bytes_per_zone"]["f32"] >= 52 * 4
