"""Stand-in for bench.py's GPU arm in the CPU test of its launcher (tests/test_bench_ranks_cpu.py): started by
bench.launcher_command under torch.distributed.run, it walks the same rank plumbing over gloo -- process group from
the environment, this rank's slab of the weak-scaling box with the global field scale agreed by all-reduce, the
max over ranks of the elapsed time, one JSON line from rank 0 -- with a sleep where the GPU arm steps a context."""
import json
import os
import sys
import time

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import numpy as np
import torch.distributed as dist

import bench
import workloads as wl


def main():
    world, rank = int(os.environ["WORLD_SIZE"]), int(os.environ["RANK"])
    dist.init_process_group("gloo")
    n = int(sys.argv[1])
    w = bench.weak_slab_workload(wl, n, rank, world, "cpu")
    t = time.perf_counter()
    time.sleep(0.01 * (1 + rank))                       # the slower rank sets the time
    ms = bench.max_over_ranks((time.perf_counter() - t) * 1e3, world, "cpu")
    bmax = bench.max_over_ranks(float(np.sqrt((w.prim8[5:8] ** 2).sum(axis=0)).max()), world, "cpu")
    dist.barrier()
    if rank == 0:
        print(json.dumps({"n_gpus": world, "ms": ms, "grid": list(w.n), "zslab": list(w.extra["zslab"]),
                          "nz_global": w.extra["nz_global"], "bmax_euclid": bmax,
                          "value": world * w.ncell * bench.SUBSTEPS_PER_STEP / (ms * 1e-3)}))
    dist.destroy_process_group()


if __name__ == "__main__":
    main()
