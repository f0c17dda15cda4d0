"""The NCCL halo transport on real hardware (pytest -m gpu): runs only where two GPUs are visible.  This pool gives
one GPU per call, so here it is collected and SKIPPED; the same exchange is validated on one GPU with all slabs in
one process (tests/test_gpu_parity.py, bitwise) and its rank logic over gloo (tests/test_slab_cpu.py).
The exchange FUSED into the substep kernel between processes (CUDA IPC mapping of the neighbour's buffers,
hz_peer_attach) needs no second GPU to be exercised: two processes share the one GPU here."""
import os
import sys

import numpy as np
import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    import torch
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import workloads as wl
    from paper_1102_5202_b200 import DistSlabHorizon
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    torch.cuda.set_device(rank)
    dist.init_process_group("nccl", rank=rank, world_size=world, device_id=torch.device("cuda", rank))
    w = wl.kerr_sweep(24)
    dsh = DistSlabHorizon(w, dtype="f64")
    dsh.substeps(w.dt, 4)
    out[rank] = (dsh.slab.sl.start, dsh.slab.sl.stop, dsh.get_primitives())
    d = dsh.diagnostics()
    if rank == 0:
        out["diag"] = d
    dsh.close()
    dist.destroy_process_group()


def test_two_ranks_over_nccl_reproduce_the_single_domain_bitwise():
    import torch
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two GPUs (the NCCL send/recv of the ghost planes between two processes)")
    import torch.multiprocessing as mp
    import workloads as wl
    from paper_1102_5202_b200 import Horizon
    w = wl.kerr_sweep(24)
    one = Horizon.from_workload(w, dtype="f64")
    one.substeps(w.dt, 4)
    ref = one.get_primitives()
    dref = one.diagnostics()
    one.close()
    with mp.Manager() as man:
        out = man.dict()
        mp.spawn(_worker, args=(2, 29763, out), nprocs=2, join=True)
        res = dict(out)
    for r in (0, 1):
        k0, k1, p = res[r]
        assert np.array_equal(p, ref[:, k0:k1]), f"rank {r}"
    for k in ("c2p_fail", "atm_reset", "p_floor"):
        assert res["diag"][k] == dref[k]
    assert abs(res["diag"]["sumD"] - dref["sumD"]) <= 1e-12 * abs(dref["sumD"])


def _worker_ipc(rank, world, port, out, dtype):
    import torch
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import workloads as wl
    from paper_1102_5202_b200 import DistSlabHorizon
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    torch.cuda.set_device(0)                      # both ranks on the one GPU; their kernels never wait on one another
    dist.init_process_group("gloo", rank=rank, world_size=world)
    w = wl.kerr_sweep(24) if dtype == "f64" else wl.alfven_wave(n=(19, 12, 20))
    dsh = DistSlabHorizon(w, dtype=dtype, device="cuda:0", fused=True)
    n0 = dsh.slab.hz.launch_count()
    dsh.substeps(w.dt, 5)
    launches = dsh.slab.hz.launch_count() - n0
    out[rank] = (dsh.slab.sl.start, dsh.slab.sl.stop, dsh.get_primitives(), launches)
    dsh.close()
    dist.destroy_process_group()


@pytest.mark.parametrize("dtype,port", [("f64", 29771), ("f32", 29772)])
def test_two_processes_with_ipc_mapped_neighbours_reproduce_the_single_domain_bitwise(dtype, port):
    """hz_peer_attach across processes: each rank opens its neighbour's state buffer through CUDA IPC and the substep
    kernel stores the planes next to the cut into it; between substeps there is a barrier and nothing else.
    f64: outflow ends (one cut); f32: periodic ring of two (both neighbours are the other rank)."""
    import torch.multiprocessing as mp
    import workloads as wl
    from paper_1102_5202_b200 import Horizon
    w = wl.kerr_sweep(24) if dtype == "f64" else wl.alfven_wave(n=(19, 12, 20))
    one = Horizon.from_workload(w, dtype=dtype)
    one.substeps(w.dt, 5)
    ref = one.get_primitives()
    one.close()
    with mp.Manager() as man:
        out = man.dict()
        mp.spawn(_worker_ipc, args=(2, port, out, dtype), nprocs=2, join=True)
        res = dict(out)
    for r in (0, 1):
        k0, k1, p, launches = res[r]
        assert launches == 5                      # the substep kernels and nothing else
        assert np.array_equal(p, ref[:, k0:k1]), f"rank {r}: max |diff| = {np.abs(p - ref[:, k0:k1]).max()}"
