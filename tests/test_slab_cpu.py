"""Host logic of the slab decomposition (paper_1102_5202_b200/slab.py) on CPU:
the z split, the boundary codes, the neighbour table, the diagnostics fold, and -- with world_size 2 and 3
over gloo -- the posting order of DistTransport's sends and receives, with a stand-in context whose
"planes" are just their global z indices.  The arithmetic path itself is tested on the GPU
(tests/test_gpu_parity.py::test_slab_decomposition_reproduces_the_single_domain_bitwise)."""
import os
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

from paper_1102_5202_b200 import binding as B  # noqa: E402
from paper_1102_5202_b200 import slab  # noqa: E402


def test_split_and_boundary_codes():
    assert slab.split_z(20, 3) == [(0, 7), (7, 14), (14, 20)]
    assert slab.split_z(8, 4) == [(0, 2), (2, 4), (4, 6), (6, 8)]
    with pytest.raises(ValueError):
        slab.split_z(7, 4)
    P, O = B.HZ_BC_PERIODIC, B.HZ_BC_OUTFLOW
    assert [slab.slab_bc(P, r, 3) for r in range(3)] == [B.HZ_BC_EXTERNAL] * 3
    assert [slab.slab_bc(O, r, 3) for r in range(3)] == [B.HZ_BC_OUTFLOW_EXTERNAL, B.HZ_BC_EXTERNAL,
                                                         B.HZ_BC_EXTERNAL_OUTFLOW]
    assert slab.slab_bc(O, 0, 1) == O and slab.slab_bc(P, 0, 1) == P
    assert [slab.neighbours(P, r, 3) for r in range(3)] == [(2, 1), (0, 2), (1, 0)]
    assert [slab.neighbours(P, r, 2) for r in range(2)] == [(1, 1), (0, 0)]
    assert [slab.neighbours(O, r, 3) for r in range(3)] == [(None, 1), (0, 2), (1, None)]


def test_diagnostics_fold():
    d1 = dict(sumD=1.0, sumSx=0.0, sumSy=0.0, sumSz=0.0, sumTau=2.0, sumBx=0.0, sumBy=0.0, sumBz=0.0, sumPsi=0.0,
              c2p_fail=1, atm_reset=2, p_floor=0, c2p_stalled=3, divB_max=3.0, max_speed_over_dx=5.0, c2p_maxit_seen=4, divB_L1=1.0)
    d2 = dict(d1, sumD=2.0, divB_max=1.0, max_speed_over_dx=7.0, divB_L1=4.0, c2p_fail=0)
    out = slab.combine_diagnostics([d1, d2], [100, 300])
    assert out["sumD"] == 3.0 and out["sumTau"] == 4.0 and out["c2p_fail"] == 1 and out["atm_reset"] == 4
    assert out["divB_max"] == 3.0 and out["max_speed_over_dx"] == 7.0
    assert out["divB_L1"] == (1.0 * 100 + 4.0 * 300) / 400


class FakeHz:
    """Stand-in for a context: one float64 per plane, value = global z index; ghosts start at -1."""

    def __init__(self, k0, k1):
        self.n = k1 - k0
        self.planes = torch.full((self.n + 4,), -1.0, dtype=torch.float64)
        self.planes[2:2 + self.n] = torch.arange(k0, k1, dtype=torch.float64)

    def halo_bytes(self, which):
        return 16

    def halo_pack(self, which, side, buf):
        src = self.planes[2:4] if side == 0 else self.planes[self.n:self.n + 2]
        buf.copy_(src.clone().view(torch.uint8))

    def halo_unpack(self, which, side, buf):
        dst = slice(0, 2) if side == 0 else slice(self.n + 2, self.n + 4)
        self.planes[dst] = buf.clone().view(torch.float64)


class FakeSlab:
    def __init__(self, bc_z, rank, parts, nz):
        k0, k1 = slab.split_z(nz, parts)[rank]
        self.hz, self.nb = FakeHz(k0, k1), slab.neighbours(bc_z, rank, parts)
        self.k0, self.k1 = k0, k1


def _worker(rank, world, port, bc_z, nz, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    s = FakeSlab(bc_z, rank, world, nz)
    tr = slab.DistTransport()
    for _ in range(2):   # twice: the buffers are reused
        tr.exchange(s, B.HZ_HALO_PRIM, device="cpu")
    out[rank] = (s.k0, s.k1, s.hz.planes.tolist())
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("world,bc_z,port", [(2, B.HZ_BC_PERIODIC, 29741), (2, B.HZ_BC_OUTFLOW, 29742),
                                             (3, B.HZ_BC_PERIODIC, 29743), (3, B.HZ_BC_OUTFLOW, 29744)])
def test_dist_transport_fills_the_right_ghost_planes(world, bc_z, port):
    nz = 13
    with mp.Manager() as man:
        out = man.dict()
        mp.spawn(_worker, args=(world, port, bc_z, nz, out), nprocs=world, join=True)
        res = dict(out)
    for rank in range(world):
        k0, k1, planes = res[rank]
        lo, hi = planes[:2], planes[-2:]
        if bc_z == B.HZ_BC_PERIODIC:
            assert lo == [float((k0 - 2) % nz), float((k0 - 1) % nz)], (rank, planes)
            assert hi == [float(k1 % nz), float((k1 + 1) % nz)], (rank, planes)
        else:
            assert lo == ([-1.0, -1.0] if rank == 0 else [float(k0 - 2), float(k0 - 1)]), (rank, planes)
            assert hi == ([-1.0, -1.0] if rank == world - 1 else [float(k1), float(k1 + 1)]), (rank, planes)
        assert planes[2:-2] == [float(k) for k in range(k0, k1)]


class FakePeerHz:
    """Stand-in for a context in the fused exchange: records what hz_peer_attach is given."""

    def __init__(self, rank):
        self._buf = torch.zeros(64, dtype=torch.uint8)
        self.rank, self.attached, self.detached, self.nsub = rank, {}, [], 0

    def prim_buffers(self):
        b = self._buf.data_ptr()
        return b + 8, b + 24, 100 + self.rank

    def peer_attach(self, side, p0, p1, fs, nz):
        self.attached[side] = (p0, p1, fs, nz)

    def peer_detach(self, side):
        self.detached.append(side)

    def substeps(self, dt, n):
        self.nsub += n

    def close(self):
        pass


class FakeMapped:
    def __init__(self, rank):
        self.rank = rank

    def data_ptr(self):
        return 10000 * (self.rank + 1)


def _worker_fused(rank, world, port, bc_z, nz, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    d = object.__new__(slab.DistSlabHorizon)           # the rank logic without a GPU context
    k0, k1 = slab.split_z(nz, world)[rank]
    sl = type("S", (), {})()
    sl.hz, sl.nb, sl.nz = FakePeerHz(rank), slab.neighbours(bc_z, rank, world), k1 - k0
    d.rank, d.parts, d.group, d.device, d.fused, d.slab = rank, world, None, "cpu", True, sl
    d._ipc_export = lambda buf: ("handle of rank", rank)          # stands in for the CUDA IPC handle
    d._ipc_open = lambda blob: FakeMapped(blob[1])
    d._attach_over_ipc()
    d.substeps(0.1, 3)
    d.close()
    out[rank] = (sl.nb, dict(sl.hz.attached), list(sl.hz.detached), sl.hz.nsub)
    dist.destroy_process_group()


@pytest.mark.parametrize("world,bc_z,port", [(2, B.HZ_BC_PERIODIC, 29745), (3, B.HZ_BC_OUTFLOW, 29746)])
def test_fused_exchange_attaches_the_right_neighbour_buffers(world, bc_z, port):
    """DistSlabHorizon(fused=True): every rank exports its buffer, gathers the handles, and attaches to each external
    side the buffers, field stride and plane count OF THAT SIDE'S NEIGHBOUR (a periodic ring of two attaches the one
    other rank on both sides); substeps are taken one at a time with a barrier after each; close detaches."""
    nz = 13
    sizes = [k1 - k0 for k0, k1 in slab.split_z(nz, world)]
    with mp.Manager() as man:
        out = man.dict()
        mp.spawn(_worker_fused, args=(world, port, bc_z, nz, out), nprocs=world, join=True)
        res = dict(out)
    for rank in range(world):
        nb, attached, detached, nsub = res[rank]
        assert nsub == 3
        assert sorted(attached) == [s for s in (0, 1) if nb[s] is not None] == sorted(detached)
        for side, (p0, p1, fs, pnz) in attached.items():
            o = nb[side]
            assert (p0, p1, fs, pnz) == (10000 * (o + 1) + 8, 10000 * (o + 1) + 24, 100 + o, sizes[o]), (rank, side)
