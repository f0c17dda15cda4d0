"""Slab decomposition along z across GPUs.

The paper's multi-GPU layer is a block decomposition with a ghost-zone exchange after EVERY substep:
pack kernel -> device-to-host -> MPI -> host-to-device -> unpack kernel.  Here the exchange never leaves
the devices: `hz_halo_pack` -> NCCL send/recv over NVLink (torch.distributed) -> `hz_halo_unpack`, two
planes of the nine primitives each way per substep (19 MB per side at 256^2 in fp64, ~25 us on NVLink 5
against a ~5 ms substep; everything is ordered on the device, the host never waits).  All arithmetic stays in the C-ABI library; this
module only splits arrays, moves buffers and orders calls.

Two transports:
  * DistTransport  -- one process per GPU (torchrun), neighbours exchanged with batched isend/irecv;
  * LocalTransport -- all slabs in ONE process on one GPU, buffers handed over directly.  This is how the
    exchange is validated on a single B200: R slabs must reproduce the single-context run bitwise.
And no transport at all (fused=True): the neighbours' primitive buffers are attached to each context
(hz_peer_attach; between processes through CUDA IPC) and the substep kernel itself stores the planes next to a cut
into the neighbour's ghost planes -- between substeps there is one barrier and no kernel.
"""
import numpy as np

from .binding import (HZ_BC_EXTERNAL, HZ_BC_EXTERNAL_OUTFLOW, HZ_BC_OUTFLOW, HZ_BC_OUTFLOW_EXTERNAL, HZ_BC_PERIODIC,
                      HZ_HALO_METRIC, HZ_HALO_PRIM, Horizon, HzParams)


def split_z(nz, parts):
    """Contiguous z ranges [k0, k1) of `parts` slabs, sizes differing by at most one plane."""
    if parts < 1 or nz < 2 * parts:
        raise ValueError(f"cannot cut nz={nz} into {parts} slabs of at least 2 planes")
    base, rem = divmod(nz, parts)
    out, k = [], 0
    for r in range(parts):
        n = base + (1 if r < rem else 0)
        out.append((k, k + n))
        k += n
    return out


def slab_bc(bc_z, rank, parts):
    """Boundary code of the z axis of slab `rank`: inner cuts are external, the domain ends keep bc_z."""
    if parts == 1:
        return bc_z
    if bc_z == HZ_BC_PERIODIC:
        return HZ_BC_EXTERNAL           # the wrap-around is a neighbour too
    if bc_z != HZ_BC_OUTFLOW:
        raise ValueError("global z boundary must be periodic or outflow")
    if rank == 0:
        return HZ_BC_OUTFLOW_EXTERNAL   # low side: domain end, high side: neighbour
    if rank == parts - 1:
        return HZ_BC_EXTERNAL_OUTFLOW
    return HZ_BC_EXTERNAL


def neighbours(bc_z, rank, parts):
    """(low, high) neighbour ranks of a slab, None at an outflow domain end."""
    if parts == 1:
        return (None, None)
    if bc_z == HZ_BC_PERIODIC:
        return ((rank - 1) % parts, (rank + 1) % parts)
    return (rank - 1 if rank > 0 else None, rank + 1 if rank < parts - 1 else None)


def slab_of(w, rank, parts):
    """Arguments of the local context of slab `rank`: (n, h, bc, slices of the input planes)."""
    k0, k1 = split_z(w.n[2], parts)[rank]
    sl = slice(k0, k1)
    n = (w.n[0], w.n[1], k1 - k0)
    bc = (w.bc[0], w.bc[1], slab_bc(w.bc[2], rank, parts))
    return n, tuple(w.h), bc, sl


class LocalTransport:
    """All slabs live in this process: a 'send' is handing the packed buffer to the neighbour's unpack."""

    def exchange(self, slabs, which):
        import torch
        bufs = {}
        for r, s in enumerate(slabs):
            nbytes = s.hz.halo_bytes(which)
            for side in (0, 1):
                if s.nb[side] is None:
                    continue
                b = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
                s.hz.halo_pack(which, side, b)
                bufs[(r, side)] = b
        for r, s in enumerate(slabs):
            for side in (0, 1):
                if s.nb[side] is None:
                    continue
                # my low ghosts are the high-side planes of the slab below me, and vice versa
                s.hz.halo_unpack(which, side, bufs[(s.nb[side], 1 - side)])
        # (no host synchronisation: packs, unpacks and the next substeps are ordered on the stream, and the caching
        # allocator reuses a freed buffer only behind them on that stream)


class DistTransport:
    """One slab per process; neighbours exchange with batched isend/irecv (NCCL on GPU tensors)."""

    def __init__(self, group=None):
        self.group = group
        self._buf = {}

    def _buffers(self, which, nbytes, device):
        import torch
        key = (which, nbytes)
        if key not in self._buf:
            self._buf[key] = [[torch.empty(nbytes, dtype=torch.uint8, device=device) for _ in range(2)]
                              for _ in range(2)]   # [send|recv][side]
        return self._buf[key]

    def exchange(self, slab, which, device="cuda"):
        import torch
        import torch.distributed as dist
        send, recv = self._buffers(which, slab.hz.halo_bytes(which), device)
        # gloo cannot send from device memory: with it (the one-GPU tests) the buffers go through the host.  NCCL,
        # the transport this module is for, sends them as they are.
        staged = torch.device(device).type == "cuda" and dist.get_backend(self.group) != "nccl"
        wire_send, wire_recv = ([None, None], [None, None]) if staged else (send, recv)
        # NCCL pairs the sends and receives between two ranks in posting order (it has no tags; none are used
        # here, so gloo in the CPU test matches the same way).  Sends go
        # low side first; receives are posted high side first, because a neighbour's low-side planes land in
        # my HIGH ghosts -- this is what makes a 2-rank periodic ring (both neighbours the same rank) pair up.
        sends, recvs = [], []
        for side in (0, 1):
            nb = slab.nb[side]
            if nb is None:
                continue
            slab.hz.halo_pack(which, side, send[side])       # on the current stream; NCCL waits for it
            if staged:
                wire_send[side] = send[side].cpu()
            sends.append(dist.P2POp(dist.isend, wire_send[side], nb, self.group))
        for side in (1, 0):
            nb = slab.nb[side]
            if nb is not None:
                if staged:
                    wire_recv[side] = torch.empty(recv[side].shape, dtype=torch.uint8)
                recvs.append(dist.P2POp(dist.irecv, wire_recv[side], nb, self.group))
        if sends or recvs:
            # With NCCL, wait() does not block the host: it makes the current stream wait for the transfer, so
            # the unpack kernels below are ordered behind it on the device and hz_step stays asynchronous.
            # (gloo, used by the CPU tests, completes the transfer inside wait().)
            for req in dist.batch_isend_irecv(sends + recvs):
                req.wait()
        for side in (0, 1):
            if slab.nb[side] is not None:
                if staged:
                    recv[side].copy_(wire_recv[side])
                slab.hz.halo_unpack(which, side, recv[side])


class Slab:
    """One slab: a Horizon context plus its place in the decomposition.

    `w` is the GLOBAL workload, of which this slab keeps its z range -- or, with local=True, already this rank's
    own planes of a global grid that no process holds as a whole (weak scaling: workloads.kerr_sweep(zslab=...));
    w.bc then still names the GLOBAL boundary kinds."""

    def __init__(self, w, rank, parts, dtype="f64", local=False, **kw):
        if local:
            n, h, sl = tuple(w.n), tuple(w.h), slice(None)
            bc = (w.bc[0], w.bc[1], slab_bc(w.bc[2], rank, parts))
        else:
            n, h, bc, sl = slab_of(w, rank, parts)
        self.rank, self.parts, self.sl = rank, parts, sl
        self.nb = neighbours(w.bc[2], rank, parts)
        self.ncell = n[0] * n[1] * n[2]
        self.nz = n[2]
        self.hz = Horizon(n, h, bc, dtype=dtype, params=HzParams.default(**w.params), **kw)
        self._w = w

    def set_metric(self):
        w, sl = self._w, self.sl
        self.hz.set_metric(np.ascontiguousarray(w.alpha[sl]), np.ascontiguousarray(w.beta3[:, sl]),
                           np.ascontiguousarray(w.gamma6[:, sl]))

    def set_primitives(self):
        self.hz.set_primitives(np.ascontiguousarray(self._w.prim8[:, self.sl]))

    def sync(self):
        import torch
        torch.cuda.current_stream().synchronize()


def attach_neighbours(slabs):
    """Mutual hz_peer_attach of slabs that live in one process (their buffers are plain device addresses; on
    several GPUs of one process they are peer-mapped addresses once peer access is enabled)."""
    for s in slabs:
        for side in (0, 1):
            if s.nb[side] is not None:
                o = slabs[s.nb[side]]
                p0, p1, fs = o.hz.prim_buffers()
                s.hz.peer_attach(side, p0, p1, fs, o.nz)


class SlabGroup:
    """R slabs in one process on one GPU, stepped in lockstep (validation of the exchange).
    `w`: the global workload, or a list of per-slab workloads (local slabs, see Slab)."""

    def __init__(self, w, parts, dtype="f64", fused=False, **kw):
        self.w, self.parts, self.fused = w, parts, fused
        if isinstance(w, (list, tuple)):
            self.slabs = [Slab(w[r], r, parts, dtype, local=True, **kw) for r in range(parts)]
        else:
            self.slabs = [Slab(w, r, parts, dtype, **kw) for r in range(parts)]
        self.tr = LocalTransport()
        for s in self.slabs:
            s.set_metric()
        self.tr.exchange(self.slabs, HZ_HALO_METRIC)
        for s in self.slabs:
            s.set_primitives()
        self.tr.exchange(self.slabs, HZ_HALO_PRIM)
        if fused:
            # fused=True: the exchange of the primitives is part of the substep kernel (hz_peer_attach): every slab
            # stores its planes next to a cut straight into the neighbour's ghost planes.  All slabs run on one
            # stream here, so a slab's next substep is ordered behind its neighbours' last one.
            attach_neighbours(self.slabs)

    def substeps(self, dt, nsub):
        for _ in range(nsub):
            for s in self.slabs:
                s.hz.substeps(dt, 1)
            if not self.fused:
                self.tr.exchange(self.slabs, HZ_HALO_PRIM)

    def get_primitives(self):
        return np.concatenate([s.hz.get_primitives() for s in self.slabs], axis=1)

    def diagnostics(self):
        return combine_diagnostics([s.hz.diagnostics() for s in self.slabs], [s.ncell for s in self.slabs])

    def close(self):
        for s in self.slabs:
            s.hz.close()


SUM_KEYS = ("sumD", "sumSx", "sumSy", "sumSz", "sumTau", "sumBx", "sumBy", "sumBz", "sumPsi",
            "c2p_fail", "atm_reset", "p_floor", "c2p_stalled")
MAX_KEYS = ("divB_max", "max_speed_over_dx", "c2p_maxit_seen")


def combine_diagnostics(ds, ncells):
    """Global reductions from per-slab ones: sums add, maxima take the max, the mean |div B| is cell-weighted."""
    out = {k: sum(d[k] for d in ds) for k in SUM_KEYS}
    out.update({k: max(d[k] for d in ds) for k in MAX_KEYS})
    out["divB_L1"] = sum(d["divB_L1"] * n for d, n in zip(ds, ncells)) / float(sum(ncells))
    return out


class DistSlabHorizon:
    """This rank's slab of a global workload under torch.distributed (one process per GPU).

    Every rank builds the same seeded global workload and keeps its z range -- or (local=True) builds only its
    own planes.  `substeps` runs one substep and one halo exchange at a time; `diagnostics` all-reduces the
    scalars.
    """

    def __init__(self, w, dtype="f64", group=None, device="cuda", local=False, fused=False):
        import torch.distributed as dist
        self.rank, self.parts = dist.get_rank(group), dist.get_world_size(group)
        self.group, self.device, self.fused = group, device, fused
        self.slab = Slab(w, self.rank, self.parts, dtype, local=local)
        self.tr = DistTransport(group)
        self.slab.set_metric()
        self.tr.exchange(self.slab, HZ_HALO_METRIC, device)
        self.slab.set_primitives()
        self.tr.exchange(self.slab, HZ_HALO_PRIM, device)
        if fused:
            self._attach_over_ipc()

    def _attach_over_ipc(self):
        """fused=True: the exchange of the primitives as part of the substep kernel across PROCESSES of one node.
        Every rank exports its state buffer as a CUDA IPC handle, the ranks gather the handles, a rank opens its
        neighbours' buffers (over NVLink they are peer memory) and attaches them (hz_peer_attach); from then on
        the only traffic between substeps is a barrier."""
        import torch
        import torch.distributed as dist
        hz = self.slab.hz
        p0, p1, fs = hz.prim_buffers()
        base = hz._buf.data_ptr()
        mine = dict(ipc=self._ipc_export(hz._buf), off0=p0 - base, off1=p1 - base, fs=fs, nz=self.slab.nz)
        infos = [None] * self.parts
        dist.all_gather_object(infos, mine, group=self.group)
        self._mapped = {}
        for side in (0, 1):
            nb = self.slab.nb[side]
            if nb is None:
                continue
            if nb not in self._mapped:
                self._mapped[nb] = self._ipc_open(infos[nb]["ipc"])   # the neighbour's state buffer in this address space
            b = self._mapped[nb].data_ptr()
            hz.peer_attach(side, b + infos[nb]["off0"], b + infos[nb]["off1"], infos[nb]["fs"], infos[nb]["nz"])
        self._token = torch.zeros(1, device=self.device)
        self._lockstep()

    @staticmethod
    def _ipc_export(buf):
        """A picklable CUDA IPC handle of the tensor `buf` (torch's own: the allocation's handle plus the offset)."""
        from torch.multiprocessing.reductions import reduce_tensor
        return reduce_tensor(buf)

    @staticmethod
    def _ipc_open(blob):
        rebuild, args = blob
        return rebuild(*args)

    def _lockstep(self):
        """No rank starts substep s + 1 before its neighbours' substep s has stored into its ghost planes.  With NCCL
        a one-element all-reduce is that barrier ON THE DEVICE (stream-ordered, the host does not wait); other
        backends (gloo in the one-GPU test) synchronise the stream and meet at a host barrier."""
        import torch
        import torch.distributed as dist
        if dist.get_backend(self.group) == "nccl":
            dist.all_reduce(self._token, group=self.group)
        else:
            if torch.device(self.device).type == "cuda":
                torch.cuda.current_stream().synchronize()
            dist.barrier(group=self.group)

    def substeps(self, dt, nsub):
        for _ in range(nsub):
            self.slab.hz.substeps(dt, 1)
            if self.fused:
                self._lockstep()
            else:
                self.tr.exchange(self.slab, HZ_HALO_PRIM, self.device)

    def step(self, dt, n):
        self.substeps(dt, 3 * n)

    def get_primitives(self):
        return self.slab.hz.get_primitives()

    def diagnostics(self):
        import torch
        import torch.distributed as dist
        d = self.slab.hz.diagnostics()
        sums = torch.tensor([float(d[k]) for k in SUM_KEYS] + [d["divB_L1"] * self.slab.ncell, float(self.slab.ncell)],
                            dtype=torch.float64, device=self.device)
        maxs = torch.tensor([float(d[k]) for k in MAX_KEYS], dtype=torch.float64, device=self.device)
        dist.all_reduce(sums, op=dist.ReduceOp.SUM, group=self.group)
        dist.all_reduce(maxs, op=dist.ReduceOp.MAX, group=self.group)
        out = {k: float(v) for k, v in zip(SUM_KEYS, sums[:len(SUM_KEYS)].tolist())}
        out.update({k: float(v) for k, v in zip(MAX_KEYS, maxs.tolist())})
        out["divB_L1"] = float(sums[-2] / sums[-1])
        for k in ("c2p_fail", "atm_reset", "p_floor", "c2p_stalled", "c2p_maxit_seen"):
            out[k] = int(round(out[k]))
        return out

    def close(self):
        if self.fused:
            # nobody unmaps a buffer a neighbour may still store into
            self._lockstep()
            for side in (0, 1):
                if self.slab.nb[side] is not None:
                    self.slab.hz.peer_detach(side)
            self._mapped = {}
            self._lockstep()
        self.slab.hz.close()


def _time_slabs(n, parts, dtype, steps):
    """One-GPU measurement of what the slab decomposition itself costs: `parts` slabs of the n^3 Kerr-Schild box as
    `parts` contexts in one process (pack kernel, device-to-device hand-over, unpack kernel after every substep, the
    extra ghost planes) against the single context.  It is NOT a multi-GPU measurement: no NCCL, no NVLink."""
    import json
    import sys
    import os
    import torch
    sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
    import workloads as wl
    w = wl.kerr_sweep(n)
    out = {}
    for name, make in (("single", lambda: Horizon.from_workload(w, dtype=dtype)), ("slabs", lambda: SlabGroup(w, parts, dtype)),
                       ("fused", lambda: SlabGroup(w, parts, dtype, fused=True))):
        obj = make()
        run = (lambda k: obj.substeps(w.dt, 3 * k))
        run(2)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        run(steps)
        e1.record()
        torch.cuda.synchronize()
        out[name] = w.ncell * 3 * steps / (e0.elapsed_time(e1) * 1e-3)
        obj.close()
    out.update(n=n, parts=parts, dtype=dtype, steps=steps, slab_over_single=out["slabs"] / out["single"],
               fused_over_single=out["fused"] / out["single"])
    print(json.dumps(out))


if __name__ == "__main__":
    import argparse
    ap = argparse.ArgumentParser(description=_time_slabs.__doc__)
    ap.add_argument("--n", type=int, default=256)
    ap.add_argument("--parts", type=int, default=2)
    ap.add_argument("--dtype", default="f64")
    ap.add_argument("--steps", type=int, default=5)
    a = ap.parse_args()
    _time_slabs(a.n, a.parts, a.dtype, a.steps)
