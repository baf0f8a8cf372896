"""Multi-GPU driver of the hot path: one process per GPU, z-slab decomposition, one halo exchange per RK
stage (reading A20).

The plan (who owns which planes, which planes move) is slab.py; the copies are igr_pull_halo of the C
library (cudaMemcpyAsync device-to-device from the neighbour's allocation, opened once with CUDA IPC:
copy engines over NVLink, no SM time, no staging).  The ORDER of a pull after the neighbours' stage, and of the
next stage after the neighbours' pulls, is stream-ordered: interprocess CUDA events (igr_event_*), waited for
with cudaStreamWaitEvent on the solver's stream.  No device synchronisation happens inside a step: the hosts only
exchange a host-side handshake (a barrier of a gloo group: "my record is enqueued") while the GPUs keep
running, so a rank's pull waits for its two neighbours and nothing else.  torch.distributed carries the
rendezvous (all-gather of the igr_export descriptions and of the event handles at start-up), those handshakes,
and the max-reduction of the wave speed (one float per step, CFL condition).
`exchange="sendrecv"` moves the same planes with torch.distributed point-to-point calls instead (NCCL
send/recv over NVLink with the nccl backend; host staging with gloo): the path for nodes where CUDA IPC
is not permitted.
"""
import ctypes as C

import numpy as np
import torch
import torch.distributed as dist

from . import igr, slab as S


class _DevMem:
    """Raw device memory as a __cuda_array_interface__ object (for torch.as_tensor)."""

    def __init__(self, ptr, nbytes):
        self.__cuda_array_interface__ = {"shape": (nbytes,), "typestr": "|u1", "data": (ptr, False), "version": 2}


def _gather_bytes(blob, group):
    """All-gather of equal-length byte strings (works on gloo and nccl)."""
    world = dist.get_world_size(group)
    t = torch.frombuffer(bytearray(blob), dtype=torch.uint8).clone()
    dev = "cuda" if dist.get_backend(group) == "nccl" else "cpu"
    t = t.to(dev)
    outs = [torch.empty_like(t) for _ in range(world)]
    dist.all_gather(outs, t, group=group)
    return [bytes(o.cpu().numpy().tobytes()) for o in outs]


class SlabSolver:
    """The solver of rank `rank`'s slab of the global workload `w` plus the exchange with its neighbours.

    exchange: "ipc" (default) | "sendrecv" | "local" (all slabs in this process: `peers` gives the other
    SlabSolver objects; single-GPU tests of the pull path)."""

    def __init__(self, w, rank=None, nranks=None, group=None, exchange="ipc", device=None, **solver_kw):
        self.group = group
        self.rank = dist.get_rank(group) if rank is None else rank
        self.nranks = dist.get_world_size(group) if nranks is None else nranks
        self.w = w
        self.slab = S.make_slab(w, self.rank, self.nranks)
        self.peer_slabs = {r: S.make_slab(w, r, self.nranks) for r in {self.slab.lo, self.slab.hi} if r >= 0}
        self.exchange_kind = exchange if self.nranks > 1 else "none"
        device = device or "cuda:%d" % torch.cuda.current_device()
        # the library owns its memory (cudaMalloc) so that the allocation has an IPC handle of its own
        self.solver = igr.Solver.for_workload(self.slab.local, device=device, own_workspace=False, **solver_kw)
        if self.nranks > 1:                       # CFL reduction over the owned planes only
            self.solver.set_wave_range(self.slab.own_lo, self.slab.own_hi)
        self._opened = []
        self._nb_events = []                      # (stage complete, pulls complete) events of the neighbours
        self._hgroup = None                       # host-only group for the handshakes of the event ordering
        self._recv = S.receives(self.slab, lambda r: self.peer_slabs[r])
        self._send = S.sends(self.slab, lambda r: self.peer_slabs[r])
        if self.exchange_kind == "ipc":
            self._connect_ipc()

    # ---- set-up
    def _connect_ipc(self):
        mine = self.solver.export_fields()
        blobs = _gather_bytes(bytes(mine), self.group)
        ok = 1
        try:
            for t in self._recv:
                peer = igr.Export.from_buffer_copy(blobs[t.peer])
                base = igr.ipc_open(peer)
                self._opened.append(base)
                self.solver.set_neighbor(t.side, peer, base, t.dst, t.src, t.count)
        except igr.IgrError:
            ok = 0
        # all ranks use the same kind of exchange: if CUDA IPC was refused anywhere, nobody uses it
        dev = self.solver.device if dist.get_backend(self.group) == "nccl" else "cpu"
        flag = torch.tensor([ok], dtype=torch.int32, device=dev)
        dist.all_reduce(flag, op=dist.ReduceOp.MIN, group=self.group)
        if int(flag.item()) == 0:
            for side in (0, 1):
                self.solver.set_neighbor(side, None, None, 0, 0, 0)
            for b in self._opened:
                igr.ipc_close(b)
            self._opened = []
            self.exchange_kind = "sendrecv"
            return
        # interprocess events: every rank publishes the handles of its two events, opens its neighbours'
        handles = _gather_bytes(self.solver.event_handle(0) + self.solver.event_handle(1), self.group)
        for r in sorted({t.peer for t in self._recv}):
            self._nb_events.append((igr.event_open(handles[r][:64]), igr.event_open(handles[r][64:])))
        # the handshakes must not enter the CUDA stream: a gloo group beside an nccl one
        self._hgroup = self.group if dist.get_backend(self.group) == "gloo" else dist.new_group(backend="gloo")

    def connect_local(self, solvers):
        """exchange="local": `solvers[r]` is the SlabSolver of rank r in this process."""
        assert self.exchange_kind == "local"
        for t in self._recv:
            peer = solvers[t.peer].solver.export_fields()
            self.solver.set_neighbor(t.side, peer, peer.base, t.dst, t.src, t.count)

    def close(self):
        for side in (0, 1):
            if self.solver._h:
                self.solver.set_neighbor(side, None, None, 0, 0, 0)
        for b in self._opened:
            igr.ipc_close(b)
        self._opened = []
        for pair in self._nb_events:
            for ev in pair:
                igr.event_close(ev)
        self._nb_events = []
        self._barrier()                            # an exporter frees its memory only after every importer unmapped it
        self.solver.close()

    # ---- state
    def set_initial_state(self):
        """Workload state of the extended slab, then the ghost planes from the neighbours."""
        q = S.local_state(self.w, self.slab, device=self.solver.device)
        self.solver.set_state(q)
        del q
        self.exchange()

    def owned_state(self):
        return self.solver.get_state()[:, self.slab.own_lo:self.slab.own_hi]

    def owned_sigma(self):
        return self.solver.get_sigma()[self.slab.own_lo:self.slab.own_hi]

    # ---- the step
    def _barrier(self):
        if self.exchange_kind in ("ipc", "sendrecv"):
            dist.barrier(group=self.group)
            if dist.get_backend(self.group) == "nccl":
                torch.cuda.synchronize(self.solver.device)    # the barrier itself is a device collective

    def exchange(self):
        """After a stage: every rank's overlap and ghost planes <- the neighbours' owned planes."""
        if self.exchange_kind == "none":
            return
        if self.exchange_kind == "local":
            self.solver.pull_halo()               # one process, one stream: already ordered
            return
        if self.exchange_kind == "ipc":
            # stream-ordered: no device synchronisation, the GPU never waits for the hosts
            self.solver.event_record(0)                           # my stage is complete (in stream order)
            dist.barrier(group=self._hgroup)                      # host only: every rank has ENQUEUED that record
            for done, _ in self._nb_events:
                self.solver.event_wait(done)                      # my pulls wait for the neighbours' stage
            self.solver.pull_halo()
            self.solver.event_record(1)                           # my pulls are complete
            dist.barrier(group=self._hgroup)
            for _, pulled in self._nb_events:
                self.solver.event_wait(pulled)                    # my next stage waits for the neighbours' pulls
            return
        self.solver.sync()
        self._barrier()                           # the neighbours' stage is complete
        self._sendrecv()
        self.solver.sync()
        self._barrier()                           # nobody overwrites planes that are still being read

    def _plane_views(self, e, first_plane, count):
        """torch uint8 views of `count` planes from `first_plane` of the six exchanged fields."""
        pb = e.plane_bytes
        offs = [e.q_offset[e.cur][c] for c in range(5)] + [e.sig_offset[e.sig_cur]]
        return [torch.as_tensor(_DevMem(e.base + o + (first_plane + S.NG) * pb, count * pb), device=self.solver.device)
                for o in offs]

    def _sendrecv(self):
        e = self.solver.export_fields()
        staged = dist.get_backend(self.group) != "nccl"           # gloo: through host memory
        ops, landing = [], []
        for t in self._send:
            buf = torch.cat(self._plane_views(e, t.src, t.count))
            ops.append(dist.P2POp(dist.isend, buf.cpu() if staged else buf, t.peer, group=self.group, tag=t.side))
        for t in self._recv:
            views = self._plane_views(e, t.dst, t.count)
            n = sum(v.numel() for v in views)
            buf = torch.empty(n, dtype=torch.uint8, device="cpu" if staged else self.solver.device)
            landing.append((views, buf))
            ops.append(dist.P2POp(dist.irecv, buf, t.peer, group=self.group, tag=t.side))
        for req in dist.batch_isend_irecv(ops):
            req.wait()
        with torch.cuda.stream(self.solver.stream):
            for views, buf in landing:
                o = 0
                for v in views:
                    v.copy_(buf[o:o + v.numel()], non_blocking=False)
                    o += v.numel()

    def max_wavespeed(self):
        """Global maximum of |u_d| + c (CFL condition): local reduction kernel, then max over ranks."""
        try:
            v = self.solver.max_wavespeed()
        except igr.IgrError as e:                  # a non-finite slab must not leave the others waiting
            if e.code != igr.ERR_NONFINITE:
                raise
            v = float("inf")
        if self.exchange_kind in ("ipc", "sendrecv"):
            dev = self.solver.device if dist.get_backend(self.group) == "nccl" else "cpu"
            t = torch.tensor([v], dtype=torch.float64, device=dev)
            dist.all_reduce(t, op=dist.ReduceOp.MAX, group=self.group)
            v = float(t.item())
        if not np.isfinite(v):
            raise igr.IgrError(igr.ERR_NONFINITE, "non-finite state on some rank")
        return v

    def step(self, dt):
        assert self.exchange_kind != "local", "slabs sharing one process advance together: step_local"
        for stage in (1, 2, 3):
            self.solver.stage(stage, dt)
            self.exchange()


def step_local(solvers, dt):
    """exchange="local": all slabs live in this process (one GPU, one stream).  Every slab runs the stage,
    then every slab pulls: the pulls read owned planes and write overlap / ghost planes only."""
    for stage in (1, 2, 3):
        for s in solvers:
            s.solver.stage(stage, dt)
        for s in solvers:
            s.exchange()


def make_local(w, nranks, **solver_kw):
    """All `nranks` slabs of `w` in this process, connected, with their initial state."""
    solvers = [SlabSolver(w, rank=r, nranks=nranks, exchange="local", **solver_kw) for r in range(nranks)]
    for s in solvers:
        s.connect_local(solvers)
    for s in solvers:
        s.solver.set_state(S.local_state(w, s.slab, device=s.solver.device))
    for s in solvers:
        s.exchange()
    return solvers
