"""NEXT-2 host logic on CPU (reading A20): the z-slab decomposition with
8 overlap planes and one exchange per RK stage reproduces the single-domain result BITWISE on the owned
planes.  The oracle stands in for the CUDA solver (same BC code EXTERNAL, same exchange plan from
paper_2505_07392_b200/slab.py); the two-rank gloo test moves the planes with torch.distributed."""
import os
import socket
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from oracle import igr_ref as R
from paper_2505_07392_b200 import slab as S
from paper_2505_07392_b200 import workloads as W
import parity

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
NGP = 3


def small_jets():
    """A 24 x 20 x 48 cut of the jets recipe: inflow patches on z-, extrapolation elsewhere."""
    import dataclasses
    w = W.jets9(n=24, radius=3, pitch=8)
    return dataclasses.replace(w, ny=20, nz=48)


def periodic_tg():
    import dataclasses
    w = W.taylor_green(16)
    return dataclasses.replace(w, nz=44, global_shape=None)


def run_global(w, dts):
    ref = parity.oracle_for(w)
    ref.set_state(W.state(w).numpy().astype(np.float64))
    for dt in dts:
        ref.step(dt)
    return ref.get_state(), ref.get_sigma()


def exchange_in_process(slabs, refs):
    """Pull plan of slab.py applied to padded oracle arrays."""
    pads = [[r.get_padded(c) for c in range(6)] for r in refs]
    new = [[a.copy() for a in p] for p in pads]
    for sl in slabs:
        for t in S.receives(sl, lambda r: slabs[r]):
            for c in range(6):
                new[sl.rank][c][t.dst + NGP:t.dst + NGP + t.count] = pads[t.peer][c][t.src + NGP:t.src + NGP + t.count]
    for r, p in zip(refs, new):
        for c in range(6):
            r.set_padded(c, p[c])


@pytest.mark.parametrize("case,nranks,n_jacobi", [("jets", 2, 5), ("jets", 3, 5), ("tg_periodic", 2, 5),
                                                   ("tg_periodic", 3, 5), ("jets", 2, 7), ("tg_periodic", 2, 3)])
def test_slabs_with_stage_exchange_equal_the_global_run_bitwise(case, nranks, n_jacobi):
    """The overlap follows the sweep count (slab.overlap_for: n_jacobi + 3): 7 sweeps need 10 planes, 3 need 6."""
    import dataclasses
    w = small_jets() if case == "jets" else periodic_tg()
    w = dataclasses.replace(w, n_jacobi=n_jacobi)
    slabs = [S.make_slab(w, r, nranks) for r in range(nranks)]
    assert all(sl.overlap == n_jacobi + 3 and sl.halo == n_jacobi + 6 for sl in slabs)
    refs = []
    for sl in slabs:
        r = parity.oracle_for(sl.local)
        r.set_state(S.local_state(w, sl).numpy().astype(np.float64))
        refs.append(r)
    exchange_in_process(slabs, refs)                       # ghost planes of the initial state
    # the global maximum is the maximum over the slabs
    g0 = parity.oracle_for(w)
    g0.set_state(W.state(w).numpy().astype(np.float64))
    assert max(r.max_wavespeed() for r in refs) == g0.max_wavespeed()
    dts = []
    for _ in range(2):
        dt = w.cfl * w.dx / max(r.max_wavespeed() for r in refs)
        dts.append(dt)
        for stage in (1, 2, 3):
            for r in refs:
                r.stage(stage, dt)
            exchange_in_process(slabs, refs)
    q, sig = run_global(w, dts)
    for sl, r in zip(slabs, refs):
        ql, sl_sig = r.get_state(), r.get_sigma()
        assert np.array_equal(ql[:, sl.own_lo:sl.own_hi], q[:, sl.z0:sl.z1])
        assert np.array_equal(sl_sig[sl.own_lo:sl.own_hi], sig[sl.z0:sl.z1])
        # the overlap planes too (they were just overwritten by the neighbours' owned planes)
        idx = np.arange(sl.e0, sl.e1) % w.nz
        assert np.array_equal(ql, q[:, idx])


def test_six_overlap_planes_are_not_enough():
    """The bound is sharp.  In the oracle the ghost planes beyond an EXTERNAL face keep the neighbour's
    previous iterate, so its first sweep is still exact there: 4 contaminated planes + 3 stencil planes = 7
    are needed and 6 fail.  (The CUDA sweeps clamp at the extended boundary in every sweep: 5 + 3 = 8,
    the value slab.py uses.)"""
    w = periodic_tg()
    slabs = [S.make_slab(w, r, 2, overlap=6) for r in range(2)]
    refs = []
    for sl in slabs:
        r = parity.oracle_for(sl.local)
        r.set_state(S.local_state(w, sl).numpy().astype(np.float64))
        refs.append(r)

    def exch():
        pads = [[r.get_padded(c) for c in range(6)] for r in refs]
        new = [[a.copy() for a in p] for p in pads]
        for sl in slabs:
            for side, dst, src in ((0, -NGP, slabs[sl.lo].own_hi - 9), (1, sl.own_hi, slabs[sl.hi].own_lo)):
                peer = sl.lo if side == 0 else sl.hi
                for c in range(6):
                    new[sl.rank][c][dst + NGP:dst + NGP + 9] = pads[peer][c][src + NGP:src + NGP + 9]
        for r, p in zip(refs, new):
            for c in range(6):
                r.set_padded(c, p[c])

    exch()
    # a nonzero Sigma warm start makes the missing neighbour visible in the first stage already
    dt = w.cfl * w.dx / max(r.max_wavespeed() for r in refs)
    for _ in range(2):
        for stage in (1, 2, 3):
            for r in refs:
                r.stage(stage, dt)
            exch()
    q, _ = run_global(w, [dt, dt])
    sl = slabs[0]
    assert not np.array_equal(refs[0].get_state()[:, sl.own_lo:sl.own_hi], q[:, sl.z0:sl.z1])


def test_split_and_plan_geometry():
    assert S.split(10, 3) == [(0, 4), (4, 7), (7, 10)]
    w = small_jets()
    a, b = S.make_slab(w, 0, 2), S.make_slab(w, 1, 2)
    assert (a.z0, a.z1, a.e0, a.e1, a.lo, a.hi) == (0, 24, 0, 32, -1, 1)
    assert (b.z0, b.z1, b.e0, b.e1, b.lo, b.hi) == (24, 48, 16, 48, 0, -1)
    assert a.local.faces[4] == w.faces[4] and a.local.faces[5] == S.EXTERNAL
    assert b.local.faces[4] == S.EXTERNAL and b.local.faces[5] == w.faces[5]
    assert 4 in a.local.patches and 4 not in b.local.patches       # the jets enter through z- of rank 0
    ra, rb = S.receives(a, lambda r: b), S.receives(b, lambda r: a)
    assert [(t.peer, t.side, t.dst, t.src, t.count) for t in ra] == [(1, 1, 24, 8, 11)]
    assert [(t.peer, t.side, t.dst, t.src, t.count) for t in rb] == [(0, 0, -3, 13, 11)]
    sa = S.sends(a, lambda r: b)
    assert [(t.peer, t.side, t.dst, t.src, t.count) for t in sa] == [(1, 0, -3, 13, 11)]
    with pytest.raises(AssertionError):
        S.make_slab(w, 0, 5)                                        # 48 / 5 < 11 planes per slab
    one = S.make_slab(w, 0, 1)
    assert one.local is w and one.lo == one.hi == -1


# ------------------------------------------------------------------ two gloo ranks
def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world),
                      OMP_NUM_THREADS="2")
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        w = periodic_tg()
        sl = S.make_slab(w, rank, world)
        peers = {r: S.make_slab(w, r, world) for r in range(world)}
        ref = parity.oracle_for(sl.local)
        ref.set_state(S.local_state(w, sl).numpy().astype(np.float64))

        def exchange():
            pads = [torch.from_numpy(ref.get_padded(c)) for c in range(6)]
            ops, bufs = [], []
            for t in S.sends(sl, lambda r: peers[r]):
                buf = torch.stack([p[t.src + NGP:t.src + NGP + t.count] for p in pads]).contiguous()
                ops.append(dist.P2POp(dist.isend, buf, t.peer, tag=t.side))
            for t in S.receives(sl, lambda r: peers[r]):
                buf = torch.empty((6, t.count) + tuple(pads[0].shape[1:]), dtype=torch.float64)
                bufs.append((t, buf))
                ops.append(dist.P2POp(dist.irecv, buf, t.peer, tag=t.side))
            for req in dist.batch_isend_irecv(ops):
                req.wait()
            for t, buf in bufs:
                for c in range(6):
                    pads[c][t.dst + NGP:t.dst + NGP + t.count] = buf[c]
            for c in range(6):
                ref.set_padded(c, pads[c].numpy())

        exchange()
        dts = []
        for _ in range(2):
            v = torch.tensor([ref.max_wavespeed()], dtype=torch.float64)
            dist.all_reduce(v, op=dist.ReduceOp.MAX)
            dt = w.cfl * w.dx / float(v)
            dts.append(dt)
            for stage in (1, 2, 3):
                ref.stage(stage, dt)
                exchange()
        q, sig = run_global(w, dts)
        ok = np.array_equal(ref.get_state()[:, sl.own_lo:sl.own_hi], q[:, sl.z0:sl.z1]) and \
            np.array_equal(ref.get_sigma()[sl.own_lo:sl.own_hi], sig[sl.z0:sl.z1])
        out.put((rank, bool(ok)))
    finally:
        dist.destroy_process_group()


def test_two_gloo_ranks_exchange_planes_and_match_the_global_run():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, out)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=300) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert res == [(0, True), (1, True)]
