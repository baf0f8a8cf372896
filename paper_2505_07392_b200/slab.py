"""z-slab domain decomposition of a workload over N ranks.

Host logic only: index arithmetic, no arithmetic of the method.  Used by the multi-GPU solver
(`paper_2505_07392_b200/dist.py`) and, with the oracle in place of the CUDA solver, by the CPU tests.

Scheme (reading A20).  The global grid is cut into N slabs of whole z-planes (z is the
slowest axis of the padded layout: a range of planes is ONE contiguous chunk per field, so the exchange
needs no pack kernels).  A rank's local solver works on its owned planes EXTENDED by `overlap` planes
on every side that has a neighbour; those faces carry the BC code EXTERNAL (ghosts are not filled by
the solver).  One RK stage computed on the extended slab is exact on the owned planes: the only wrong
inputs are the Sigma neighbours beyond the extended boundary, they contaminate one more plane per
Jacobi sweep, and the flux stencil reaches 3 planes: overlap = n_jacobi + 3 (8 with the 5 sweeps of every
configuration; `overlap_for`).  After every stage each rank overwrites its overlap and ghost planes
(overlap + 3 per side, q and Sigma) with the neighbour's owned planes.  Redundant work: 2 x overlap planes
per rank (1.6 % at 1024 planes).  The result on the owned planes is bitwise the single-domain result."""
from dataclasses import dataclass, replace

from .workloads import Workload, _state_slab

NG = 3               # ghost layers = planes the flux stencil reaches
EXTERNAL = 3         # BC code of a face shared with a neighbour (include/igr.h IGR_BC_EXTERNAL)
PERIODIC = 0


@dataclass
class Slab:
    rank: int
    nranks: int
    z0: int              # owned global planes [z0, z1)
    z1: int
    e0: int              # extended global planes [e0, e1) (beyond [0, nz) when the global z axis is periodic)
    e1: int
    lo: int              # neighbour rank below / above, or -1
    hi: int
    local: Workload      # the workload the local solver is created for (nz = e1 - e0)
    nz_global: int
    overlap: int = 0     # planes of redundant computation per side with a neighbour

    @property
    def own_lo(self):    # local index of the first owned plane
        return self.z0 - self.e0

    @property
    def own_hi(self):    # local index one past the last owned plane
        return self.z1 - self.e0

    @property
    def halo(self):      # planes received per side
        return self.overlap + NG


def overlap_for(w):
    """Planes of redundant computation per side with a neighbour: one per Jacobi sweep (the sweeps clamp at the
    extended boundary, the error moves one plane per sweep) plus the reach of the flux stencil."""
    return w.n_jacobi + NG


def split(nz, nranks):
    """Owned ranges: nranks contiguous slabs, sizes differing by at most one plane."""
    base, rem = divmod(nz, nranks)
    out, z = [], 0
    for r in range(nranks):
        n = base + (1 if r < rem else 0)
        out.append((z, z + n))
        z += n
    return out


def make_slab(w, rank, nranks, overlap=None):
    """The slab of global workload `w` owned by `rank` of `nranks`.  `overlap` defaults to `overlap_for(w)`;
    a smaller value is accepted only so that the tests can show that the bound is sharp."""
    assert 0 <= rank < nranks
    if overlap is None:
        overlap = overlap_for(w)
    periodic = w.faces[4] == PERIODIC
    if nranks == 1:
        return Slab(0, 1, 0, w.nz, 0, w.nz, -1, -1, w, w.nz, overlap)
    z0, z1 = split(w.nz, nranks)[rank]
    sizes = [b - a for a, b in split(w.nz, nranks)]
    assert min(sizes) >= overlap + NG, "slabs thinner than %d planes cannot feed their neighbours" % (overlap + NG)
    lo = rank - 1 if rank > 0 else (nranks - 1 if periodic else -1)
    hi = rank + 1 if rank < nranks - 1 else (0 if periodic else -1)
    e0 = z0 - (overlap if lo >= 0 else 0)
    e1 = z1 + (overlap if hi >= 0 else 0)
    faces = list(w.faces)
    faces[4] = EXTERNAL if lo >= 0 else w.faces[4]
    faces[5] = EXTERNAL if hi >= 0 else w.faces[5]
    patches = {}
    for f, plist in w.patches.items():
        a = f // 2
        if a == 2:                                   # z faces: only on the rank that has the domain face
            if (f == 4 and lo < 0) or (f == 5 and hi < 0):
                patches[f] = list(plist)
        else:                                        # x / y faces: the second transverse axis is z
            patches[f] = [(p[0], p[1] - e0) + tuple(p[2:]) for p in plist]
    gshape = w.global_shape or (w.nx, w.ny, w.nz)
    local = replace(w, name="%s_slab%dof%d" % (w.name, rank, nranks), nz=e1 - e0, faces=tuple(faces),
                    patches=patches, origin=(w.origin[0], w.origin[1], w.origin[2] + e0), global_shape=gshape)
    return Slab(rank, nranks, z0, z1, e0, e1, lo, hi, local, w.nz, overlap)


def local_state(w, slab, device="cpu", dtype=None):
    """Initial state of the extended slab, [5][e1-e0][ny][nx]: the global generator evaluated on wrapped
    global plane indices (so that periodic images are bitwise the planes they copy)."""
    import torch
    dtype = dtype or torch.float32
    chunk = max(1, (1 << 24) // (w.nx * w.ny))
    out = torch.empty((5, slab.e1 - slab.e0, w.ny, w.nx), dtype=dtype, device=torch.device(device))
    k = slab.e0
    while k < slab.e1:
        g = k % w.nz                                  # wrapped start
        n = min(slab.e1 - k, w.nz - g, chunk)
        out[:, k - slab.e0:k - slab.e0 + n] = _state_slab(w, device, dtype, g, n)
        k += n
    return out


@dataclass
class Transfer:
    """`count` planes of every exchanged field: the receiver's local planes [dst, dst + count) take the
    sender's local planes [src, src + count) (interior-relative plane indices: ghost planes are < 0 or
    >= nz; add NG for the index into the padded array)."""
    peer: int
    side: int            # 0: my low side, 1: my high side
    dst: int
    src: int
    count: int


def receives(slab, peer_slab_of):
    """What `slab` pulls after every stage.  `peer_slab_of(rank)` returns the neighbour's Slab."""
    out = []
    n = slab.halo
    if slab.lo >= 0:                                   # my planes [-NG, own_lo) <- their last n owned planes
        p = peer_slab_of(slab.lo)
        out.append(Transfer(slab.lo, 0, -NG, p.own_hi - n, n))
    if slab.hi >= 0:                                   # my planes [own_hi, nz + NG) <- their first n owned planes
        p = peer_slab_of(slab.hi)
        out.append(Transfer(slab.hi, 1, slab.own_hi, p.own_lo, n))
    return out


def sends(slab, peer_slab_of):
    """The transfers of my neighbours that read from me (for two-sided exchanges): Transfer.peer is the
    receiver, side the RECEIVER's side, src are MY planes, dst THEIR planes."""
    out = []
    n = slab.halo
    for nb in sorted({r for r in (slab.lo, slab.hi) if r >= 0}):
        p = peer_slab_of(nb)
        if p.lo == slab.rank:                          # I am below them: they take my last n owned planes
            out.append(Transfer(nb, 0, -NG, slab.own_hi - n, n))
        if p.hi == slab.rank:                          # I am above them: they take my first n owned planes
            out.append(Transfer(nb, 1, p.own_hi, slab.own_lo, n))
    return out
