"""Seeded synthetic inputs for the five configurations of BASELINE.json.

This module serves BOTH the oracle tests and the CUDA path, and therefore holds none of the
method's arithmetic: it only samples initial conditions at cell centres (reading A13), converts
the given primitive state (rho, u, p) to the conserved state with the ideal-gas law (PAPER.md
eq. 4) and produces counter-based noise.  It imports neither the oracle nor the CUDA
library.  The paper's own cases (Mach-14 two-fluid jet, L274; ~1500-engine array, L343) are MFC
case files that are not available; configs 4-5 imitate their structure (many circular supersonic
inflow jets on one plane into gas at rest).

Arrays are generated with torch so that the large cases can be created directly in device
memory; layout [5][nz][ny][nx], x fastest, fp32 values derived from fp64 formulas.
"""
from dataclasses import dataclass, field, replace
import math

import torch

PERIODIC, EXTRAP, INFLOW = 0, 1, 2
_M32 = 0xFFFFFFFF


@dataclass
class Workload:
    name: str
    nx: int
    ny: int
    nz: int
    dx: float
    gamma: float = 1.4
    alpha: float = 0.0            # set to 10*dx^2 by the constructors below
    order: int = 5
    n_jacobi: int = 5
    faces: tuple = (0, 0, 0, 0, 0, 0)       # x-,x+,y-,y+,z-,z+
    patches: dict = field(default_factory=dict)  # face -> [(c0,c1,radius,edge,rho,u,v,w,p)]
    cfl: float = 0.5
    n_steps: int = 0
    t_end: float = 0.0
    origin: tuple = (0, 0, 0)     # global index of local cell (0,0,0) (sub-boxes)
    global_shape: tuple = None    # (nx,ny,nz) of the full domain the noise is indexed on
    kind: str = ""
    params: dict = field(default_factory=dict)
    gamma2: float = 0.0           # > 1: the two-fluid variant (NEXT-3, reading A21): `gamma` is fluid 1's exponent

    @property
    def n_cells(self):
        return self.nx * self.ny * self.nz

    @property
    def nf(self):                 # fields of the conserved state
        return 7 if self.gamma2 else 5


# --------------------------------------------------------------------------- noise
def _mix32(x):
    """32-bit integer finaliser (Wellons' lowbias32) evaluated in int64 tensors."""
    x = ((x ^ (x >> 16)) * 0x7FEB352D) & _M32
    x = ((x ^ (x >> 15)) * 0x846CA68B) & _M32
    return x ^ (x >> 16)


def hash_noise(gi, gj, gk, gshape, comp, seed):
    """Uniform noise in [-1, 1) as a pure function of the GLOBAL cell index, the component and
    the seed (counter-based, so any sub-box reproduces the full-domain values exactly)."""
    gnx, gny, _ = gshape
    lin = (gi + gnx * (gj + gny * gk)) & _M32
    h = _mix32(lin ^ ((seed * 0x9E3779B1 + comp * 0x85EBCA77) & _M32))
    h = _mix32((h + 0x6C8E9CF5 * (comp + 1)) & _M32)
    return h.to(torch.float64) * (2.0 / 4294967296.0) - 1.0


def _index_grids(w, device, kz0=0, nk=None):
    i0, j0, k0 = w.origin
    nk = w.nz if nk is None else nk
    gi = torch.arange(w.nx, dtype=torch.int64, device=device).view(1, 1, -1) + i0
    gj = torch.arange(w.ny, dtype=torch.int64, device=device).view(1, -1, 1) + j0
    gk = torch.arange(nk, dtype=torch.int64, device=device).view(-1, 1, 1) + (k0 + kz0)
    return gi, gj, gk


def _conserved(w, rho, u, v, ww, p, out_dtype, nk):
    """(rho, u, p) -> (rho, rho u, E) with E = p/(gamma-1) + rho |u|^2 / 2 (eq. 4)."""
    shape = (nk, w.ny, w.nx)
    rho, u, v, ww, p = (torch.broadcast_to(t, shape) for t in (rho, u, v, ww, p))
    q = torch.empty((5,) + shape, dtype=out_dtype, device=rho.device)
    q[0] = rho
    q[1] = rho * u
    q[2] = rho * v
    q[3] = rho * ww
    q[4] = p / (w.gamma - 1.0) + 0.5 * rho * (u * u + v * v + ww * ww)
    return q


def _conserved2(w, a1, rho1, rho2, u, v, ww, p, out_dtype, nk):
    """Two fluids (reading A21): (a1, rho1, rho2, u, p) -> (a1 rho1, a2 rho2, rho u, E, a1) with the isobaric
    mixture rule E = p Gamma + rho |u|^2 / 2, Gamma = a1/(gamma1 - 1) + (1 - a1)/(gamma2 - 1)."""
    shape = (nk, w.ny, w.nx)
    a1, rho1, rho2, u, v, ww, p = (torch.broadcast_to(t, shape) for t in (a1, rho1, rho2, u, v, ww, p))
    q = torch.empty((7,) + shape, dtype=out_dtype, device=a1.device)
    m1, m2 = a1 * rho1, (1.0 - a1) * rho2
    rho = m1 + m2
    q[0], q[1] = m1, m2
    q[2], q[3], q[4] = rho * u, rho * v, rho * ww
    q[5] = p * (a1 / (w.gamma - 1.0) + (1.0 - a1) / (w.gamma2 - 1.0)) + 0.5 * rho * (u * u + v * v + ww * ww)
    q[6] = a1
    return q


def state(w, device="cpu", dtype=torch.float32, slab=None):
    """Initial conserved state of workload `w`, [5][nz][ny][nx], generated on `device` (in z-slabs
    so that the fp64 temporaries of the large cases stay small)."""
    if slab is None:
        slab = max(1, min(w.nz, (1 << 24) // (w.nx * w.ny) or 1))
    if slab >= w.nz:
        return _state_slab(w, device, dtype, 0, w.nz)
    q = torch.empty((w.nf, w.nz, w.ny, w.nx), dtype=dtype, device=torch.device(device))
    for k0 in range(0, w.nz, slab):
        nk = min(slab, w.nz - k0)
        q[:, k0:k0 + nk] = _state_slab(w, device, dtype, k0, nk)
    return q


def state_planes(w, k0, nk, device="cpu", dtype=torch.float32):
    """Planes [k0, k0 + nk) of the initial state, [5][nk][ny][nx] (for grids filled slab by slab)."""
    return _state_slab(w, device, dtype, k0, nk)


def _state_slab(w, device, dtype, kz0, nk):
    dev = torch.device(device)
    gi, gj, gk = _index_grids(w, dev, kz0, nk)
    f64 = torch.float64
    one = torch.ones((), dtype=f64, device=dev)
    x = (gi.to(f64) + 0.5) * w.dx
    y = (gj.to(f64) + 0.5) * w.dx
    z = (gk.to(f64) + 0.5) * w.dx
    gshape = w.global_shape or (w.nx, w.ny, w.nz)
    P = w.params
    if w.kind == "entropy_wave":
        rho = 1.0 + 0.2 * torch.sin(2.0 * math.pi * (x + y + z))
        return _conserved(w, rho, one, one, one, one, dtype, nk)
    if w.kind == "sod":
        # the interface is smoothed over `smooth` cells (tanh half-width): the purely linear
        # scheme does not survive a grid-sharp start with alpha = 10 dx^2 (recipe)
        if P["smooth"] > 0:
            sl = 0.5 * (1.0 - torch.tanh((x - 0.5) / (P["smooth"] * w.dx)))
        else:
            sl = torch.where(x < 0.5, 1.0 * one, 0.0 * one)
        rho = 0.125 + (1.0 - 0.125) * sl
        p = 0.1 + (1.0 - 0.1) * sl
        if P["noise"] > 0:
            rho = rho * (1.0 + P["noise"] * hash_noise(gi, gj, gk, gshape, 0, P["seed"]))
        zero = 0.0 * one
        return _conserved(w, rho, zero, zero, zero, p, dtype, nk)
    if w.kind == "taylor_green":
        p0 = 1.0 / (w.gamma * P["mach"] ** 2)
        u = torch.sin(x) * torch.cos(y) * torch.cos(z)
        v = -torch.cos(x) * torch.sin(y) * torch.cos(z)
        p = p0 + (torch.cos(2 * x) + torch.cos(2 * y)) * (torch.cos(2 * z) + 2.0) / 16.0
        return _conserved(w, one, u, v, 0.0 * one, p, dtype, nk)
    if w.kind == "jets":
        amp, seed = P["noise"], P["seed"]
        # ambient at rest + a smoothed jet column above every inflow patch: the linear scheme
        # cannot start from a grid-sharp Mach-3 discontinuity (input recipe), so the
        # primitive state blends from the patch state to the ambient with a tanh profile of
        # half-width `delta` cells about the patch edge; by default the columns run through the
        # whole domain height (no impulsive-start vortex ring), else up to z = stub_height.
        # stub_delta = 0 is the configuration AS BASELINE.json STATES IT: grid-sharp patches (edge 0) into gas
        # at rest, no columns -- kept so that the tests can show where the scheme loses positivity on it.
        delta = P["stub_delta"]
        gx, gy, gz = gi.to(f64) + 0.5, gj.to(f64) + 0.5, gk.to(f64) + 0.5
        h = P.get("stub_height")               # None: columns through the whole domain
        s = torch.zeros((1, w.ny, w.nx), dtype=f64, device=dev)
        if delta > 0:
            sz = 1.0 if h is None else 0.5 * (1.0 - torch.tanh((gz - h) / delta))
            for cx, cy, rad in P["jet_centers"]:          # GLOBAL cell units (sub-box independent)
                rr = torch.sqrt((gx - cx) ** 2 + (gy - cy) ** 2)
                s = torch.maximum(s, 0.5 * (1.0 - torch.tanh((rr - rad) / delta)))
            s = s * sz
        rho_j, w_j, p_j = P["jet_state"]
        rho = 1.0 + (rho_j - 1.0) * s
        p = 1.0 + (p_j - 1.0) * s
        u = amp * hash_noise(gi, gj, gk, gshape, 1, seed)
        v = amp * hash_noise(gi, gj, gk, gshape, 2, seed)
        ww = amp * hash_noise(gi, gj, gk, gshape, 3, seed) + w_j * s
        if w.gamma2:
            # two fluids: the jet gas is fluid 1 (gamma), the gas at rest fluid 2 (gamma2); the volume fraction
            # follows the same profile s, kept inside (eps, 1 - eps) so that both partial densities stay positive
            eps = P.get("a1_floor", 1e-3)
            a1 = eps + (1.0 - 2.0 * eps) * s
            return _conserved2(w, a1, rho_j * one, 1.0 * one, u, v, ww, p, dtype, nk)
        return _conserved(w, rho, u, v, ww, p, dtype, nk)
    if w.kind == "two_fluid_vortex":
        # smooth periodic two-fluid test state: Taylor-Green-like velocity at Mach ~0.5, a smooth blob of fluid 1
        a1 = 0.5 + 0.4 * torch.sin(x) * torch.sin(y) * torch.cos(z)
        u = 0.5 * torch.sin(x) * torch.cos(y) * torch.cos(z) + 0.2
        v = -0.5 * torch.cos(x) * torch.sin(y) * torch.cos(z) - 0.1
        ww = 0.3 * torch.sin(z) * torch.cos(x)
        p = 1.0 + 0.1 * (torch.cos(2 * x) + torch.cos(2 * y)) * (torch.cos(2 * z) + 2.0) / 4.0
        return _conserved2(w, a1, 1.0 * one, 0.3 * one, u, v, ww, p, dtype, nk)
    if w.kind == "uniform":
        return _conserved(w, P["rho"] * one, P["u"] * one, P["v"] * one, P["w"] * one,
                          P["p"] * one, dtype, nk)
    raise ValueError(w.kind)


# --------------------------------------------------------------------------- the five configs
def entropy_wave(n=32):
    """Config 1: periodic entropy wave on [0,1]^3, rho = 1 + 0.2 sin(2 pi (x+y+z)), u=v=w=1, p=1."""
    dx = 1.0 / n
    return Workload("entropy_wave_%d" % n, n, n, n, dx, alpha=10 * dx * dx, n_steps=20,
                    kind="entropy_wave")


def entropy_wave_exact_rho(w, t, device="cpu"):
    """Exact translated wave rho(x,t) = 1 + 0.2 sin(2 pi (x+y+z-3t)) at cell centres (P10)."""
    gi, gj, gk = _index_grids(w, torch.device(device))
    s = (gi + gj + gk).to(torch.float64) * w.dx + 1.5 * w.dx
    return (1.0 + 0.2 * torch.sin(2.0 * math.pi * (s - 3.0 * t))).expand(w.nz, w.ny, w.nx)


def sod(nx=512, ny=32, nz=32, noise=1e-4, seed=2, smooth=4.0):
    """Config 2: planar Sod tube along x on [0,1], extrapolation in x, periodic in y, z."""
    dx = 1.0 / nx
    return Workload("sod_%dx%dx%d" % (nx, ny, nz), nx, ny, nz, dx, alpha=10 * dx * dx,
                    faces=(EXTRAP, EXTRAP, PERIODIC, PERIODIC, PERIODIC, PERIODIC), t_end=0.2,
                    kind="sod", params={"noise": noise, "seed": seed, "smooth": smooth})


def taylor_green(n=256, n_steps=200):
    """Config 3: inviscid compressible Taylor-Green vortex on [0,2 pi]^3, Mach 0.1."""
    dx = 2.0 * math.pi / n
    return Workload("taylor_green_%d" % n, n, n, n, dx, alpha=10 * dx * dx, n_steps=n_steps,
                    kind="taylor_green", params={"mach": 0.1})


def _jet_patches(centers, radius, edge, rho_j, p_j, mach, gamma):
    w_j = mach * math.sqrt(gamma * p_j / rho_j)
    return [(float(cx), float(cy), float(radius), float(edge), rho_j, 0.0, 0.0, w_j, p_j)
            for cx, cy in centers]


def jets9(n=512, n_steps=500, radius=10, pitch=60, noise=1e-3, seed=4, stub_delta=2.0):
    """Config 4: 3x3 array of underexpanded Mach-3 jets entering on z=0; dx = 1."""
    c = n // 2
    centers = [(c + pitch * a, c + pitch * b) for b in (-1, 0, 1) for a in (-1, 0, 1)]
    faces = (EXTRAP, EXTRAP, EXTRAP, EXTRAP, INFLOW, EXTRAP)
    return Workload("jets9_%d" % n, n, n, n, 1.0, alpha=10.0, faces=faces,
                    patches={4: _jet_patches(centers, radius, stub_delta, 0.5, 2.0, 3.0, 1.4)},
                    n_steps=n_steps, kind="jets", global_shape=(n, n, n),
                    params={"noise": noise, "seed": seed, "stub_delta": stub_delta,
                            "jet_centers": [(cx, cy, radius) for cx, cy in centers],
                            "jet_state": (0.5, 3.0 * math.sqrt(1.4 * 2.0 / 0.5), 2.0)})


def jets33(n=1024, n_steps=100, radius=8, rings=((14, 3), (44, 10), (84, 20)), noise=1e-3,
           seed=5, stub_delta=2.0):
    """Config 5: 33 jets in concentric rings of 3, 10, 20 (ring radii 14/44/84 cells: SURVEY 8(d),
    the config gives only counts and the patch radius); integer patch centres."""
    c = n // 2
    centers = []
    for R, cnt in rings:
        for m in range(cnt):
            th = 2.0 * math.pi * m / cnt
            centers.append((round(c + R * math.cos(th)), round(c + R * math.sin(th))))
    faces = (EXTRAP, EXTRAP, EXTRAP, EXTRAP, INFLOW, EXTRAP)
    return Workload("jets33_%d" % n, n, n, n, 1.0, alpha=10.0, faces=faces,
                    patches={4: _jet_patches(centers, radius, stub_delta, 0.5, 3.0, 3.0, 1.4)},
                    n_steps=n_steps, kind="jets", global_shape=(n, n, n),
                    params={"noise": noise, "seed": seed, "stub_delta": stub_delta,
                            "jet_centers": [(cx, cy, radius) for cx, cy in centers],
                            "jet_state": (0.5, 3.0 * math.sqrt(1.4 * 3.0 / 0.5), 3.0)})


def two_fluid_vortex(n=32, gamma1=1.4, gamma2=1.67):
    """Smooth periodic two-fluid state on [0, 2 pi]^3 (parity tests of the two-fluid variant)."""
    dx = 2.0 * math.pi / n
    return Workload("two_fluid_vortex_%d" % n, n, n, n, dx, gamma=gamma1, alpha=10 * dx * dx, kind="two_fluid_vortex",
                    gamma2=gamma2)


def two_fluid(w, gamma1=1.3, gamma2=1.4, a1_floor=1e-3):
    """The two-fluid variant of a jets workload (the paper's timed problem is a two-fluid jet, L274): the jet gas
    is fluid 1 (gamma1), the gas at rest fluid 2 (gamma2); the patches carry (a1, rho2) = (1 - a1_floor, 1)."""
    assert w.kind == "jets"
    patches = {f: [tuple(p[:9]) + (1.0 - a1_floor, 1.0) for p in pl] for f, pl in w.patches.items()}
    return replace(w, name=w.name.replace("jets", "jets2f"), gamma=gamma1, gamma2=gamma2, patches=patches,
                   params={**w.params, "a1_floor": a1_floor})


def uniform(nx, ny, nz, dx, rho, u, v, w, p, faces=(0, 0, 0, 0, 0, 0), patches=None):
    return Workload("uniform", nx, ny, nz, dx, alpha=10 * dx * dx, faces=faces,
                    patches=patches or {}, kind="uniform",
                    params={"rho": rho, "u": u, "v": v, "w": w, "p": p})


def subbox(w, lo, hi):
    """Dependency-cone sub-box [lo, hi) of a jets workload (SURVEY 8(c) "oracle reach"): the same
    global noise, patch centres shifted, the true BC on faces that coincide with a domain face
    and extrapolation (clamp) on the artificial ones."""
    assert w.kind == "jets"
    full = (w.nx, w.ny, w.nz)
    faces = []
    for a in range(3):
        faces.append(w.faces[2 * a] if lo[a] == 0 else EXTRAP)
        faces.append(w.faces[2 * a + 1] if hi[a] == full[a] else EXTRAP)
    patches = {}
    for f, plist in w.patches.items():
        a = f // 2
        on_face = (lo[a] == 0) if f % 2 == 0 else (hi[a] == full[a])
        if not on_face:
            continue
        t0, t1 = [b for b in range(3) if b != a]
        patches[f] = [(p[0] - lo[t0], p[1] - lo[t1]) + tuple(p[2:]) for p in plist]
    return replace(w, name=w.name + "_sub", nx=hi[0] - lo[0], ny=hi[1] - lo[1], nz=hi[2] - lo[2],
                   faces=tuple(faces), patches=patches,
                   origin=tuple(w.origin[a] + lo[a] for a in range(3)))
