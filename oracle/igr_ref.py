"""ctypes binding of the fp64 CPU oracle (oracle/igr_ref.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this module.  It imports nothing from the
CUDA package and shares no code with it.  See igr_ref.h for the citations.
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "igr_ref.c")
_SRC2 = os.path.join(_HERE, "igr_ref2.c")        # two-fluid variant (NEXT-3)
_LIB = os.path.join(_HERE, "libigr_ref.so")

PERIODIC, EXTRAP, INFLOW, EXTERNAL = 0, 1, 2, 3
STORE_F64, STORE_F32, STORE_F16, STORE_BF16 = 0, 1, 2, 3


def build(force=False):
    """Compile the oracle with gcc (plain C99, OpenMP on outer loops, no FMA contraction)."""
    if (not force and os.path.exists(_LIB)
            and os.path.getmtime(_LIB) >= max(os.path.getmtime(_SRC), os.path.getmtime(_SRC2),
                                              os.path.getmtime(os.path.join(_HERE, "igr_ref.h")))):
        return _LIB
    cmd = ["gcc", "-O2", "-fopenmp", "-ffp-contract=off", "-fPIC", "-shared", "-std=c99",
           "-Wall", "-Wextra", "-o", _LIB, _SRC, _SRC2, "-lm"]
    subprocess.check_call(cmd, cwd=_HERE)
    return _LIB


class _Patch(C.Structure):
    _fields_ = [(n, C.c_double) for n in ("c0", "c1", "radius", "edge", "rho", "u", "v", "w", "p")]


class _BC(C.Structure):
    _fields_ = [("face", C.c_int * 6), ("n_patches", C.c_int * 6),
                ("patches", C.POINTER(_Patch) * 6)]


class _Patch2(C.Structure):
    _fields_ = [(n, C.c_double) for n in ("c0", "c1", "radius", "edge", "a1rho1", "a2rho2", "a1", "u", "v", "w", "p")]


class _BC2(C.Structure):
    _fields_ = [("face", C.c_int * 6), ("n_patches", C.c_int * 6),
                ("patches", C.POINTER(_Patch2) * 6)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        dp = C.POINTER(C.c_double)
        vp = C.c_void_p
        _lib.igr_ref_create.argtypes = [C.c_int] * 3 + [C.c_double] * 3 + [C.c_int] * 2 + \
            [C.POINTER(_BC), C.POINTER(vp)]
        _lib.igr_ref_destroy.argtypes = [vp]
        _lib.igr_ref_destroy.restype = None
        _lib.igr_ref_set_storage.argtypes = [vp, C.c_int]
        _lib.igr_ref_set_viscosity.argtypes = [vp, C.c_double, C.c_double]
        _lib.igr_ref_viscous_flux.argtypes = [C.c_int, C.c_double, C.c_double, dp, dp, dp]
        _lib.igr_ref_viscous_flux.restype = None
        for name in ("set_state", "get_state", "set_sigma", "get_sigma", "get_source", "get_rhs",
                     "set_source",
                     "max_wavespeed"):
            getattr(_lib, "igr_ref_" + name).argtypes = [vp, dp]
        _lib.igr_ref_get_padded.argtypes = [vp, C.c_int, dp]
        _lib.igr_ref_set_padded.argtypes = [vp, C.c_int, dp]
        _lib.igr_ref_step.argtypes = [vp, C.c_double]
        _lib.igr_ref_stage.argtypes = [vp, C.c_int, C.c_double]
        for name in ("fill_ghosts", "source", "jacobi_sweep", "solve_sigma", "fill_sigma_ghosts",
                     "rhs", "eval_rhs"):
            getattr(_lib, "igr_ref_" + name).argtypes = [vp]
        _lib.igr_ref_rk_combine.argtypes = [C.c_double, dp, C.c_double, dp, C.c_double, dp, dp,
                                            C.c_long]
        _lib.igr_ref_rk_combine.restype = None
        _lib.igr_ref_reconstruct.argtypes = [C.c_int, dp, dp, dp]
        _lib.igr_ref_reconstruct.restype = None
        _lib.igr_ref_lf_flux.argtypes = [C.c_int, C.c_double, dp, dp, C.c_double, C.c_double,
                                         C.c_double, dp]
        _lib.igr_ref_lf_flux.restype = None
        _lib.igr_ref_round_storage.argtypes = [C.c_double, C.c_int]
        _lib.igr_ref_round_storage.restype = C.c_double
        _lib.igr_ref2_create.argtypes = [C.c_int] * 3 + [C.c_double] * 4 + [C.c_int] * 2 + \
            [C.POINTER(_BC2), C.POINTER(vp)]
        _lib.igr_ref2_destroy.argtypes = [vp]
        _lib.igr_ref2_destroy.restype = None
        for name in ("set_state", "get_state", "get_rhs", "get_sigma", "set_sigma", "get_source", "max_wavespeed"):
            getattr(_lib, "igr_ref2_" + name).argtypes = [vp, dp]
        _lib.igr_ref2_get_padded.argtypes = [vp, C.c_int, dp]
        _lib.igr_ref2_step.argtypes = [vp, C.c_double]
        _lib.igr_ref2_stage.argtypes = [vp, C.c_int, C.c_double]
        for name in ("fill_ghosts", "source", "solve_sigma", "rhs", "eval_rhs"):
            getattr(_lib, "igr_ref2_" + name).argtypes = [vp]
    return _lib


def _dptr(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _make_bc(faces, patches):
    """faces: 6 ints (x-,x+,y-,y+,z-,z+); patches: {face_index: [(c0,c1,radius,edge,rho,u,v,w,p), ...]}"""
    bc = _BC()
    keep = []
    for f in range(6):
        bc.face[f] = int(faces[f])
        plist = (patches or {}).get(f, [])
        bc.n_patches[f] = len(plist)
        if plist:
            arr = (_Patch * len(plist))(*[_Patch(*map(float, p)) for p in plist])
            keep.append(arr)
            bc.patches[f] = C.cast(arr, C.POINTER(_Patch))
    return bc, keep


class RefSolver:
    """The oracle's solver object: igr_ref_create / set_state / max_wavespeed / step / get_state
    plus the per-piece calls of one RHS evaluation."""

    def __init__(self, nx, ny, nz, dx, gamma, alpha, order=5, n_jacobi=5,
                 faces=(0, 0, 0, 0, 0, 0), patches=None, storage=STORE_F64):
        self.shape = (nz, ny, nx)
        self.nx, self.ny, self.nz = nx, ny, nz
        bc, keep = _make_bc(faces, patches)
        h = C.c_void_p()
        rc = lib().igr_ref_create(nx, ny, nz, dx, gamma, alpha, order, n_jacobi, C.byref(bc),
                                  C.byref(h))
        if rc != 0:
            raise ValueError("igr_ref_create failed with code %d" % rc)
        self._h = h
        if storage != STORE_F64:
            self.set_storage(storage)

    def __del__(self):
        if getattr(self, "_h", None):
            lib().igr_ref_destroy(self._h)
            self._h = None

    def set_storage(self, mode):
        assert lib().igr_ref_set_storage(self._h, mode) == 0

    def set_viscosity(self, mu, zeta=0.0):
        assert lib().igr_ref_set_viscosity(self._h, float(mu), float(zeta)) == 0

    def set_state(self, q):
        q = np.ascontiguousarray(q, dtype=np.float64)
        assert q.shape == (5,) + self.shape, q.shape
        assert lib().igr_ref_set_state(self._h, _dptr(q)) == 0

    def _get(self, name, lead=()):
        out = np.empty(lead + self.shape, dtype=np.float64)
        assert getattr(lib(), "igr_ref_" + name)(self._h, _dptr(out)) == 0
        return out

    def get_state(self):
        return self._get("get_state", (5,))

    def get_sigma(self):
        return self._get("get_sigma")

    def get_source(self):
        return self._get("get_source")

    def get_rhs(self):
        return self._get("get_rhs", (5,))

    def set_sigma(self, sig):
        sig = np.ascontiguousarray(sig, dtype=np.float64)
        assert sig.shape == self.shape
        assert lib().igr_ref_set_sigma(self._h, _dptr(sig)) == 0

    def set_source(self, b):
        b = np.ascontiguousarray(b, dtype=np.float64)
        assert b.shape == self.shape
        assert lib().igr_ref_set_source(self._h, _dptr(b)) == 0

    def get_padded(self, c):
        out = np.empty((self.nz + 6, self.ny + 6, self.nx + 6), dtype=np.float64)
        assert lib().igr_ref_get_padded(self._h, c, _dptr(out)) == 0
        return out

    def max_wavespeed(self):
        v = C.c_double()
        assert lib().igr_ref_max_wavespeed(self._h, C.byref(v)) == 0
        return v.value

    def set_padded(self, c, a):
        a = np.ascontiguousarray(a, dtype=np.float64)
        assert a.shape == (self.nz + 6, self.ny + 6, self.nx + 6)
        assert lib().igr_ref_set_padded(self._h, c, _dptr(a)) == 0

    def step(self, dt):
        assert lib().igr_ref_step(self._h, float(dt)) == 0

    def stage(self, stage, dt):
        assert lib().igr_ref_stage(self._h, int(stage), float(dt)) == 0

    def fill_ghosts(self):
        lib().igr_ref_fill_ghosts(self._h)

    def source(self):
        lib().igr_ref_source(self._h)

    def jacobi_sweep(self):
        lib().igr_ref_jacobi_sweep(self._h)

    def solve_sigma(self):
        lib().igr_ref_solve_sigma(self._h)

    def fill_sigma_ghosts(self):
        lib().igr_ref_fill_sigma_ghosts(self._h)

    def rhs(self):
        lib().igr_ref_rhs(self._h)

    def eval_rhs(self):
        lib().igr_ref_eval_rhs(self._h)


def rk_combine(a, qn, b, qs, dt, r):
    qn, qs, r = (np.ascontiguousarray(x, dtype=np.float64) for x in (qn, qs, r))
    out = np.empty_like(qn)
    lib().igr_ref_rk_combine(a, _dptr(qn), b, _dptr(qs), dt, _dptr(r), _dptr(out), qn.size)
    return out


def reconstruct(order, f6):
    f6 = np.ascontiguousarray(f6, dtype=np.float64)
    assert f6.shape == (6,)
    fl, fr = C.c_double(), C.c_double()
    lib().igr_ref_reconstruct(order, _dptr(f6), C.byref(fl), C.byref(fr))
    return fl.value, fr.value


def lf_flux(d, gamma, UL, UR, sigL, sigR, lam):
    UL = np.ascontiguousarray(UL, dtype=np.float64)
    UR = np.ascontiguousarray(UR, dtype=np.float64)
    F = np.empty(5)
    lib().igr_ref_lf_flux(d, gamma, _dptr(UL), _dptr(UR), sigL, sigR, lam, _dptr(F))
    return F


def viscous_flux(d, mu, zeta, G9, u3):
    G9 = np.ascontiguousarray(G9, dtype=np.float64).reshape(9)
    u3 = np.ascontiguousarray(u3, dtype=np.float64)
    F = np.empty(5)
    lib().igr_ref_viscous_flux(d, mu, zeta, _dptr(G9), _dptr(u3), _dptr(F))
    return F


def round_storage(x, mode):
    return lib().igr_ref_round_storage(float(x), mode)


class RefSolver2:
    """The two-fluid oracle (igr_ref2.c, reading A21).  State [7][nz][ny][nx] =
    (a1 rho1, a2 rho2, rho u, rho v, rho w, E, a1); patches: {face: [(c0, c1, radius, edge, a1rho1, a2rho2, a1,
    u, v, w, p), ...]}."""
    NF = 7

    def __init__(self, nx, ny, nz, dx, gamma1, gamma2, alpha, order=5, n_jacobi=5, faces=(0,) * 6, patches=None):
        self.shape = (nz, ny, nx)
        self.nx, self.ny, self.nz = nx, ny, nz
        bc, self._keep = _BC2(), []
        for f in range(6):
            bc.face[f] = int(faces[f])
            plist = (patches or {}).get(f, [])
            bc.n_patches[f] = len(plist)
            if plist:
                arr = (_Patch2 * len(plist))(*[_Patch2(*map(float, p)) for p in plist])
                self._keep.append(arr)
                bc.patches[f] = C.cast(arr, C.POINTER(_Patch2))
        h = C.c_void_p()
        rc = lib().igr_ref2_create(nx, ny, nz, dx, gamma1, gamma2, alpha, order, n_jacobi, C.byref(bc), C.byref(h))
        if rc != 0:
            raise ValueError("igr_ref2_create failed with code %d" % rc)
        self._h = h

    def __del__(self):
        if getattr(self, "_h", None):
            lib().igr_ref2_destroy(self._h)
            self._h = None

    def set_state(self, q):
        q = np.ascontiguousarray(q, dtype=np.float64)
        assert q.shape == (7,) + self.shape, q.shape
        assert lib().igr_ref2_set_state(self._h, _dptr(q)) == 0

    def _get(self, name, lead=()):
        out = np.empty(lead + self.shape, dtype=np.float64)
        assert getattr(lib(), "igr_ref2_" + name)(self._h, _dptr(out)) == 0
        return out

    def get_state(self):
        return self._get("get_state", (7,))

    def get_rhs(self):
        return self._get("get_rhs", (7,))

    def get_sigma(self):
        return self._get("get_sigma")

    def get_source(self):
        return self._get("get_source")

    def set_sigma(self, sig):
        sig = np.ascontiguousarray(sig, dtype=np.float64)
        assert sig.shape == self.shape
        assert lib().igr_ref2_set_sigma(self._h, _dptr(sig)) == 0

    def get_padded(self, c):
        out = np.empty((self.nz + 6, self.ny + 6, self.nx + 6), dtype=np.float64)
        assert lib().igr_ref2_get_padded(self._h, c, _dptr(out)) == 0
        return out

    def max_wavespeed(self):
        v = C.c_double()
        assert lib().igr_ref2_max_wavespeed(self._h, C.byref(v)) == 0
        return v.value

    def step(self, dt):
        assert lib().igr_ref2_step(self._h, float(dt)) == 0

    def stage(self, stage, dt):
        assert lib().igr_ref2_stage(self._h, int(stage), float(dt)) == 0

    def fill_ghosts(self):
        lib().igr_ref2_fill_ghosts(self._h)

    def source(self):
        lib().igr_ref2_source(self._h)

    def solve_sigma(self):
        lib().igr_ref2_solve_sigma(self._h)

    def rhs(self):
        lib().igr_ref2_rhs(self._h)

    def eval_rhs(self):
        lib().igr_ref2_eval_rhs(self._h)
