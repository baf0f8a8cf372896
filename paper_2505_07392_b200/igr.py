"""Thin Python binding of libigr.so (include/igr.h): argument marshalling only.

Every step of the hot path runs in the CUDA kernels of the library.  PyTorch is used for device
memory (the solver's workspace is a torch tensor) and for the stream.  There is no CPU fallback:
loading fails loudly if the library has not been built, and igr_create fails without a GPU.
Names follow include/igr.h (igr_create -> Solver(...), igr_step -> Solver.step, ...).
"""
import ctypes as C
import os

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libigr.so")

OK, ERR_ARG, ERR_BC, ERR_ALLOC, ERR_CUDA, ERR_NONFINITE = 0, -1, -2, -3, -4, -5
BC_PERIODIC, BC_EXTRAP, BC_INFLOW, BC_EXTERNAL = 0, 1, 2, 3
STORE_F32, STORE_F16, STORE_BF16, STORE_F64 = 0, 1, 2, 3
VARIANT_TILED, VARIANT_SIMPLE = 0, 1
_STATUS = {0: "IGR_OK", -1: "IGR_ERR_ARG", -2: "IGR_ERR_BC", -3: "IGR_ERR_ALLOC", -4: "IGR_ERR_CUDA",
           -5: "IGR_ERR_NONFINITE"}

EXPORTS = ["igr_workspace_bytes", "igr_create", "igr_create_ex", "igr_destroy", "igr_set_state",
           "igr_get_state", "igr_set_sigma", "igr_get_sigma", "igr_max_wavespeed", "igr_step",
           "igr_sync", "igr_last_error", "igr_halo_bc", "igr_sigma_source", "igr_jacobi", "igr_rhs",
           "igr_rk_update", "igr_get_source", "igr_set_source", "igr_get_rhs", "igr_get_padded",
           "igr_kernel_launches", "igr_profile", "igr_profile_read", "igr_set_viscosity", "igr_stage",
           "igr_export_fields", "igr_ipc_open", "igr_ipc_close", "igr_set_neighbor", "igr_pull_halo", "igr_set_wave_range", "igr_set_state_planes",
           "igr_get_state_planes", "igr_set_state_f64", "igr_get_state_f64", "igr_get_sigma_f64",
           "igr_event_handle", "igr_event_open", "igr_event_close", "igr_event_record", "igr_event_wait",
           "igr_max_wavespeed_noalloc"]
NOALLOC_MAX_CELLS = 1 << 30      # igr.h IGR_NOALLOC_MAX_CELLS


class IgrError(RuntimeError):
    def __init__(self, code, msg=""):
        self.code = code
        super().__init__("%s (%d) %s" % (_STATUS.get(code, "?"), code, msg))


class Patch(C.Structure):
    _fields_ = [(n, C.c_double) for n in ("c0", "c1", "radius", "edge", "rho", "u", "v", "w", "p", "a1", "rho2")]


class BC(C.Structure):
    _fields_ = [("face", C.c_int32 * 6), ("n_patches", C.c_int32 * 6),
                ("patches", C.POINTER(Patch) * 6)]


class Options(C.Structure):
    _fields_ = [("storage", C.c_int32), ("fused", C.c_int32), ("variant", C.c_int32),
                ("n_fluids", C.c_int32), ("stream", C.c_void_p),
                ("workspace", C.c_void_p), ("workspace_bytes", C.c_size_t), ("gamma2", C.c_double)]


class Export(C.Structure):
    """igr_export (include/igr.h): plain bytes, can be shipped to another rank as they are."""
    _fields_ = [("ipc_handle", C.c_ubyte * 64), ("base", C.c_uint64), ("q_offset", (C.c_uint64 * 5) * 3),
                ("sig_offset", C.c_uint64 * 2), ("plane_bytes", C.c_uint64), ("nz", C.c_int32),
                ("storage", C.c_int32), ("cur", C.c_int32), ("sig_cur", C.c_int32),
                ("owns_memory", C.c_int32), ("reserved", C.c_int32)]


_lib = None


def lib():
    """Load libigr.so; raises if it has not been built (python -m paper_2505_07392_b200.build)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError("libigr.so is missing: build it with `python -m paper_2505_07392_b200.build` "
                              "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        vp, fp = C.c_void_p, C.c_void_p          # float pointers are passed as raw addresses
        L.igr_workspace_bytes.argtypes = [C.c_int] * 3 + [C.POINTER(Options)]
        L.igr_workspace_bytes.restype = C.c_size_t
        L.igr_create.argtypes = [C.c_int] * 3 + [C.c_double] * 3 + [C.c_int] * 2 + [C.POINTER(BC), C.POINTER(vp)]
        L.igr_create_ex.argtypes = [C.c_int] * 3 + [C.c_double] * 3 + [C.c_int] * 2 + \
            [C.POINTER(BC), C.POINTER(Options), C.POINTER(vp)]
        L.igr_destroy.argtypes = [vp]
        L.igr_destroy.restype = None
        for n in ("igr_set_state", "igr_get_state", "igr_set_sigma", "igr_get_sigma", "igr_get_source",
                  "igr_set_source", "igr_get_rhs"):
            getattr(L, n).argtypes = [vp, fp]
        L.igr_get_padded.argtypes = [vp, C.c_int, fp]
        for n in ("igr_set_state_f64", "igr_get_state_f64", "igr_get_sigma_f64"):
            getattr(L, n).argtypes = [vp, vp]
        L.igr_set_state_planes.argtypes = [vp, C.c_int, C.c_int, fp]
        L.igr_get_state_planes.argtypes = [vp, C.c_int, C.c_int, fp]
        L.igr_max_wavespeed.argtypes = [vp, C.POINTER(C.c_double)]
        L.igr_step.argtypes = [vp, C.c_double]
        L.igr_rk_update.argtypes = [vp, C.c_int, C.c_double]
        for n in ("igr_sync", "igr_halo_bc", "igr_sigma_source", "igr_jacobi", "igr_rhs"):
            getattr(L, n).argtypes = [vp]
        L.igr_kernel_launches.argtypes = [vp, C.POINTER(C.c_longlong)]
        L.igr_profile.argtypes = [vp, C.c_int]
        L.igr_set_viscosity.argtypes = [vp, C.c_double, C.c_double]
        L.igr_profile_read.argtypes = [vp, C.POINTER(C.c_double), C.POINTER(C.c_longlong)]
        L.igr_stage.argtypes = [vp, C.c_int, C.c_double]
        L.igr_export_fields.argtypes = [vp, C.POINTER(Export)]
        L.igr_ipc_open.argtypes = [C.POINTER(Export), C.POINTER(vp)]
        L.igr_ipc_close.argtypes = [vp]
        L.igr_set_neighbor.argtypes = [vp, C.c_int, C.POINTER(Export), vp, C.c_int, C.c_int, C.c_int]
        L.igr_pull_halo.argtypes = [vp]
        L.igr_set_wave_range.argtypes = [vp, C.c_int, C.c_int]
        L.igr_event_handle.argtypes = [vp, C.c_int, C.POINTER(C.c_ubyte * 64)]
        L.igr_event_open.argtypes = [C.POINTER(C.c_ubyte * 64), C.POINTER(vp)]
        L.igr_event_close.argtypes = [vp]
        L.igr_event_record.argtypes = [vp, C.c_int]
        L.igr_event_wait.argtypes = [vp, vp]
        L.igr_last_error.argtypes = [vp]
        L.igr_last_error.restype = C.c_char_p
        L.igr_max_wavespeed_noalloc.argtypes = [fp] + [C.c_int] * 3 + [C.c_double, fp, vp, C.c_char_p, C.c_size_t]
        _lib = L
    return _lib


def make_bc(faces, patches=None):
    """faces: 6 codes (x-,x+,y-,y+,z-,z+); patches: {face: [(c0,c1,radius,edge,rho,u,v,w,p[,a1,rho2]), ...]}
    (a1, rho2: two fluids only, igr.h igr_patch; default 1, 0)."""
    bc, keep = BC(), []
    for f in range(6):
        bc.face[f] = int(faces[f])
        plist = (patches or {}).get(f, [])
        bc.n_patches[f] = len(plist)
        if plist:
            arr = (Patch * len(plist))(*[Patch(*map(float, tuple(p) + (1.0, 0.0)[len(p) - 9:])) for p in plist])
            keep.append(arr)
            bc.patches[f] = C.cast(arr, C.POINTER(Patch))
    return bc, keep


def _addr(a, shape, writable=False, f64=False):
    """Raw address of a contiguous fp32 (f64: fp64) torch tensor (cpu or cuda) or numpy array of `shape`."""
    if isinstance(a, torch.Tensor):
        assert a.dtype == (torch.float64 if f64 else torch.float32) and a.is_contiguous() \
            and tuple(a.shape) == tuple(shape), (a.dtype, a.shape, shape)
        return a.data_ptr()
    assert isinstance(a, np.ndarray) and a.dtype == (np.float64 if f64 else np.float32) and a.flags.c_contiguous \
        and a.shape == tuple(shape), (type(a), getattr(a, "shape", None), shape)
    if writable:
        assert a.flags.writeable
    return a.ctypes.data


def max_wavespeed_noalloc(q, gamma, out, stream=None, shape=None):
    """igr_max_wavespeed_noalloc (igr.h): the CFL wave speed of the unpadded fp32 CUDA tensor q [5][nz][ny][nx] into
    the 2-element fp32 CUDA tensor `out` (out[0] = speed, out[1] = non-finite flag), on `stream` (a raw cudaStream_t;
    default: torch's current stream).  Nothing is allocated and nothing is waited for.  `shape` = (nz, ny, nx)
    overrides q's own extents (the size check comes first: a refused size never touches q)."""
    nz, ny, nx = (int(v) for v in (shape if shape is not None else q.shape[1:]))
    if shape is None:
        assert q.is_cuda and out.is_cuda
        qa = _addr(q, (5, nz, ny, nx))
    else:
        qa = q.data_ptr()
    oa = _addr(out, (2,), True)
    if stream is None:
        stream = torch.cuda.current_stream(out.device).cuda_stream
    err = C.create_string_buffer(256)
    rc = lib().igr_max_wavespeed_noalloc(qa, nx, ny, nz, float(gamma), oa, stream, err, len(err))
    if rc != OK:
        raise IgrError(rc, err.value.decode())


def ipc_open(peer):
    """Address in this process of another process's allocation described by `peer` (an Export)."""
    base = C.c_void_p()
    rc = lib().igr_ipc_open(C.byref(peer), C.byref(base))
    if rc != OK:
        raise IgrError(rc, "igr_ipc_open")
    return base.value


def event_open(handle_bytes):
    """This process's handle of another process's interprocess event (64-byte CUDA IPC handle)."""
    buf = (C.c_ubyte * 64).from_buffer_copy(handle_bytes)
    ev = C.c_void_p()
    rc = lib().igr_event_open(C.byref(buf), C.byref(ev))
    if rc != OK:
        raise IgrError(rc, "igr_event_open")
    return ev.value


def event_close(ev):
    rc = lib().igr_event_close(C.c_void_p(ev))
    if rc != OK:
        raise IgrError(rc, "igr_event_close")


def ipc_close(base):
    rc = lib().igr_ipc_close(C.c_void_p(base))
    if rc != OK:
        raise IgrError(rc, "igr_ipc_close")


class Solver:
    """igr_create_ex / igr_destroy and the calls of include/igr.h on one solver object."""

    def __init__(self, nx, ny, nz, dx, gamma, alpha, order=5, n_jacobi=5, faces=(0,) * 6, patches=None,
                 storage=STORE_F32, fused=1, variant=VARIANT_TILED, device="cuda:0", own_workspace=True,
                 n_fluids=1, gamma2=0.0):
        L = lib()
        self.nx, self.ny, self.nz = nx, ny, nz
        self.shape = (nz, ny, nx)
        self.nf = 7 if n_fluids == 2 else 5          # fields of "the state" (igr.h, igr_options.n_fluids)
        self.device = torch.device(device)
        self._h = None
        opt = Options()
        opt.storage, opt.fused, opt.variant = storage, fused, variant
        opt.n_fluids, opt.gamma2 = n_fluids, gamma2
        if not torch.cuda.is_available():
            raise IgrError(ERR_CUDA, "no CUDA device: libigr has no CPU fallback")
        torch.cuda.set_device(self.device)
        self.stream = torch.cuda.current_stream(self.device)
        opt.stream = self.stream.cuda_stream
        if own_workspace:
            nbytes = L.igr_workspace_bytes(nx, ny, nz, C.byref(opt))
            self._ws = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
            base = (self._ws.data_ptr() + 255) // 256 * 256
            opt.workspace, opt.workspace_bytes = base, nbytes
        bc, self._keep = make_bc(faces, patches)
        h = C.c_void_p()
        rc = L.igr_create_ex(nx, ny, nz, dx, gamma, alpha, order, n_jacobi, C.byref(bc), C.byref(opt),
                             C.byref(h))
        if rc != OK:
            raise IgrError(rc, "igr_create_ex")
        self._h = h

    @classmethod
    def for_workload(cls, w, **kw):
        if getattr(w, "gamma2", 0.0):
            kw = dict(n_fluids=2, gamma2=w.gamma2, **kw)
        return cls(w.nx, w.ny, w.nz, w.dx, w.gamma, w.alpha, order=w.order, n_jacobi=w.n_jacobi,
                   faces=w.faces, patches=w.patches, **kw)

    def close(self):
        if self._h:
            lib().igr_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, rc):
        if rc != OK:
            raise IgrError(rc, lib().igr_last_error(self._h).decode())

    # ---- igr.h calls
    def set_state(self, q):
        if q.dtype in (np.float64, torch.float64):           # fp64 arrays: the fp64 mode only (igr_set_state_f64)
            self._check(lib().igr_set_state_f64(self._h, _addr(q, (self.nf,) + self.shape, f64=True)))
            return
        self._check(lib().igr_set_state(self._h, _addr(q, (self.nf,) + self.shape)))

    def get_state_f64(self, out=None):
        out = np.empty((self.nf,) + self.shape, np.float64) if out is None else out
        self._check(lib().igr_get_state_f64(self._h, _addr(out, (self.nf,) + self.shape, True, f64=True)))
        return out

    def get_sigma_f64(self, out=None):
        out = np.empty(self.shape, np.float64) if out is None else out
        self._check(lib().igr_get_sigma_f64(self._h, _addr(out, self.shape, True, f64=True)))
        return out

    def get_state(self, out=None):
        out = np.empty((self.nf,) + self.shape, np.float32) if out is None else out
        self._check(lib().igr_get_state(self._h, _addr(out, (self.nf,) + self.shape, True)))
        return out

    def set_state_planes(self, k0, q):
        """q: [5][nk][ny][nx], planes k0 .. k0 + nk - 1 (Sigma is left as it is)."""
        nk = int(q.shape[1])
        self._check(lib().igr_set_state_planes(self._h, int(k0), nk, _addr(q, (self.nf, nk, self.ny, self.nx))))

    def get_state_planes(self, k0, nk, out=None):
        out = np.empty((self.nf, nk, self.ny, self.nx), np.float32) if out is None else out
        self._check(lib().igr_get_state_planes(self._h, int(k0), int(nk),
                                               _addr(out, (self.nf, nk, self.ny, self.nx), True)))
        return out

    def set_sigma(self, f):
        self._check(lib().igr_set_sigma(self._h, _addr(f, self.shape)))

    def _scalar_out(self, fn, out):
        out = np.empty(self.shape, np.float32) if out is None else out
        self._check(fn(self._h, _addr(out, self.shape, True)))
        return out

    def get_sigma(self, out=None):
        return self._scalar_out(lib().igr_get_sigma, out)

    def get_source(self, out=None):
        return self._scalar_out(lib().igr_get_source, out)

    def set_source(self, f):
        self._check(lib().igr_set_source(self._h, _addr(f, self.shape)))

    def get_rhs(self, out=None):
        out = np.empty((5,) + self.shape, np.float32) if out is None else out
        self._check(lib().igr_get_rhs(self._h, _addr(out, (5,) + self.shape, True)))
        return out

    def get_padded(self, c, out=None):
        shp = (self.nz + 6, self.ny + 6, self.nx + 6)
        out = np.empty(shp, np.float32) if out is None else out
        self._check(lib().igr_get_padded(self._h, c, _addr(out, shp, True)))
        return out

    # ---- interprocess events (igr.h): which = 0 "stage complete", 1 "pulls complete"
    def event_handle(self, which):
        buf = (C.c_ubyte * 64)()
        self._check(lib().igr_event_handle(self._h, int(which), C.byref(buf)))
        return bytes(buf)

    def event_record(self, which):
        self._check(lib().igr_event_record(self._h, int(which)))

    def event_wait(self, ev):
        self._check(lib().igr_event_wait(self._h, C.c_void_p(ev)))

    def max_wavespeed(self):
        v = C.c_double()
        self._check(lib().igr_max_wavespeed(self._h, C.byref(v)))
        return v.value

    def step(self, dt):
        self._check(lib().igr_step(self._h, float(dt)))

    def sync(self):
        self._check(lib().igr_sync(self._h))

    def halo_bc(self):
        self._check(lib().igr_halo_bc(self._h))

    def sigma_source(self):
        self._check(lib().igr_sigma_source(self._h))

    def jacobi(self):
        self._check(lib().igr_jacobi(self._h))

    def rhs(self):
        self._check(lib().igr_rhs(self._h))

    def rk_update(self, stage, dt):
        self._check(lib().igr_rk_update(self._h, int(stage), float(dt)))

    # ---- NEXT-2: slab exchange (include/igr.h)
    def stage(self, stage, dt):
        self._check(lib().igr_stage(self._h, int(stage), float(dt)))

    def export_fields(self):
        e = Export()
        self._check(lib().igr_export_fields(self._h, C.byref(e)))
        return e

    def set_neighbor(self, side, peer, peer_base, dst_plane, src_plane, count):
        """peer: Export of the neighbour (None: drop it); peer_base: its allocation as addressable here."""
        if peer is None:
            self._check(lib().igr_set_neighbor(self._h, int(side), None, None, 0, 0, 0))
        else:
            self._check(lib().igr_set_neighbor(self._h, int(side), C.byref(peer), C.c_void_p(peer_base),
                                               int(dst_plane), int(src_plane), int(count)))

    def pull_halo(self):
        self._check(lib().igr_pull_halo(self._h))

    def set_wave_range(self, k0, k1):
        self._check(lib().igr_set_wave_range(self._h, int(k0), int(k1)))

    ROWS = ("halo_bc", "sigma_source", "jacobi", "rhs", "rk_update", "max_wavespeed")

    def set_viscosity(self, mu, zeta=0.0):
        self._check(lib().igr_set_viscosity(self._h, float(mu), float(zeta)))

    def kernel_launches(self):
        v = C.c_longlong()
        self._check(lib().igr_kernel_launches(self._h, C.byref(v)))
        return v.value

    def profile(self, enable):
        self._check(lib().igr_profile(self._h, int(bool(enable))))

    def profile_read(self):
        """{row: (total_ms, calls)} of the rows timed since profile(True)."""
        ms, cnt = (C.c_double * 6)(), (C.c_longlong * 6)()
        self._check(lib().igr_profile_read(self._h, ms, cnt))
        return {r: (ms[i], cnt[i]) for i, r in enumerate(self.ROWS)}
