"""NEXT-1 on the GPU: viscous fluxes (eqs. 2, 3, 5) through the C ABI against the
fp64 oracle, same seeded inputs, same tolerances as the inviscid rows (fp32: max-rel <= 1e-4)."""
import numpy as np
import pytest

from oracle import igr_ref as R
from paper_2505_07392_b200 import igr
from paper_2505_07392_b200 import workloads as W
import parity
from test_gpu_kernels import BCS, smooth_state, G

pytestmark = pytest.mark.gpu
MU, ZETA = 0.02, 0.01


def pair(shape, bc, **kw):
    nx, ny, nz = shape
    faces, patches = BCS[bc]
    dx = 1.0 / nx
    g = igr.Solver(nx, ny, nz, dx, G, 10 * dx * dx, faces=faces, patches=patches, **kw)
    r = R.RefSolver(nx, ny, nz, dx, G, 10 * dx * dx, faces=faces, patches=patches)
    g.set_viscosity(MU, ZETA)
    r.set_viscosity(MU, ZETA)
    return g, r


@pytest.mark.parametrize("variant", [igr.VARIANT_TILED, igr.VARIANT_SIMPLE])
@pytest.mark.parametrize("bc", ["periodic", "mixed", "inflow_x"])
@pytest.mark.parametrize("shape", [(37, 20, 13), (64, 16, 16)])
def test_rhs_with_viscous_fluxes(shape, bc, variant):
    g, r = pair(shape, bc, variant=variant)
    q = smooth_state(*shape, seed=4)
    sig = (0.05 * np.random.default_rng(44).uniform(0, 1, shape[::-1])).astype(np.float32)
    g.set_state(q); r.set_state(q.astype(np.float64))
    g.set_sigma(sig); r.set_sigma(sig.astype(np.float64))
    g.halo_bc(); g.sigma_source()                     # the source kernel also writes the gradients
    r.fill_ghosts(); r.fill_sigma_ghosts()
    g.rhs(); r.rhs()
    mx, l1 = parity.worst(g.get_rhs(), r.get_rhs())
    assert mx <= 1e-4 and l1 <= 2e-5, (mx, l1)
    # the viscous part alone (difference to the inviscid RHS) also agrees
    g0, r0 = pair(shape, bc, variant=variant)
    g0.set_viscosity(0, 0); r0.set_viscosity(0, 0)
    g0.set_state(q); r0.set_state(q.astype(np.float64))
    g0.set_sigma(sig); r0.set_sigma(sig.astype(np.float64))
    g0.halo_bc(); g0.sigma_source(); r0.fill_ghosts(); r0.fill_sigma_ghosts()
    g0.rhs(); r0.rhs()
    dv_g = g.get_rhs().astype(np.float64) - g0.get_rhs()
    dv_r = r.get_rhs() - r0.get_rhs()
    assert np.abs(dv_r[1:]).max() > 1e-3
    assert np.abs(dv_g - dv_r)[1:].max() <= 2e-3 * np.abs(dv_r[1:]).max()


@pytest.mark.parametrize("fused", [0, 1])
def test_viscous_taylor_green_five_steps(fused):
    w = W.taylor_green(48)
    g = igr.Solver.for_workload(w, fused=fused)
    g.set_viscosity(MU, ZETA)
    ref = parity.oracle_for(w)
    ref.set_viscosity(MU, ZETA)
    q0 = W.state(w).numpy()
    g.set_state(q0); ref.set_state(q0.astype(np.float64))
    for _ in range(5):
        dt = w.cfl * w.dx / g.max_wavespeed()
        g.step(dt); ref.step(dt)
    mx, l1 = parity.worst(g.get_state(), ref.get_state())
    assert mx <= 1e-4, (mx, l1)
    # viscosity does something at this Reynolds number: compare with the inviscid oracle
    inv = parity.oracle_for(w)
    inv.set_state(q0.astype(np.float64))
    for _ in range(5):
        inv.step(dt)
    assert parity.worst(ref.get_state(), inv.get_state())[0] > 1e-4


def test_zero_viscosity_is_the_default_path_bitwise():
    shape = (37, 20, 13)
    q = smooth_state(*shape, seed=6)
    out = []
    for setv in (False, True):
        g, _ = pair(shape, "mixed", fused=1)
        g.set_viscosity(0.0, 0.0) if setv else g.set_viscosity(MU, ZETA)
        if not setv:
            g.set_viscosity(0.0, 0.0)
        g.set_state(q)
        for _ in range(2):
            g.step(0.3 / shape[0] / g.max_wavespeed())
        out.append(g.get_state())
    g2 = igr.Solver(shape[0], shape[1], shape[2], 1.0 / shape[0], G, 10.0 / shape[0] ** 2, faces=BCS["mixed"][0],
                    patches=BCS["mixed"][1], fused=1)
    g2.set_state(q)
    for _ in range(2):
        g2.step(0.3 / shape[0] / g2.max_wavespeed())
    assert np.array_equal(out[0], out[1]) and np.array_equal(out[0], g2.get_state())
