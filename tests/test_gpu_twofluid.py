"""GPU parity of the two-fluid variant (reading A21): igr_options.n_fluids = 2 through
the C ABI against the two-fluid oracle (oracle/igr_ref2.c, pinned in tests/test_oracle_twofluid.py) on the same
seeded inputs, with the dt replay of reading A16.  Tolerances as for one fluid (north_star): fp32 vs fp64 oracle,
max-rel <= 1e-4 on smooth cases, L1-rel <= 1e-3 on the jets; norms per field group (tests/parity.py)."""
import dataclasses

import numpy as np
import pytest

from paper_2505_07392_b200 import igr
from paper_2505_07392_b200 import workloads as W
import parity
from test_gpu_configs import FULL, _subbox_parity

pytestmark = pytest.mark.gpu


def test_two_fluid_vortex_five_steps_match_the_oracle():
    w = W.two_fluid_vortex(40)                    # 40^3: several RHS tiles and a ragged tail, quad and blocked Jacobi regions
    g = igr.Solver.for_workload(w)
    assert g.nf == 7
    qg, qr, sg, sr, dts = parity.run_pair(w, g, n_steps=5)
    mx, l1 = parity.worst(qg, qr)
    assert mx <= 1e-4, (mx, l1, parity.norms(qg, qr))
    assert parity.scalar_norms(sg, sr)[0] <= 1e-3 and np.abs(sr).max() > 1e-4


@pytest.mark.parametrize("shape", [(37, 20, 13), (70, 45, 40)])
def test_two_fluid_jets_three_steps_match_the_oracle(shape):
    w = W.two_fluid(W.jets9(n=shape[0], radius=4, pitch=11))
    w = dataclasses.replace(w, ny=shape[1], nz=shape[2], global_shape=None)
    g = igr.Solver.for_workload(w)
    qg, qr, sg, sr, dts = parity.run_pair(w, g, n_steps=3)
    mx, l1 = parity.worst(qg, qr)
    assert l1 <= 1e-3 and mx <= 2e-3, (mx, l1, parity.norms(qg, qr))
    assert qr[1].min() > 0 and qr[0].min() > 0                     # both partial densities present everywhere
    assert np.ptp(qr[6]) > 0.9                                     # and a real interface


@pytest.mark.skipif(not FULL, reason="full-size configs disabled")
def test_two_fluid_jets33_1024_subbox_first_3_steps():
    """The workload `bench.py --workload jets2f33_1024` times, in its launch configuration, against the two-fluid
    oracle on the dependency-cone sub-box over the lip of an inner-ring jet (as for config 5 with one fluid)."""
    w = W.two_fluid(W.jets33())
    got, want, rho_min = _subbox_parity(w, (496, 480, 0), 64, 80, 3)
    mx, l1 = parity.worst(got, want)
    assert l1 <= 1e-3, (mx, l1, parity.norms(got, want))
    assert rho_min > 0 and np.ptp(want[6]) > 0.9                    # an interface crosses the sub-box


def test_two_fluid_interface_advection_keeps_u_and_p_uniform():
    """T2 of the oracle pins on the GPU: uniform u, p across a material interface stay uniform (to fp32 round-off)."""
    w = W.two_fluid_vortex(32)
    q = W.state(w).numpy().astype(np.float64)
    a1 = q[6]
    u0, p0 = (0.7, -0.4, 0.9), 1.3
    rho = a1 * 1.0 + (1 - a1) * 0.3
    G = a1 / (w.gamma - 1) + (1 - a1) / (w.gamma2 - 1)
    q0 = np.stack([a1 * 1.0, (1 - a1) * 0.3, rho * u0[0], rho * u0[1], rho * u0[2],
                   p0 * G + 0.5 * rho * sum(c * c for c in u0), a1]).astype(np.float32)
    g = igr.Solver.for_workload(w)
    g.set_state(q0)
    for _ in range(5):
        g.step(w.cfl * w.dx / g.max_wavespeed())
    out = g.get_state().astype(np.float64)
    rho = out[0] + out[1]
    for a in range(3):
        assert np.abs(out[2 + a] / rho - u0[a]).max() <= 2e-5
    G = out[6] / (w.gamma - 1) + (1 - out[6]) / (w.gamma2 - 1)
    p = (out[5] - 0.5 * (out[2] ** 2 + out[3] ** 2 + out[4] ** 2) / rho) / G
    assert np.abs(p - p0).max() <= 5e-5 * p0
    assert np.abs(out[6] - a1).max() > 0.02                        # the interface did move


def test_two_fluid_partial_masses_are_conserved():
    w = W.two_fluid_vortex(32)
    q0 = W.state(w).numpy()
    g = igr.Solver.for_workload(w)
    g.set_state(q0)
    for _ in range(5):
        g.step(w.cfl * w.dx / g.max_wavespeed())
    out = g.get_state().astype(np.float64)
    tot0, tot = q0.astype(np.float64).reshape(7, -1).sum(1), out.reshape(7, -1).sum(1)
    scale = np.abs(q0.astype(np.float64)).reshape(7, -1).sum(1)
    scale[2:5] = scale[2:5].sum()
    assert np.all(np.abs(tot - tot0)[:6] <= 2e-7 * scale[:6]), (tot - tot0) / scale


def test_two_fluid_single_fluid_limit_on_the_gpu():
    """a1 = 1, no second fluid, gamma2 = gamma: the two-fluid kernels reproduce the one-fluid kernels to fp32
    round-off (different instruction sequences: mass flux rho1 u_d against m_d, 1/Gamma against gamma - 1)."""
    w1 = W.taylor_green(32)
    q1 = W.state(w1).numpy()
    w2 = dataclasses.replace(w1, gamma2=w1.gamma)
    q2 = np.stack([q1[0], 0 * q1[0], q1[1], q1[2], q1[3], q1[4], 1 + 0 * q1[0]]).astype(np.float32)
    g1, g2 = igr.Solver.for_workload(w1), igr.Solver.for_workload(w2)
    g1.set_state(q1); g2.set_state(q2)
    for _ in range(4):
        lam = g1.max_wavespeed()
        assert abs(g2.max_wavespeed() - lam) <= 2e-6 * lam
        g1.step(w1.cfl * w1.dx / lam); g2.step(w1.cfl * w1.dx / lam)
    a, b = g1.get_state(), g2.get_state()
    assert np.all(b[1] == 0.0) and np.abs(b[6] - 1).max() <= 1e-6
    mx, _ = parity.worst(b[[0, 2, 3, 4, 5]], a)
    assert mx <= 2e-6, mx


def test_two_fluid_is_refused_where_it_is_not_built():
    w = W.two_fluid_vortex(16)
    for kw in (dict(storage=igr.STORE_F16), dict(fused=0), dict(variant=igr.VARIANT_SIMPLE)):
        with pytest.raises(igr.IgrError) as ei:
            igr.Solver.for_workload(w, **kw)
        assert ei.value.code == igr.ERR_ARG
    g = igr.Solver.for_workload(w)
    for call in (g.rhs, lambda: g.set_viscosity(0.1, 0.0), g.export_fields):
        with pytest.raises(igr.IgrError) as ei:
            call()
        assert ei.value.code == igr.ERR_ARG
