"""The four acceptance gates of BASELINE.json's north_star for the fp64 oracle (SURVEY P7, P8, P10,
P11), checked before any GPU code is trusted.  CPU only."""
import math
import os

import numpy as np
import pytest
import torch

from oracle import igr_ref as R
from paper_2505_07392_b200 import workloads as W
import exact_riemann as ER

HERE = os.path.dirname(os.path.abspath(__file__))


def solver_for(w, **kw):
    return R.RefSolver(w.nx, w.ny, w.nz, w.dx, w.gamma, w.alpha, order=w.order,
                       n_jacobi=w.n_jacobi, faces=w.faces, patches=w.patches, **kw)


def state64(w):
    return W.state(w, dtype=torch.float64).numpy()


# ------------------------------------------------------------------ gate 1 (P7): uniform state
@pytest.mark.parametrize("faces", [(0,) * 6, (1,) * 6, (1, 1, 0, 0, 2, 1), (2, 1, 1, 2, 0, 0)])
def test_gate1_uniform_state_is_preserved_bitwise(faces):
    rho, u, v, w_, p = 0.9, 0.3, -0.7, 1.1, 1.3
    patches = {f: [(4.0, 5.0, 3.0, e, rho, u, v, w_, p)] for f, e in zip(range(6), (0, 2, 0, 2, 0, 2))
               if faces[f] == 2}
    w = W.uniform(10, 9, 8, 0.1, rho, u, v, w_, p, faces=faces, patches=patches)
    q0 = state64(w)
    s = solver_for(w)
    s.set_state(q0)
    for _ in range(4):
        s.step(0.5 * w.dx / s.max_wavespeed())
    assert np.array_equal(s.get_state(), q0)
    assert np.all(s.get_sigma() == 0.0)
    assert np.all(s.get_rhs() == 0.0)


# ------------------------------------------------------------------ gate 2 (P8): conservation
def test_gate2_conservation_on_periodic_grid():
    n = 16
    c = (np.arange(n) + 0.5) / n
    z, y, x = np.meshgrid(c, c, c, indexing="ij")
    tw = 2 * np.pi
    rho = 1 + 0.3 * np.sin(tw * x) * np.cos(tw * y) + 0.2 * np.sin(tw * z)
    vel = [0.5 * np.sin(tw * (x + y)), 0.4 * np.cos(tw * (y - z)) - 0.2, 0.3 * np.sin(tw * (z + x))]
    p = 1 + 0.2 * np.cos(tw * (x + y + z))
    q = np.stack([rho, rho * vel[0], rho * vel[1], rho * vel[2],
                  p / 0.4 + 0.5 * rho * sum(v * v for v in vel)])
    s = R.RefSolver(n, n, n, 1.0 / n, 1.4, 10.0 / n ** 2)
    s.set_state(q)
    tot0 = q.reshape(5, -1).sum(axis=1)
    scale = np.abs(q).reshape(5, -1).sum(axis=1)
    for _ in range(10):
        s.step(0.5 / n / s.max_wavespeed())
        tot = s.get_state().reshape(5, -1).sum(axis=1)
        assert np.all(np.abs(tot - tot0) <= 1e-13 * scale)
    assert np.abs(s.get_sigma()).max() > 1e-4      # the entropic pressure was active


# ------------------------------------------------------------------ gate 3 (P10): entropy wave
def _wave_error(n, dt, t_end):
    w = W.entropy_wave(n)
    s = solver_for(w)
    s.set_state(state64(w))
    ns = int(round(t_end / dt))
    for _ in range(ns):
        s.step(t_end / ns)
    exact = W.entropy_wave_exact_rho(w, t_end).numpy()
    st = s.get_state()
    # in exact arithmetic u = 1 and p = 1 stay constant and Sigma stays 0 (pure advection of rho)
    assert np.abs(st[1] / st[0] - 1).max() < 1e-12 and np.abs(s.get_sigma()).max() < 1e-12
    return np.abs(st[0] - exact).max()


def test_gate3_entropy_wave_converges_at_design_order():
    t_end, dt16 = 0.1, 0.5 * (1 / 16) / 2.33
    e = [_wave_error(n, dt16 * (16 / n) ** (5 / 3), t_end) for n in (16, 32, 64)]
    o1, o2 = math.log2(e[0] / e[1]), math.log2(e[1] / e[2])
    assert 4.7 < o1 < 5.5 and 4.7 < o2 < 5.3, (e, o1, o2)      # spatial order 5 (dt ~ dx^(5/3))
    e = [_wave_error(n, 0.5 * (1 / n) / 2.33, t_end) for n in (16, 32, 64)]
    assert math.log2(e[1] / e[2]) > 2.9                         # fixed CFL: time error, order 3


def test_gate3_config1_error_vs_exact_after_20_steps():
    w = W.entropy_wave(32)
    s = solver_for(w)
    s.set_state(state64(w))
    t = 0.0
    dt = w.cfl * w.dx / s.max_wavespeed()
    for _ in range(w.n_steps):
        s.step(dt)
        t += dt
    err = np.abs(s.get_state()[0] - W.entropy_wave_exact_rho(w, t).numpy()).max()
    assert err < 6e-5, err           # SURVEY P10 predicts ~4e-5 at 32^3 after 20 steps


# ------------------------------------------------------------------ gate 4 (P11): Sod
def test_exact_riemann_helper_matches_published_star_values():
    gold = {}
    for line in open(os.path.join(HERE, "golden", "toro_sod_star.txt")):
        if not line.startswith("#") and line.strip():
            k, v = line.split()
            gold[k] = float(v)
    ps, us, rl, rr = ER.star_state(1, 0, 1, 0.125, 0, 0.1)
    for got, key in ((ps, "p_star"), (us, "u_star"), (rl, "rho_star_L"), (rr, "rho_star_R")):
        assert abs(got - gold[key]) <= 0.6e-5 * max(1, abs(gold[key])) + 5e-6, (key, got)


def _sod_l1(nx):
    w = W.sod(nx, 4, 4, noise=0.0)
    s = solver_for(w)
    s.set_state(state64(w))
    t = 0.0
    while t < w.t_end - 1e-14:
        dt = min(w.cfl * w.dx / s.max_wavespeed(), w.t_end - t)
        s.step(dt)
        t += dt
    st = s.get_state()
    assert np.array_equal(st, np.broadcast_to(st[:, :1, :1, :], st.shape))   # stays planar
    rho = st[0, 0, 0]
    x = (np.arange(nx) + 0.5) * w.dx
    rex, _, _ = ER.sample((x - 0.5) / w.t_end, 1, 0, 1, 0.125, 0, 0.1)
    return np.abs(rho - rex).sum() * w.dx, rho, x


def test_gate4_sod_matches_exact_riemann_solution_in_l1():
    l1 = {}
    for nx in (128, 256, 512):
        l1[nx], rho, x = _sod_l1(nx)
    assert l1[512] <= 1e-2, l1
    assert math.log2(l1[128] / l1[256]) > 0.55 and math.log2(l1[256] / l1[512]) > 0.6, l1
    # Fig. 2 (L115): the regularised shock is a smooth monotone profile at the grid scale
    seg = rho[np.searchsorted(x, 0.5 + 0.2 * 1.3):]
    jump = 0.26557 - 0.125
    assert np.diff(seg).max() <= 0.01 * jump
    # no Gibbs oscillation anywhere: global bounds within 2 % of the shock jump (the residual
    # is the start-up pulse of the smoothed interface at the rarefaction head)
    assert rho.min() >= 0.125 - 0.02 * jump and rho.max() <= 1.0 + 0.02 * jump


# ------------------------------------------------------------------ inflow patches, jets
def test_soft_edged_inflow_patch_ghosts_blend_fixed_state_and_interior():
    n = 16
    pt = (8.0, 7.0, 4.0, 1.0, 0.5, 0.0, 0.0, 6.0, 2.0)
    s = R.RefSolver(n, n, n, 1.0, 1.4, 10.0, faces=(1, 1, 1, 1, 2, 1), patches={4: [pt]})
    rng = np.random.default_rng(2)
    q = np.stack([1 + 0.1 * rng.uniform(-1, 1, (n, n, n)) for _ in range(5)])
    q[4] += 3.0
    s.set_state(q)
    s.fill_ghosts()
    jj, ii = np.meshgrid(np.arange(n), np.arange(n), indexing="ij")
    r = np.hypot(ii + 0.5 - pt[0], jj + 0.5 - pt[1])
    wgt = np.where(r >= pt[2] + 4 * pt[3], 0.0, 0.5 * (1 - np.tanh((r - pt[2]) / pt[3])))
    fixed = [0.5, 0.0, 0.0, 3.0, 2.0 / 0.4 + 0.5 * 0.5 * 36.0]
    assert wgt.max() > 0.99 and (wgt == 0).sum() > 20
    for c in range(5):
        P = s.get_padded(c)
        for g in range(3):
            np.testing.assert_allclose(P[g, 3:-3, 3:-3], wgt * fixed[c] + (1 - wgt) * q[c][0],
                                       rtol=1e-14, atol=1e-15)


def test_small_jet_workload_stays_finite_and_positive():
    w = W.jets33(n=40, radius=6, rings=((0, 1),), n_steps=30)
    s = solver_for(w)
    s.set_state(state64(w))
    for _ in range(w.n_steps):
        lam = s.max_wavespeed()
        assert np.isfinite(lam) and lam > 0
        s.step(w.cfl * w.dx / lam)
    st = s.get_state()
    p = 0.4 * (st[4] - 0.5 * (st[1] ** 2 + st[2] ** 2 + st[3] ** 2) / st[0])
    assert np.isfinite(st).all() and st[0].min() > 0 and p.min() > 0
    assert st[3].max() > 1.0 and np.abs(s.get_sigma()).max() > 1e-3


def test_subbox_reproduces_full_domain_in_dependency_cone():
    """SURVEY 8(c) "oracle reach": per RHS evaluation the result depends on data within +-8 cells
    (3 reconstruction + 5 sweeps), so after one step (3 evaluations) a sub-box with pad 24 equals
    the full-domain run on its core."""
    w = W.jets33(n=72, radius=6, rings=((12, 3),))
    s = solver_for(w)
    q = state64(w)
    s.set_state(q)
    dt = 0.5 / s.max_wavespeed()
    s.step(dt)
    full = s.get_state()
    lo, hi = (10, 14, 0), (10 + 56, 14 + 52, 40)        # touches z = 0 (inflow face) only
    wb = W.subbox(w, lo, hi)
    qb = state64(wb)
    assert np.array_equal(qb, q[:, lo[2]:hi[2], lo[1]:hi[1], lo[0]:hi[0]])
    sb = solver_for(wb)
    sb.set_state(qb)
    sb.step(dt)
    pad = 24
    core = sb.get_state()[:, :hi[2] - lo[2] - pad, pad:-pad, pad:-pad]
    ref = full[:, lo[2]:hi[2] - pad, lo[1] + pad:hi[1] - pad, lo[0] + pad:hi[0] - pad]
    assert np.array_equal(core, ref)
