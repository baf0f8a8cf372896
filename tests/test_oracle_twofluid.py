"""Pins of the two-fluid oracle (oracle/igr_ref2.c, reading A21).  CPU only.

The paper gives no two-fluid equations (Alg. 1 L147, L196, L210, L228 only show that a volume fraction is
reconstructed, enters the flux and is updated like the conserved variables), so what pins this oracle is what the
five-equation model of two ideal gases is KNOWN to do, none of it computed with the oracle's own pieces:
  T1  single-fluid limit: a1 = 1, a2 rho2 = 0 reproduces the pinned single-fluid oracle (bitwise with
      gamma = 1.5, where 1/Gamma = gamma - 1 exactly; to round-off with gamma = 1.4);
  T2  a material interface advected by a uniform flow keeps u and p uniform to round-off (the defining property
      of the isobaric mixture rule Gamma = sum a_i/(gamma_i - 1); a linearly mixed gamma breaks it);
  T3  each partial mass, the momentum and the energy are conserved to round-off on a periodic box;
  T4  the non-conservative term a1 div u: in a uniform dilatation a uniform a1 stays uniform, while the
      divergence form alone would change it at the rate -3 s a1;
  T5  the mixture wave speed max_d|u_d| + sqrt((1 + 1/Gamma) p / rho) against its closed form."""
import math

import numpy as np
import pytest

from oracle import igr_ref as R


def gam(a1, g1, g2):
    return a1 / (g1 - 1) + (1 - a1) / (g2 - 1)


def cons2(a1, rho1, rho2, u, v, w, p, g1, g2):
    """(a1 rho1, a2 rho2, rho u, rho v, rho w, E, a1) from the primitive fields."""
    a1, rho1, rho2, u, v, w, p = (np.asarray(x, dtype=np.float64) for x in (a1, rho1, rho2, u, v, w, p))
    m1, m2 = a1 * rho1, (1 - a1) * rho2
    rho = m1 + m2
    return np.stack([m1, m2, rho * u, rho * v, rho * w, p * gam(a1, g1, g2) + 0.5 * rho * (u * u + v * v + w * w),
                     a1 + 0 * rho])


def smooth(n, seed):
    rng = np.random.default_rng(seed)
    z, y, x = np.meshgrid(*(3 * [(np.arange(n) + 0.5) / n]), indexing="ij")
    tw = 2 * np.pi
    ph = rng.uniform(0, tw, 8)
    rho = 1 + 0.3 * np.sin(tw * x + ph[0]) * np.cos(tw * y + ph[1]) + 0.2 * np.sin(tw * z + ph[2])
    u = 0.5 * np.sin(tw * (x + y) + ph[3]) + 0.1
    v = 0.4 * np.cos(tw * (y - z) + ph[4]) - 0.2
    w = 0.3 * np.sin(tw * (z + x) + ph[5]) * np.cos(tw * y)
    p = 1 + 0.2 * np.cos(tw * (x + y + z) + ph[6])
    a1 = 0.5 + 0.4 * np.sin(tw * x + ph[7]) * np.sin(tw * y) * np.cos(tw * z)
    return rho, u, v, w, p, a1


# ------------------------------------------------------------------------------------------ T1
@pytest.mark.parametrize("gamma,bitwise", [(1.5, True), (1.4, False)])
@pytest.mark.parametrize("bc", ["periodic", "inflow"])
def test_t1_single_fluid_limit_reproduces_the_single_fluid_oracle(gamma, bitwise, bc):
    n, dx = 12, 1.0 / 12
    rho, u, v, w, p, _ = smooth(n, 1)
    st = (0.6, 0.1, -0.2, 1.5, 1.2)                      # rho, u, v, w, p of the inflow patches
    faces = (0,) * 6 if bc == "periodic" else (1, 1, 0, 0, 2, 1)
    p1 = {4: [(5.0, 6.0, 3.0, 0.0) + st, (9.0, 4.0, 2.0, 1.0) + st]} if bc == "inflow" else None
    p2 = {4: [(c0, c1, r, e, st[0], 0.0, 1.0) + st[1:] for c0, c1, r, e in ((5.0, 6.0, 3.0, 0.0), (9.0, 4.0, 2.0, 1.0))]} \
        if bc == "inflow" else None
    one = R.RefSolver(n, n, n, dx, gamma, 10 * dx * dx, faces=faces, patches=p1)
    two = R.RefSolver2(n, n, n, dx, gamma, 1.67, 10 * dx * dx, faces=faces, patches=p2)
    q1 = np.stack([rho, rho * u, rho * v, rho * w, p / (gamma - 1) + 0.5 * rho * (u * u + v * v + w * w)])
    q2 = np.stack([q1[0], 0 * rho, q1[1], q1[2], q1[3], q1[4], 1 + 0 * rho])
    one.set_state(q1); two.set_state(q2)
    for _ in range(3):
        lam = one.max_wavespeed()
        assert two.max_wavespeed() == pytest.approx(lam, rel=0 if bitwise else 1e-14)
        dt = 0.5 * dx / lam
        one.step(dt); two.step(dt)
    a, b = one.get_state(), two.get_state()
    assert np.all(b[1] == 0.0) and np.all(b[6] == 1.0)   # no second fluid appears, a1 stays exactly 1
    got = b[[0, 2, 3, 4, 5]]
    if bitwise:
        assert np.array_equal(got, a)
        assert np.array_equal(one.get_sigma(), two.get_sigma())
    else:
        assert np.abs(got - a).max() <= 1e-13 * np.abs(a).max()
        assert np.abs(one.get_sigma() - two.get_sigma()).max() <= 1e-13 * max(np.abs(one.get_sigma()).max(), 1e-3)


# ------------------------------------------------------------------------------------------ T2
def test_t2_uniform_velocity_and_pressure_survive_a_material_interface():
    n, dx = 16, 1.0 / 16
    g1, g2 = 1.4, 1.67
    u0, p0 = (0.7, -0.4, 0.9), 1.3
    _, _, _, _, _, a1 = smooth(n, 2)
    one = np.ones_like(a1)
    s = R.RefSolver2(n, n, n, dx, g1, g2, 10 * dx * dx)
    s.set_state(cons2(a1, 1.0 * one, 0.2 * one, u0[0] * one, u0[1] * one, u0[2] * one, p0 * one, g1, g2))
    a_start = a1.copy()
    for _ in range(5):
        s.step(0.5 * dx / s.max_wavespeed())
    q = s.get_state()
    rho = q[0] + q[1]
    for a in range(3):
        assert np.abs(q[2 + a] / rho - u0[a]).max() <= 1e-13
    ke = 0.5 * (q[2] ** 2 + q[3] ** 2 + q[4] ** 2) / rho
    p = (q[5] - ke) / gam(q[6], g1, g2)
    assert np.abs(p - p0).max() <= 1e-12
    assert np.abs(s.get_sigma()).max() <= 1e-12                    # no velocity gradients: no entropic pressure
    assert np.abs(q[6] - a_start).max() > 0.05                     # the interface did move
    # the pin discriminates: the pressure a LINEARLY mixed gamma would read off the same state is far from uniform
    g_lin = q[6] * g1 + (1 - q[6]) * g2
    assert np.ptp((g_lin - 1) * (q[5] - ke)) > 1e-2 * p0


# ------------------------------------------------------------------------------------------ T3
def test_t3_partial_masses_momentum_and_energy_are_conserved():
    n, dx = 12, 1.0 / 12
    g1, g2 = 1.4, 1.67
    rho, u, v, w, p, a1 = smooth(n, 3)
    s = R.RefSolver2(n, n, n, dx, g1, g2, 10 * dx * dx)
    q0 = cons2(a1, rho, 0.3 * rho, u, v, w, p, g1, g2)
    s.set_state(q0)
    tot0 = q0.reshape(7, -1).sum(axis=1)
    scale = np.abs(q0).reshape(7, -1).sum(axis=1)
    scale[2:5] = scale[2:5].sum()
    for _ in range(3):
        s.step(0.5 * dx / s.max_wavespeed())
        tot = s.get_state().reshape(7, -1).sum(axis=1)
        assert np.all(np.abs(tot - tot0)[:6] <= 1e-13 * scale[:6]), (tot - tot0) / scale
    assert abs(tot[6] - tot0[6]) > 1e-8 * scale[6]                  # the volume fraction is advected, not conserved
    assert np.abs(s.get_sigma()).max() > 1e-4                       # and the entropic pressure was active


# ------------------------------------------------------------------------------------------ T4
def test_t4_uniform_volume_fraction_stays_uniform_in_a_dilatation():
    n, dx, srate = 14, 0.1, 0.3
    g1, g2 = 1.4, 1.67
    z, y, x = np.meshgrid(*(3 * [(np.arange(n) + 0.5) * dx]), indexing="ij")
    one = np.ones_like(x)
    a0 = 0.37
    s = R.RefSolver2(n, n, n, dx, g1, g2, 10 * dx * dx, faces=(1,) * 6)
    s.set_state(cons2(a0 * one, 1.0 * one, 0.2 * one, srate * x, srate * y, srate * z, 2.0 * one, g1, g2))
    s.eval_rhs()
    r = s.get_rhs()
    inner = (slice(4, -4),) * 3                                      # away from the clamped ghosts
    assert np.abs(r[6][inner]).max() <= 1e-13
    # the divergence form alone: d(a1)/dt = -div(a1 u) = -3 s a1, which is what the partial masses feel
    for c, val in ((0, a0 * 1.0), (1, (1 - a0) * 0.2)):
        assert r[c][inner] == pytest.approx(-3 * srate * val, rel=1e-12)


# ------------------------------------------------------------------------------------------ T5
def test_t5_mixture_wavespeed_is_the_closed_form():
    g1, g2 = 1.4, 1.67
    a1, rho1, rho2, u, v, w, p = 0.3, 1.1, 0.25, 0.2, -0.9, 0.4, 1.7
    s = R.RefSolver2(5, 4, 3, 0.1, g1, g2, 0.1)
    one = np.ones((3, 4, 5))
    s.set_state(cons2(a1 * one, rho1 * one, rho2 * one, u * one, v * one, w * one, p * one, g1, g2))
    rho = a1 * rho1 + (1 - a1) * rho2
    G = a1 / 0.4 + 0.7 / 0.67
    assert s.max_wavespeed() == pytest.approx(0.9 + math.sqrt((1 + 1 / G) * p / rho), rel=1e-13)
    # neither pure-fluid sound speed
    for g in (g1, g2):
        assert abs(0.9 + math.sqrt(g * p / rho) - s.max_wavespeed()) > 1e-2
