"""NEXT-1: pins of the oracle's viscous fluxes (eqs. 2, 3, 5, L55-L67; Alg. 1
L164-L173, L191) against textbook results.  CPU only."""
import numpy as np
import pytest

from oracle import igr_ref as R

G = 1.4


def cons(rho, u, v, w, p):
    return np.stack([rho, rho * u, rho * v, rho * w, p / (G - 1) + 0.5 * rho * (u * u + v * v + w * w)])


def test_stress_tensor_textbook_cases():
    mu, zeta = 0.7, 0.3
    u0 = np.zeros(3)
    om = np.array([0.3, -0.5, 0.8])                       # rigid rotation: no viscous stress at all
    Arot = np.array([[0, -om[2], om[1]], [om[2], 0, -om[0]], [-om[1], om[0], 0]])
    for d in range(3):
        assert np.abs(R.viscous_flux(d, mu, zeta, Arot, u0)).max() < 1e-15
    s = 0.9                                               # uniform dilatation: tau = 3 zeta s I (mu drops out)
    for d in range(3):
        F = R.viscous_flux(d, mu, zeta, s * np.eye(3), u0)
        expect = np.zeros(5)
        expect[1 + d] = -3 * zeta * s
        np.testing.assert_allclose(F, expect, atol=1e-15)
    A = np.zeros((3, 3))                                  # simple shear du_x/dy = s: tau_xy = tau_yx = mu s
    A[0, 1] = s
    uf = np.array([2.0, -1.0, 0.5])
    Fy = R.viscous_flux(1, mu, zeta, A, uf)               # flux along y carries -tau_xy in x-momentum
    np.testing.assert_allclose(Fy, [0, -mu * s, 0, 0, -uf[0] * mu * s], atol=1e-15)
    Fx = R.viscous_flux(0, mu, zeta, A, uf)               # symmetric: flux along x carries -tau_yx in y-momentum
    np.testing.assert_allclose(Fx, [0, 0, -mu * s, 0, -uf[1] * mu * s], atol=1e-15)
    np.testing.assert_allclose(R.viscous_flux(2, mu, zeta, A, uf), 0, atol=1e-15)


def _solver(n, dx, mu, zeta, faces=(0,) * 6, alpha=None):
    s = R.RefSolver(n[0], n[1], n[2], dx, G, 10 * dx * dx if alpha is None else alpha, faces=faces)
    s.set_viscosity(mu, zeta)
    return s


def test_zero_viscosity_is_the_inviscid_scheme_bitwise():
    rng = np.random.default_rng(0)
    n = 8
    q = cons(1 + 0.1 * rng.uniform(-1, 1, (n, n, n)), *(0.3 * rng.uniform(-1, 1, (3, n, n, n))), np.ones((n, n, n)))
    a, b = _solver((n, n, n), 1 / n, 0.0, 0.0), R.RefSolver(n, n, n, 1 / n, G, 10 / n ** 2)
    for s in (a, b):
        s.set_state(q)
        s.step(0.01)
    assert np.array_equal(a.get_state(), b.get_state())


def test_linear_velocity_field_heating_equals_tau_contracted_with_grad_u():
    """u = A x with constant rho, p: the reconstructed gradient is A exactly, so the viscous momentum
    flux is constant (no force) and the energy equation gains div(u . tau) = tau : grad u (eq. 3)."""
    rng = np.random.default_rng(1)
    n, dx, mu, zeta = 12, 0.1, 0.4, 0.25
    A = rng.uniform(-1, 1, (3, 3))
    c = (np.arange(n) + 0.5) * dx
    z, y, x = np.meshgrid(c, c, c, indexing="ij")
    vel = np.einsum("ab,bzyx->azyx", A, np.stack([x, y, z]))
    q = cons(np.full_like(x, 1.3), vel[0], vel[1], vel[2], np.full_like(x, 2.0))
    r = []
    for m_, z_ in ((mu, zeta), (0.0, 0.0)):
        s = _solver((n, n, n), dx, m_, z_, faces=(1,) * 6)
        s.set_state(q)
        s.fill_ghosts(); s.fill_sigma_ghosts()
        s.rhs()
        r.append(s.get_rhs())
    dv = (r[0] - r[1])[:, 4:-4, 4:-4, 4:-4]               # clamp ghosts break linearity near the rim
    tau = mu * (A + A.T) + (zeta - 2 * mu / 3) * np.trace(A) * np.eye(3)
    np.testing.assert_allclose(dv[1:4], 0.0, atol=1e-11)
    np.testing.assert_allclose(dv[0], 0.0, atol=1e-13)
    np.testing.assert_allclose(dv[4], np.sum(tau * A), rtol=1e-10)


def test_shear_wave_decays_at_the_discrete_viscous_rate():
    """rho = 1, u_y = a sin(2 pi x): a pure shear wave (no dilatation, Sigma = 0) decays as
    exp(-nu k^2 t); checked against the exact amplification factor of the discrete operator."""
    n, mu, amp, nsteps = 32, 0.02, 1e-5, 40
    dx = 1.0 / n
    x = (np.arange(n) + 0.5) * dx
    uy = amp * np.sin(2 * np.pi * x)[None, None, :] * np.ones((4, 4, 1))
    one = np.ones_like(uy)
    q = cons(one, 0 * one, uy, 0 * one, 10 * one)
    dt = 0.2 * dx / np.sqrt(1.4 * 10)
    amps = []
    for m_ in (mu, 0.0):
        s = _solver((n, 4, 4), dx, m_, 0.0)
        s.set_state(q)
        for _ in range(nsteps):
            s.step(dt)
        my = s.get_state()[2, 0, 0]
        amps.append(2 * np.abs(np.fft.rfft(my)[1]) / n)
        assert np.abs(s.get_sigma()).max() < 1e-12
    # discrete symbol: central difference -> face value (mean of the L and R reconstructions) -> divergence
    th = 2 * np.pi / n
    cbar = 0.5 * (np.array([2, -13, 47, 27, -3, 0]) + np.array([0, -3, 27, 47, -13, 2])) / 60.0
    face = sum(cbar[t] * np.exp(1j * (t - 2) * th) for t in range(6))       # relative to cell i (face i+1/2)
    lam = mu * (1j * np.sin(th) / dx) * face * (1 - np.exp(-1j * th)) / dx
    assert abs(lam.imag) < 1e-9 * abs(lam.real) and lam.real < 0
    assert lam.real == pytest.approx(-mu * (2 * np.pi) ** 2, rel=2e-2)      # -> -nu k^2 as dx -> 0
    z_ = lam.real * dt
    g = 1 + z_ + z_ ** 2 / 2 + z_ ** 3 / 6
    assert amps[0] / amps[1] == pytest.approx(g ** nsteps, rel=1e-6)
    assert amps[0] / amps[1] < 0.98


def test_conservation_with_viscosity_on_periodic_grid():
    n = 12
    c = (np.arange(n) + 0.5) / n
    z, y, x = np.meshgrid(c, c, c, indexing="ij")
    tw = 2 * np.pi
    q = cons(1 + 0.2 * np.sin(tw * x) * np.cos(tw * y), 0.5 * np.sin(tw * (x + y)), 0.4 * np.cos(tw * (y - z)),
             0.3 * np.sin(tw * (z + x)), 1 + 0.2 * np.cos(tw * (x + y + z)))
    s = _solver((n, n, n), 1 / n, 0.01, 0.005)
    s.set_state(q)
    tot0, scale = q.reshape(5, -1).sum(1), np.abs(q).reshape(5, -1).sum(1)
    for _ in range(5):
        s.step(0.3 / n / s.max_wavespeed())
    assert np.all(np.abs(s.get_state().reshape(5, -1).sum(1) - tot0) <= 1e-13 * scale)
