"""Pins of the two places where the oracle forms a wave speed (CPU only).

P15  igr_ref_max_wavespeed (the CFL speed, reading A9: max over INTERIOR cells of max_d |u_d| + sqrt(gamma p / rho))
     against the closed form on states where every plausible mistake gives another number: gamma dropped from
     the sound speed, the Euclidean norm of u in place of the largest component, a signed velocity, the
     kinetic energy left in the pressure, ghost cells entering the maximum.
P16  the cell-centred sound speed and the local Lax-Friedrichs speed inside igr_ref_rhs (reading A5:
     lambda = max over the two cells beside a face of |u_d| + sqrt(gamma p / rho), p without Sigma) against the
     TEXTBOOK Rusanov flux worked out here by hand: a y-z-uniform density jump with constant u and p is pure
     linear advection of rho, so r beside the jump follows from face values of the unique quartic with the
     given cell averages (solved here with numpy, no coefficient table) and from
     F^ = (F_L + F_R)/2 - lambda (U_R - U_L)/2.
Nothing here calls a piece of the oracle to form an expected value."""
import math

import numpy as np
import pytest

from oracle import igr_ref as R

G = 1.4


def cons(rho, u, v, w, p):
    rho, u, v, w, p = (np.asarray(a, dtype=np.float64) for a in (rho, u, v, w, p))
    return np.stack([rho, rho * u, rho * v, rho * w, p / (G - 1) + 0.5 * rho * (u * u + v * v + w * w)])


# --------------------------------------------------------------------------------------- P15
def test_p15_wavespeed_of_a_uniform_state_is_the_closed_form():
    rho, u, v, w, p = 0.9, 0.3, -0.7, 1.1, 1.3
    s = R.RefSolver(6, 5, 4, 0.1, G, 0.1)
    s.set_state(cons(*(np.full((4, 5, 6), a) for a in (rho, u, v, w, p))))
    want = 1.1 + math.sqrt(1.4 * 1.3 / 0.9)                        # = 2.5220486...
    assert want == pytest.approx(2.5220486, abs=1e-7)
    assert s.max_wavespeed() == pytest.approx(want, rel=1e-14)
    # what the plausible mistakes would have returned
    wrong = [1.1 + math.sqrt(1.3 / 0.9),                            # gamma dropped
             math.sqrt(0.3 ** 2 + 0.7 ** 2 + 1.1 ** 2) + math.sqrt(1.4 * 1.3 / 0.9),   # |u|_2
             1.1 + math.sqrt(1.4 * (1.3 + 0.4 * 0.5 * 0.9 * (0.09 + 0.49 + 1.21)) / 0.9)]  # kinetic energy in p
    assert all(abs(x - want) > 1e-2 for x in wrong)


@pytest.mark.parametrize("axis", [0, 1, 2])
def test_p15_wavespeed_picks_the_largest_component_of_the_fastest_interior_cell(axis):
    """One cell carries the maximum, through a NEGATIVE velocity component along `axis` that is larger in
    magnitude than the other two (which are not zero, so a Euclidean norm would show)."""
    nx, ny, nz = 7, 6, 5
    rho = np.full((nz, ny, nx), 1.0); p = np.full_like(rho, 1.0)
    vel = [np.full_like(rho, 0.1), np.full_like(rho, 0.2), np.full_like(rho, 0.05)]
    k, j, i = 3, 2, 4
    rho[k, j, i], p[k, j, i] = 0.5, 2.0
    comp = [1.0, -0.8, 0.6]
    comp[axis] = -2.5
    for a in range(3):
        vel[a][k, j, i] = comp[a]
    s = R.RefSolver(nx, ny, nz, 0.1, G, 0.1)
    s.set_state(cons(rho, vel[0], vel[1], vel[2], p))
    want = 2.5 + math.sqrt(1.4 * 2.0 / 0.5)
    assert s.max_wavespeed() == pytest.approx(want, rel=1e-14)
    assert math.sqrt(sum(c * c for c in comp)) + math.sqrt(1.4 * 2.0 / 0.5) - want > 0.1     # |u|_2 differs
    assert want - (max(comp) + math.sqrt(1.4 * 2.0 / 0.5)) > 1.0                              # signed max differs


def test_p15_ghost_cells_do_not_enter_the_maximum():
    """An inflow patch far faster than the interior: after the ghosts are filled they hold the jet state, the
    CFL speed is still the interior one ("max over interior cells")."""
    nx = ny = nz = 8
    patch = (4.0, 4.0, 3.0, 0.0, 0.5, 0.0, 0.0, 9.0, 3.0)            # c0, c1, radius, edge, rho, u, v, w, p
    s = R.RefSolver(nx, ny, nz, 1.0, G, 10.0, faces=(1, 1, 1, 1, 2, 1), patches={4: [patch]})
    one = np.ones((nz, ny, nx))
    s.set_state(cons(one, 0.2 * one, 0.0 * one, -0.1 * one, one))
    s.fill_ghosts()
    assert s.get_padded(3)[2, 3 + 4, 3 + 4] == pytest.approx(0.5 * 9.0)      # the ghost holds the jet
    assert s.max_wavespeed() == pytest.approx(0.2 + math.sqrt(1.4), rel=1e-14)


# --------------------------------------------------------------------------------------- P16
def face_values(avg6):
    """Left / right value at the face between cells 0 and 1 of the degree-4 polynomials whose cell averages
    over unit cells -2..2 (left-biased) and -1..3 (right-biased) are the given ones: the DEFINITION of the
    fifth-order finite-volume reconstruction, solved numerically."""
    out = []
    for cells in (range(-2, 3), range(-1, 4)):
        A = np.array([[((c + 0.5) ** (k + 1) - (c - 0.5) ** (k + 1)) / (k + 1) for k in range(5)] for c in cells])
        coef = np.linalg.solve(A, np.array([avg6[c + 2] for c in cells]))
        out.append(sum(coef[k] * 0.5 ** k for k in range(5)))
    return out


@pytest.mark.parametrize("U", [0.3, -0.45])
def test_p16_rusanov_flux_beside_a_density_jump(U):
    nx, ny, nz, dx = 16, 4, 4, 0.125
    P, ra, rb, jump = 1.3, 1.0, 0.25, 8
    rho1d = np.where(np.arange(nx) < jump, ra, rb)
    rho = np.broadcast_to(rho1d, (nz, ny, nx)).copy()
    one = np.ones_like(rho)
    s = R.RefSolver(nx, ny, nz, dx, G, 10 * dx * dx, faces=(1, 1, 0, 0, 0, 0))
    s.set_state(cons(rho, U * one, 0 * one, 0 * one, P * one))
    s.eval_rhs()                                   # ghosts, source (zero: u is constant), sweeps, r
    assert np.abs(s.get_sigma()).max() == 0.0
    r = s.get_rhs()

    # textbook: linear advection of rho at speed U; Rusanov flux with the LOCAL speed of the two cells
    rho_ext = np.concatenate([np.full(3, ra), rho1d, np.full(3, rb)])          # extrapolation ghosts

    def cell_speed(i):
        return abs(U) + math.sqrt(G * P / rho_ext[i + 3])

    def flux(i):                                   # numerical fluxes at face i + 1/2, (rho, m_x, E)
        rl, rr = face_values(rho_ext[i + 3 - 2:i + 3 + 4])
        lam = max(cell_speed(i), cell_speed(i + 1))
        UL = np.array([rl, rl * U, P / (G - 1) + 0.5 * rl * U * U])
        UR = np.array([rr, rr * U, P / (G - 1) + 0.5 * rr * U * U])
        FL = np.array([rl * U, rl * U * U + P, (UL[2] + P) * U])
        FR = np.array([rr * U, rr * U * U + P, (UR[2] + P) * U])
        return 0.5 * (FL + FR) - 0.5 * lam * (UR - UL)

    lam_jump = abs(U) + math.sqrt(G * P / rb)      # the lighter gas is the faster one
    assert max(cell_speed(jump - 1), cell_speed(jump)) == lam_jump
    for i in range(jump - 3, jump + 3):            # every cell whose faces feel the jump
        want = -(flux(i) - flux(i - 1)) / dx
        got = r[[0, 1, 4], 1, 2, i]
        assert got == pytest.approx(want, rel=1e-11, abs=1e-12), (i, got, want)
        assert r[2, 1, 2, i] == 0.0 and r[3, 1, 2, i] == 0.0
    # the pin discriminates: with the speed of the HEAVIER side, without gamma, or without |u| the mass
    # residual beside the jump would differ in the second digit
    i = jump - 1
    rl, rr = face_values(rho_ext[i + 3 - 2:i + 3 + 4])
    for lam_wrong in (abs(U) + math.sqrt(G * P / ra), abs(U) + math.sqrt(P / rb), math.sqrt(G * P / rb)):
        assert abs(0.5 * (lam_wrong - lam_jump) * (rr - rl) / dx) > 1e-2 * abs(r[0, 1, 2, i])
