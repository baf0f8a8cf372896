"""Finding F1 under test: what the scheme AS READ does on the inputs AS BASELINE.json STATES
THEM, with the oracle.  CPU only.

The purely linear fifth-order reconstruction with a local Lax-Friedrichs flux, alpha = 10 dx^2 and five
warm-started sweeps from Sigma = 0 has no limiter and no floor (reading A10).  These tests record, as
reproducible facts and not as prose, that it does not survive grid-sharp data, what the smallest changes are
that do survive, and the numbers behind the smoothing the input recipe uses (section 3 of DESIGN.md).
Nothing here is a parity tolerance: the expected values are step counts and overshoots measured with the oracle,
asserted with margins, so that a change of the oracle's arithmetic that moves them is noticed."""
import dataclasses
import math
import os
import sys

import numpy as np
import pytest
import torch

from oracle import igr_ref as R
from paper_2505_07392_b200 import workloads as W

sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))
import exact_riemann as ER   # noqa: E402


def lifetime(w, n_max, lam_floor=0.0, t_end=None):
    """Steps the oracle takes before the state stops being finite and positive (rho, p > 0), at most n_max.
    Returns (steps, alive, solver, time)."""
    s = R.RefSolver(w.nx, w.ny, w.nz, w.dx, w.gamma, w.alpha, order=w.order, n_jacobi=w.n_jacobi, faces=w.faces,
                    patches=w.patches)
    s.set_state(W.state(w, dtype=torch.float64).numpy())
    t = 0.0
    for n in range(n_max):
        q = s.get_state()
        p = (w.gamma - 1) * (q[4] - 0.5 * (q[1] ** 2 + q[2] ** 2 + q[3] ** 2) / q[0])
        if not (np.isfinite(q).all() and q[0].min() > 0 and p.min() > 0):
            return n, False, s, t
        if t_end is not None and t >= t_end - 1e-14:
            return n, True, s, t
        dt = w.cfl * w.dx / max(s.max_wavespeed(), lam_floor)
        if t_end is not None:
            dt = min(dt, t_end - t)
        s.step(dt)
        t += dt
    return n_max, True, s, t


def sod(nx, smooth, alpha_dx2=10.0):
    w = W.sod(nx, 4, 4, noise=0.0, smooth=smooth)
    return dataclasses.replace(w, alpha=alpha_dx2 * w.dx * w.dx)


def test_f1_config2_as_stated_loses_positivity_after_ten_steps():
    """Config 2 with the one-cell interface of BASELINE.json (left state for x < 0.5, right state otherwise),
    256 cells, alpha = 10 dx^2, CFL 0.5: negative pressure at step 10."""
    n, alive, _, t = lifetime(sod(256, 0.0), 60, t_end=0.2)
    assert not alive and 8 <= n <= 12, (n, alive)
    assert t < 0.012                                # 5 % of the run
    # more sweeps do not help (the advisor's question: five sweeps from Sigma = 0 are far from converged)
    n20, alive20, _, _ = lifetime(dataclasses.replace(sod(256, 0.0), n_jacobi=20), 60, t_end=0.2)
    assert not alive20 and 7 <= n20 <= 12, n20


def test_f1_config2_survives_with_half_the_regularisation_or_a_one_cell_ramp():
    """The same sharp start survives with alpha = 5 dx^2; with alpha = 10 dx^2 a tanh ramp of half-width one
    cell survives too -- but leaves a start-up pulse of 13 % of rho_L at the head of the rarefaction, against
    0.1 % with the half-width of 4 cells that the input recipe uses.  4 is the smallest of (1, 2, 3, 4) that
    keeps the profile within gate 4's bound (2 % of the shock's density jump, Fig. 2 / L115: "smooth profiles at
    the grid scale"), which is why the recipe uses it and not the smallest ramp that merely survives."""
    jump = 0.26557 - 0.125
    n, alive, _, _ = lifetime(sod(256, 0.0, alpha_dx2=5.0), 600, t_end=0.2)
    assert alive and n > 200
    over = {}
    for half_width in (1.0, 2.0, 3.0, 4.0):
        n, alive, s, t = lifetime(sod(256, half_width), 600, t_end=0.2)
        assert alive and abs(t - 0.2) < 1e-12
        rho = s.get_state()[0, 0, 0]
        over[half_width] = rho.max() - 1.0
        x = (np.arange(256) + 0.5) / 256
        rex, _, _ = ER.sample((x - 0.5) / 0.2, 1, 0, 1, 0.125, 0, 0.1)
        l1 = np.abs(rho - rex).sum() / 256
        assert l1 < (0.02 if half_width < 2 else 0.01), (half_width, l1)
    assert 0.10 < over[1.0] < 0.16 and 0.03 < over[2.0] < 0.06 and 0.008 < over[3.0] < 0.016, over
    assert over[4.0] <= 0.02 * jump < over[3.0], over


def test_f1_jets_as_stated_violate_their_own_cfl_bound_then_lose_positivity():
    """Configs 4 / 5 as stated: grid-sharp Mach-3 patches (edge 0) into gas AT REST (no columns).  (a) The CFL
    speed of the interior (reading A9) knows nothing of the inflow ghosts, which are 8 times faster than the
    sound speed of the gas at rest: the first step is taken at an effective CFL number of ~4 and the state is
    not finite after it.  (b) With dt bounded by the patch speed as well (a harness-side fix, not part of the
    method) the under-expanded jet loses positivity at the patch lip within 20 steps.  With the recipe's
    tanh-edged patches and pre-filled columns the same replica lives ~90 steps (F1: 338 / 137 steps at
    the full sizes of configs 4 / 5)."""
    stated = W.jets9(n=40, radius=5, pitch=12, stub_delta=0.0)
    assert stated.patches[4][0][3] == 0.0                                   # sharp mask
    q0 = W.state(stated, dtype=torch.float64).numpy()
    assert np.abs(q0[3]).max() < 2e-3 and abs(q0[0].max() - 1) < 1e-12     # at rest but for the seeded noise
    n, alive, _, _ = lifetime(stated, 10)
    assert not alive and n <= 2, n
    lam_jet = 4.0 * math.sqrt(1.4 * 2.0 / 0.5)                              # |w_j| + c_j
    n, alive, _, _ = lifetime(stated, 60, lam_floor=lam_jet)
    assert not alive and 8 <= n <= 20, n
    n, alive, _, _ = lifetime(W.jets9(n=40, radius=5, pitch=12), 60)
    assert alive and n == 60
