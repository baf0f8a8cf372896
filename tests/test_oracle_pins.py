"""Pins of the fp64 oracle against what the paper and the mathematics fix (SURVEY 8(c) P1-P6,
P9, P12, P13).  CPU only.  None of these re-types the oracle's formula: each checks a closed
form, an invariant, a dense solve, or a special case that reduces to a textbook result."""
import math

import numpy as np
import pytest

from oracle import igr_ref as R
from paper_2505_07392_b200 import workloads as W

G = 1.4


def cons(rho, u, v, w, p):
    return np.stack([rho, rho * u, rho * v, rho * w, p / (G - 1) + 0.5 * rho * (u * u + v * v + w * w)])


def make(nx, ny, nz, dx=None, faces=(0,) * 6, patches=None, alpha=None, n_jacobi=5, order=5):
    dx = dx if dx is not None else 1.0 / nx
    alpha = alpha if alpha is not None else 10 * dx * dx
    return R.RefSolver(nx, ny, nz, dx, G, alpha, order=order, n_jacobi=n_jacobi, faces=faces,
                       patches=patches)


# ---------------------------------------------------------------------------------- P1, P2
@pytest.mark.parametrize("order,exact_deg", [(5, 4), (3, 2)])
def test_p1_reconstruction_exact_on_monomial_cell_averages(order, exact_deg):
    """PAPER.md L132 "fifth-order accurate finite volume": from exact cell averages of x^k the
    face value is reproduced to round-off for k <= 4 and not for k = 5 (order 3: k <= 2)."""
    dx, xf = 0.37, 0.5 * 0.37   # cells q=-2..3 centred at q*dx; face between cells 0 and 1

    def avg(k, qc):
        a, b = (qc - 0.5) * dx, (qc + 0.5) * dx
        return (b ** (k + 1) - a ** (k + 1)) / ((k + 1) * dx)

    for k in range(exact_deg + 2):
        f6 = np.array([avg(k, qc) for qc in range(-2, 4)])
        fl, fr = R.reconstruct(order, f6)
        errs = (abs(fl - xf ** k), abs(fr - xf ** k))
        if k <= exact_deg:
            assert max(errs) < 1e-14, (k, errs)
        else:
            assert min(errs) > 1e-6 * dx ** k, (k, errs)


def test_p2_jump_is_fifth_undivided_difference():
    """U_R - U_L = (-1, 5, -10, 10, -5, 1)/30 on cells -2..3: LF dissipation is O(dx^5)."""
    expect = np.array([-1, 5, -10, 10, -5, 1]) / 30.0
    for t in range(6):
        e = np.zeros(6)
        e[t] = 1.0
        fl, fr = R.reconstruct(5, e)
        assert abs((fr - fl) - expect[t]) < 1e-15
    fl, fr = R.reconstruct(5, np.ones(6))      # partition of unity
    assert abs(fl - 1) < 1e-15 and abs(fr - 1) < 1e-15
    fl, fr = R.reconstruct(5, np.array([0, 0, 1.0, 0, 0, 0]))   # upwind bias: L weights cell 0 most
    assert fl == pytest.approx(47 / 60) and fr == pytest.approx(27 / 60)


# ---------------------------------------------------------------------------------- P3
@pytest.mark.parametrize("d", [0, 1, 2])
def test_p3_lf_flux_consistency_and_upwind_limit(d):
    rng = np.random.default_rng(3)
    rho, p, sig = 0.7, 1.3, 0.21
    vel = rng.uniform(-1, 1, 3)
    U = cons(np.float64(rho), *vel, np.float64(p))
    F = R.lf_flux(d, G, U, U, sig, sig, 5.0)
    # consistency F^(U,U) = F(U): Euler flux of eqs (6)-(8) written from the primitives
    H = U[4] + p + sig
    expect = np.array([rho * vel[d]] + [rho * vel[a] * vel[d] + (p + sig) * (a == d) for a in range(3)]
                      + [H * vel[d]])
    np.testing.assert_allclose(F, expect, rtol=1e-14, atol=1e-15)
    # constant u, p with a density jump and lambda = |u_d|: the mass flux is exact upwinding
    rl, rr = 1.0, 0.3
    UL, UR = cons(np.float64(rl), *vel, np.float64(p)), cons(np.float64(rr), *vel, np.float64(p))
    F = R.lf_flux(d, G, UL, UR, 0.0, 0.0, abs(vel[d]))
    up = rl if vel[d] > 0 else rr
    assert F[0] == pytest.approx(vel[d] * up, rel=1e-14)
    # Sigma enters the normal momentum and the energy flux only, and gets no dissipation
    F0 = R.lf_flux(d, G, UL, UR, 0.0, 0.0, 2.0)
    F1 = R.lf_flux(d, G, UL, UR, 0.4, 0.6, 2.0)
    dF = F1 - F0
    expect = np.zeros(5)
    expect[1 + d] = 0.5
    expect[4] = 0.5 * (0.4 + 0.6) * vel[d]
    np.testing.assert_allclose(dF, expect, atol=1e-14)


# ---------------------------------------------------------------------------------- P4
def test_p4_ssprk3_third_order_on_linear_ode():
    """y' = -y with the stage combinations of ref. 17 (L389) converges at order 3 and one step
    equals the degree-3 Taylor polynomial of exp(-dt)."""
    def step(y, dt):
        yn = np.array([y])
        y1 = R.rk_combine(0.0, yn, 1.0, yn, dt, -yn)
        y2 = R.rk_combine(0.75, yn, 0.25, y1, dt, -y1)
        return R.rk_combine(1 / 3, yn, 2 / 3, y2, dt, -y2)[0]

    dt = 0.3
    assert step(1.0, dt) == pytest.approx(1 - dt + dt ** 2 / 2 - dt ** 3 / 6, rel=1e-15)
    errs = []
    for n in (10, 20, 40):
        y = 1.0
        for _ in range(n):
            y = step(y, 1.0 / n)
        errs.append(abs(y - math.exp(-1.0)))
    assert 2.8 < math.log2(errs[0] / errs[1]) < 3.2 and 2.8 < math.log2(errs[1] / errs[2]) < 3.2


# ---------------------------------------------------------------------------------- P5
def _source_for_linear_field(A, n=8, dx=0.1, alpha=0.37):
    s = make(n, n, n, dx=dx, alpha=alpha, faces=(1,) * 6)
    c = (np.arange(n) + 0.5) * dx
    z, y, x = np.meshgrid(c, c, c, indexing="ij")
    pos = np.stack([x, y, z])
    vel = np.einsum("ab,bzyx->azyx", A, pos)
    rho = 1.0 + 0.1 * np.sin(3 * x + y) * np.cos(z)     # non-uniform density must not matter
    s.set_state(cons(rho, vel[0], vel[1], vel[2], np.ones_like(x)))
    s.fill_ghosts()
    s.source()
    return s.get_source()[1:-1, 1:-1, 1:-1]          # clamp ghosts break linearity at the rim


def test_p5_source_on_linear_velocity_fields():
    """eq. (9) left side (L127): b = alpha (tr(A^2) + tr(A)^2) exactly for u = A x."""
    rng = np.random.default_rng(5)
    alpha = 0.37
    A = rng.uniform(-1, 1, (3, 3))
    b = _source_for_linear_field(A, alpha=alpha)
    np.testing.assert_allclose(b, alpha * (np.trace(A @ A) + np.trace(A) ** 2), rtol=1e-11)
    om = np.array([0.3, -0.5, 0.8])                  # pure rotation: b = -alpha |omega|^2 / 2
    Arot = np.array([[0, -om[2], om[1]], [om[2], 0, -om[0]], [-om[1], om[0], 0]])
    b = _source_for_linear_field(Arot, alpha=alpha)
    np.testing.assert_allclose(b, -alpha * 2 * om.dot(om), rtol=1e-11)   # |vorticity| = 2|om|
    sdil = 0.7                                        # uniform dilatation: 3 s^2 + 9 s^2
    b = _source_for_linear_field(sdil * np.eye(3), alpha=alpha)
    np.testing.assert_allclose(b, alpha * 12 * sdil ** 2, rtol=1e-11)
    # a transposed-operand mistake (G_ab G_ab instead of G_ab G_ba) would fail the rotation case


# ---------------------------------------------------------------------------------- P6
def _dense_operator(rho, dx, alpha):
    """Matrix of Sigma/rho - alpha div(grad Sigma / rho) on a periodic grid, 6-point stencil,
    face density = arithmetic mean: assembled face by face (independent of the oracle)."""
    nz, ny, nx = rho.shape
    N = rho.size
    A = np.zeros((N, N))
    lin = np.arange(N).reshape(rho.shape)
    k2 = alpha / dx ** 2
    A[np.arange(N), np.arange(N)] += 1.0 / rho.ravel()
    for ax in range(3):
        nb = np.roll(lin, -1, axis=ax)
        rf = 0.5 * (rho + np.roll(rho, -1, axis=ax))
        for i, n_, r in zip(lin.ravel(), nb.ravel(), rf.ravel()):
            # flux through the face between i and n: (Sigma_n - Sigma_i)/(rho_f dx)
            A[i, i] += k2 / r
            A[i, n_] -= k2 / r
            A[n_, n_] += k2 / r
            A[n_, i] -= k2 / r
    return A


def test_p6_jacobi_matches_dense_solve_on_4cubed():
    rng = np.random.default_rng(6)
    n, dx = 4, 0.25
    alpha = 10 * dx * dx
    rho = rng.uniform(0.5, 2.0, (n, n, n))
    sig_star = rng.uniform(-1, 1, (n, n, n))
    A = _dense_operator(rho, dx, alpha)
    assert np.allclose(A, A.T) and np.linalg.eigvalsh(A).min() > 0          # SPD
    b = (A @ sig_star.ravel()).reshape(rho.shape)
    s = make(n, n, n, dx=dx, alpha=alpha, n_jacobi=1)
    zero = np.zeros_like(rho)
    s.set_state(cons(rho, zero, zero, zero, np.ones_like(rho)))
    s.fill_ghosts()
    s.source()
    assert np.all(s.get_source() == 0)             # gas at rest: b = 0
    s.set_source(b)                                # test hook: drive the sweeps with b* = A Sigma*
    first = None
    for it in range(3000):
        s.jacobi_sweep()
        if it == 0:
            first = s.get_sigma().copy()
    # (i) 3000 sweeps from 0 return Sigma*; (ii) equal to the dense solve
    np.testing.assert_allclose(s.get_sigma(), sig_star, rtol=0, atol=1e-12)
    np.testing.assert_allclose(s.get_sigma().ravel(), np.linalg.solve(A, b.ravel()), atol=1e-12)
    # one sweep from 0 is D^-1 b; a second sweep from x is x + D^-1 (b - A x)
    D = np.diag(A)
    np.testing.assert_allclose(first.ravel(), b.ravel() / D, rtol=1e-13)
    x = rng.uniform(-1, 1, rho.size)
    s.set_sigma(x.reshape(rho.shape))
    s.jacobi_sweep()
    np.testing.assert_allclose(s.get_sigma().ravel(), x + (b.ravel() - A @ x) / D, rtol=1e-12, atol=1e-14)


def test_p6_constant_mode_contraction_is_60_over_61():
    """rho = 1, alpha = 10 dx^2: a constant Sigma is multiplied by 60/61 per sweep (b = 0)."""
    n = 6
    s = make(n, n, n)
    one = np.ones((n, n, n))
    s.set_state(cons(one, 0 * one, 0 * one, 0 * one, one))
    s.fill_ghosts()
    s.source()
    s.set_sigma(one)
    s.jacobi_sweep()
    np.testing.assert_allclose(s.get_sigma(), 60.0 / 61.0, rtol=1e-15)


def test_p6_constant_rho_constant_b_gives_sigma_rho_b():
    """rho, b constant => the converged Sigma is rho*b (the divergence term vanishes).  b is made
    constant with the uniform dilatation field of P5 on the interior; checked through the fixed
    point: Sigma = rho*b is returned unchanged by a sweep where its neighbours are interior."""
    n, dx, alpha, sdil, rho0 = 10, 0.1, 0.05, 0.7, 1.7
    s = make(n, n, n, dx=dx, alpha=alpha, faces=(1,) * 6)
    c = (np.arange(n) + 0.5) * dx
    z, y, x = np.meshgrid(c, c, c, indexing="ij")
    rho = np.full_like(x, rho0)
    s.set_state(cons(rho, sdil * x, sdil * y, sdil * z, np.ones_like(x)))
    s.fill_ghosts()
    s.source()
    b0 = alpha * 12 * sdil ** 2
    s.set_sigma(np.full_like(x, rho0 * b0))
    s.jacobi_sweep()
    np.testing.assert_allclose(s.get_sigma()[2:-2, 2:-2, 2:-2], rho0 * b0, rtol=1e-12)


# ---------------------------------------------------------------------------------- P9
def _random_state(rng, n, smooth=True):
    c = (np.arange(n) + 0.5) / n
    z, y, x = np.meshgrid(c, c, c, indexing="ij")
    tw = 2 * np.pi
    rho = 1 + 0.3 * np.sin(tw * x) * np.cos(tw * y) + 0.2 * np.sin(tw * (z + 0.1))
    u = 0.5 * np.sin(tw * (x + 2 * y)) + 0.1
    v = 0.4 * np.cos(tw * (y - z)) - 0.2
    w = 0.3 * np.sin(tw * (z + x)) * np.cos(tw * y)
    p = 1 + 0.2 * np.cos(tw * (x + y + z))
    if not smooth:
        rho = rho + 0.05 * rng.uniform(-1, 1, rho.shape)
    return cons(rho, u, v, w, p)


def test_p9_scale_covariance_pins_sigma_over_rho_form():
    """Reading A1: with Sigma/rho - alpha div(grad Sigma/rho) = b every operation is homogeneous
    of degree 1 under (rho, m, E, Sigma) -> k (rho, m, E, Sigma); k = 4 makes it bitwise.  The
    rho*Sigma form of north_star's wording breaks this."""
    rng = np.random.default_rng(9)
    n = 8
    q = _random_state(rng, n, smooth=False)
    outs = []
    for k in (1.0, 4.0):
        s = make(n, n, n)
        s.set_state(k * q)
        lam = s.max_wavespeed()
        for _ in range(2):
            s.step(0.3 / n / 2.5)
        outs.append((s.get_state(), s.get_sigma(), lam))
    assert np.abs(outs[0][1]).max() > 1e-6            # Sigma is actually exercised
    assert outs[0][2] == outs[1][2]
    assert np.array_equal(4.0 * outs[0][0], outs[1][0])
    assert np.array_equal(4.0 * outs[0][1], outs[1][1])


# ---------------------------------------------------------------------------------- P12
def test_p12_axis_permutation_symmetry():
    rng = np.random.default_rng(12)
    n = 8
    q = _random_state(rng, n, smooth=False)
    dt = 0.3 / n / 2.5

    def run(q0):
        s = make(n, n, n)
        s.set_state(q0)
        for _ in range(2):
            s.step(dt)
        return s.get_state(), s.get_sigma()

    qa, sa = run(q)
    # swap the x and z axes: arrays are [c][z][y][x]; momentum components x<->z swap too
    qp = q[[0, 3, 2, 1, 4]].transpose(0, 3, 2, 1)
    qb, sb = run(qp)
    np.testing.assert_allclose(qb[[0, 3, 2, 1, 4]].transpose(0, 3, 2, 1), qa, rtol=1e-12, atol=1e-13)
    np.testing.assert_allclose(sb.transpose(2, 1, 0), sa, rtol=1e-10, atol=1e-14)
    # cyclic permutation x->y->z->x
    qc = q[[0, 3, 1, 2, 4]].transpose(0, 2, 3, 1)     # new[z'][y'][x'] = old[z=y'][y=x'][x=z']
    qd, _ = run(qc)
    np.testing.assert_allclose(qd[[0, 2, 3, 1, 4]].transpose(0, 3, 1, 2), qa, rtol=1e-12, atol=1e-13)


def test_p12_yz_uniform_input_stays_yz_uniform_bitwise():
    w = W.sod(64, 4, 4, noise=0.0)
    q = W.state(w).numpy().astype(np.float64)
    s = R.RefSolver(w.nx, w.ny, w.nz, w.dx, w.gamma, w.alpha, faces=w.faces)
    s.set_state(q)
    for _ in range(5):
        s.step(0.4 * w.dx / s.max_wavespeed())
    out = s.get_state()
    assert np.array_equal(out, np.broadcast_to(out[:, :1, :1, :], out.shape))
    assert np.all(out[2] == 0) and np.all(out[3] == 0)


# ---------------------------------------------------------------------------------- P13
def test_p13_periodic_run_equals_doubled_copy():
    rng = np.random.default_rng(13)
    n = 6
    q = _random_state(rng, n, smooth=False)
    dt = 0.3 / n / 2.5
    s1 = make(n, n, n, dx=1.0 / n)
    s1.set_state(q)
    s2 = make(2 * n, n, n, dx=1.0 / n)
    s2.set_state(np.concatenate([q, q], axis=3))
    for _ in range(3):
        s1.step(dt)
        s2.step(dt)
    a, b = s1.get_state(), s2.get_state()
    assert np.array_equal(b[..., :n], a) and np.array_equal(b[..., n:], a)


def test_p13_ghost_values_per_bc_type():
    n = 12
    patch = (6.0, 5.0, 3.0, 0.0, 0.5, 0.1, -0.2, 7.0, 2.0)  # (c0,c1,r,edge,rho,u,v,w,p), z- face
    faces = (0, 0, 1, 1, 2, 1)                          # x periodic, y extrap, z- inflow, z+ extrap
    s = R.RefSolver(n, n, n, 1.0, G, 10.0, faces=faces, patches={4: [patch]})
    rng = np.random.default_rng(131)
    q = _random_state(rng, n, smooth=False)
    s.set_state(q)
    s.fill_ghosts()
    for c in range(5):
        P = s.get_padded(c)
        I = P[3:-3, 3:-3, 3:-3]
        assert np.array_equal(I, q[c])
        # periodic x: ghost i=-1..-3 equals interior n-1..n-3
        assert np.array_equal(P[3:-3, 3:-3, 0:3], I[:, :, n - 3:n])
        assert np.array_equal(P[3:-3, 3:-3, n + 3:n + 6], I[:, :, 0:3])
        # extrapolation y: all ghost layers equal the nearest interior layer
        for g in range(3):
            assert np.array_equal(P[3:-3, g, 3:-3], I[:, 0, :])
            assert np.array_equal(P[3:-3, n + 3 + g, 3:-3], I[:, n - 1, :])
            assert np.array_equal(P[n + 3 + g, 3:-3, 3:-3], I[n - 1, :, :])
    # inflow z-: inside the circle the fixed state in ALL ghost layers, clamp outside
    jj, ii = np.meshgrid(np.arange(n), np.arange(n), indexing="ij")
    mask = (ii + 0.5 - patch[0]) ** 2 + (jj + 0.5 - patch[1]) ** 2 <= patch[2] ** 2
    lattice = sum(1 for j in range(n) for i in range(n)
                  if (2 * i + 1 - 12) ** 2 + (2 * j + 1 - 10) ** 2 <= 36)   # integer form x4
    assert mask.sum() == lattice and lattice > 0
    rho_j, u_j, v_j, w_j, p_j = patch[4:]
    fixed = [rho_j, rho_j * u_j, rho_j * v_j, rho_j * w_j,
             p_j / (G - 1) + 0.5 * rho_j * (u_j ** 2 + v_j ** 2 + w_j ** 2)]
    for c in range(5):
        P = s.get_padded(c)
        for g in range(3):
            layer = P[g, 3:-3, 3:-3]
            assert np.allclose(layer[mask], fixed[c], rtol=1e-15)
            assert np.array_equal(layer[~mask], q[c][0][~mask])
    # Sigma ghosts: wrap on periodic faces, clamp elsewhere -- also under inflow patches
    sig = rng.uniform(-1, 1, (n, n, n))
    s.set_sigma(sig)
    s.fill_sigma_ghosts()
    P = s.get_padded(5)
    assert np.array_equal(P[3:-3, 3:-3, 0:3], sig[:, :, n - 3:n])
    for g in range(3):
        assert np.array_equal(P[g, 3:-3, 3:-3], sig[0])
        assert np.array_equal(P[3:-3, n + 3 + g, 3:-3], sig[:, n - 1, :])


def test_storage_rounding_matches_numpy_half_and_bf16_definition():
    rng = np.random.default_rng(7)
    xs = np.concatenate([rng.normal(0, 1, 2000), rng.normal(0, 1e-6, 500), rng.normal(0, 3e4, 500),
                         [0.0, 65504.0, 65519.9, 65520.0, 1e-8, 6e-8, -2.5]])
    for x in xs:
        with np.errstate(over="ignore"):
            assert R.round_storage(x, R.STORE_F16) == float(np.float64(x).astype(np.float16))
        assert R.round_storage(x, R.STORE_F32) == float(np.float32(x))
        # bf16: 8 significant bits -> half an ulp <= 2^-8 relative, and idempotent
        y = R.round_storage(x, R.STORE_BF16)
        assert abs(y - x) <= abs(x) * 2.0 ** -8 + 1e-300
        assert R.round_storage(y, R.STORE_BF16) == y
        assert np.float32(y).view(np.uint32) & 0xFFFF == 0      # representable in bf16
    assert R.round_storage(1.0 + 2.0 ** -8, R.STORE_BF16) == 1.0             # tie -> even
    assert R.round_storage(1.0 + 3 * 2.0 ** -8, R.STORE_BF16) == 1.0 + 2.0 ** -6


def test_create_rejects_bad_arguments():
    with pytest.raises(ValueError):
        R.RefSolver(8, 8, 8, 0.1, G, 0.1, order=4)
    with pytest.raises(ValueError):
        R.RefSolver(8, 8, 8, 0.1, G, 0.1, faces=(0, 1, 0, 0, 0, 0))   # periodic on one side only
