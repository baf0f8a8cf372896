"""Helpers shared by the GPU parity tests: error norms of DESIGN.md reading A15 and the dt-replay
protocol of reading A16 (the GPU's wave speed chooses dt; the oracle replays the same dt values)."""
import numpy as np
import torch

from oracle import igr_ref as R
from paper_2505_07392_b200 import workloads as W


def norms(got, ref):
    """Per-field (max-rel, L1-rel); the three momentum components share one denominator."""
    got = np.asarray(got, dtype=np.float64)
    ref = np.asarray(ref, dtype=np.float64)
    if ref.shape[0] == 5:
        groups = [[0], [1, 2, 3], [4]]
    elif ref.shape[0] == 7:                       # two fluids: (a1 rho1, a2 rho2, m, E, a1)
        groups = [[0], [1], [2, 3, 4], [5], [6]]
    else:
        groups = [[c] for c in range(ref.shape[0])]
    out = {}
    for grp in groups:
        d = np.abs(got[grp] - ref[grp])
        out[tuple(grp)] = (d.max() / np.abs(ref[grp]).max(), d.sum() / np.abs(ref[grp]).sum())
    return out


def worst(got, ref):
    n = norms(got, ref)
    return max(v[0] for v in n.values()), max(v[1] for v in n.values())


def scalar_norms(got, ref, floor=0.0):
    got = np.asarray(got, dtype=np.float64)
    ref = np.asarray(ref, dtype=np.float64)
    d = np.abs(got - ref)
    return d.max() / max(np.abs(ref).max(), floor), d.sum() / max(np.abs(ref).sum(), floor * ref.size)


def oracle_for(w, storage=R.STORE_F64):
    if getattr(w, "gamma2", 0.0):                 # two fluids (igr_ref2.c): patches (.., a1 rho1, a2 rho2, a1, u, v, w, p)
        patches = {f: [tuple(p[:4]) + (p[9] * p[4], (1.0 - p[9]) * p[10], p[9]) + tuple(p[5:9]) for p in pl]
                   for f, pl in w.patches.items()}
        return R.RefSolver2(w.nx, w.ny, w.nz, w.dx, w.gamma, w.gamma2, w.alpha, order=w.order, n_jacobi=w.n_jacobi,
                            faces=w.faces, patches=patches)
    return R.RefSolver(w.nx, w.ny, w.nz, w.dx, w.gamma, w.alpha, order=w.order, n_jacobi=w.n_jacobi,
                       faces=w.faces, patches=w.patches, storage=storage)


def run_pair(w, gpu, n_steps=None, t_end=None, q0=None, check_wave=True):
    """Advance the GPU solver and the oracle together from the same fp32 initial state.  Returns
    (q_gpu, q_oracle, sigma_gpu, sigma_oracle, dts)."""
    q0 = W.state(w).numpy() if q0 is None else q0           # fp32 array handed to BOTH sides
    ref = oracle_for(w)
    ref.set_state(q0.astype(np.float64))
    gpu.set_state(q0)
    dts, t = [], 0.0
    while True:
        if n_steps is not None and len(dts) >= n_steps:
            break
        if t_end is not None and t >= t_end - 1e-14:
            break
        lam = gpu.max_wavespeed()
        if check_wave:
            lam_ref = ref.max_wavespeed()
            assert abs(lam - lam_ref) <= 1e-5 * lam_ref + 1e-6, (lam, lam_ref)
        dt = w.cfl * w.dx / lam
        if t_end is not None:
            dt = min(dt, t_end - t)
        gpu.step(dt)
        ref.step(dt)
        dts.append(dt)
        t += dt
    return gpu.get_state(), ref.get_state(), gpu.get_sigma(), ref.get_sigma(), dts
