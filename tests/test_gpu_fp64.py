"""GPU parity of the fp64 mode (IGR_STORE_F64): fp64 storage and arithmetic against the fp64 oracle
on the same inputs, dt replayed (reading A16).  Both sides evaluate the same formulas in fp64; they differ only in
the order of a few sums and in fused multiply-adds, so the tolerance is 1e-12 relative to the largest value of
each field group (a few hundred ulps after several steps)."""
import dataclasses

import numpy as np
import pytest
import torch

from paper_2505_07392_b200 import igr
from paper_2505_07392_b200 import workloads as W
import parity

pytestmark = pytest.mark.gpu


def run_pair64(w, n_steps):
    q0 = W.state(w, dtype=torch.float64).numpy()
    g = igr.Solver.for_workload(w, storage=igr.STORE_F64)
    ref = parity.oracle_for(w)
    g.set_state(q0); ref.set_state(q0)
    for _ in range(n_steps):
        lam = g.max_wavespeed()
        assert abs(lam - ref.max_wavespeed()) <= 1e-13 * lam
        dt = w.cfl * w.dx / lam
        g.step(dt); ref.step(dt)
    return g, ref


@pytest.mark.parametrize("case", ["entropy_wave", "taylor_green", "sod", "jets"])
def test_fp64_mode_matches_the_oracle_to_1e_12(case):
    w = {"entropy_wave": lambda: W.entropy_wave(24),
         "taylor_green": lambda: W.taylor_green(24),
         "sod": lambda: W.sod(96, 6, 5),
         "jets": lambda: dataclasses.replace(W.jets9(n=37, radius=4, pitch=11), ny=20, nz=13, global_shape=None)}[case]()
    g, ref = run_pair64(w, 5)
    mx, l1 = parity.worst(g.get_state_f64(), ref.get_state())
    assert mx <= 1e-12, (mx, l1)
    sr = ref.get_sigma()
    assert np.abs(g.get_sigma_f64() - sr).max() <= 1e-12 * max(np.abs(sr).max(), 1e-6)
    # the fp32 calls convert at the boundary
    assert np.array_equal(g.get_state(), g.get_state_f64().astype(np.float32))


def test_fp64_uniform_state_is_preserved_bitwise():
    w = W.uniform(20, 12, 9, 0.1, 0.9, 0.3, -0.7, 1.1, 1.3)
    q0 = W.state(w, dtype=torch.float64).numpy()
    g = igr.Solver.for_workload(w, storage=igr.STORE_F64)
    g.set_state(q0)
    for _ in range(3):
        g.step(0.5 * w.dx / g.max_wavespeed())
    assert np.array_equal(g.get_state_f64(), q0) and np.all(g.get_sigma_f64() == 0.0)


def test_fp64_arrays_are_refused_by_the_other_storage_types():
    w = W.entropy_wave(16)
    g = igr.Solver.for_workload(w)
    with pytest.raises(igr.IgrError) as ei:
        g.set_state(W.state(w, dtype=torch.float64).numpy())
    assert ei.value.code == igr.ERR_ARG
