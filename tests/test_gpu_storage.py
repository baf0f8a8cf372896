"""Reduced-precision storage (FP32 compute, FP16 storage): q and Sigma
stored as fp16 / bf16, arithmetic fp32, C ABI fp32.  Parity against (a) the storage-emulating oracle
(fp64 arithmetic, q rounded to the storage format after set_state and every RK stage, Sigma after every
solve) and (b) the pure fp64 oracle with the looser bounds of DESIGN.md section 7."""
import os

import numpy as np
import pytest
import torch

from oracle import igr_ref as R
from paper_2505_07392_b200 import igr
from paper_2505_07392_b200 import workloads as W
import parity

pytestmark = pytest.mark.gpu
FULL = os.environ.get("IGR_TEST_FULL", "1") != "0"

FMT = {
    "f16": dict(gpu=igr.STORE_F16, ref=R.STORE_F16, np=np.float16, pbits=11, l1=2e-3, mx=1e-2),
    "bf16": dict(gpu=igr.STORE_BF16, ref=R.STORE_BF16, np=None, pbits=8, l1=1.6e-2, mx=5e-2),
}


def ulp_of(x, pbits):
    """Spacing of the storage format at |x| (normal range)."""
    e = np.floor(np.log2(np.maximum(np.abs(x), 1e-30)))
    return 2.0 ** (e - (pbits - 1))


def compare_stored(got, emu, pbits, floor=1e-2):
    """Fraction of identical stored values, fraction within 1 ulp and the largest difference in ulps
    of the storage format; values below floor * max|field| are measured in ulps at that floor (a
    value near zero is the rounded result of a cancellation, its own ulp is not the error scale)."""
    got = np.asarray(got, np.float64)
    same = got == emu
    mag = np.maximum(np.maximum(np.abs(got), np.abs(emu)), floor * np.abs(emu).max())
    ulps = np.abs(got - emu) / ulp_of(mag, pbits)
    return same.mean(), (ulps <= 1.0 + 1e-6).mean(), ulps.max()


def run_three(w, fmt, mode, q0=None, steps=3):
    f = FMT[fmt]
    q0 = W.state(w).numpy() if q0 is None else q0
    g = igr.Solver.for_workload(w, storage=f["gpu"], **mode)
    emu = parity.oracle_for(w, storage=f["ref"])
    pure = parity.oracle_for(w)
    g.set_state(q0)
    emu.set_state(q0.astype(np.float64))
    pure.set_state(q0.astype(np.float64))
    for _ in range(steps):
        dt = w.cfl * w.dx / g.max_wavespeed()
        g.step(dt); emu.step(dt); pure.step(dt)
    return g, emu, pure


@pytest.mark.parametrize("mode", [dict(fused=1), dict(fused=0), dict(variant=igr.VARIANT_SIMPLE)],
                         ids=["tiled_fused", "tiled", "simple"])
@pytest.mark.parametrize("fmt", ["f16", "bf16"])
def test_set_get_roundtrip_is_the_storage_rounding(fmt, mode):
    w = W.taylor_green(16)
    q0 = W.state(w).numpy()
    g = igr.Solver.for_workload(w, storage=FMT[fmt]["gpu"], **mode)
    g.set_state(q0)
    got = g.get_state()
    want = np.vectorize(lambda x: R.round_storage(x, FMT[fmt]["ref"]))(q0.astype(np.float64))
    assert np.array_equal(got.astype(np.float64), want)


@pytest.mark.parametrize("mode", [dict(fused=1), dict(fused=0)], ids=["tiled_fused", "tiled"])
@pytest.mark.parametrize("fmt", ["f16", "bf16"])
@pytest.mark.parametrize("case", ["jets", "tgv", "tgv_m01"])
def test_three_steps_vs_emulating_and_pure_oracle(case, fmt, mode):
    f = FMT[fmt]
    if case == "jets":
        w = W.jets33(n=64, radius=6, rings=((10, 3),))
    else:
        w = W.taylor_green(48)
        # "tgv": Mach 0.5, p0 ~ 2.9, well inside the resolution of the 2-byte formats.  "tgv_m01": config 3's own
        # Mach 0.1 (p0 ~ 71, E ~ 178): one ulp of fp16 at E is 0.125, more than the whole pressure variation of the
        # vortex -- the stored field barely moves (PAPER.md L351 sees the same effect), but GPU and the
        # storage-emulating oracle must still round alike
        if case == "tgv":
            w.params["mach"] = 0.5
    g, emu, pure = run_three(w, fmt, mode)
    got = g.get_state()
    # (a) storage-emulating oracle: the stored values agree except for rare 1-ulp rounding flips
    same, within1, worst = compare_stored(got, emu.get_state(), f["pbits"])
    same_s, within1_s, worst_s = compare_stored(g.get_sigma(), emu.get_sigma(), f["pbits"])
    print("stored q: identical %.4f within-1-ulp %.5f worst %.1f ulp; Sigma: %.4f %.5f %.1f"
          % (same, within1, worst, same_s, within1_s, worst_s))
    # a flipped rounding (fp32 vs fp64 arithmetic before the store) is 1 ulp; it can grow by a few
    # ulps through the following stages, never more.  Bounds as in DESIGN.md section 7; measured on the B200
    # (profiles/r02_storage_fractions.txt): identical 0.975-0.995, within 1 ulp >= 0.9998, worst 4.0 ulp.  At
    # Mach 0.1 the increments dt r are a fraction of an ulp of fp16, so many stores sit near a rounding tie:
    # identical 0.909 (f16) / 0.970 (bf16), but every value within 1 ulp (worst 0.5)
    min_same = 0.90 if case == "tgv_m01" else 0.97
    assert same >= min_same and within1 >= 0.999 and worst <= 8.0, (same, within1, worst)
    assert within1_s >= 0.99 and worst_s <= 16.0, (same_s, within1_s, worst_s)
    # (b) pure fp64 oracle: looser bounds from 9 stores x half an ulp.  At Mach 0.1 the increments dt r are smaller
    # than half an ulp of the stored momentum and energy: they are not rounded at random, they vanish (the effect the
    # paper reports for FP16 storage, L351), so the distance to the pure oracle is ~3 times the random-walk bound
    # (measured: L1-rel 5.6e-3 in fp16, 2.1e-2 in bf16)
    mx, l1 = parity.worst(got, pure.get_state())
    slack = 3.0 if case == "tgv_m01" else 1.0
    assert l1 <= slack * f["l1"] and mx <= slack * f["mx"], (mx, l1)


@pytest.mark.skipif(not FULL, reason="full-size configs disabled")
@pytest.mark.parametrize("fmt", ["f16", "bf16"])
def test_config5_jets33_1024_subbox_reduced_storage(fmt):
    """Config 5 in reduced-precision storage: full 1024^3 on the GPU in the launch configuration
    bench.py times, first 3 steps compared on the 64^3 sub-region through the dependency-cone sub-box."""
    f = FMT[fmt]
    w = W.jets33()
    target, size, pad, steps = (496, 480, 0), 64, 80, 3
    full = (w.nx, w.ny, w.nz)
    lo = tuple(max(0, target[a] - pad) for a in range(3))
    hi = tuple(min(full[a], target[a] + size + pad) for a in range(3))
    wb = W.subbox(w, lo, hi)
    g = igr.Solver.for_workload(w, storage=f["gpu"], fused=1)
    q0 = W.state(w, device="cuda")
    g.set_state(q0)
    qb = q0[:, lo[2]:hi[2], lo[1]:hi[1], lo[0]:hi[0]].contiguous().cpu().numpy()
    del q0
    emu = parity.oracle_for(wb, storage=f["ref"])
    pure = parity.oracle_for(wb)
    emu.set_state(qb.astype(np.float64)); pure.set_state(qb.astype(np.float64))
    for _ in range(steps):
        dt = w.cfl * w.dx / g.max_wavespeed()
        g.step(dt); emu.step(dt); pure.step(dt)
    out = torch.empty((5, w.nz, w.ny, w.nx), dtype=torch.float32, device="cuda")
    g.get_state(out)
    assert torch.isfinite(out).all()
    sl = tuple(slice(target[a], target[a] + size) for a in (2, 1, 0))
    got = out[(slice(None),) + sl].cpu().numpy()
    del out
    rl = tuple(slice(target[a] - lo[a], target[a] - lo[a] + size) for a in (2, 1, 0))
    same, within1, worst = compare_stored(got, emu.get_state()[(slice(None),) + rl], f["pbits"])
    assert same >= 0.97 and within1 >= 0.999 and worst <= 8.0, (same, within1, worst)
    mx, l1 = parity.worst(got, pure.get_state()[(slice(None),) + rl])
    assert l1 <= f["l1"] and mx <= f["mx"], (mx, l1)
