#!/usr/bin/env python
"""bench.py -- grind time of one SSP-RK3 step of the 3D IGR Euler hot path on B200.

    python bench.py --gpus N --steps K --warmup W [--impl reference] [--workload jets33_1024]
                    [--storage f32|f16|bf16] [--fused 0|1]

A "step" is one pass of the whole hot path (halo/BC, source, Jacobi, RHS, RK update, x3 stages) over
the synthetic many-jet workload (config 5 of BASELINE.json at N=1).  Prints ONE JSON line.
metric = grind time ns/(cell*eqn*RHS) = t_step / (cells * 5 * 3); lower is better.
Multi-GPU (--gpus N under torchrun, one rank per GPU): weak scaling by z slabs: the
job is the workload stacked N times along z, every rank owns one copy's planes plus n_jacobi + 3 overlap planes per
neighbour and pulls its halo planes from the neighbours after every RK stage (CUDA IPC peer copies, or
torch.distributed send/recv); value = time / (total OWNED cells * equations * 3), time = max over ranks.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "grind time ns/(cell*eqn*RHS), 3D IGR Euler SSP-RK3 step"
UNIT = "ns/(cell*eqn*RHS)"


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="jets33_1024")
    ap.add_argument("--storage", default="f32", choices=["f32", "f16", "bf16", "f64"],
                    help="f16 / bf16: reduced-precision storage, fp32 arithmetic (L264); f64: fp64 storage AND arithmetic "
                         "(NEXT-4: one thread per cell, for the paper's FP64 column)")
    ap.add_argument("--fused", type=int, default=1)
    ap.add_argument("--e2e-steps", type=int, default=2)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--row-power", type=float, default=0.0, metavar="SECONDS",
                    help="N = 1: also loop every main row alone for SECONDS and report its time, board power and SM "
                         "clock (`row_power`): which kernel runs into the power limit")
    ap.add_argument("--exchange", default="ipc", choices=["ipc", "sendrecv"],
                    help="N > 1: halo planes by CUDA IPC peer copies (falls back to sendrecv if IPC is refused) "
                         "or by torch.distributed send/recv")
    ap.add_argument("--backend", default="nccl", choices=["nccl", "gloo"], help="N > 1: rendezvous backend")
    ap.add_argument("--one-gpu", action="store_true",
                    help="N > 1: every rank on cuda:0 (functional check of the exchange path on a 1-GPU box; "
                         "use with --backend gloo; the timing is meaningless)")
    ap.add_argument("--wavespeed-every", type=int, default=1,
                    help="query igr_max_wavespeed (CFL) every N steps and reuse dt in between (SURVEY 8(d) times both "
                         "1 and 10; the fused stage-3 reduction makes the query a 8-byte read)")
    ap.add_argument("--mu", type=float, default=0.0, help="shear viscosity (NEXT-1; 0 = Euler, the headline)")
    ap.add_argument("--zeta", type=float, default=0.0, help="bulk viscosity")
    return ap.parse_args()


def make_workload(name):
    from paper_2505_07392_b200 import workloads as W
    kind, n = name.rsplit("_", 1)
    n = int(n)
    if kind in ("jets2f33", "jets2f9"):          # two-fluid variant (NEXT-3): the same jets, 7 equations
        return W.two_fluid(make_workload(kind.replace("2f", "") + "_%d" % n))
    if kind == "jets33":
        scale = n / 1024.0
        if n >= 1024:
            return W.jets33(n=n)
        rings = tuple((max(2, round(R * scale * 2)), c) for R, c in ((14, 3), (44, 10), (84, 20)))
        return W.jets33(n=n, radius=max(4, round(8 * max(scale * 2, 0.5))), rings=rings)
    if kind == "jets9":
        return W.jets9(n=n) if n >= 512 else W.jets9(n=n, radius=max(4, n // 50), pitch=max(16, n // 8))
    if kind == "taylor_green":
        return W.taylor_green(n)
    raise SystemExit("unknown workload " + name)


class ClockSampler(threading.Thread):
    """nvidia-smi clocks and throttle reasons DURING the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap,power.limit")

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.rows, self.proc = index, [], None

    def run(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            for line in self.proc.stdout:
                self.rows.append([x.strip() for x in line.split(",")])
        except Exception:
            pass

    def stop(self):
        if self.proc:
            self.proc.terminate()
        self.join(timeout=2)
        sm = sorted(int(float(r[0])) for r in self.rows if r and r[0].replace(".", "").isdigit())
        mx = [int(float(r[1])) for r in self.rows if len(r) > 1 and r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for i, n in enumerate(names) if any(len(r) > 3 + i and r[3 + i] == "Active" for r in self.rows)]
        def num(x):
            try:
                return float(x)
            except ValueError:
                return None
        pw = sorted(v for v in (num(r[2]) for r in self.rows if len(r) > 2) if v is not None)
        lim = [v for v in (num(r[7]) for r in self.rows if len(r) > 7) if v is not None]
        # (power: the fp32 step sits at the board's limit, which is what pulls the SM clock below its maximum)
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": reasons, "samples": len(sm), "power_w": pw[len(pw) // 2] if pw else None,
                "power_limit_w": max(lim) if lim else None}


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def cpu_baseline(w, n_box=96, steps=2):
    """The oracle, as it stands, on a bounded sample of the same workload: an n_box^3 sub-box on the
    inflow plane around the first jet, `steps` steps, all host cores (OpenMP)."""
    import numpy as np
    from paper_2505_07392_b200 import workloads as W
    cores = len(os.sched_getaffinity(0))
    os.environ.setdefault("OMP_NUM_THREADS", str(cores))
    from oracle import igr_ref as R
    if w.kind == "jets":
        cx, cy, _ = w.params["jet_centers"][0]
        lo = [int(max(0, min(w.nx - n_box, cx - n_box // 2))), int(max(0, min(w.ny - n_box, cy - n_box // 2))), 0]
        nb = min(n_box, w.nx)
        wb = W.subbox(w, tuple(lo), (lo[0] + nb, lo[1] + nb, nb))
    else:
        wb = type(w)(**{**w.__dict__, "nx": min(n_box, w.nx), "ny": min(n_box, w.ny), "nz": min(n_box, w.nz)})
    q = W.state(wb).numpy().astype(np.float64)
    if wb.gamma2:        # two fluids: oracle/igr_ref2.c, patches (c0, c1, radius, edge, a1 rho1, a2 rho2, a1, u, v, w, p)
        pt = {f: [tuple(p[:4]) + (p[9] * p[4], (1.0 - p[9]) * p[10], p[9]) + tuple(p[5:9]) for p in pl]
              for f, pl in wb.patches.items()}
        s = R.RefSolver2(wb.nx, wb.ny, wb.nz, wb.dx, wb.gamma, wb.gamma2, wb.alpha, order=wb.order,
                         n_jacobi=wb.n_jacobi, faces=wb.faces, patches=pt)
    else:
        s = R.RefSolver(wb.nx, wb.ny, wb.nz, wb.dx, wb.gamma, wb.alpha, order=wb.order, n_jacobi=wb.n_jacobi,
                        faces=wb.faces, patches=wb.patches)
    s.set_state(q)
    dt = wb.cfl * wb.dx / s.max_wavespeed()
    s.step(dt)                                   # untimed first touch
    t0 = time.perf_counter()
    for _ in range(steps):
        s.step(wb.cfl * wb.dx / s.max_wavespeed())
    dt_wall = time.perf_counter() - t0
    cells = wb.nx * wb.ny * wb.nz
    return {"value": dt_wall / steps / (cells * wb.nf * 3) * 1e9, "unit": UNIT, "cores": int(os.environ["OMP_NUM_THREADS"]),
            "kind": "oracle", "sample": "%dx%dx%d sub-box of %s on the inflow plane, %d steps, fp64, OpenMP"
            % (wb.nx, wb.ny, wb.nz, w.name, steps), "ms_per_step": dt_wall / steps * 1e3}


def alg_bytes(row, storage, fused=1, nf=5):
    """Algorithmic HBM bytes per cell per launch, averaged over the three stages:
    q and Sigma in the storage type (s bytes), b and r in fp32.  source: 4 q reads + b write; jacobi
    (5 sweeps blocked): rho + b + Sigma in + Sigma out; rhs: 5 q + Sigma reads, then either 5 r writes
    (unfused) or the fused update: q_n reads in stages 2, 3 and 5 q writes; rk_update (unfused only)."""
    if storage == "f64":    # fp64 mode: every field 8 bytes, one launch per Jacobi sweep, unfused update
        return {"sigma_source": 4 * 8 + 8, "jacobi": 5 * 4 * 8, "rhs": 6 * 8 + 5 * 8,
                "rk_update": (5 * 24 + 2 * 5 * 32) / 3.0}[row]
    s = 4 if storage == "f32" else 2
    if nf == 7:         # two fluids, fp32, fused: source reads 5 fields and writes b and the mixture density (which
        #                 is then read with its ghosts); jacobi reads that density; rhs moves 7 fields and Sigma
        return {"sigma_source": 5 * 4 + 4 + 2 * 4, "jacobi": 16, "rhs": 8 * 4 + 7 * 4 + 2 * 7 * 4 / 3.0,
                "rk_update": 0.0}[row]
    rhs = 6 * s + (5 * s + 2 * 5 * s / 3.0 if fused else 20)
    return {"sigma_source": 4 * s + 4, "jacobi": 3 * s + 4, "rhs": rhs,
            "rk_update": (5 * (s + 4 + s) + 2 * 5 * (2 * s + 4 + s)) / 3.0}[row]


# Algorithmic fp32 operations per cell per launch (FMA = 2), counted on the oracle's formulas
# (DESIGN.md section 5): rhs = 3 faces x (reconstruction 108 + two side fluxes 48 + LF 25 + lambda 2)
# + cell wave speeds 15 + divergence 30 + RK stage 20; jacobi = 5 sweeps x 14 + coefficients 20;
# source = 9 differences + velocities + traces.
ALG_FLOP = {"sigma_source": 45.0, "jacobi": 90.0, "rhs": 614.0, "rk_update": 20.0}
TRAFFIC_CSV = os.path.join(ROOT, "profiles", "dram_traffic.csv")


def ncu_traffic(workload, storage, row):
    """DRAM bytes per launch of `row` (dram__bytes_read.sum + dram__bytes_write.sum of one `ncu --set full`
    capture, profiles/dram_traffic.md), averaged over the launches of one step that were captured -- or None
    if profiles/dram_traffic.csv holds no capture of exactly this workload and storage type.  Nothing is
    scaled from another size."""
    import csv
    if not os.path.exists(TRAFFIC_CSV):
        return None, None
    vals = []
    with open(TRAFFIC_CSV) as f:
        for r in csv.DictReader(line for line in f if not line.startswith("#")):
            if r["workload"] == workload and r["storage"] == storage and r["row"] == row:
                vals.append((float(r["dram_read_bytes"]) + float(r["dram_write_bytes"]), r["stage"]))
    if not vals:
        return None, None
    return sum(v for v, _ in vals) / len(vals), "+".join(st for _, st in vals)


def alu_peak_tflops():
    """Plain FP32 ALU peak of a B200: 148 SMs x 128 lanes x 2 flop (FMA) x SM clock."""
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    mhz = float(json.load(open(p)).get("sm_max_mhz", 1965.0)) if os.path.exists(p) else 1965.0
    return 148 * 128 * 2 * mhz * 1e6 / 1e12


def reduce_max(value, world, device="cpu"):
    """Max over ranks of a host scalar (multi-GPU timing rule: the slowest rank counts)."""
    if world <= 1:
        return float(value)
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(value)], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_numbers(ms_step, cells_per_rank, world, neq=5):
    """Whole-job metric of `world` ranks that each advance `cells_per_rank` owned cells in ms_step (max
    over ranks): grind time per (cell*eqn*RHS) of the job (neq equations, 3 RHS evaluations per step) and
    aggregate cell updates per second."""
    total = cells_per_rank * world
    return {"grind_ns": ms_step * 1e6 / (total * neq * 3), "cell_updates_per_s": total / (ms_step * 1e-3)}


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2505_07392_b200 import igr, workloads as W
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if args.one_gpu:
        local = 0
    torch.cuda.set_device(local)
    dev = "cuda:%d" % local
    if world > 1:
        if args.backend == "nccl":
            dist.init_process_group("nccl", device_id=torch.device(dev))
        else:
            dist.init_process_group("gloo")
    rdev = dev if args.backend == "nccl" else "cpu"      # where the scalar reductions live
    w = make_workload(args.workload)
    storage = {"f32": igr.STORE_F32, "f16": igr.STORE_F16, "bf16": igr.STORE_BF16, "f64": igr.STORE_F64}[args.storage]
    if args.storage == "f64":
        args.fused = 0                    # the fp64 mode runs one kernel per row
    cells = w.n_cells                     # cells OWNED per rank (weak scaling: the job has world x cells)
    ss = None
    if world > 1:
        # z-slab decomposition: the job is the workload stacked `world` times along z,
        # every rank owns w.nz planes and computes n_jacobi + 3 overlap planes per neighbour on top of them
        import dataclasses
        from paper_2505_07392_b200 import dist as D, slab as S
        wg = dataclasses.replace(w, name="%s_x%dz" % (w.name, world), nz=w.nz * world)
        ss = D.SlabSolver(wg, exchange=args.exchange, device=dev, storage=storage, fused=args.fused)
        g = ss.solver
        q0 = S.local_state(wg, ss.slab, device=dev)
    else:
        g = igr.Solver.for_workload(w, storage=storage, fused=args.fused, device=dev)
        # the fp32 copy of the initial state stays on the device for restarts only if it fits beside the solver
        free_b = torch.cuda.mem_get_info(torch.device(dev))[0]
        q0 = W.state(w, device=dev) if free_b > w.nf * cells * 4 + (12 << 30) else None
    if args.mu > 0 or args.zeta > 0:
        g.set_viscosity(args.mu, args.zeta)
    filled = [False]

    def load_initial():
        if q0 is not None:
            g.set_state(q0)
        else:                             # slab by slab through igr_set_state_planes (large grids)
            nk = max(1, (1 << 24) // (w.nx * w.ny))
            for k0 in range(0, w.nz, nk):
                g.set_state_planes(k0, W.state_planes(w, k0, min(nk, w.nz - k0), device=dev))
            if filled[0]:                 # restart: Sigma back to zero (a fresh solver has it zero already)
                g.set_sigma(torch.zeros((w.nz, w.ny, w.nx), dtype=torch.float32, device=dev))
            filled[0] = True
        if ss:
            ss.exchange()                 # ghost planes from the neighbours

    load_initial()
    g.sync()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    resets = [0]
    resets_timed = [0]                    # restarts that fell between the two timing events
    solver = ss if ss else g              # max_wavespeed (max over ranks) and step (+ exchange per stage)

    dt_cache = [None, 0]                  # dt in use, steps since it was computed

    def one_step():
        if dt_cache[0] is not None and dt_cache[1] < args.wavespeed_every:
            dt_cache[1] += 1
            solver.step(dt_cache[0])
            return
        # The purely linear scheme eventually loses positivity on the under-resolved jets (F1:
        # config 5 after ~137 steps).  The library reports it (IGR_ERR_NONFINITE, on every rank after the
        # max-reduction); a long benchmark then restarts from the device-resident initial state and says so
        # in the JSON line ("resets").
        try:
            lam = solver.max_wavespeed()
        except igr.IgrError as e:
            if e.code != igr.ERR_NONFINITE:
                raise
            load_initial()
            resets[0] += 1
            lam = solver.max_wavespeed()
        dt_cache[0], dt_cache[1] = w.cfl * w.dx / lam, 1
        solver.step(dt_cache[0])

    for _ in range(max(args.warmup, 3)):
        one_step()
    sampler = ClockSampler(local)
    sampler.start()
    barrier()
    l0 = g.kernel_launches()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(g.stream)
    r_before = resets[0]
    for _ in range(args.steps):
        one_step()
    e1.record(g.stream)
    resets_timed[0] = resets[0] - r_before
    barrier()
    ms = e0.elapsed_time(e1)
    launches = g.kernel_launches() - l0
    clocks = sampler.stop()
    ms = reduce_max(ms, world, rdev)
    ms_step = ms / args.steps
    job = job_numbers(ms_step, cells, world, w.nf)
    grind = job["grind_ns"]

    # per-row CUDA-event timing on the solver's stream (separate region, same state)
    nprof = max(1, min(args.steps, 5))
    g.profile(True)
    t_ex = [0.0]
    if ss:                                # host time of the exchanges (syncs, barriers, peer copies)
        inner = ss.exchange

        def timed_exchange():
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            inner()
            t_ex[0] += time.perf_counter() - t0
        ss.exchange = timed_exchange
    for _ in range(nprof):
        one_step()
    if ss:
        ss.exchange = inner
    rows = g.profile_read()
    g.profile(False)
    row_ms = {r: (v[0] / v[1] if v[1] else 0.0) for r, v in rows.items()}
    step_ms_prof = sum(v[0] for v in rows.values()) / nprof
    dom = max(("sigma_source", "jacobi", "rhs", "rk_update"), key=lambda r: rows[r][0])
    peak, peak_src = measured_peaks()
    main_rows = [r for r in ("sigma_source", "jacobi", "rhs", "rk_update") if row_ms[r] > 0]
    hbm_gbs = {r: alg_bytes(r, args.storage, args.fused, w.nf) * cells / (row_ms[r] * 1e-3) / 1e9 for r in main_rows}
    alu_tf = {r: ALG_FLOP[r] * cells / (row_ms[r] * 1e-3) / 1e12 for r in main_rows}
    alu_peak = alu_peak_tflops()
    # the dominant kernel is reported against the roofline that binds it: the larger of the two fractions
    if alu_tf[dom] / alu_peak > hbm_gbs[dom] / peak:
        roofline = {"bound": "alu", "kernel": dom, "achieved": alu_tf[dom], "peak": alu_peak, "unit": "TFLOP/s",
                    "frac": alu_tf[dom] / alu_peak,
                    "peak_source": "148 SM x 128 fp32 lanes x 2 x sm_max_mhz (DESIGN.md section 5)",
                    "alg_flop_per_cell": ALG_FLOP[dom]}
    else:
        roofline = {"bound": "hbm", "kernel": dom, "achieved": hbm_gbs[dom], "peak": peak, "unit": "GB/s",
                    "frac": hbm_gbs[dom] / peak, "peak_source": peak_src}
    traffic, traffic_stages = (None, None) if ss else ncu_traffic(w.name, args.storage, dom)
    roofline.update({
        "traffic": traffic,
        "traffic_unit": ("bytes per launch, mean of the captured stages %s (ncu --set full, profiles/dram_traffic.csv)"
                         % traffic_stages) if traffic else "no ncu capture of this workload / storage in profiles/",
        "alg_bytes_per_cell": alg_bytes(dom, args.storage, args.fused, w.nf),
        "hbm": {"achieved_gbs": hbm_gbs[dom], "peak_gbs": peak, "frac": hbm_gbs[dom] / peak, "peak_source": peak_src,
                "frac_of_nominal_8tbs": hbm_gbs[dom] / 8000.0},
        "avg_launch_ms": row_ms[dom], "share_of_step": rows[dom][0] / nprof / step_ms_prof,
        "rows_ms_per_call": row_ms,
        "rows_hbm_frac": {r: hbm_gbs[r] / peak for r in main_rows},
        "rows_alu_frac": {r: alu_tf[r] / alu_peak for r in main_rows},
        "step_hbm_frac": sum(3 * alg_bytes(r, args.storage, args.fused, w.nf) for r in main_rows) * cells
        / (ms_step * 1e-3) / 1e9 / peak})

    # end to end through the C ABI with HOST buffers: set_state (H2D) + wave speed + step + get_state (D2H)
    e2e = None
    if args.e2e_steps > 0:
        lw = ss.slab.local if ss else w      # the arrays the rank's C-ABI calls move (extended slab)
        try:
            host = torch.empty((w.nf, lw.nz, lw.ny, lw.nx), dtype=torch.float32, pin_memory=True)
            pinned = True
        except RuntimeError:
            host = torch.empty((w.nf, lw.nz, lw.ny, lw.nx), dtype=torch.float32)
            pinned = False
        load_initial()                           # a fresh state: the e2e steps never meet a reset
        g.get_state(host)
        barrier()
        t0 = time.perf_counter()
        for _ in range(args.e2e_steps):
            g.set_state(host)
            if ss:
                ss.exchange()
            solver.step(w.cfl * w.dx / solver.max_wavespeed())
            g.get_state(host)
        barrier()
        t_e2e = (time.perf_counter() - t0) / args.e2e_steps
        t_e2e = reduce_max(t_e2e, world, rdev)
        nbytes = w.nf * lw.n_cells * 4
        e2e = {"value": job_numbers(t_e2e * 1e3, cells, world, w.nf)["grind_ns"], "unit": UNIT, "h2d_bytes_per_step": nbytes,
               "d2h_bytes_per_step": nbytes + 8, "ms_per_step": t_e2e * 1e3, "pinned_host": pinned}

    row_power = None
    if args.row_power > 0 and world == 1 and not ss:
        row_power = {}
        load_initial()
        g.halo_bc()
        for name, fn in (("sigma_source", g.sigma_source), ("jacobi", g.jacobi), ("rhs", g.rhs), ("step", one_step)):
            if name == "rhs" and w.nf != 5:
                continue                                   # (the unfused RHS exists for one fluid only)
            for _ in range(3):
                fn()
            g.sync()
            smp = ClockSampler(local)
            smp.start()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            t0, n = time.perf_counter(), 0
            e0.record(g.stream)
            while time.perf_counter() - t0 < args.row_power:
                for _ in range(5):
                    fn()
                g.sync()
                n += 5
            e1.record(g.stream)
            g.sync()
            c = smp.stop()
            row_power[name] = {"ms_per_call": e0.elapsed_time(e1) / n, "power_w": c["power_w"], "sm_mhz": c["sm_mhz"],
                               "reasons": c["reasons"]}
        row_power["note"] = ("each row looped alone; rhs = the unfused kernel (writes r, no q_n read); power_limit_w in "
                             "`clocks`")

    out = {"metric": METRIC, "value": grind, "unit": UNIT, "n_gpus": world, "steps": args.steps,
           "warmup": max(args.warmup, 3), "ms_per_step": ms_step, "higher_is_better": False,
           "scaling": "weak", "vs_baseline": None, "dtype": "f64" if args.storage == "f64" else "f32",
           "storage_dtype": args.storage, "data": "synthetic",
           "config": {"workload": w.name, "grid": [w.nx, w.ny, w.nz], "cells_per_gpu": cells,
                      "equations": w.nf, "storage": args.storage, "fused": args.fused, "mu": args.mu, "zeta": args.zeta, "n_jacobi": w.n_jacobi, "order": w.order,
                      "cfl": w.cfl,
                      "parallelism": ("z slabs: %d ranks x %d owned planes + %d overlap planes per neighbour, one halo "
                                      "exchange per RK stage (%s)" % (world, w.nz, ss.slab.overlap, ss.exchange_kind))
                      if ss else "single GPU",
                      "exchange_ms_per_step": (t_ex[0] * 1e3 / nprof) if ss else 0.0,
                      "l2": "inputs larger than L2 (no flush needed)" if cells * 4 > (126 << 20) else "inputs fit L2",
                      "wavespeed_query_every_step": args.wavespeed_every == 1, "wavespeed_every": args.wavespeed_every,
                      "resets": resets[0]},
           "cell_updates_per_s": job["cell_updates_per_s"],
           "clocks": clocks, "e2e": e2e, "gpu_launches": launches, "roofline": roofline}
    if row_power:
        out["row_power"] = row_power
    if resets_timed[0]:
        # the state was reloaded inside the timed region (positivity lost, F1): the line is flagged
        out["invalid"] = "%d restart(s) from the initial state inside the timed region" % resets_timed[0]
        print("bench.py: WARNING: " + out["invalid"], file=sys.stderr)
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        out["cpu_baseline"] = cpu_baseline(w)
    if rank == 0:
        print(json.dumps(out))
    if world > 1:
        barrier()
        ss.close()
        dist.destroy_process_group()


def run_reference(args):
    """The oracle as it stands on the host cores, on a bounded sample of the same workload."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    w = make_workload(args.workload)
    steps = max(1, min(args.steps, 3))
    cb = cpu_baseline(w, n_box=96, steps=steps)
    out = {"impl": "reference", "metric": METRIC, "value": cb["value"], "unit": UNIT,
           "n_gpus": int(os.environ.get("WORLD_SIZE", "1")), "steps": steps, "warmup": 1,
           "ms_per_step": cb["ms_per_step"], "higher_is_better": False, "scaling": "weak", "vs_baseline": None,
           "dtype": "f64", "data": "synthetic",
           "config": {"workload": w.name, "grid": [w.nx, w.ny, w.nz], "sample": cb["sample"]},
           "cpu_baseline": {"value": cb["value"], "unit": UNIT, "kind": "oracle", "cores": cb["cores"],
                            "sample": cb["sample"]},
           "e2e": {"value": cb["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
           "gpu_launches": 0}
    print(json.dumps(out))


if __name__ == "__main__":
    a = parse()
    if a.impl == "reference":
        run_reference(a)
    else:
        run_ours(a)
