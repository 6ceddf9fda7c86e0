#!/usr/bin/env python
"""bench.py — throughput of the Poisson hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--small]

A STEP is one pass over every row of the hot path, each on the full-size grid of the BASELINE.json
config that exercises it, with seeded synthetic inputs (paper_2605_03563_b200/workloads.py):

    grid "c3"  256^3 Cartesian, Dirichlet ghosts (config 3):  multipole_bc(lmax 8), apply_laplacian, red-black SOR
               sweeps, fp64 V-cycles, mixed-precision V-cycles, residual norm
    grid "c4"  512^3 periodic, 19-point 6th-order star (config 4): CG, fixed 500 iterations (BASELINE: "fixed 500
               iterations for timing")
    grid "c5"  256x128x256 spherical (config 5): multipole_bc(lmax 8) + Jacobi-scaled BiCGSTAB, fixed 200 iterations

metric = grid-point updates per second (paper's s_s = N^3 / t_iteration): a point-update is one grid
point passing through one solver iteration / sweep / V-cycle (counted on finest-level points) / operator application.
`value` = all point-updates of the step / device time, inputs resident in HBM.  `e2e` = the same step through the
*_host C-ABI entry points: pinned host buffers, host->device and device->host copies inside the timed region.
Per-row throughput and roofline fractions are in "rows"; "roofline" describes the dominant kernel (cg_pass_a).

N > 1 ("replicas only"): every rank runs the same step on its own GPU, no collective in the
data path; value = point-updates of all ranks / max-over-ranks time.

--impl reference: the CPU oracle (oracle/, as it stands) timed on the host cores on a bounded sample of the same
step; rank 0 only.
"""
import argparse
import json
import math
import os
import statistics
import subprocess
import sys
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

from paper_2605_03563_b200 import workloads as wl  # noqa: E402

METRIC = "grid-point updates per second per solver iteration (rows of the hot path on 256^3-512^3 grids)"
UNIT = "Gpoint-updates/s"

# Algorithmic bytes per point per unit.
ROW_BYTES = {
    "multipole_bc": 8, "apply_laplacian": 16, "rbsor_sweep": 12,   # 24/T, T = 2 sweeps per HBM pass (NHS = 4) on grids >= 2^21 points
    "mg_vcycle_f64": 75, "mg_vcycle_mixed": 66,
    "residual_norm": 16, "cg_iteration_19pt": 72, "multipole_bc_spherical": 8, "bicgstab_iteration": 136,
    # SURVEY.md §8(f) rows (measured after the timed step; not part of `value`):
    "spai_smooth": 24,              # f1: read x, b; write x
    "mgv_vcycle_f64": 94,           # f2: V(1,1): (2 x 24 smoothing + 17 residual/restriction + 17 prolongation) x 8/7
    "mgv_vcycle_mixed": 88,         # f2: the same with the coarse levels (1/7 of the points) stored in fp32
    "pcg_iteration": 88,            # f3: pass A 48 + pass B 24 + fused symmetric GS sweep from zero with r.z 16
    "rbsor_cheby_sweep": 12,        # f4: the fused kernel with one omega per half-step: 24/T, T = 2
    "rbsor_local_sweep": 48,        # f4: spherical, position-dependent omega: two unfused half-sweeps
    "mgv_vcycle_f64_511": 94,       # f2 at the paper's own size (Table 2: 511^3, seven coarse levels, nu = 1)
    "spai_smooth_o6": 24,           # f1: the SPAI step on the compact 27-point sixth-order operator (same bytes, 27-point A)
    "mgv_vcycle_o6_511": 94,        # f1 + f2: Table 2, order 6: 511^3, V(1,1)
}
ROW_CITE = {
    "multipole_bc": "a6 PAPER.md:213-222", "apply_laplacian": "a1 PAPER.md:43-49", "rbsor_sweep": "a2 PAPER.md:59-63",
    "mg_vcycle_f64": "a5 PAPER.md:125-152", "mg_vcycle_mixed": "a5 PAPER.md:205", "residual_norm": "a7 PAPER.md:55",
    "cg_iteration_19pt": "a3 PAPER.md:95-105,172", "multipole_bc_spherical": "a6 PAPER.md:222",
    "bicgstab_iteration": "a4 PAPER.md:105",
    "spai_smooth": "f1 PAPER.md:154-184", "mgv_vcycle_f64": "f2 PAPER.md:125-152", "mgv_vcycle_mixed": "f2 PAPER.md:205",
    "pcg_iteration": "f3 PAPER.md:107-123", "rbsor_cheby_sweep": "f4 PAPER.md:81-88", "rbsor_local_sweep": "f4 PAPER.md:88-93",
    "mgv_vcycle_f64_511": "f2 PAPER.md:186-195 Table 2 (paper: 34.8 ms per V(1,1) cycle = 3.83 Gzups, hardware not stated)",
    "spai_smooth_o6": "f1 PAPER.md:172-182 (compact order 6, Table 1 row 6)",
    "mgv_vcycle_o6_511": "f1 PAPER.md:186-195 Table 2 order 6 (paper: 35.3 ms per V(1,1) cycle)",
}


def plan(small):
    """Units of each row per step."""
    if small:
        return dict(n3=64, n4=64, n5=(32, 16, 32), apply=2, sor=4, vc64=2, vcmx=2, resn=1, cg=20, bicg=10)
    return dict(n3=256, n4=512, n5=(256, 128, 256), apply=10, sor=20, vc64=10, vcmx=10, resn=1, cg=500, bicg=200)


def row_units(p):
    n3, n4 = p["n3"] ** 3, p["n4"] ** 3
    n5 = p["n5"][0] * p["n5"][1] * p["n5"][2]
    return [  # (row, points, units per step)
        ("multipole_bc", n3, 1), ("apply_laplacian", n3, p["apply"]), ("rbsor_sweep", n3, p["sor"]),
        ("mg_vcycle_f64", n3, p["vc64"]), ("mg_vcycle_mixed", n3, p["vcmx"]), ("residual_norm", n3, p["resn"]),
        ("cg_iteration_19pt", n4, p["cg"]), ("multipole_bc_spherical", n5, 1), ("bicgstab_iteration", n5, p["bicg"]),
    ]


def measured_peak():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        try:
            return float(json.load(open(path))["hbm_gbs"]), "MEASURED_PEAKS.json hbm_gbs (driver-measured copy)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


def stored_traffic():
    """DRAM bytes from the committed ncu captures (profiles/traffic.csv, lines `key,bytes`): `cg_pass_a` etc. = bytes per
    launch of that kernel class, `row:<name>` = bytes per point-update of that bench row (dram__bytes_read.sum +
    dram__bytes_write.sum of all its kernels / its point-updates).  ncu cannot run inside the timed bench, so these are
    the stored figures of the capture profiles/README.md names, not a measurement of this run."""
    path = os.path.join(ROOT, "profiles", "traffic.csv")
    out = {}
    try:
        for line in open(path):
            f = [x.strip() for x in line.split(",")]
            if len(f) >= 2 and f[0] and not f[0].startswith(("#", '"')):
                try:
                    out[f[0]] = float(f[1])
                except ValueError:
                    pass   # header line
    except OSError:
        return None
    return out or None


def max_over_ranks(values, world, device="cpu"):
    """Replicas only: the only cross-rank traffic of the bench is this MAX over the ranks' device
    times (nccl on GPUs; gloo in the CPU test).  Returns the list of per-entry maxima."""
    if world <= 1:
        return [float(v) for v in values]
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(v) for v in values], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(v) for v in t.cpu()]


def aggregate_value(units_per_rank, world, ms_max, steps):
    """Whole-job throughput in Gpoint-updates/s: every rank did `units_per_rank` point-updates per step."""
    return world * units_per_rank * steps / (ms_max * 1e-3) / 1e9


class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.proc, self.path = index, None, "/tmp/bench_clocks_%d_%d.csv" % (os.getpid(), index)

    def start(self):
        try:
            self.fh = open(self.path, "w")
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"], stdout=self.fh,
                                         stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        self.fh.close()
        sm, mx, reasons, pw = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in open(self.path):
            f = [x.strip() for x in line.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0]))
                mx.append(float(f[1]))
                pw.append(float(f[2]))
            except ValueError:
                continue
            for nme, val in zip(names, f[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(nme)
        try:
            os.remove(self.path)
        except OSError:
            pass
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


# ---------------------------------------------------------------------------------------------------------------------
def build_inputs(p):
    w3 = wl.config3(p["n3"])
    w4 = wl.config4(p["n4"])
    w5 = wl.config5(*p["n5"])
    return w3, w4, w5


ALL_ROWS = list(ROW_BYTES)
_marker = {}


def row_marker(args, torch, index):
    """--mark (profiling aid): index + 1 consecutive launches of a tiny torch kernel (int32 add) announce the row that
    follows, so that a kernel list captured by ncu can be cut into rows (profiles/README.md)."""
    if not args.mark:
        return
    if "t" not in _marker:
        _marker["t"] = torch.zeros(8, device="cuda", dtype=torch.int32)
    for _ in range(index + 1):
        _marker["t"].add_(1)


def measure_next_rows(p, args, pb, torch, stream, g3, g5, d, omega3):
    """SURVEY.md §8(f) rows, each timed on its own after the step (CUDA events, warm-up + repeats); not in `value`."""
    light = args.small or args.divide > 1   # functional / profiling runs: few units, one repeat
    reps = 1 if light else 3

    def timed(fn, units, name):
        row_marker(args, torch, ALL_ROWS.index(name))
        fn()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(reps):
            fn()
        e1.record()
        torch.cuda.synchronize()
        row_marker(args, torch, len(ALL_ROWS))
        return e0.elapsed_time(e1) / reps

    out = []
    # f1 / f2: the paper's own multigrid on the vertex-centred 2^N k - 1 grid next to config 3's (255^3), two-sphere density
    nv = p["n3"] - 1
    wv = wl.two_spheres(nv, cell_centred=False)
    gv = pb.Poisson(wv["shape"], wv["spacing"], wv["origin"], bc=wv["bc"], stream=stream.cuda_stream)
    gv.set_ghost_faces([torch.from_numpy(f).cuda() for f in wl.analytic_ghost_faces(wv, wv["potential"])])
    rhs = torch.from_numpy(np.ascontiguousarray(wv["rhs"])).cuda()
    phi = torch.zeros_like(rhs)
    nsm, ncyc = (2, 2) if light else (8, 10)
    out.append(("spai_smooth", nv ** 3, nsm, timed(lambda: gv.spai_smooth(phi, rhs, nsteps=nsm), nsm, "spai_smooth")))
    for name, prec in (("mgv_vcycle_f64", pb.F64), ("mgv_vcycle_mixed", pb.MIXED)):
        def cyc():
            phi.zero_()
            gv.mgv_vcycle(phi, rhs, nu1=1, nu2=1, precision=prec, ncycles=ncyc, want_resnorms=False)
        out.append((name, nv ** 3, ncyc, timed(cyc, ncyc, name)))
    del gv
    gv = pb.Poisson((nv,) * 3, (2.0 / (nv + 1),) * 3, (-1 + 2.0 / (nv + 1),) * 3, bc=(0,) * 6, stream=stream.cuda_stream)
    gv.set_option(pb.OPT_COMPACT_ORDER, 6)
    out.append(("spai_smooth_o6", nv ** 3, nsm, timed(lambda: gv.spai_smooth(phi, rhs, nsteps=nsm), nsm, "spai_smooth_o6")))
    del gv, rhs, phi
    if not light:
        # the paper's own Table 2 configuration: 511^3, seven coarse levels, V(1,1), order 2, fp64
        n5v = 2 * p["n3"] - 1
        wv = wl.two_spheres(n5v, cell_centred=False)
        gv = pb.Poisson(wv["shape"], wv["spacing"], wv["origin"], bc=wv["bc"], stream=stream.cuda_stream)
        gv.set_ghost_faces([torch.from_numpy(f).cuda() for f in wl.analytic_ghost_faces(wv, wv["potential"])])
        rhs = torch.from_numpy(np.ascontiguousarray(wv["rhs"])).cuda()
        del wv
        phi = torch.zeros_like(rhs)

        def cyc511():
            phi.zero_()
            gv.mgv_vcycle(phi, rhs, nu1=1, nu2=1, precision=pb.F64, ncycles=ncyc, want_resnorms=False)
        out.append(("mgv_vcycle_f64_511", n5v ** 3, ncyc, timed(cyc511, ncyc, "mgv_vcycle_f64_511")))
        # f1: the compact sixth-order discretisation (zero boundary values, right-hand side taken as it is)
        del gv
        gv = pb.Poisson((n5v,) * 3, (2.0 / (n5v + 1),) * 3, (-1 + 2.0 / (n5v + 1),) * 3, bc=(0,) * 6, stream=stream.cuda_stream)
        gv.set_option(pb.OPT_COMPACT_ORDER, 6)
        out.append(("mgv_vcycle_o6_511", n5v ** 3, ncyc, timed(cyc511, ncyc, "mgv_vcycle_o6_511")))
        del gv, rhs, phi
    # f3: Gauss-Seidel-preconditioned CG, f4: Chebyshev omega sequence, both on the config-3 grid (7-point, Dirichlet)
    npcg, nsw = (5, 4) if light else (50, 20)

    def pcg():
        d["phi3"].zero_()
        res = g3.pcg_solve(d["phi3"], d["rhs3"], fixed_iters=npcg)
        if res["status"] != pb.OK or res["iters"] != npcg:
            raise SystemExit("bench: PCG ended early (status %d, %d iterations)" % (res["status"], res["iters"]))
    out.append(("pcg_iteration", p["n3"] ** 3, npcg, timed(pcg, npcg, "pcg_iteration")))
    out.append(("rbsor_cheby_sweep", p["n3"] ** 3, nsw,
                timed(lambda: g3.rbsor_cheby(d["sor3"], d["rhs3"], nsw), nsw, "rbsor_cheby_sweep")))
    n5 = p["n5"][0] * p["n5"][1] * p["n5"][2]
    nloc = 4
    out.append(("rbsor_local_sweep", n5, nloc,
                timed(lambda: g5.rbsor_local(d["phi5"], d["rhs5"], nloc), nloc, "rbsor_local_sweep")))
    return out


def run_ours(args):
    import torch
    import torch.distributed as dist

    from paper_2605_03563_b200 import binding as pb

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback); use --impl reference for the oracle")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    pb.lib()
    p = plan(args.small)
    if args.divide > 1:
        for key in ("apply", "sor", "vc64", "vcmx", "cg", "bicg"):
            p[key] = max(1, p[key] // args.divide)
    if args.rows:   # profiling aid: a subset of the rows (the reported value then covers only those)
        keep = set(args.rows.split(","))
        if "cg_iteration_19pt" not in keep:
            p["n4"] = 32          # grids of unselected rows are shrunk so that set-up stays short
        if not keep & {"multipole_bc_spherical", "bicgstab_iteration"}:
            p["n5"] = (32, 16, 32)
        if keep <= {"cg_iteration_19pt", "multipole_bc_spherical", "bicgstab_iteration"}:
            p["n3"] = 32
    w3, w4, w5 = build_inputs(p)
    units = row_units(p)
    if args.rows:
        units = [u for u in units if u[0] in keep]
    kids = pb.kernel_classes()
    stream = torch.cuda.current_stream()
    mk = lambda w: pb.Poisson(w["shape"], w.get("spacing"), w.get("origin"), edges=w.get("edges"),
                              coord=w.get("coord", 0), order=w.get("order", 2), bc=w["bc"], stream=stream.cuda_stream)
    g3, g4, g5 = mk(w3), mk(w4), mk(w5)
    if args.path is not None:
        for g in (g3, g4, g5):
            g.set_option(pb.OPT_KERNEL_PATH, args.path)
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    h = dict(rho3=pin(w3["rho"]), rhs3=pin(w3["rhs"]), rhs4=pin(w4["rhs"]), rho5=pin(w5["rho"]), rhs5=pin(w5["rhs"]))
    d = {k: v.cuda(non_blocking=True) for k, v in h.items()}
    z = lambda ref: torch.zeros_like(ref)
    d.update(phi3=z(d["rhs3"]), out3=z(d["rhs3"]), sor3=z(d["rhs3"]), mx3=z(d["rhs3"]), phi4=z(d["rhs4"]),
             phi5=z(d["rhs5"]))
    h.update(phi3=pin(np.zeros_like(w3["rhs"])), out3=pin(np.zeros_like(w3["rhs"])),
             phi4=pin(np.zeros_like(w4["rhs"])), phi5=pin(np.zeros_like(w5["rhs"])))
    del w3["exact"], w4["rhs"]
    torch.cuda.synchronize()
    omega3 = 2.0 / (1.0 + math.sin(math.pi / (p["n3"] + 1)))
    row_names = [u[0] for u in units]

    def krylov_ok(what, res, fixed):
        # a BREAKDOWN in fixed mode sets the device `done` flag and every later pass returns at once: that would time
        # empty launches.  A timed solve must have run all its iterations.
        if res["status"] != pb.OK or res["iters"] != fixed:
            raise SystemExit("bench: %s ended with status %d after %d of %d iterations — timing would be invalid"
                             % (what, res["status"], res["iters"], fixed))

    def _apply():
        for _ in range(p["apply"]):
            g3.apply_laplacian(d["phi3"], d["out3"])

    def _resn():
        for _ in range(p["resn"]):
            g3.residual_norm(d["phi3"], d["rhs3"])

    row_fn = {
        "multipole_bc": lambda: g3.multipole_bc(d["rho3"], 1.0, 8, want_moments=False),
        "apply_laplacian": _apply,
        "rbsor_sweep": lambda: g3.rbsor_sweep(d["sor3"], d["rhs3"], omega3, p["sor"]),
        "mg_vcycle_f64": lambda: g3.mg_vcycle(d["phi3"], d["rhs3"], ncycles=p["vc64"], precision=pb.F64,
                                              want_resnorms=False),
        "mg_vcycle_mixed": lambda: g3.mg_vcycle(d["mx3"], d["rhs3"], ncycles=p["vcmx"], precision=pb.MIXED,
                                                want_resnorms=False),
        "residual_norm": _resn,
        "cg_iteration_19pt": lambda: krylov_ok("CG", g4.cg_solve(d["phi4"], d["rhs4"], fixed_iters=p["cg"]), p["cg"]),
        "multipole_bc_spherical": lambda: g5.multipole_bc(d["rho5"], 1.0, 8, want_moments=False),
        "bicgstab_iteration": lambda: krylov_ok("BiCGSTAB", g5.bicgstab_solve(d["phi5"], d["rhs5"],
                                                                             fixed_iters=p["bicg"]), p["bicg"]),
    }

    def step_device(ev=None):
        mark = (lambda: (ev.append(torch.cuda.Event(enable_timing=True)), ev[-1].record())) if ev is not None \
            else (lambda: None)
        mark()
        for name in row_names:
            row_marker(args, torch, ALL_ROWS.index(name))
            row_fn[name]()
            mark()
        row_marker(args, torch, len(ALL_ROWS))   # "no row": what follows belongs to the harness

    def _apply_host():
        for _ in range(p["apply"]):
            g3.apply_laplacian_host(h["phi3"], h["out3"])

    n3b, n4b, n5b = d["rhs3"].numel() * 8, d["rhs4"].numel() * 8, d["rhs5"].numel() * 8
    # the same rows through the host-buffer entry points: every input crosses PCIe, every result comes back
    host_fn = {  # name -> (call, h2d bytes, d2h bytes)
        "multipole_bc": (lambda: g3.multipole_bc_host(h["rho3"], 1.0, 8, want_moments=False), n3b, 0),
        "apply_laplacian": (_apply_host, n3b * p["apply"], n3b * p["apply"]),
        "rbsor_sweep": (lambda: g3.rbsor_sweep_host(h["phi3"], h["rhs3"], omega3, p["sor"]), 2 * n3b, n3b),
        "mg_vcycle_f64": (lambda: g3.mg_vcycle_host(h["phi3"], h["rhs3"], ncycles=p["vc64"], precision=pb.F64,
                                                    want_resnorms=False), 2 * n3b, n3b),
        "mg_vcycle_mixed": (lambda: g3.mg_vcycle_host(h["phi3"], h["rhs3"], ncycles=p["vcmx"], precision=pb.MIXED,
                                                      want_resnorms=False), 2 * n3b, n3b),
        # residual norm of host data: zero sweeps + the norm
        "residual_norm": (lambda: g3.rbsor_sweep_host(h["phi3"], h["rhs3"], 1.0, 0, want_resnorm=True), 2 * n3b, n3b),
        "cg_iteration_19pt": (lambda: krylov_ok("CG (host)", g4.cg_solve_host(h["phi4"], h["rhs4"],
                                                                             fixed_iters=p["cg"]), p["cg"]), 2 * n4b, n4b),
        "multipole_bc_spherical": (lambda: g5.multipole_bc_host(h["rho5"], 1.0, 8, want_moments=False), n5b, 0),
        "bicgstab_iteration": (lambda: krylov_ok("BiCGSTAB (host)", g5.bicgstab_solve_host(
            h["phi5"], h["rhs5"], fixed_iters=p["bicg"]), p["bicg"]), 2 * n5b, n5b),
    }

    def step_host():
        for k in ("phi3", "phi4", "phi5"):
            h[k].zero_()
        for name in row_names:
            host_fn[name][0]()

    h2d = sum(host_fn[nm][1] for nm in row_names)
    d2h = sum(host_fn[nm][2] for nm in row_names)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def zero_state():
        for k in ("phi3", "sor3", "mx3", "phi4", "phi5"):
            d[k].zero_()

    # ---- device-resident timing ----
    for _ in range(args.warmup):
        zero_state()
        step_device()
    barrier()
    dom = kids.index("cg_pass_a")
    g4.set_option(pb.OPT_TIME_KERNELS, dom)
    g4.reset_kernel_times()
    launches0 = sum(g.kernel_launches() for g in (g3, g4, g5))
    sampler = ClockSampler(local)
    sampler.start()
    evs = []
    barrier()
    t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t0.record()
    for _ in range(args.steps):
        ev = []
        zero_state()   # every timed step starts from the same cold state (phi = 0) as the warm-up steps
        step_device(ev)
        evs.append(ev)
    t1.record()
    barrier()
    clocks = sampler.stop()
    ms_total = t0.elapsed_time(t1)
    launches = sum(g.kernel_launches() for g in (g3, g4, g5)) - launches0
    dom_ms, dom_cnt = g4.kernel_time(dom)
    g4.set_option(pb.OPT_TIME_KERNELS, -1)
    row_ms = [statistics.mean(ev[i].elapsed_time(ev[i + 1]) for ev in evs) for i in range(len(row_names))]
    # ---- end-to-end timing (host buffers) ----
    e2e_steps = max(1, min(args.steps, 2))
    step_host()
    barrier()
    t2, t3 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t2.record()
    for _ in range(e2e_steps):
        step_host()
    t3.record()
    barrier()
    ms_e2e = t2.elapsed_time(t3)
    # ---- a separate pass with every kernel class event-timed (not part of `value`) ----
    for g in (g3, g4, g5):
        g.set_option(pb.OPT_TIME_KERNELS, -2)
        g.reset_kernel_times()
    step_device()
    torch.cuda.synchronize()
    ktab = {}
    for g, gname in ((g3, "c3"), (g4, "c4"), (g5, "c5")):
        for i, kname in enumerate(kids):
            ms, cnt = g.kernel_time(i)
            if cnt:
                ktab["%s:%s" % (gname, kname)] = {"launches": cnt, "avg_ms": ms / cnt, "total_ms": ms}
        g.set_option(pb.OPT_TIME_KERNELS, -1)

    next_rows = measure_next_rows(p, args, pb, torch, stream, g3, g5, d, omega3) if not args.rows else []

    ms_total, ms_e2e = max_over_ranks([ms_total, ms_e2e], world, "cuda")
    total_updates = sum(pts * u for _, pts, u in units)
    peak, peak_src = measured_peak()
    tr = stored_traffic() or {}
    rows = {}

    def add_row(name, pts, u, ms, in_value):
        # per row: Gpoint-updates/s, algorithmic B/point, achieved algorithmic GB/s, fraction of the measured HBM peak,
        # and the DRAM bytes per point-update ncu counted for the row's kernels (profiles/traffic.csv), with the GB/s
        # that figure implies
        gpts = pts * u / (ms * 1e-3) / 1e9
        gbs = gpts * ROW_BYTES[name]
        dram = tr.get("row:" + name)
        row = {"cite": ROW_CITE[name], "pts": pts, "units": u, "ms": round(ms, 4), "gpts": round(gpts, 2),
               "B_pt": ROW_BYTES[name], "alg_gbs": round(gbs), "frac": round(gbs / peak, 3),
               "dram_B_pt": dram, "dram_gbs": round(gpts * dram) if dram else None, "in_value": in_value}
        if name.startswith("multipole_bc"):
            # the moments are line sums since round 2 (z lines / radial lines: lmax + 1 multiply-adds per point, DESIGN.md
            # §6): an HBM-bound pass of 8 B/point, no longer the fp64-ALU-bound one of the point-by-point kernel
            row.update(bound="hbm")
        rows[name] = row

    for (name, pts, u), ms in zip(units, row_ms):
        add_row(name, pts, u, ms, True)
    for name, pts, u, ms in next_rows:
        add_row(name, pts, u, ms, False)
    n4 = p["n4"] ** 3
    achieved = 48.0 * n4 / (dom_ms / max(dom_cnt, 1) * 1e-3) / 1e9 if dom_cnt else None
    out = {
        "metric": METRIC, "value": round(aggregate_value(total_updates, world, ms_total, args.steps), 3),
        "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": round(ms_total / args.steps, 3), "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "rows": rows,
        "roofline": {"kernel": "cg_pass_a (19-point, 512^3): x += a p_old; p = r + b p_old; q = L p; sum p.q",
                     "bound": "hbm", "achieved": round(achieved, 1) if achieved else None, "peak": peak,
                     "unit": "GB/s", "frac": round(achieved / peak, 4) if achieved else None,
                     "traffic": tr.get("cg_pass_a"), "traffic_source": "profiles/traffic.csv (ncu --set full, stored)",
                     "algorithmic_bytes_per_launch": 48 * n4, "avg_launch_ms": round(dom_ms / max(dom_cnt, 1), 4),
                     "launches_timed": dom_cnt, "peak_source": peak_src},
        "e2e": {"value": round(aggregate_value(total_updates, world, ms_e2e, e2e_steps), 3), "unit": UNIT,
                "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h, "steps": e2e_steps,
                "ms_per_step": round(ms_e2e / e2e_steps, 3)},
        "config": {"workload": "one pass over all hot-path rows: config 3 grid 256^3 (multipole lmax 8, apply x%d, "
                               "RB-SOR x%d sweeps, V(2,2) x%d fp64 + x%d mixed, residual norm), config 4 grid 512^3 "
                               "periodic 19-point CG x%d iterations, config 5 grid 256x128x256 spherical multipole "
                               "+ BiCGSTAB x%d iterations" % (p["apply"], p["sor"], p["vc64"], p["vcmx"], p["cg"],
                                                              p["bicg"]) if not args.small else "small smoke plan",
                   "point_updates_per_step": total_updates, "l2": "working sets larger than L2 (256^3 fp64 array = "
                   "134 MB, 512^3 = 1.07 GB, several live per row); no explicit flush",
                   "parallelism": "replicas only" if world > 1 else "single GPU"},
        "gpu_launches": launches,
        "clocks": clocks,
        "kernels": {k: [v["launches"], round(v["avg_ms"], 4)] for k, v in ktab.items()},   # class: [launches, avg ms]
    }
    if rank == 0:
        if not args.no_cpu and world == 1:
            out["cpu_baseline"] = cpu_baseline(p, quick=args.small)
        print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


# ---------------------------------------------------------------------------------------------------------------------
def oracle_rates(p, quick=False):
    """Per-row oracle rates (point-updates/s) on a bounded sample of the step's workload.  The oracle runs as it
    stands (OpenMP over pointwise loops); slabs keep the xy extent of the full grid and shorten z."""
    sys.path.insert(0, os.path.join(ROOT, "oracle"))
    import pyoracle as po

    rates, notes = {}, []
    n3 = p["n3"]
    w3 = wl.config3(n3)
    o3 = po.Oracle(w3["shape"], w3["spacing"], w3["origin"], bc=w3["bc"])
    # multipole moments on a z-slab (trigonometric long-double oracle: ~2 us per point)
    nz = max(4, n3 // 8)
    os_ = po.Oracle((n3, n3, nz), w3["spacing"], w3["origin"], bc=w3["bc"])
    t = time.perf_counter()
    os_.multipole_bc(np.ascontiguousarray(w3["rho"][:nz]), 1.0, 8)
    rates["multipole_bc"] = n3 * n3 * nz / (time.perf_counter() - t)
    notes.append("multipole: %dx%dx%d slab" % (n3, n3, nz))
    phi = np.zeros_like(w3["rhs"])
    t = time.perf_counter()
    o3.apply(phi)
    rates["apply_laplacian"] = phi.size / (time.perf_counter() - t)
    t = time.perf_counter()
    o3.rbsor(phi, w3["rhs"], 1.5, 2)
    rates["rbsor_sweep"] = 2 * phi.size / (time.perf_counter() - t)
    t = time.perf_counter()
    o3.vcycle(phi, w3["rhs"], ncycles=1)
    dt = time.perf_counter() - t
    t = time.perf_counter()
    rn = o3.residual_norm(phi, w3["rhs"])
    dtr = time.perf_counter() - t
    rates["residual_norm"] = phi.size / dtr
    rates["mg_vcycle_f64"] = phi.size / max(dt - 2 * dtr, 1e-9)  # the oracle call also takes two residual norms
    t = time.perf_counter()
    o3.vcycle(phi, w3["rhs"], ncycles=1, precision=1)
    rates["mg_vcycle_mixed"] = phi.size / max(time.perf_counter() - t - 2 * dtr, 1e-9)
    notes.append("apply/SOR(2 sweeps)/V-cycle(1+1)/residual: full %d^3" % n3)
    del phi, o3, w3
    # CG, 19-point periodic: slab of the config-4 grid, per-iteration time from the difference of two runs
    n4 = p["n4"]
    nz = max(8, n4 // 8)
    rhs = wl.random_field((n4, n4, nz), 4)
    rhs -= rhs.mean()
    o4 = po.Oracle((n4, n4, nz), (1.0 / n4,) * 3, (0.0,) * 3, order=6, bc=(po.BC_PERIODIC,) * 6)
    x = np.zeros_like(rhs)
    t = time.perf_counter()
    o4.cg(x, rhs, fixed_iters=1)
    d1 = time.perf_counter() - t
    x[:] = 0
    t = time.perf_counter()
    o4.cg(x, rhs, fixed_iters=4)
    d4 = time.perf_counter() - t
    rates["cg_iteration_19pt"] = 3 * rhs.size / max(d4 - d1, 1e-9)
    notes.append("CG 19-pt: %dx%dx%d periodic slab, (4 its - 1 it)/3" % (n4, n4, nz))
    del rhs, x, o4
    w5 = wl.config5(*p["n5"])
    o5 = po.Oracle(w5["shape"], edges=w5["edges"], coord=1, bc=w5["bc"])
    nr, nt, nph = p["n5"]
    npz = max(4, nph // 8)
    w5s = wl.config5(nr, nt, npz)
    o5s = po.Oracle(w5s["shape"], edges=w5s["edges"], coord=1, bc=w5s["bc"])
    t = time.perf_counter()
    o5s.multipole_bc(w5s["rho"], 1.0, 8)
    rates["multipole_bc_spherical"] = w5s["rho"].size / (time.perf_counter() - t)
    x = np.zeros_like(w5["rhs"])
    t = time.perf_counter()
    o5.bicgstab(x, w5["rhs"], fixed_iters=1)
    d1 = time.perf_counter() - t
    x[:] = 0
    t = time.perf_counter()
    o5.bicgstab(x, w5["rhs"], fixed_iters=4)
    d4 = time.perf_counter() - t
    rates["bicgstab_iteration"] = 3 * x.size / max(d4 - d1, 1e-9)
    notes.append("BiCGSTAB: full %dx%dx%d, (4 its - 1 it)/3; spherical multipole: %d phi-planes" % (nr, nt, nph, npz))
    return rates, notes, po.get_threads()


def projected_value(p, rates):
    """Whole-step throughput implied by per-row rates: total point-updates / sum_rows(updates_row / rate_row)."""
    units = row_units(p)
    tot = sum(pts * u for _, pts, u in units)
    tsec = sum(pts * u / rates[name] for name, pts, u in units)
    return tot / tsec / 1e9


def cpu_baseline(p, quick=False):
    rates, notes, cores = oracle_rates(p, quick)
    return {"value": round(projected_value(p, rates), 5), "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": "per-row oracle rates on bounded samples, combined with the step's row weights "
                      "(total updates / sum(updates_row / rate_row)); " + "; ".join(notes),
            "rows": {k: round(v / 1e9, 5) for k, v in rates.items()}}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    p = plan(args.small)
    for _ in range(min(args.warmup, 1)):
        oracle_rates(p)
    vals, t0 = [], time.perf_counter()
    last = None
    for _ in range(args.steps):
        rates, notes, cores = oracle_rates(p)
        vals.append(projected_value(p, rates))
        last = (rates, notes, cores)
    dt = time.perf_counter() - t0
    rates, notes, cores = last
    v = statistics.mean(vals)
    total_updates = sum(pts * u for _, pts, u in row_units(p))
    sample = ("each step = one bounded-sample pass of the oracle over every row; value = total updates / "
              "sum(updates_row / rate_row); " + "; ".join(notes))
    out = {"impl": "reference", "metric": METRIC, "value": round(v, 5), "unit": UNIT, "n_gpus": args.gpus,
           "steps": args.steps, "warmup": args.warmup, "ms_per_step": round(total_updates / (v * 1e9) * 1e3, 1),
           "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           "config": {"workload": "same rows and grids as the CUDA arm (projected from bounded samples)",
                      "point_updates_per_step": total_updates, "sample_wall_s_per_step": round(dt / args.steps, 2)},
           "gpu_launches": 0,
           "cpu_baseline": {"value": round(v, 5), "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
           "e2e": {"value": round(v, 5), "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(out))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--small", action="store_true", help="tiny grids: a functional check, not a measurement")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--path", type=int, default=None, help="force POISSON_OPT_KERNEL_PATH (1 generic, 2 plane)")
    ap.add_argument("--rows", default=None, help="comma list of row names: time only these (profiling aid)")
    ap.add_argument("--divide", type=int, default=1, help="divide the per-row unit counts (profiling aid)")
    ap.add_argument("--mark", action="store_true", help="launch a marker kernel before every row (profiling aid)")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
