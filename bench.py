#!/usr/bin/env python
"""bench.py -- SPH pair interactions/s of the full density + hydro + FLD pass (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload c5] [--impl ours|reference]

A step = one pass of the whole hot path over one synthetic particle set (BASELINE.json configs, workloads/):
spray_build_cells -> spray_density -> spray_hydro_rhs_limiter (hydro right-hand sides + limiter pre-sweep in one sweep) ->
spray_fld_apply(FROZEN) (operator apply); --separate-calls runs spray_hydro_rhs -> spray_fld_apply(UPDATE_LIMITER) instead
(the same outputs bit for bit, tests/test_gpu_fused.py).
`value` = pair interactions per second with inputs resident in HBM; `e2e` = the same through the C-ABI with pinned
HOST buffers (H2D of every input and D2H of every output inside the timed region).  Multi-GPU: the path does not
shard (BASELINE.json: one GPU, no collectives) -> N independent replicas, "weak" scaling, no data-path collective.
Prints ONE JSON line on rank 0.  DESIGN.md §6 states the roofline arithmetic used below.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "SPH pair interactions/sec (density+hydro+FLD pass, fp64)"
UNIT = "pair interactions/s"

# Algorithmic flops per in-support ordered pair and sweep, counted from the defining formulas (DESIGN.md §6,
# frozen in BASELINE.md §2): add/sub/mul/compare = 1, FMA = 2, div = 1, sqrt = 1; distance + predicate included.
FLOPS = {0: dict(density=20, hydro=58, hydro_visc=25, limiter=32, apply=46),     # cubic spline
         1: dict(density=23, hydro=60, hydro_visc=25, limiter=33, apply=48)}     # Wendland C2
# Algorithmic HBM bytes per particle and pass: build 32 + sort 3*16 + reorder 64; gathers of 13
# caller-order fields at 16 B; sweep reads 40/104/64/64 B and writes 12/40/8+8/24 B (outputs + perm).
BYTES_PER_PARTICLE = 32 + 48 + 64 + 13 * 16 + (40 + 104 + 64 + 64) + (12 + 44 + 20 + 28)
FP64_NOMINAL_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12    # 148 SMs x 64 DFMA/clk x 2 flop x 1.965 GHz = 37.2


def peaks():
    try:
        return json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json"))), "measured"
    except Exception:
        return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0}, "fallback"


def traffic_table(workload):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch from the committed ncu --set full capture of this workload
    (profiles/r02_traffic.csv: workload, kernel, read bytes, written bytes, commit).  Empty when there is no capture."""
    out = {}
    try:
        for line in open(os.path.join(ROOT, "profiles", "r02_traffic.csv")):
            f = [c.strip() for c in line.split(",")]
            if len(f) >= 4 and f[0] == workload:
                out[f[1]] = float(f[2]) + float(f[3])
    except Exception:
        pass
    return out


def approaching_fraction(workload):
    """Fraction of ordered neighbour pairs with v_ab . x_ab < 0 (the pairs that take the viscous branch, eqs. (41)-(43)), MEASURED
    on the reduced-size preset of the same recipe (same lattice, jitter and velocity law, so the same fraction): the neighbour
    lists of the 48^3 set from the library's own export, the dot products in torch."""
    import numpy as np
    import torch
    import workloads as W
    import paper_2604_20124_b200 as P
    small = {"c5_v": "c5_mid", "c5": "c5_mid", "c4": "c4_mid", "c3": "c3_mid", "c2": "c2_mid", "c1": "c1"}.get(workload, workload)
    w = W.make(small)
    dev = torch.device("cuda", torch.cuda.current_device())
    t = {f: torch.from_numpy(np.ascontiguousarray(getattr(w, f))).to(dev) for f in ("x", "y", "z", "h", "vx", "vy", "vz")}
    sp = P.Spray(w.n, w.grid.ncell_total, device=dev.index or 0)
    sp.build_cells(w.grid, w.kernel, t["x"], t["y"], t["z"], t["h"])
    off, nbr = sp.neighbor_lists(True)
    a = torch.repeat_interleave(torch.arange(w.n, device=dev), (off[1:] - off[:-1]).to(torch.int64))
    b = nbr.to(torch.int64)
    dot = torch.zeros(a.shape[0], dtype=torch.float64, device=dev)
    for k, (c, v) in enumerate((("x", "vx"), ("y", "vy"), ("z", "vz"))):
        dx = t[c][a] - t[c][b]
        if w.grid.periodic[k]:
            L = float(w.grid.hi[k]) - float(w.grid.lo[k])
            dx = dx - L * torch.round(dx / L)
        dot += dx * (t[v][a] - t[v][b])
    return float((dot < 0).double().mean().item())


def cpu_model():
    try:
        for line in open("/proc/cpuinfo"):
            if line.lower().startswith("model name"):
                return line.split(":", 1)[1].strip()
    except Exception:
        pass
    return "unknown"


class ClockSampler:
    """nvidia-smi clocks + throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons, pw = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1])); pw.append(float(r[2]))
                for nm, v in zip(names, r[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(nm)
            except Exception:
                pass
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


def max_over_ranks(seconds, world, device=None):
    """Multi-GPU timing rule: the job's time is the MAX over ranks (one all-reduce of a scalar, outside the timed
    region).  Replicas only: this and the barrier are the only collectives of the bench."""
    if world <= 1:
        return float(seconds)
    import torch
    import torch.distributed as dist
    t = torch.tensor([seconds], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_value(world, pairs_per_pass, steps, seconds):
    """Whole-job throughput: every rank runs `steps` full passes over its own replica (weak scaling)."""
    return world * pairs_per_pass * steps / seconds


def oracle_sample_pass(w, targets):
    """The oracle as it stands on a bounded sample of the workload (its cell-list variant restricted to `targets`;
    rho = recipe density and mu = c/(3 rho kappa) as inputs).  Returns (seconds, pair interactions)."""
    import numpy as np
    import oracle as O
    a = (w.grid, w.kernel, w.x, w.y, w.z, w.h, w.m)
    mu = w.c_light / (3.0 * w.rho_nom * w.kappa)
    t0 = time.perf_counter()
    d = O.density(*a, targets=targets)
    O.hydro(*a, w.rho_nom, w.p, w.cs, w.vx, w.vy, w.vz, w.alpha, w.beta, targets=targets)
    O.limiter(*a, w.rho_nom, w.kappa, w.E, w.c_light, targets=targets)
    O.fld_apply(*a, w.rho_nom, mu, w.E, sym_mode=True, targets=targets)
    dt = time.perf_counter() - t0
    cg = d["nnbr"].astype(np.int64).sum()
    cs = O.neighbor_counts(w.grid, w.x, w.y, w.z, w.h, O.SYM, targets=targets).astype(np.int64).sum()
    return dt, int(2 * cg + 2 * cs + len(targets))


def run_reference(args, w, rank):
    """--impl reference: the CPU oracle (this tier's reference arm), rank 0 only, bounded sample per step."""
    import numpy as np
    import oracle as O
    if rank != 0:
        return
    rng = np.random.default_rng(0)
    ns = min(w.n, args.cpu_sample)
    targets = np.sort(rng.choice(w.n, size=ns, replace=False)).astype(np.int64)
    for _ in range(args.warmup):
        oracle_sample_pass(w, targets[: max(1, ns // 8)])
    tot_t, tot_p = 0.0, 0
    for _ in range(args.steps):
        dt, pairs = oracle_sample_pass(w, targets)
        tot_t += dt; tot_p += pairs
    v = tot_p / tot_t
    sample = f"{ns} of {w.n} target particles of {w.name} per step (all neighbours), oracle cell-list variant, long-double sums"
    print(json.dumps({"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
                      "warmup": args.warmup, "ms_per_step": 1e3 * tot_t / args.steps, "higher_is_better": True, "scaling": "weak",
                      "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": {"workload": w.name, "n_particles": w.n},
                      "cpu_baseline": {"value": v, "unit": UNIT, "cores": O.num_threads(), "kind": "oracle", "sample": sample},
                      "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="c5", help="workloads.PRESETS name; c5 = BASELINE.json's roofline config (16.7 M particles)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--path", type=int, default=None, help="pair-kernel implementation (spray_set_path); default = library default")
    ap.add_argument("--cpu-sample", type=int, default=200000, help="target particles per oracle step (cpu_baseline / reference arm)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--separate-calls", action="store_true",
                    help="pass = build, density, spray_hydro_rhs, spray_fld_apply(UPDATE_LIMITER) (two sweeps) instead of the default "
                         "build, density, spray_hydro_rhs_limiter (hydro + limiter in one sweep), spray_fld_apply(FROZEN): same outputs, bitwise")
    ap.add_argument("--no-n1", action="store_true", help="skip the row-N1/N3 measurements (spray_rad_jacobi iterations, spray_kgc_continuity)")
    ap.add_argument("--no-levels", action="store_true", help="do not set up the internal levels of the tiled path for variable-h workloads")
    ap.add_argument("--no-variants", action="store_true", help="skip the c5_v variant (v ~ N(0, 0.01^2): the viscous branch at full size)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup

    # --gpus N without a launcher: start the N replica ranks ourselves (one process per GPU, torchrun on 127.0.0.1)
    if args.impl == "ours" and args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        port = 29500 + os.getpid() % 2000
        os.execv(sys.executable, [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
                                  "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:])

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))

    import numpy as np
    import workloads as W
    w = W.make(args.workload)

    if args.impl == "reference":
        run_reference(args, w, rank)
        return

    import torch
    import torch.distributed as dist
    import paper_2604_20124_b200 as P

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the SPRAY pass has no CPU fallback (use --impl reference for the oracle)")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=dev)

    fields = ("x", "y", "z", "h", "m", "p", "cs", "vx", "vy", "vz", "alpha", "E", "kappa")
    host = {f: torch.from_numpy(np.ascontiguousarray(getattr(w, f))).pin_memory() for f in fields}
    d = {f: host[f].to(dev) for f in fields}
    n = w.n
    sp = P.Spray(n, w.grid.ncell_total, device=local_rank)
    if args.path is not None:
        sp.set_path(args.path)
    levels = []
    if float(w.h.min()) != float(w.h.max()) and not args.no_levels:
        # variable h (BASELINE.json configs 2 and 4): internal levels of the tiled path, cell edges from the h range (workloads.level_edges)
        levels = W.level_edges(w.h)
        sp.set_levels(w.grid, levels)
    f64 = torch.float64
    out = {k: torch.empty(n, dtype=f64, device=dev) for k in ("rho", "ax", "ay", "az", "dudt", "divv", "mu", "y", "diag", "offd")}
    hout = {k: torch.empty(n, dtype=f64).pin_memory() for k in out}

    fused = not args.separate_calls

    def hydro_and_fld(src, o, between=None):
        """rows (a6)-(a8): hydro right-hand sides, limiter pre-sweep, operator apply -- as two calls either way"""
        hy = [o["ax"], o["ay"], o["az"], o["dudt"], o["divv"]]
        if fused:
            sp.hydro_rhs_limiter(src["m"], o["rho"], src["p"], src["cs"], src["vx"], src["vy"], src["vz"], src["alpha"], src["E"], src["kappa"],
                                 beta=w.beta, c_light=w.c_light, out=hy, mu=o["mu"])
            if between: between()
            sp.fld_apply(src["m"], o["rho"], None, src["E"], w.c_light, lmode=P.FLD_FROZEN_CHAINED, mu=o["mu"], y=o["y"], diag=o["diag"], offd=o["offd"])
        else:
            sp.hydro_rhs(src["m"], o["rho"], src["p"], src["cs"], src["vx"], src["vy"], src["vz"], src["alpha"], w.beta, out=hy)
            if between: between()
            sp.fld_apply(src["m"], o["rho"], src["kappa"], src["E"], w.c_light, mu=o["mu"], y=o["y"], diag=o["diag"], offd=o["offd"])

    def one_pass(src, ev=None):
        sp.build_cells(w.grid, w.kernel, src["x"], src["y"], src["z"], src["h"])
        if ev: ev[1].record()
        sp.density(src["m"], rho=out["rho"])
        if ev: ev[2].record()
        hydro_and_fld(src, out, (lambda: ev[3].record()) if ev else None)
        if ev: ev[4].record()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # pair counts of this workload (outside the timed region)
    one_pass(d)
    cg = int(sp.neighbor_counts(False).to(torch.int64).sum().item())
    cs = int(sp.neighbor_counts(True).to(torch.int64).sum().item())
    assert sp.check() == 0, "device status flags set"
    pstats = sp.path_stats_full()
    n_tiles, n_fast = pstats["tiles"], pstats["n_fast"]
    pairs = {"density": cg + n, "hydro": cs, "limiter": cg, "apply": cs}
    p_pass = sum(pairs.values())

    for _ in range(args.warmup):
        one_pass(d)
    l0 = sp.launch_count()
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(5)] for _ in range(args.steps)]
    sampler = ClockSampler(local_rank)
    sampler.start()
    barrier()
    for s in range(args.steps):
        evs[s][0].record()
        one_pass(d, evs[s])
    barrier()
    clocks = sampler.stop()
    launches = sp.launch_count() - l0
    t_total = evs[0][0].elapsed_time(evs[-1][4]) * 1e-3
    seg = np.array([[e[i].elapsed_time(e[i + 1]) for i in range(4)] for e in evs]) * 1e-3     # build, density, hydro, fld
    t_total = max_over_ranks(t_total, world, dev)
    value = aggregate_value(world, p_pass, args.steps, t_total)

    # ---- e2e: pinned host buffers, H2D of every input and D2H of every output inside the timed region
    e2e = None
    if not args.no_e2e:
        # The four C-ABI calls need their inputs at different times, so a caller overlaps the copies with the kernels:
        # a copy-in stream uploads the fields in the order of need (one event per call), a copy-out stream downloads each
        # call's results while the next call runs.  Device inputs and outputs are double-buffered, so the uploads of step
        # k+1 (an independent batch) run under the kernels of step k and the downloads of step k under those of step k+1.
        # Every byte still crosses PCIe inside the timed region, every step.
        main = torch.cuda.current_stream()
        s_in, s_out = torch.cuda.Stream(), torch.cuda.Stream()
        if fused:
            groups = [("x", "y", "z", "h"), ("m",), ("p", "cs", "vx", "vy", "vz", "alpha", "E", "kappa"), ()]
            outs = [(), ("rho",), ("ax", "ay", "az", "dudt", "divv", "mu"), ("y", "diag", "offd")]
        else:
            groups = [("x", "y", "z", "h"), ("m",), ("p", "cs", "vx", "vy", "vz", "alpha"), ("E", "kappa")]
            outs = [(), ("rho",), ("ax", "ay", "az", "dudt", "divv"), ("mu", "y", "diag", "offd")]
        dbuf = [d, {f: torch.empty_like(d[f]) for f in fields}]
        obuf = [out, {o: torch.empty_like(out[o]) for o in out}]
        in_free = [torch.cuda.Event(), torch.cuda.Event()]     # kernels of the step that last read dbuf[b] are done
        out_free = [torch.cuda.Event(), torch.cuda.Event()]    # results of the step that last wrote obuf[b] are in host memory

        def e2e_pass(b):
            dd, oo = dbuf[b], obuf[b]
            ev_in = []
            with torch.cuda.stream(s_in):
                s_in.wait_event(in_free[b])
                for grp in groups:
                    for f in grp:
                        dd[f].copy_(host[f], non_blocking=True)
                    ev = torch.cuda.Event(); ev.record(s_in); ev_in.append(ev)

            def done(k):                        # results of call k go home on the copy-out stream
                ev = torch.cuda.Event(); ev.record(main)
                with torch.cuda.stream(s_out):
                    s_out.wait_event(ev)
                    for o in outs[k]:
                        hout[o].copy_(oo[o], non_blocking=True)

            main.wait_event(out_free[b])
            main.wait_event(ev_in[0])
            sp.build_cells(w.grid, w.kernel, dd["x"], dd["y"], dd["z"], dd["h"])
            main.wait_event(ev_in[1])
            sp.density(dd["m"], rho=oo["rho"])
            done(1)
            main.wait_event(ev_in[2])

            def between():
                done(2)
                main.wait_event(ev_in[3])
            hydro_and_fld(dd, oo, between)
            done(3)
            in_free[b].record(main)
            out_free[b].record(s_out)

        for b in (0, 1):
            e2e_pass(b)
        main.wait_stream(s_out)
        barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ksteps = max(2, min(args.steps, 5))
        e0.record()
        for k in range(ksteps):
            e2e_pass(k & 1)
        main.wait_stream(s_out)                 # the last step ends when its last result is in host memory
        e1.record()
        barrier()
        te = e0.elapsed_time(e1) * 1e-3
        te = max_over_ranks(te, world, dev)
        e2e = {"value": aggregate_value(world, p_pass, ksteps, te), "unit": UNIT, "h2d_bytes_per_step": 8 * n * len(fields),
               "d2h_bytes_per_step": 8 * n * len(out), "ms_per_step": 1e3 * te / ksteps}

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- FP64 peak probe (MEASURED_PEAKS.json has no FP64 entry): sustained DFMA rate, same job
    pk, pk_src = peaks()
    pb = torch.empty(148 * 8 * 256, dtype=f64, device=dev)
    iters = 4000
    P.fp64_peak_probe(local_rank, 148 * 8, 256, 200, pb)
    torch.cuda.synchronize()
    p0, p1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    p0.record()
    for _ in range(10):
        P.fp64_peak_probe(local_rank, 148 * 8, 256, iters, pb)
    p1.record()
    torch.cuda.synchronize()
    fp64_meas = 10 * 148 * 8 * 256 * iters * 64 * 2 / (p0.elapsed_time(p1) * 1e-3) / 1e12

    # ---- row N1: Jacobi iterations of the implicit radiation step on the same particle set, with the
    #      neighbour lists of the last spray_build_cells; outside the timed region of the headline metric
    n1 = None
    if not args.no_n1:
        u_n = d["p"] / ((w.gamma - 1.0) * out["rho"])
        T_n = (w.gamma - 1.0) * u_n
        dTdu = torch.full_like(u_n, w.gamma - 1.0)
        nit = 20
        dt_rad = 0.3 * float(w.h.min()) ** 2 / float(out["mu"].max().item())
        sp.rad_jacobi(d["m"], out["rho"], out["mu"], d["kappa"], d["E"], u_n, T_n, dTdu, dt_rad, w.c_light, 1.0, niter=2)
        torch.cuda.synchronize()
        r0, r1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        r0.record()
        rj = sp.rad_jacobi(d["m"], out["rho"], out["mu"], d["kappa"], d["E"], u_n, T_n, dTdu, dt_rad, w.c_light, 1.0, niter=nit)
        r1.record()
        torch.cuda.synchronize()
        t_it = r0.elapsed_time(r1) * 1e-3 / nit
        n1 = {"call": "spray_rad_jacobi", "iterations": nit, "ms_per_iteration": 1e3 * t_it, "iterations_per_s": 1.0 / t_it,
              "pair_interactions_per_s": pairs["apply"] / t_it,
              "flop_roofline_frac": pairs["apply"] * FLOPS[w.kernel]["apply"] / t_it / (fp64_meas * 1e12),
              "resid_last": float(rj["resid"][-1].item()), "note": "includes the one-off prologue of the call (1/%d per iteration)" % nit}

    # ---- row N2: thermal conduction (spray_conduction: one symmetric frozen sweep of the apply kernel with mu = k, E = T) and the
    #      matrix-free operator of the implicit two-temperature system, eqs. (28)-(34) (spray_conduction_implicit: two sweeps, one
    #      per species); k proportional to T^(5/2) (Spitzer-like), same lists; apply flops per ordered pair
    n2 = None
    if not args.no_n1:
        u_g = d["p"] / ((w.gamma - 1.0) * out["rho"])
        T_g = (w.gamma - 1.0) * u_g
        T_e = 1.1 * T_g
        k_i = 0.02 * (T_g / T_g.mean()) ** 2.5 + 1e-3
        k_e = 0.05 * (T_e / T_e.mean()) ** 2.5 + 1e-3
        kei = torch.full_like(u_g, 0.5)
        tau = torch.full_like(u_g, w.gamma - 1.0)
        u_e = T_e / (w.gamma - 1.0)
        dt_c = 0.3 * float(w.h.min()) ** 2 / float(k_e.max().item())
        def _time(fn, nrep=5):
            fn(); fn()
            torch.cuda.synchronize()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            for _ in range(nrep):
                fn()
            b.record()
            torch.cuda.synchronize()
            return a.elapsed_time(b) * 1e-3 / nrep
        t_c = _time(lambda: sp.conduction(d["m"], out["rho"], k_i, T_g))
        t_o = _time(lambda: sp.conduction_implicit(d["m"], out["rho"], k_i, k_e, kei, tau, tau, None, None, u_g, u_e, dt_c, 0))
        fa = FLOPS[w.kernel]["apply"]
        n2 = {"call": "spray_conduction", "ms_per_call": 1e3 * t_c, "pair_interactions_per_s": pairs["apply"] / t_c,
              "flop_roofline_frac": pairs["apply"] * fa / t_c / (fp64_meas * 1e12),
              "implicit_operator": {"call": "spray_conduction_implicit(SPRAY_COND_OPERATOR)", "ms_per_application": 1e3 * t_o,
                                    "pair_interactions_per_s": 2 * pairs["apply"] / t_o,
                                    "flop_roofline_frac": 2 * pairs["apply"] * fa / t_o / (fp64_meas * 1e12),
                                    "note": "two symmetric frozen sweeps (ions, electrons) + per-particle form/combine kernels"}}
        del u_g, T_g, T_e, k_i, k_e, kei, tau, u_e

    # ---- row N3: continuity equation with the KGC filter (spray_kgc_continuity), same lists; 60 flops per in-support ordered pair
    #      over N_gather (distance 9, sqrt + 1/r + F 12, grad W and V_b 6, moment matrix 12, v_ab 3, velocity moments 18)
    n3 = None
    if not args.no_n1:
        for _ in range(2):
            sp.kgc_continuity(d["m"], out["rho"], d["vx"], d["vy"], d["vz"], want_L=False, want_raw=False)
        torch.cuda.synchronize()
        r0, r1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        nrep = 5
        r0.record()
        for _ in range(nrep):
            sp.kgc_continuity(d["m"], out["rho"], d["vx"], d["vy"], d["vz"], want_L=False, want_raw=False)
        r1.record()
        torch.cuda.synchronize()
        t_k = r0.elapsed_time(r1) * 1e-3 / nrep
        n3 = {"call": "spray_kgc_continuity", "ms_per_call": 1e3 * t_k, "pair_interactions_per_s": pairs["limiter"] / t_k,
              "flops_per_pair": 60, "flop_roofline_frac": pairs["limiter"] * 60 / t_k / (fp64_meas * 1e12)}

    # ---- row N4: mesh-free laser ray tracing and deposition (spray_ray_deposit) on the same particle set and cell table: a beam
    #      of 65 536 rays entering at the low-z face with a small divergence, 128 steps of one lattice spacing; f = n_e/n_c
    #      proportional to rho (0.8 in the densest fluid), kib proportional to f^2.  Counted: ray steps, and in-support
    #      ray-particle interactions (neighbour count of a particle = particles within 2h = interactions per ray step, uniform h).
    n4 = None
    if not args.no_n1:
        nr, nst = 65536, 128
        gen = torch.Generator(device=dev); gen.manual_seed(1234)
        lo = [float(v) for v in w.grid.lo]
        Lb = [float(b) - float(a) for a, b in zip(w.grid.lo, w.grid.hi)]
        u = torch.rand((5, nr), generator=gen, device=dev, dtype=f64)
        rays = torch.stack([lo[0] + Lb[0] * u[0], lo[1] + Lb[1] * u[1], torch.full((nr,), lo[2] + 0.05 * Lb[2], dtype=f64, device=dev),
                            0.1 * (u[2] - 0.5), 0.1 * (u[3] - 0.5), torch.ones(nr, dtype=f64, device=dev), 1.0 + u[4]]).contiguous()
        fq = 0.8 * out["rho"] / out["rho"].max()
        kib = 20.0 * (0.05 + fq * fq)
        dt_ray = Lb[2] / round(n ** (1.0 / 3.0))
        sp.ray_deposit(d["m"], out["rho"], fq, kib, rays, dt_ray, 4, c_light=1.0, want_gradn=False)
        torch.cuda.synchronize()
        r0, r1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        r0.record()
        rr = sp.ray_deposit(d["m"], out["rho"], fq, kib, rays, dt_ray, nst, c_light=1.0, want_gradn=False)
        r1.record()
        torch.cuda.synchronize()
        t_r = r0.elapsed_time(r1) * 1e-3
        # the same call without rays: the gradient sweep over all particles (prologue + SW_GRADN) and the deposit scatter alone
        g0, g1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        norays = rays[:, :0].contiguous()
        sp.ray_deposit(d["m"], out["rho"], fq, kib, norays, dt_ray, nst, c_light=1.0, want_gradn=False)   # untimed: allocator warm-up
        torch.cuda.synchronize()
        g0.record()
        for _ in range(3):
            sp.ray_deposit(d["m"], out["rho"], fq, kib, norays, dt_ray, nst, c_light=1.0, want_gradn=False)
        g1.record()
        torch.cuda.synchronize()
        t_g = g0.elapsed_time(g1) * 1e-3 / 3
        steps_taken = int(rr["steps"].sum().item())
        nb_mean = pairs["limiter"] / n + 1.0
        n4 = {"call": "spray_ray_deposit", "rays": nr, "max_steps": nst, "ray_steps": steps_taken, "ms_per_call": 1e3 * t_r,
              "ms_gradient_sweep_and_scatter": 1e3 * t_g, "ms_ray_kernel": 1e3 * (t_r - t_g),
              "ray_steps_per_s": steps_taken / t_r, "ray_particle_interactions_per_s": steps_taken * nb_mean / t_r,
              "energy_balance_rel": float(abs(rr["edep"].sum() + rr["rays"][6].sum() - rays[6].sum()) / rays[6].sum()),
              "absorbed_fraction": float(rr["edep"].sum() / rays[6].sum()),
              "note": "includes the gradient sweep over all particles (prologue + SW_GRADN) and the deposit scatter"}

    # ---- variant of SURVEY 8(d) config 5: the same particle set with v ~ N(0, 0.01^2), so that about half of the pairs take the
    #      viscous branch of eqs. (41)-(43); same pass, timed the same way (headline stays the literal v = 0 config)
    variants = None
    if w.name.startswith("c5") and not (np.any(w.vx) or np.any(w.vy) or np.any(w.vz)) and not args.no_variants and not args.no_n1:
        wv = W.make("c5_v")
        dv = dict(d)
        for f in ("vx", "vy", "vz"):
            dv[f] = torch.from_numpy(np.ascontiguousarray(getattr(wv, f))).to(dev)
        for _ in range(3):
            one_pass(dv)
        torch.cuda.synchronize()
        v0, v1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        nv = max(3, min(args.steps, 10))
        v0.record()
        for _ in range(nv):
            one_pass(dv)
        v1.record()
        torch.cuda.synchronize()
        t_v = v0.elapsed_time(v1) * 1e-3 / nv
        fv = approaching_fraction("c5_v")
        flv = FLOPS[w.kernel]
        flops_v = (pairs["density"] * flv["density"] + pairs["hydro"] * (flv["hydro"] + fv * flv["hydro_visc"]) +
                   pairs["limiter"] * flv["limiter"] + pairs["apply"] * flv["apply"])
        variants = {"c5_v": {"workload": wv.name, "ms_per_pass": 1e3 * t_v, "pair_interactions_per_s": p_pass / t_v,
                             "approaching_pair_fraction": fv, "flops": flops_v, "frac": flops_v / (fp64_meas * 1e12) / t_v,
                             "note": "v ~ N(0, 0.01^2): the +25-flop viscous term weighted by the measured fraction of approaching pairs"}}
        del wv, dv

    # ---- roofline.  Top level = the WHOLE PASS, the quantity BASELINE.json's north_star targets;
    #      `kernels` lists every part of the pass with its measured time, share, algorithmic work and fraction of its own bound.
    fl = FLOPS[w.kernel]
    moving = bool(np.any(w.vx) or np.any(w.vy) or np.any(w.vz))
    visc_frac = approaching_fraction(args.workload) if moving else 0.0
    flops = {"density": pairs["density"] * fl["density"], "hydro": pairs["hydro"] * (fl["hydro"] + visc_frac * fl["hydro_visc"]),
             "limiter": pairs["limiter"] * fl["limiter"], "apply": pairs["apply"] * fl["apply"]}
    seg_mean = seg.mean(axis=0)
    t_step = t_total / args.steps
    t_alu = sum(flops.values()) / (fp64_meas * 1e12)
    t_hbm = BYTES_PER_PARTICLE * n / (pk["hbm_gbs"] * 1e9)
    calls = {"build": seg_mean[0], "density": seg_mean[1], "hydro": seg_mean[2], "fld": seg_mean[3]}
    hyd_flops = flops["hydro"] + (flops["limiter"] if fused else 0.0)
    fld_flops = flops["apply"] + (0.0 if fused else flops["limiter"])
    # parts of spray_build_cells from the events the call records on its stream (spray_build_timing), a few extra passes
    bt = np.zeros(3)
    for _ in range(3):
        sp.build_cells(w.grid, w.kernel, d["x"], d["y"], d["z"], d["h"])
        bt += np.array(sp.build_timing())
    bt *= 1e-3 / 3
    hbm = pk["hbm_gbs"] * 1e9
    pk64 = fp64_meas * 1e12
    b_cells = (32 + 48 + 64) * n                       # keys, three sort passes, reorder
    b_lists = (2 * 32 + 2 * (pairs["hydro"] / max(n, 1))) * n      # candidates read once per tile row (32 B twice) + 2 B per neighbour written
    tr = traffic_table(w.name)
    def part(name, kernel, sec, bound, work, peak, extra=None):
        e = {"part": name, "kernel": kernel, "ms": 1e3 * float(sec), "share": float(sec) / t_step, "bound": bound,
             "algorithmic": work, "unit": "flop" if bound == "alu" else "B",
             "frac": (work / max(float(sec), 1e-12)) / peak if work else 0.0, "traffic": tr.get(kernel)}
        if extra:
            e.update(extra)
        return e
    kernels = [
        part("cell list (a1-a4)", "k_cell_key..k_ref_sweep<4>", bt[0], "hbm", b_cells, hbm),
        part("tiles + tables", "k_mark_coincident..k_tile_tables", bt[1], "hbm", 0, hbm, {"note": "index work only"}),
        part("neighbour lists", "k_build_lists", bt[2], "hbm", b_lists, hbm,
             {"note": "a search: zero algorithmic flops; bound in practice by shared-memory wavefronts and issue (profiles/r02*)"}),
        part("density (a5)", "k_prep_density + k_tiled_sweep<0>", calls["density"], "alu", flops["density"], pk64),
        part("hydro + limiter (a6, a7)" if fused else "hydro (a6)", "k_prep_hydro + k_tiled_sweep<10>" if fused else "k_prep_hydro + k_tiled_sweep<1>",
             calls["hydro"], "alu", hyd_flops, pk64),
        part("apply (a8)" if fused else "limiter + apply (a7, a8)", "k_prep_fld + k_tiled_sweep<3>", calls["fld"], "alu", fld_flops, pk64),
    ]
    dom = max(kernels, key=lambda e: e["ms"])
    roofline = {"bound": "alu", "kernel": "whole pass (density + hydro + FLD incl. the cell-list and neighbour-list build): north_star's target quantity",
                "achieved": sum(flops.values()) / t_step / 1e12, "peak": fp64_meas, "unit": "TFLOP/s",
                "frac": max(t_alu, t_hbm) / t_step,
                "peak_source": "DFMA-chain probe measured in this run (spray_fp64_peak_probe); nominal 148x64x2x1.965GHz = %.1f" % FP64_NOMINAL_TFLOPS,
                "traffic": dom["traffic"], "dominant": dom["part"] + " (" + dom["kernel"] + ")",
                "kernels": kernels,
                "pass": {"flops": sum(flops.values()), "bytes": BYTES_PER_PARTICLE * n, "t_alu_ms": 1e3 * t_alu, "t_hbm_ms": 1e3 * t_hbm,
                         "t_pass_ms": 1e3 * t_step, "frac": max(t_alu, t_hbm) / t_step, "hbm_peak_gbs": pk["hbm_gbs"], "hbm_peak_source": pk_src,
                         "approaching_pair_fraction": visc_frac},
                "per_call_ms": {k: 1e3 * float(v) for k, v in calls.items()},
                "per_call_tflops": {"density": flops["density"] / calls["density"] / 1e12, "hydro": hyd_flops / calls["hydro"] / 1e12,
                                    "fld": fld_flops / calls["fld"] / 1e12},
                "calls": (["spray_build_cells", "spray_density", "spray_hydro_rhs_limiter", "spray_fld_apply(FROZEN_CHAINED)"] if fused else
                          ["spray_build_cells", "spray_density", "spray_hydro_rhs", "spray_fld_apply(UPDATE_LIMITER)"])}

    cpu = None
    if not args.no_cpu_baseline:
        import oracle as O
        rng = np.random.default_rng(0)
        ns = min(n, args.cpu_sample)
        targets = np.sort(rng.choice(n, size=ns, replace=False)).astype(np.int64)
        dt, pr = oracle_sample_pass(w, targets)
        # the same oracle on ONE thread, on a sample sized for ~10 s (single thread and all hardware threads)
        nthr = O.num_threads()
        ns1 = max(1, min(ns, int(ns * 10.0 / max(dt * nthr, 1e-9))))
        O.set_threads(1)
        dt1, pr1 = oracle_sample_pass(w, targets[:: max(1, ns // ns1)][:ns1])
        O.set_threads(nthr)
        cpu = {"value": pr / dt, "unit": UNIT, "cores": nthr, "kind": "oracle", "seconds": dt,
               "sample": f"{ns} of {n} target particles of {w.name} (all their neighbours), oracle cell-list variant, long-double sums",
               "single_thread": {"value": pr1 / dt1, "unit": UNIT, "seconds": dt1, "targets": int(min(ns1, ns))},
               "cpu_model": cpu_model(),
               "note": "the oracle is a parity checker (x87 long-double sums, -O2 -ffp-contract=off, normaliser sums), not a tuned CPU code: "
                       "GPU/oracle ratios are ratios against a checker"}

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": 1e3 * t_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic",
            "config": {"workload": w.name, "n_particles": n, "kernel": ["cubic_spline", "wendland_c2"][w.kernel], "grid": list(w.grid.ncell),
                       "pairs_per_pass": p_pass, "unique_ordered_pairs": cs, "unique_pairs_per_s": world * cs * args.steps / t_total,
                       "l2": "inputs larger than L2 (%.1f GB of caller arrays + %.1f GB of library scratch resident per replica)"
                             % (8e-9 * n * (len(fields) + len(out)), 1e-9 * pstats["scratch_bytes"]),
                       "scratch_bytes": pstats["scratch_bytes"], "declined": pstats["declined"], "level_edges": levels,
                       "parallelism": "replicas only" if world > 1 else "1 GPU", "path": args.path,
                       "tiles": n_tiles, "tiled_fraction": n_fast / max(n, 1)},
            "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline, "cpu_baseline": cpu,
            "fp64_probe_tflops": fp64_meas, "variants": variants, "next_rows": {"N1_rad_jacobi": n1, "N2_conduction": n2, "N3_kgc_continuity": n3, "N4_ray_deposit": n4}}
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
