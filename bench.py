#!/usr/bin/env python
"""bench.py -- throughput of the ADI time step (all S0-S9 rows of DESIGN.md) on BASELINE.json config 3.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl b200|reference]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N ... bench.py --gpus N ...

A "step" is one tf_step (b^n, then pseudo-Newton iterations of y-sweep + x-sweep + residual until
res < tol) on the 8192x8192 spinodal film of config 3.  value = grid points x steps / seconds over all
ranks (weak scaling: every rank advances its own 8192^2 replica; the path has no exchange step on one
GPU).  Prints ONE JSON line on rank 0.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_1806_10550_b200 import inputs  # noqa: E402

METRIC = "grid-point ADI steps/sec (fp64)"
UNIT = "grid-point-steps/s"
# algorithmic HBM bytes per grid point per launch
ALG_BYTES = {"y_forward": 40, "y_backward": 32, "x_forward": 40, "x_backward_update": 40}


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--config", type=int, default=3, help="BASELINE.json config index; 3 is the headline, 4 the isolated solver (side measurement)")
    ap.add_argument("--fixed-iters", type=int, default=0, help="fixed Newton count per step (0: converge to tol)")
    ap.add_argument("--pressure", default="power", choices=["power", "nlc"],
                    help="power: BASELINE.json's Pi (headline); nlc: the paper's NLC pressure (1.8)-(1.9) with (1.11), on the "
                         "same grid with the paper's spacing 0.05 and a 0.2 film (side measurement, row f-1)")
    ap.add_argument("--nsys", type=int, default=0, help="config 4 only: number of systems (0: the config's 16384)")
    ap.add_argument("--variant", default="lu", choices=["lu", "partition", "pcr"],
                    help="config 4 only: tf_penta_solve_ex variant (pcr: parallel cyclic reduction, systems along rows, length <= 2048)")
    ap.add_argument("--length", type=int, default=0, help="config 4 only: unknowns per system (0: the config's 16384)")
    ap.add_argument("--nparts", type=int, default=0, help="config 4 only: chunks per system of the partition variant (0: automatic)")
    ap.add_argument("--cusparse", action="store_true", help="config 4 only: also time cuSPARSE's interleaved-batch routine (context)")
    ap.add_argument("--slabs", action="store_true",
                    help="config 4 only: every system spread over the ranks (paper_1806_10550_b200/dist.py: one NCCL "
                         "all-gather of the interface values); strong scaling, launch with torchrun for --gpus N > 1")
    ap.add_argument("--distributed", action="store_true",
                    help="ONE film spread over the ranks (paper_1806_10550_b200/dist_step.py: two all-to-alls and one "
                         "all-reduce per Newton iteration) instead of one replica per rank; strong scaling")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-side", action="store_true", help="skip the short side measurements of configs 0, 1, 2 and 4")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    return ap.parse_args()


class ClockSampler:
    """nvidia-smi clocks / throttle reasons of one GPU every 200 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows, self.proc = [], None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), [t.strip() for t in line.split(",")]))

    def stop(self, t0, t1):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        self.th.join(timeout=2)
        rows = [r for t, r in self.rows if t0 <= t <= t1 and len(r) >= 7] or [r for _, r in self.rows if len(r) >= 7]
        if not rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        sm = sorted(float(r[0]) for r in rows)
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for k, n in enumerate(names) if any(r[3 + k].lower().startswith("active") for r in rows)]
        pw = [float(r[2]) for r in rows if r[2].replace(".", "", 1).isdigit()]
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": float(rows[0][1]), "reasons": reasons,
                "samples": len(rows), "power_w_max": max(pw) if pw else None}


def measured_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


NCU_SUMMARY = os.path.join("profiles", "r03_ncu_full_summary.csv")
NCU_KERNEL = {"y_forward": "yfwd_ws_kernel", "y_backward": "ybwd2_tma_kernel", "x_forward": "xfwd_ws_kernel",
              "x_backward_update": "xbwd2_tma_kernel"}


def ncu_traffic(kernel):
    """dram__bytes_read.sum + dram__bytes_write.sum of one launch of `kernel` at 8192^2, from the committed
    ncu --set full summary (profiles/r02_ncu.md names the command), or None."""
    import csv
    p = os.path.join(ROOT, NCU_SUMMARY)
    try:
        for row in csv.DictReader(open(p)):
            if row["kernel"].startswith(NCU_KERNEL[kernel]):
                return int(round((float(row["dram_read_GB"]) + float(row["dram_write_GB"])) * 1e9))
    except (OSError, KeyError, ValueError):
        return None
    return None


def ncu_fp64_thread_instructions(kernel):
    """fp64-pipe instructions of one launch of `kernel` at 8192^2, per thread: smsp__inst_executed_pipe_fp64.sum (warp
    instructions) x 32 lanes, from the same committed summary, or None."""
    import csv
    try:
        for row in csv.DictReader(open(os.path.join(ROOT, NCU_SUMMARY))):
            if row["kernel"].startswith(NCU_KERNEL[kernel]):
                return 32 * int(float(row["fp64_warp_inst"]))
    except (OSError, KeyError, ValueError):
        return None
    return None


# ----------------------------------------------------------------------------------------- CPU oracle legs
def oracle_sample_run(cfg, n, steps, warmup, fixed_iters, omp=False):
    """Times the CPU oracle AS IT STANDS (serial build; omp=True: its OpenMP build, one thread per line) on an
    n x n cut of the config's recipe."""
    from oracle import tfo
    o = tfo.ThinFilmOracle(n, n, cfg["dx"], cfg["dy"], cfg["kappa"], cfg["hstar"], cfg["n"], cfg["m"], omp=omp)
    o.set_newton(cfg["tol"], cfg["max_iter"], fixed_iters)
    o.set_state(inputs.initial_condition(cfg, n, n))
    for _ in range(warmup):
        o.step(cfg["dt"])
    t0 = time.perf_counter()
    iters = 0
    for _ in range(steps):
        st, it, _ = o.step(cfg["dt"])
        iters += it
    dt = time.perf_counter() - t0
    return dict(seconds=dt, iters=iters, pts=n * n, steps=steps, cores=tfo.num_threads(omp))


def run_reference(args, cfg):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    n = min(1024 if (args.steps + args.warmup) <= 30 else 512, cfg["nx"], cfg["ny"])
    r = oracle_sample_run(cfg, n, args.steps, args.warmup, args.fixed_iters)
    value = r["pts"] * r["steps"] / r["seconds"]
    sample = f"{n}x{n} cut of {cfg['name']} (same dx, dt, IC recipe and seed), {args.steps} steps after {args.warmup} warm-up"
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * r["seconds"] / r["steps"],
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": cfg["name"], "grid": [cfg["nx"], cfg["ny"]], "dt": cfg["dt"], "tol": cfg["tol"],
                   "note": "CPU oracle (oracle/tfo.c, serial, untuned) on a bounded sample; size-independent unit"},
        "newton_iters_total": r["iters"],
        "point_iterations_per_s": r["pts"] * r["iters"] / r["seconds"],
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": r["cores"], "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


# ----------------------------------------------------------------------------------------- multi-rank bookkeeping
def max_over_ranks(seconds, world, device):
    """The job's time is the slowest rank's device time (replicas: no data-path collective)."""
    if world <= 1:
        return float(seconds)
    import torch
    import torch.distributed as dist
    t = torch.tensor([seconds], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(npts, steps, world, seconds):
    """grid-point steps per second over all ranks: every rank advances its own npts-point film `steps` times."""
    return world * npts * steps / seconds


# ----------------------------------------------------------------------------------------- side measurements
def side_measurements():
    """Short runs of the other BASELINE.json configs (parity-test cases, not the headline), so that the driver's own
    bench run records them: ms per step and per Newton iteration of configs 0 and 1 (fixed dt, 50 steps after 30),
    config 2 (40 accepted adaptive steps, decisions on the device), and the isolated solver of config 4."""
    import torch
    from paper_1806_10550_b200 import tf
    out = {}

    def timed(fn):
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        ev0.record()
        r = fn()
        ev1.record()
        torch.cuda.synchronize()
        return ev0.elapsed_time(ev1), r

    for idx in (0, 1):
        cfg = inputs.config(idx)
        g = tf.ThinFilm(cfg["nx"], cfg["ny"], cfg["dx"], cfg["dy"], cfg["kappa"], cfg["hstar"], cfg["n"], cfg["m"])
        g.set_newton(cfg["tol"], cfg["max_iter"], 0)
        g.set_state(torch.from_numpy(inputs.initial_condition(cfg)).cuda())
        for _ in range(30):
            g.step(cfg["dt"])
        ms, its = timed(lambda: sum(g.step(cfg["dt"])[1] for _ in range(50)))
        out[cfg["name"]] = {"ms_per_step": ms / 50, "newton_iters_per_step": its / 50, "ms_per_iteration": ms / its,
                            "grid_point_steps_per_s": cfg["nx"] * cfg["ny"] * 50 / (ms * 1e-3), "graph_replays": g.graph_replays(),
                            "note": "steps 31-80 of the config's run (L2-resident: time to solution, no roofline)"}
        g.close()
    cfg = inputs.config(2)
    g = tf.ThinFilm(cfg["nx"], cfg["ny"], cfg["dx"], cfg["dy"], cfg["kappa"], cfg["hstar"], cfg["n"], cfg["m"])
    g.set_newton(cfg["tol"], cfg["max_iter"], 0)
    h2 = torch.from_numpy(inputs.initial_condition(cfg)).cuda()
    for dev in (False, True):
        g.set_state(h2)
        ms, r = timed(lambda: tf.advance_adaptive(g, cfg["dt"], 40, cfg["grow"], cfg["shrink"], cfg["dt_max"], cfg["dt_min"],
                                                  on_device=dev))
        its = sum(x[2] for x in r[2])
        out[cfg["name"] + ("_device_controller" if dev else "_host_controller")] = {
            "ms_per_accepted_step": ms / 40, "attempts": len(r[2]), "newton_iters_total": its, "ms_per_iteration": ms / its,
            "point_iterations_per_s": cfg["nx"] * cfg["ny"] * its / (ms * 1e-3)}
    g.close()
    del h2
    cfg = inputs.config(4)
    n = cfg["nrow"]
    gen = torch.Generator(device="cuda").manual_seed(cfg["seed"])
    peak, _ = measured_peak()
    for direction, name in ((1, "columns_y"), (0, "rows_x")):
        U = lambda lo, hi: torch.rand(n, n, dtype=torch.float64, device="cuda", generator=gen) * (hi - lo) + lo
        e, c, a, b, y = U(-1, 1), U(-1, 1), U(-1, 1), U(-1, 1), U(-1, 1)
        d = 1 + e.abs() + c.abs() + a.abs() + b.abs() + U(0, 1)
        ws = torch.empty(tf.lib().tf_penta_workspace_bytes(n, n), dtype=torch.uint8, device="cuda")
        x = torch.empty_like(e)
        solve = lambda: tf.penta_solve(direction, e, c, d, a, b, y, out=x, workspace=ws)
        for _ in range(3):
            solve()
        ms, _ = timed(lambda: [solve() for _ in range(5)])
        ms /= 5
        out[cfg["name"] + "_" + name] = {"ms": ms, "unknowns_per_s": n * n / (ms * 1e-3), "alg_bytes_per_unknown": 104,
                                         "alg_gbs": 104 * n * n / (ms * 1e-3) / 1e9, "frac_of_peak": 104 * n * n / (ms * 1e-3) / 1e9 / peak}
        del e, c, a, b, y, d, ws, x
    torch.cuda.empty_cache()
    return out


# ----------------------------------------------------------------------------------------- B200 arm
def run_b200(args, cfg):
    import torch
    import torch.distributed as dist
    from paper_1806_10550_b200 import tf

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py --impl b200 needs a CUDA device (no CPU fallback)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    nx, ny, dt = cfg["nx"], cfg["ny"], cfg["dt"]
    npts = nx * ny
    if args.pressure == "nlc":
        # the paper's own model and scales (PAPER.md:99-105 (1.11), 453: spacing 0.05), film 0.2 (1 + 0.01 U[-1,1])
        cfg = dict(cfg, dx=0.05, dy=0.05, name=cfg["name"] + "_nlc")
        dt = 1e-3
        h_host = torch.from_numpy(0.2 * inputs.noise_ic(nx, ny, cfg["seed"])).pin_memory()
    else:
        h_host = torch.from_numpy(inputs.initial_condition(cfg)).pin_memory()     # every rank: its own replica
    h_dev = h_host.cuda(non_blocking=True)
    ctx = tf.ThinFilm(nx, ny, cfg["dx"], cfg["dy"], cfg["kappa"], cfg["hstar"], cfg["n"], cfg["m"])
    if args.pressure == "nlc":
        ctx.set_pressure(tf.PI_NLC, (0.0857, 1.0 / 0.0857, 36.0, 0.01, 1.67, 1.0, 0.05))
    ctx.set_newton(cfg["tol"], cfg["max_iter"], args.fixed_iters)

    def timed_run(e2e, profile=True):
        """W warm-up + K timed steps from the initial condition; returns (seconds, iters, launches, t0, t1)."""
        ctx.set_state(h_dev)
        hbuf = h_host.clone().pin_memory() if e2e else None

        def one():
            if e2e:
                ctx.set_state(hbuf)              # H2D of the step's input from pinned host memory
            st, it, res = ctx.step(dt)
            if st != tf.OK:
                raise SystemExit(f"tf_step did not converge (status {st}, iters {it}, res {res})")
            if e2e:
                ctx.get_state(hbuf)              # D2H of the step's result
            return it

        for _ in range(args.warmup):
            one()
        ctx.set_profiling(profile and not e2e)
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        l0, w0 = tf.kernel_launches(), time.time()
        ev0.record()
        iters = sum(one() for _ in range(args.steps))
        ev1.record()
        barrier()
        w1 = time.time()
        sec = ev0.elapsed_time(ev1) / 1e3
        sec = max_over_ranks(sec, world, "cuda")
        return sec, iters, tf.kernel_launches() - l0, w0, w1

    fp64_burst = tf.fp64_peak(5)[0] if rank == 0 else None          # DFMA micro-benchmark on the cool GPU, best of 5
    sampler = ClockSampler(local) if rank == 0 else None
    sec, iters, launches, w0, w1 = timed_run(e2e=False)
    fp64_hot = tf.fp64_peak(5)[1] if rank == 0 else None            # ... and right behind the timed steps, mean of 5
    clocks = sampler.stop(w0, w1) if sampler else None
    prof = ctx.get_profile()
    # the same run without the per-kernel CUDA events (5 event records per iteration) and with graph replay allowed
    usec, uiters, _, _, _ = timed_run(e2e=False, profile=False)
    mass_drift = None
    if rank == 0:
        m1 = ctx.mass()
        m0 = float(h_host.sum(dtype=torch.float64).item()) * cfg["dx"] * cfg["dy"]
        mass_drift = abs(m1 - m0) / m0
    e2e = None
    if not args.no_e2e:
        esec, eiters, _, _, _ = timed_run(e2e=True)
        e2e = {"value": whole_job_value(npts, args.steps, world, esec), "unit": UNIT, "h2d_bytes_per_step": npts * 8,
               "d2h_bytes_per_step": npts * 8, "ms_per_step": 1e3 * esec / args.steps, "newton_iters_total": eiters}
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    peak, peak_src = measured_peak()
    kern = {}
    for name, (ms, n) in prof.items():
        if n:
            avg = ms / n
            kern[name] = {"avg_ms": avg, "launches": n, "alg_bytes_per_launch": ALG_BYTES[name] * npts,
                          "alg_gbs": ALG_BYTES[name] * npts / (avg * 1e-3) / 1e9}
    dom = max(kern, key=lambda k: kern[k]["avg_ms"] * kern[k]["launches"]) if kern else None
    roofline = None
    if dom:
        # two ceilings for the dominant kernel: HBM (algorithmic bytes against the measured copy peak) and the fp64 pipe
        # (fp64 instructions of one launch, counted by ncu, against the DFMA rate measured behind the timed steps);
        # `roofline` is the one the kernel is nearer to, the other one rides along as `roofline.other`
        a = kern[dom]["alg_gbs"]
        hbm = {"bound": "hbm", "kernel": dom, "achieved": a, "peak": peak, "unit": "GB/s", "frac": a / peak,
               "peak_source": peak_src, "traffic": ncu_traffic(dom) if (nx, ny) == (8192, 8192) else None,
               "traffic_source": NCU_SUMMARY,
               "alg_bytes_per_launch": kern[dom]["alg_bytes_per_launch"], "avg_launch_ms": kern[dom]["avg_ms"]}
        inst = ncu_fp64_thread_instructions(dom) if (nx, ny) == (8192, 8192) and args.pressure == "power" else None
        alu = None
        if inst and fp64_hot:
            ach = inst / (kern[dom]["avg_ms"] * 1e-3) / 1e12
            alu = {"bound": "alu", "kernel": dom, "achieved": ach, "peak": fp64_hot / 1e12, "unit": "T fp64 thread-instructions/s",
                   "frac": ach / (fp64_hot / 1e12), "traffic": None,
                   "peak_source": "tf_fp64_peak (DFMA micro-benchmark of this library) right behind the timed steps, mean of 5 launches",
                   "peak_burst": fp64_burst / 1e12, "peak_nominal": "148 SMs x 64 DFMA lanes x 1.965 GHz = 18.6",
                   "fp64_thread_instructions_per_launch": inst, "instructions_source": NCU_SUMMARY,
                   "avg_launch_ms": kern[dom]["avg_ms"]}
        roofline = dict(alu, other=hbm) if alu and alu["frac"] > hbm["frac"] else dict(hbm, other=alu)
    ksum = sum(k["avg_ms"] * k["launches"] for k in kern.values())
    line = {
        "metric": METRIC, "value": whole_job_value(npts, args.steps, world, sec), "unit": UNIT, "n_gpus": world,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * sec / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": cfg["name"], "grid": [nx, ny], "dx": cfg["dx"], "dt": dt, "tol": cfg["tol"],
                   "max_iter": cfg["max_iter"], "fixed_iters": args.fixed_iters, "pressure": args.pressure,
                   "ic": "1 + 0.01 U[-1,1] seeded noise", "parallelism": f"replicas x{world} (no exchange step)",
                   "l2": "working set 7 fields x 512 MiB >> 126 MB L2: every launch streams from HBM, no flush needed"},
        "newton_iters_total": iters, "newton_iters_per_step": iters / args.steps,
        "point_iterations_per_s": world * npts * iters / sec,
        "penta_unknowns_per_s": 2 * world * npts * iters / sec,
        "iteration_model": {"bytes_per_point_iter": 152, "gbs": 152 * npts * iters / sec / 1e9,
                            "frac_of_peak": 152 * npts * iters / sec / 1e9 / peak,
                            "compulsory_48B_gbs": 48 * npts * iters / sec / 1e9,
                            "compulsory_48B_frac_of_peak": 48 * npts * iters / sec / 1e9 / peak},
        "unprofiled": {"value": whole_job_value(npts, args.steps, world, usec), "ms_per_step": 1e3 * usec / args.steps,
                       "newton_iters_total": uiters,
                       "note": "same steps timed again without the per-kernel CUDA events of the headline run"},
        "kernels": kern, "kernel_time_share_of_step": ksum / (sec * 1e3) if kern else None,
        "roofline": roofline, "clocks": clocks, "e2e": e2e, "gpu_launches": launches,
        "mass_rel_drift": mass_drift,
    }
    if world == 1 and not args.no_side and args.pressure == "power" and (nx, ny) == (8192, 8192):
        ctx.close()
        del h_dev
        torch.cuda.empty_cache()
        try:
            line["side"] = side_measurements()
        except Exception as exc:                         # a side measurement must never cost the headline line
            line["side"] = {"error": repr(exc)}
    if world == 1 and not args.no_cpu_baseline and args.pressure == "power":
        n = 2048 if min(nx, ny) >= 2048 else min(nx, ny)
        r = oracle_sample_run(cfg, n, 1, 0, args.fixed_iters)
        line["cpu_baseline"] = {
            "value": r["pts"] * r["steps"] / r["seconds"], "unit": UNIT, "cores": r["cores"], "kind": "oracle",
            "sample": f"{n}x{n} cut of {cfg['name']} (same dx, dt, IC recipe, seed), first step, {r['iters']} Newton "
                      f"iterations, {r['seconds']:.1f} s",
            "point_iterations_per_s": r["pts"] * r["iters"] / r["seconds"]}
        r = oracle_sample_run(cfg, n, 1, 0, args.fixed_iters, omp=True)      # same sample, the oracle's OpenMP build
        line["cpu_baseline_all_cores"] = {
            "value": r["pts"] * r["steps"] / r["seconds"], "unit": UNIT, "cores": r["cores"], "kind": "oracle (OpenMP build)",
            "sample": f"{n}x{n} cut, first step, {r['iters']} Newton iterations, {r['seconds']:.1f} s",
            "point_iterations_per_s": r["pts"] * r["iters"] / r["seconds"]}
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


# ----------------------------------------------------------------------------------------- vendor library, context only
def cusparse_gpsv_interleaved(e, c, d, a, b, y, steps):
    """cuSPARSE's interleaved-batch pentadiagonal solver (cusparseDgpsvInterleavedBatch, algo 0) on the column layout
    ([len][nsys] = element i of system j at i*nsys + j, exactly its "interleaved" format).  Context for config 4
    (SURVEY.md 8(d)): a library call, not part of the product path.  The routine overwrites its inputs, so every timed
    call gets fresh copies made outside the timed region.  Returns (mean ms, solution of the last call) or None."""
    import ctypes
    import glob
    import torch
    libs = glob.glob(os.path.join(os.path.dirname(torch.__file__), "..", "nvidia", "cusparse", "lib", "libcusparse.so*")) + \
        glob.glob("/usr/local/cuda/lib64/libcusparse.so*")
    if not libs:
        return None
    L = ctypes.CDLL(libs[0])
    vp, ci = ctypes.c_void_p, ctypes.c_int
    L.cusparseCreate.argtypes = [ctypes.POINTER(vp)]
    L.cusparseSetStream.argtypes = [vp, vp]
    L.cusparseDgpsvInterleavedBatch_bufferSizeExt.argtypes = [vp, ci, ci] + [vp] * 6 + [ci, ctypes.POINTER(ctypes.c_size_t)]
    L.cusparseDgpsvInterleavedBatch.argtypes = [vp, ci, ci] + [vp] * 6 + [ci, vp]
    L.cusparseDestroy.argtypes = [vp]
    h = vp()
    if L.cusparseCreate(ctypes.byref(h)) != 0:
        return None
    L.cusparseSetStream(h, vp(torch.cuda.current_stream().cuda_stream))
    m, nsys = e.shape

    def fresh():
        ts = [t.clone() for t in (e, c, d, a, b, y)]
        ts[0][:2] = 0.0; ts[1][:1] = 0.0; ts[3][-1:] = 0.0; ts[4][-2:] = 0.0     # the routine wants the outside entries zero
        return ts
    ts = fresh()
    size = ctypes.c_size_t(0)
    if L.cusparseDgpsvInterleavedBatch_bufferSizeExt(h, 0, m, *[t.data_ptr() for t in ts], nsys, ctypes.byref(size)) != 0:
        L.cusparseDestroy(h)
        return None
    buf = torch.empty(max(size.value, 8), dtype=torch.uint8, device="cuda")
    total, x = 0.0, None
    for k in range(steps + 1):                      # first call untimed
        if k:
            ts = fresh()
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ev0.record()
        rc = L.cusparseDgpsvInterleavedBatch(h, 0, m, *[t.data_ptr() for t in ts], nsys, buf.data_ptr())
        ev1.record()
        torch.cuda.synchronize()
        if rc != 0:
            L.cusparseDestroy(h)
            return None
        if k:
            total += ev0.elapsed_time(ev1)
        x = ts[5]
    L.cusparseDestroy(h)
    return total / steps, x


# ----------------------------------------------------------------------------------------- config 4 (side measurement)
def run_distributed(args, cfg):
    """The headline workload as ONE film over all ranks: strong scaling, max over ranks."""
    import torch
    import torch.distributed as dist
    from paper_1806_10550_b200 import dist_step as ds
    rank, world = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))
    torch.cuda.set_device(int(os.environ.get("LOCAL_RANK", "0")))
    own_group = not dist.is_initialized()
    if own_group:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29532")
        dist.init_process_group("nccl", rank=rank, world_size=world)
    nx, ny, dt = cfg["nx"], cfg["ny"], cfg["dt"]
    f = ds.DistributedFilm(nx, ny, cfg["dx"], cfg["dy"], cfg["kappa"], cfg["hstar"], cfg["n"], cfg["m"], tol=cfg["tol"],
                           max_iter=cfg["max_iter"])
    j0, j1 = f.lay.rows[rank]
    f.set_state_rows(inputs.initial_condition(cfg)[j0:j1].copy())
    for _ in range(args.warmup):
        f.step(dt)
    dist.barrier()
    torch.cuda.synchronize()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record()
    iters = 0
    for _ in range(args.steps):
        st, k, _ = f.step(dt)
        iters += k
    ev1.record()
    torch.cuda.synchronize()
    dist.barrier()
    sec = max_over_ranks(ev0.elapsed_time(ev1) * 1e-3, world, "cuda")
    if rank == 0:
        print(json.dumps({"metric": "grid-point ADI steps/sec (fp64)", "value": nx * ny * args.steps / sec,
                          "unit": "grid-point-steps/s", "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
                          "ms_per_step": sec * 1e3 / args.steps, "higher_is_better": True, "scaling": "strong",
                          "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                          "config": {"workload": cfg["name"], "grid": [nx, ny], "dt": dt, "tol": cfg["tol"],
                                     "parallelism": f"one film over {world} ranks: row blocks (x-sweep) / column blocks "
                                                    "(y-sweep), 2 all-to-alls + 1 all-reduce per Newton iteration"},
                          "newton_iters_total": iters, "gpu_launches": 4 * iters}), flush=True)
    if own_group:
        dist.destroy_process_group()


def run_penta_slabs(args, cfg):
    """Config 4 with every system cut into one slab of rows per rank (direction 1: systems = columns): the slab solver
    of DESIGN.md section 8 -- interface pass, NCCL all-gather of 20 * nparts doubles per system and rank, reduced +
    chunk solves.  Strong scaling: the 16384 x 16384 problem is fixed, each rank holds 1/N of every system."""
    import torch
    import torch.distributed as dist
    from paper_1806_10550_b200 import dist as tfdist, tf
    rank, world = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))
    torch.cuda.set_device(int(os.environ.get("LOCAL_RANK", "0")))
    own_group = not dist.is_initialized()
    if own_group:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29531")
        dist.init_process_group("nccl", rank=rank, world_size=world)
    n = cfg["nrow"]
    nsys = args.nsys or n
    lo, hi = tfdist.slab_bounds(n, world, rank)
    gen = torch.Generator(device="cuda").manual_seed(cfg["seed"] + 1000 * rank)
    U = lambda a, b: torch.rand(hi - lo, nsys, dtype=torch.float64, device="cuda", generator=gen) * (b - a) + a
    e, c, a, b, y = U(-1, 1), U(-1, 1), U(-1, 1), U(-1, 1), U(-1, 1)
    d = 1 + e.abs() + c.abs() + a.abs() + b.abs() + U(0, 1)
    nparts = max(1, args.nparts)
    solve = lambda: tfdist.penta_solve_slabs(1, nparts, e, c, d, a, b, y)
    for _ in range(max(args.warmup, 3)):
        solve()
    dist.barrier()
    torch.cuda.synchronize()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record()
    for _ in range(args.steps):
        solve()
    ev1.record()
    torch.cuda.synchronize()
    dist.barrier()
    sec = max_over_ranks(ev0.elapsed_time(ev1) * 1e-3 / args.steps, world, "cuda")
    if rank == 0:
        print(json.dumps({"metric": "pentadiagonal unknowns/s (fp64), isolated solve, systems spread over the ranks",
                          "unit": "unknowns/s", "n_gpus": world, "value": nsys * n / sec, "ms_per_step": sec * 1e3,
                          "steps": args.steps, "warmup": max(args.warmup, 3), "dtype": "f64", "scaling": "strong",
                          "data": "synthetic (config 4 recipe drawn on the GPU)", "higher_is_better": True,
                          "config": {"workload": cfg["name"], "systems": nsys, "length": n, "variant": "slabs",
                                     "chunks_per_rank": nparts, "exchange": "all-gather of 20*chunks doubles per system and rank",
                                     "alg_bytes_per_unknown": 200},
                          "gpu_launches": 4 * args.steps}), flush=True)
    if own_group:
        dist.destroy_process_group()


def run_penta(args, cfg):
    """Isolated batched pentadiagonal solve (BASELINE.json config 4), both directions, device-resident inputs of
    the config's recipe drawn on the GPU (torch generator, seed 4): not the headline line, a kernel measurement."""
    import torch
    from paper_1806_10550_b200 import tf
    if int(os.environ.get("RANK", "0")) != 0:
        return
    torch.cuda.set_device(int(os.environ.get("LOCAL_RANK", "0")))
    n = args.length or (1024 if args.variant == "pcr" else cfg["nrow"])     # the cyclic-reduction variant holds a system in shared memory
    nsys = args.nsys or cfg["nrow"]
    variant = {"partition": tf.PENTA_PARTITION, "pcr": tf.PENTA_PCR}.get(args.variant, tf.PENTA_LU)
    gen = torch.Generator(device="cuda").manual_seed(cfg["seed"])
    peak, peak_src = measured_peak()
    small = 7 * nsys * n * 8 < 4 * 126e6          # working set not far above L2: flush between timed solves
    flush = torch.empty(64 * 1024 * 1024, dtype=torch.float64, device="cuda") if small else None
    res = {}
    for direction, name in ((1, "along_columns_y"), (0, "along_rows_x")):
        if variant == tf.PENTA_PCR and direction == 1:
            continue                                    # the cyclic-reduction variant exists for the x-sweep shape only
        nrow, ncol = (nsys, n) if direction == 0 else (n, nsys)
        U = lambda lo, hi: torch.rand(nrow, ncol, dtype=torch.float64, device="cuda", generator=gen) * (hi - lo) + lo
        e, c, a, b, y = U(-1, 1), U(-1, 1), U(-1, 1), U(-1, 1), U(-1, 1)
        d = 1 + e.abs() + c.abs() + a.abs() + b.abs() + U(0, 1)
        ws = torch.empty(tf.lib().tf_penta_workspace_bytes_ex(nrow, ncol, direction, variant, args.nparts),
                         dtype=torch.uint8, device="cuda")
        out = torch.empty_like(e)
        chunks = tf.penta_partition_chunks(nrow, ncol, direction, args.nparts) if variant == tf.PENTA_PARTITION else 1
        solve = lambda: tf.penta_solve(direction, e, c, d, a, b, y, out=out, workspace=ws, variant=variant, nparts=args.nparts)
        for _ in range(max(args.warmup, 3)):
            solve()
        torch.cuda.synchronize()
        if small:
            evs = []
            for _ in range(args.steps):
                flush.fill_(0.0)
                ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                ev0.record()
                solve()
                ev1.record()
                evs.append((ev0, ev1))
            torch.cuda.synchronize()
            ms = sum(a0.elapsed_time(a1) for a0, a1 in evs) / args.steps
        else:
            ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            ev0.record()
            for _ in range(args.steps):
                solve()
            ev1.record()
            torch.cuda.synchronize()
            ms = ev0.elapsed_time(ev1) / args.steps
        bpu = 104 if chunks == 1 else 200          # partition: 2 x 48 B interface pass + 104 B chunk solves
        if variant == tf.PENTA_PCR:
            bpu = 56                                # six arrays in, one out: the compulsory traffic
        res[name] = {"ms": ms, "chunks": chunks, "unknowns_per_s": nsys * n / (ms * 1e-3), "alg_bytes_per_unknown": bpu,
                     "alg_gbs": bpu * nsys * n / (ms * 1e-3) / 1e9, "frac_of_peak": bpu * nsys * n / (ms * 1e-3) / 1e9 / peak}
        if args.cusparse and direction == 1:
            lib_run = cusparse_gpsv_interleaved(e, c, d, a, b, y, min(args.steps, 5))
            if lib_run is None:
                res[name]["cusparse_gpsvInterleavedBatch"] = "unavailable"
            else:
                solve()
                torch.cuda.synchronize()
                res[name]["cusparse_gpsvInterleavedBatch"] = {
                    "ms": lib_run[0], "unknowns_per_s": nsys * n / (lib_run[0] * 1e-3),
                    "max_rel_diff_to_ours": float((lib_run[1] - out).abs().max() / out.abs().max()),
                    "note": "vendor library, QR-based (algo 0), in-place; context only"}
        del e, c, a, b, y, d, ws, out
    print(json.dumps({"metric": "pentadiagonal unknowns/s (fp64), isolated solve", "unit": "unknowns/s", "n_gpus": 1,
                      "value": min(r["unknowns_per_s"] for r in res.values()), "steps": args.steps, "warmup": max(args.warmup, 3),
                      "dtype": "f64", "data": "synthetic (config 4 recipe drawn on the GPU)", "higher_is_better": True,
                      "config": {"workload": cfg["name"], "systems": nsys, "length": n, "variant": args.variant,
                                 "l2": "512 MiB flush write between timed solves" if small else
                                 f"inputs 6 x {nsys * n * 8 / 2**20:.0f} MiB >> 126 MB L2"},
                      "directions": res, "peak": peak, "peak_source": peak_src,
                      "gpu_launches": (4 if variant == tf.PENTA_PARTITION else 2) * 2 * args.steps}), flush=True)


def main():
    args = parse()
    cfg = inputs.config(args.config)
    if args.config == 4 and args.slabs and args.impl == "b200":
        return run_penta_slabs(args, cfg)
    if args.config == 4:
        return run_penta(args, cfg) if args.impl == "b200" else print(json.dumps(
            {"impl": "reference", "unavailable": "config 4 is a side measurement of the B200 arm only"}))
    if args.impl == "reference":
        run_reference(args, cfg)
    elif args.distributed:
        run_distributed(args, cfg)
    else:
        run_b200(args, cfg)


if __name__ == "__main__":
    main()
