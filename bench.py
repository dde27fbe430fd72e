#!/usr/bin/env python
"""bench.py -- V-cycles/s and smoother HBM GB/s of the MHS multigrid hot path (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config I] [--boundary-only M]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N ... bench.py --gpus N ...

--config I (0..4) runs BASELINE.json configs[I] instead of configs[2]; --boundary-only M times the 2D boundary Poisson
multigrid alone on an M x M plane (configs[4]: "also time the 2D boundary Poisson MG alone on 4097^2 fp32").  Every mode
prints the same contract line; the metric string names the grid.

A "step" is one pass of the whole hot path over one synthetic magnetogram:
mhs_solve_boundary (2D V-cycles) -> mhs_solve_interior to the config's tolerance (3D V-cycles) ->
mhs_fields (B, p, rho).  Workload: BASELINE.json configs[2] (257^3 fp64, the configuration the metric
is quoted on).  `value` = 3D V-cycles done by all ranks in the K timed steps / device time of those
steps (so the 2D solve and the field recovery are inside the denominator); inputs are resident in HBM.
`e2e` = the same through the *_host entry points of the C ABI: pinned-host Bz0 in, pinned-host
B, p, rho out, copies inside the timed region.  N > 1: one process per GPU, independent magnetograms
per rank ("replicas only", no data-path collective), max-over-ranks time.

--impl reference times the CPU oracle (oracle/, as it stands) on this box's host cores on a bounded
sample of the same workload; rank 0 only.
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

METRIC = "V-cycles/s (3D, whole path: boundary solve + interior solve to tol + fields) at 257^3 fp64"


def metric_name(w):
    """BASELINE.json's metric is quoted on configs[2] (257^3 fp64, the default); other --config values say their own size."""
    if (w.nx, w.ny, w.nz, w.dtype) == (257, 257, 257, "f64"):
        return METRIC
    return METRIC.replace("257^3 fp64", "%dx%dx%d %s" % (w.nx, w.ny, w.nz, "fp64" if w.dtype == "f64" else "fp32"))
FALLBACK_HBM_GBS = 6650.0   # /opt/skills/guides/B200_PROFILING.md fallback


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


def reduce_over_ranks(ms, cycles, world, device="cuda"):
    """(max over ranks of the device time, sum over ranks of the cycles done): the only cross-rank
    traffic of a replica run.  `device="cpu"` serves the gloo test (tests/test_replicas_gloo.py)."""
    if world <= 1:
        return ms, cycles
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    c = torch.tensor([cycles], device=device, dtype=torch.float64)
    dist.all_reduce(c, op=dist.ReduceOp.SUM)
    return float(t.item()), int(c.item())


def read_traffic(key):
    """profiles/traffic.csv: `key,value` rows copied from the committed `ncu --set full` capture
    (dram__bytes_read.sum + dram__bytes_write.sum per launch of the named kernel); None if absent."""
    p = os.path.join(ROOT, "profiles", "traffic.csv")
    try:
        for line in open(p):
            k, _, v = line.strip().partition(",")
            if k == key:
                return float(v)
    except Exception:
        pass
    return None


def read_traffic_source():
    """First comment line of profiles/traffic.csv: which capture (command, commit) the numbers come from."""
    try:
        for line in open(os.path.join(ROOT, "profiles", "traffic.csv")):
            if line.startswith("#"):
                return "profiles/traffic.csv: " + line[1:].strip()
    except Exception:
        pass
    return "profiles/traffic.csv (static: copied from the committed ncu --set full capture, not measured by this run)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index = index
        self.rows = []
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
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
        time.sleep(0.25)
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
                for n, v in zip(names, r[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(n)
            except Exception:
                continue
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": max(mx), "power_w_max": max(pw), "samples": len(sm),
                "reasons": sorted(reasons)}


def oracle_sample(w, cycles, min_seconds=0.0):
    """The oracle as it stands on a bounded sample: the 2D boundary solve (cheap) to set up, then
    at least `cycles` 3D V-cycles at full size -- and as many more as it takes to fill `min_seconds` --
    timed.  Returns (V-cycles/s, seconds, threads, cycles done)."""
    import numpy as np
    import oracle
    P0, _ = oracle.solve_boundary(w.Bz0, (w.Lx, w.Ly), omega=w.omega, n_pre=w.n_pre, n_post=w.n_post, tol=w.tol)
    P = np.zeros(w.shape); P[0] = P0
    c = 1.0 + w.f
    t0 = time.perf_counter()
    done = 0
    while done < cycles or time.perf_counter() - t0 < min_seconds:
        P = oracle.vcycle3(P, None, c, w.alpha, w.L, omega=w.omega, n_pre=w.n_pre, n_post=w.n_post)
        done += 1
    dt = time.perf_counter() - t0
    return done / dt, dt, oracle.num_threads(), done


def run_reference(args, w, cfg):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    per_step = 1 if w.npoints > 5e7 else 2
    for _ in range(args.warmup and 1):
        oracle_sample(w, 1)
    tot_c, tot_t, thr = 0, 0.0, 1
    for _ in range(args.steps):
        v, dt, thr, _ = oracle_sample(w, per_step)
        tot_c += per_step; tot_t += dt
    val = tot_c / tot_t
    sample = "%d V-cycles of the 3D interior solve per step at full size (%dx%dx%d), 2D solve and fields untimed" % (
        per_step, w.nx, w.ny, w.nz)
    out = {"impl": "reference", "metric": metric_name(w), "value": val, "unit": "V-cycles/s", "n_gpus": args.gpus,
           "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * tot_t / args.steps, "higher_is_better": True,
           "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": cfg,
           "cpu_baseline": {"value": val, "unit": "V-cycles/s", "cores": thr, "kind": "oracle", "sample": sample},
           "e2e": {"value": val, "unit": "V-cycles/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
           "gpu_launches": 0}
    print(json.dumps(out))
    return 0


def run_boundary_only(args):
    """BASELINE configs[4]: "also time the 2D boundary Poisson MG alone on 4097^2 fp32".  A step = mhs_solve_boundary on one
    seeded M x M magnetogram (domain [0,4]^2, the configs[4] patch recipe) to its tolerance (fp32: 1e-6 or the stagnation
    rule, C20; fp64: 1e-10).  value = 2D V-cycles / device time.  Roofline: the 2D levels above 513^2 run one kernel per
    multigrid component (the levels below run inside one cluster-kernel launch), so the bytes are SURVEY 8(d)'s
    one-kernel-per-operator count in 2D: 4 sweeps x 3w + residual 3w + restriction 1.25w + prolongation 2.25w = 18.5w per
    node per cycle, x 4/3 for the coarse levels."""
    from paper_1307_6720_b200 import inputs
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    M = args.boundary_only
    dtn = args.dtype or "f32"
    w = inputs.boundary_only(M, dtype=dtn)
    metric = "2D V-cycles/s (boundary Poisson solve alone, eq 11) at %d^2 %s" % (M, "fp32" if dtn == "f32" else "fp64")
    cfg = {"workload": "BASELINE.json configs[4], 2D part: boundary Poisson multigrid alone on %dx%d %s, domain [0,4]^2, 256 seeded "
                       "Gaussian patches, V(2,2), omega=2/3, tol %g%s" % (M, M, dtn, w.tol, " or stagnation (C20)" if dtn == "f32" else ""),
           "grid": [M, M, 1], "parallelism": "replicas x%d" % world,
           "l2": "L2 flushed between steps (a 256 MB device buffer is overwritten): the %.0f MB working set fits the 126 MB L2" % (3 * M * M * (4 if dtn == "f32" else 8) / 1e6)}
    if args.impl == "reference":
        if rank != 0:
            return 0
        import oracle
        tot_c, tot_t = 0, 0.0
        for it in range(args.warmup and 1):
            oracle.solve_boundary(w.Bz0, (w.Lx, w.Ly), tol=1e-10, max_cycles=1)
        for it in range(args.steps):
            t0 = time.perf_counter()
            _, oi = oracle.solve_boundary(w.Bz0, (w.Lx, w.Ly), tol=1e-10, max_cycles=2)
            tot_t += time.perf_counter() - t0; tot_c += oi["cycles"]
        val = tot_c / tot_t
        sample = "2 V-cycles of the 2D solve per step at full size (%dx%d)" % (M, M)
        print(json.dumps({"impl": "reference", "metric": metric, "value": val, "unit": "V-cycles/s", "n_gpus": args.gpus, "steps": args.steps,
                          "warmup": args.warmup, "ms_per_step": 1e3 * tot_t / args.steps, "higher_is_better": True, "scaling": "weak",
                          "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": cfg,
                          "cpu_baseline": {"value": val, "unit": "V-cycles/s", "cores": oracle.num_threads(), "kind": "oracle", "sample": sample},
                          "e2e": {"value": val, "unit": "V-cycles/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}, "gpu_launches": 0}))
        return 0
    import torch
    import torch.distributed as dist
    from paper_1307_6720_b200 import binding
    if not torch.cuda.is_available():
        raise SystemExit("bench.py --impl ours needs a CUDA device (no CPU fallback)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    dt = torch.float32 if dtn == "f32" else torch.float64
    es = 4 if dtn == "f32" else 8
    S = binding.Solver.from_workload(w, dtype=dt, profile=0, flags=args.flags)
    bz_dev = torch.as_tensor(w.Bz0, dtype=dt, device="cuda").contiguous()
    bz_host = torch.as_tensor(w.Bz0, dtype=dt).contiguous().pin_memory()
    p0_host = torch.empty((M, M), dtype=dt).pin_memory()
    flush = torch.empty(64 * 1024 * 1024, dtype=torch.float32, device="cuda")

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def timed(host, steps):
        """Sum over steps of the event time of each step (the L2 flush between steps is outside the events)."""
        tot, cyc, last = 0.0, 0, None
        for _ in range(steps):
            flush.fill_(1.0)
            barrier()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            last = S.solve_boundary(bz_host if host else bz_dev)
            if host:
                S.get_boundary(p0_host)
            e1.record()
            barrier()
            tot += e0.elapsed_time(e1); cyc += last["cycles"]
        tot, cyc_all = reduce_over_ranks(tot, cyc, world)
        return tot, cyc, cyc_all, last

    for _ in range(max(args.warmup, 0)):
        S.solve_boundary(bz_dev)
    S.solve_boundary(bz_host); S.get_boundary(p0_host)
    S.reset_profile()
    clocks = ClockSampler(local)
    if rank == 0:
        clocks.start()
    ms, cyc, cyc_all, last = timed(False, args.steps)
    nlaunch = S.profile()["total_launches"]
    by_class = S.profile()["launches"]
    clk = clocks.stop() if rank == 0 else None
    ms_e2e, _, cyc_e2e, _ = timed(True, args.steps)
    peak, peak_src = peaks()
    n_int = (M - 2) * (M - 2)
    per_cycle = 18.5 * es * n_int * 4.0 / 3.0
    achieved = per_cycle * cyc / (ms * 1e-3) / 1e9
    roof = {"bound": "hbm", "kernel": "the 2D V(2,2) cycle as launched: one kernel per multigrid component on the levels above 513^2, "
                                      "one cluster-kernel launch for the rest",
            "achieved": achieved, "peak": peak, "peak_source": peak_src, "unit": "GB/s", "frac": achieved / peak,
            "traffic": None, "algorithmic_bytes_per_cycle": per_cycle,
            "note": "bytes = SURVEY 8(d) one-kernel-per-operator count in 2D (18.5 w per node per cycle x 4/3); the fine levels "
                    "(67 MB per array in fp32) live in the 126 MB L2 within a step, so this is not a DRAM-bound figure"}
    out = {"metric": metric, "value": cyc_all / (ms * 1e-3), "unit": "V-cycles/s", "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
           "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": dtn, "data": "synthetic",
           "config": cfg, "cycles_per_step": {"boundary_2d": cyc / args.steps}, "converged": bool(last["converged"]),
           "stagnated": bool(last["stagnated"]), "r_final_over_r0": last["r_final"] / last["r0"] if last["r0"] else 0.0, "clocks": clk,
           "roofline": roof,
           "e2e": {"value": cyc_e2e / (ms_e2e * 1e-3), "unit": "V-cycles/s", "ms_per_step": ms_e2e / args.steps,
                   "h2d_bytes_per_step": M * M * es, "d2h_bytes_per_step": M * M * es,
                   "api": "mhs_solve_boundary_host (pinned host Bz0 in) + mhs_get_boundary_host (P(x,y,0) out to pinned host memory)"},
           "gpu_launches": nlaunch, "kernel_launches_by_class": by_class}
    S.close()
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        import oracle
        t0 = time.perf_counter()
        n = 0
        P0 = None
        while n < 1 or time.perf_counter() - t0 < args.cpu_baseline_seconds:
            _, oi = oracle.solve_boundary(w.Bz0, (w.Lx, w.Ly), tol=1e-10, max_cycles=2)
            n += oi["cycles"]
        dtm = time.perf_counter() - t0
        out["cpu_baseline"] = {"value": n / dtm, "unit": "V-cycles/s", "cores": oracle.num_threads(), "kind": "oracle",
                               "sample": "%d V-cycles of the 2D solve at %dx%d (%.1f s of CPU work)" % (n, M, M, dtm)}
    if rank == 0:
        print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=2, help="index into BASELINE.json configs (default 2 = 257^3 fp64)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-baseline-seconds", type=float, default=12.0, help="CPU work of the oracle sample (default ~12 s)")
    ap.add_argument("--flags", type=int, default=0, help="mhs_options.flags (1 = reference kernels)")
    ap.add_argument("--boundary-only", type=int, default=0, metavar="M",
                    help="time the 2D boundary solve alone on an M x M plane (configs[4]: M = 4097)")
    ap.add_argument("--dtype", default=None, choices=["f32", "f64"], help="--boundary-only: element type (default f32, as configs[4])")
    ap.add_argument("--fmg", type=int, default=0, help="mhs_options.fmg_cycles (full-multigrid start; changes the iterates)")
    ap.add_argument("--smoother", type=int, default=0, help="mhs_options.smoother (1 = z-line Jacobi; changes the iterates)")
    args = ap.parse_args()
    if args.boundary_only:
        return run_boundary_only(args)

    from paper_1307_6720_b200 import inputs
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    w = inputs.config(args.config, replica=rank)
    cfg = {"workload": "BASELINE.json configs[%d]: %dx%dx%d %s, f(z)=%g*exp(-%g z), alpha=%g, V(%d,%d), omega=2/3, tol %g; "
                       "one seeded magnetogram per rank" % (args.config, w.nx, w.ny, w.nz, w.dtype, w.a, w.kappa, w.alpha,
                                                            w.n_pre, w.n_post, w.tol),
           "grid": [w.nx, w.ny, w.nz], "parallelism": "replicas x%d (no collective on the data path)" % world,
           "l2": "no flush: per-step working set (2 x %.0f MB iterate buffers + 5 x %.0f MB outputs) exceeds the 126 MB L2"
                 % (w.npoints * 8 / 1e6, w.npoints * 8 / 1e6)}
    if args.impl == "reference":
        return run_reference(args, w, cfg)

    import torch
    import torch.distributed as dist
    from paper_1307_6720_b200 import binding

    if not torch.cuda.is_available():
        raise SystemExit("bench.py --impl ours needs a CUDA device (no CPU fallback)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    dt = torch.float64 if w.dtype == "f64" else torch.float32
    es = 8 if w.dtype == "f64" else 4
    N = w.npoints
    S = binding.Solver.from_workload(w, profile=1, flags=args.flags, fmg_cycles=args.fmg, smoother=args.smoother,
                                     **({"omega": 0.8} if args.smoother else {}))
    bz_dev = torch.as_tensor(w.Bz0, dtype=dt, device="cuda").contiguous()
    bz_host = torch.as_tensor(w.Bz0, dtype=dt).contiguous().pin_memory()
    Bd = torch.empty(3 * N, dtype=dt, device="cuda"); pd = torch.empty(N, dtype=dt, device="cuda"); rd = torch.empty(N, dtype=dt, device="cuda")
    # two sets of pinned host output buffers: the pipelined end-to-end leg fills one while the other is still arriving
    hostbufs = [(torch.empty(3 * N, dtype=dt).pin_memory(), torch.empty(N, dtype=dt).pin_memory(), torch.empty(N, dtype=dt).pin_memory())
                for _ in range(2)]
    Bh, ph, rh = hostbufs[0]

    nstep = [0]

    def step(host):
        """host = False: device-resident; "block": mhs_fields_host (returns when B, p, rho are in host memory);
        "pipe": mhs_fields_host_async (the copy of this step's results overlaps the next step's solve)."""
        ib = S.solve_boundary(bz_host if host else bz_dev)
        ii = S.solve_interior(w.tol, w.max_cycles)
        if host == "pipe":
            b = hostbufs[nstep[0] % 2]
            nstep[0] += 1
            S.fields(b[0], b[1], b[2], host=True, wait=False)
        elif host:
            S.fields(Bh, ph, rh, host=True)
        else:
            S.fields(Bd, pd, rd)
        return ib["cycles"], ii["cycles"], ii

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def timed(host, steps):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        e0.record()
        c2 = c3 = 0
        last = None
        for _ in range(steps):
            a, b, last = step(host)
            c2 += a; c3 += b
        if host == "pipe":
            S.host_sync()      # the last step's results have landed before the clock stops
        e1.record()
        barrier()
        ms = e0.elapsed_time(e1)
        ms, c3_all = reduce_over_ranks(ms, c3, world)
        return ms, c2, c3, c3_all, last

    for _ in range(max(args.warmup, 0)):
        step(False)
    step("block")  # warm the host path (staging buffer allocation) outside the timed regions
    # Timed region 1 (`value`): K steps with NO event records between kernels -- they undo the overlap of dependent
    # launches and cost ~1 % -- bracketed by two events on the stream.
    S.set_profiling(0)
    S.reset_profile()
    clocks = ClockSampler(local)
    if rank == 0:
        clocks.start()
    ms, c2, c3, c3_all, last = timed(False, args.steps)
    nlaunch = S.profile()["total_launches"]
    by_class = S.profile()["launches"]
    # Timed region 2 (roofline): the same K steps again with CUDA events around every finest-level smoothing /
    # prolongation launch on the library's stream; its own ms/step is reported next to the kernel numbers.
    S.set_profiling(1)
    S.reset_profile()
    ms_prof, _, _, _, _ = timed(False, args.steps)
    prof = S.profile()
    # Timed region 3 (shares): the same K steps with CUDA events around EVERY kernel class (serialises dependent launches)
    S.set_profiling(2)
    S.reset_profile()
    ms_cls, _, _, _, _ = timed(False, args.steps)
    prof2 = S.profile()
    class_ms = {k: v / args.steps for k, v in prof2["ms"].items()}
    clk = clocks.stop() if rank == 0 else None
    S.set_profiling(0)   # (the end-to-end legs: event records would also serialise against the copy stream)
    S.reset_profile()
    ms_e2e, _, _, c3_all_e2e, _ = timed("pipe", args.steps)
    ms_blk, _, _, c3_all_blk, _ = timed("block", args.steps)

    # ---- roofline of the dominant kernel: k_zsweep, the temporally blocked finest-level smoother.
    # It runs as two kinds of launch: plain passes (class smooth_l0: read u, write u', S sweeps) and prolongation-fused
    # post-smoothing passes (class prolong_l0 when fused_prolong_l0 > 0: read u and e_c, write u').  Algorithmic bytes
    # per launch: 2w per node, + w/8 for the coarse correction; whatever the number of sweeps fused in it.
    peak, peak_src = peaks()
    n_int = (w.nx - 2) * (w.ny - 2) * (w.nz - 2)
    sweeps = prof["sweeps_l0"]
    l_plain, t_plain = prof["launches"]["smooth_l0"], prof["ms"]["smooth_l0"]
    l_fused = prof["fused_prolong_l0"]
    fused_all = l_fused > 0 and l_fused == prof["launches"]["prolong_l0"]
    t_fused = prof["ms"]["prolong_l0"] if fused_all else 0.0
    b_plain, b_fused = 2.0 * es * n_int, (2.0 + 0.125) * es * n_int
    launches = l_plain + (l_fused if fused_all else 0)
    t_smooth_ms = t_plain + t_fused
    alg_bytes = b_plain * l_plain + (b_fused * l_fused if fused_all else 0.0)
    achieved = alg_bytes / (t_smooth_ms * 1e-3) / 1e9 if t_smooth_ms > 0 else 0.0
    tr_p = read_traffic("smooth_l0_dram_bytes_per_launch_%d" % w.nx) if w.nx == w.ny == w.nz else None
    tr_f = read_traffic("prolong_smooth_l0_dram_bytes_per_launch_%d" % w.nx) if w.nx == w.ny == w.nz else None
    traffic = tr_p
    if fused_all and tr_p is not None and tr_f is not None and launches:
        traffic = (tr_p * l_plain + tr_f * l_fused) / launches
    roof = {"bound": "hbm", "kernel": "k_zsweep: finest-level weighted-Jacobi smoother, 2 sweeps per HBM pass "
                                      "(plain passes + prolongation-fused post-smoothing passes)",
            "achieved": achieved, "peak": peak, "peak_source": peak_src, "unit": "GB/s", "frac": achieved / peak,
            "frac_of_8TBs_nominal": achieved / 8000.0, "traffic": traffic,
            "traffic_source": (read_traffic_source() if traffic is not None else None),
            "frac_from_traffic": ((traffic * launches / (t_smooth_ms * 1e-3) / 1e9 / peak) if traffic and t_smooth_ms > 0 else None),
            "launches": launches, "sweeps": sweeps, "sweeps_per_launch": (sweeps / launches) if launches else None,
            "avg_launch_us": 1e3 * t_smooth_ms / launches if launches else None,
            "algorithmic_bytes_per_launch": alg_bytes / launches if launches else None,
            "smoother_gpts_per_s": n_int * sweeps / (t_smooth_ms * 1e-3) / 1e9 if t_smooth_ms > 0 else 0.0,
            "smoother_share_of_step": t_smooth_ms / ms_prof,
            "note": (None if launches else "no finest-level smoother launch: the whole solve of this grid runs inside one "
                                           "cluster-kernel launch (shared memory / L2 resident, latency-bound)"),
            "timed_in": "a second pass of the same K steps with CUDA events around every launch of this kernel (%.3f ms/step; "
                        "`value` comes from the pass without them)" % (ms_prof / args.steps),
            "plain_pass": {"launches": l_plain, "avg_us": 1e3 * t_plain / l_plain if l_plain else None,
                           "algorithmic_bytes": b_plain, "gbs": b_plain * l_plain / (t_plain * 1e-3) / 1e9 if t_plain > 0 else None},
            "prolong_fused_pass": ({"launches": l_fused, "avg_us": 1e3 * t_fused / l_fused, "algorithmic_bytes": b_fused,
                                    "gbs": b_fused * l_fused / (t_fused * 1e-3) / 1e9} if fused_all and t_fused > 0 else None)}

    out = {"metric": metric_name(w), "value": c3_all / (ms * 1e-3), "unit": "V-cycles/s", "n_gpus": world, "steps": args.steps,
           "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak",
           "vs_baseline": None, "dtype": w.dtype, "data": "synthetic", "config": cfg,
           "cycles_per_step": {"boundary_2d": c2 / args.steps, "interior_3d": c3 / args.steps},
           "converged": bool(last["converged"]), "r_final_over_r0": last["r_final"] / last["r0"] if last["r0"] else 0.0,
           "clocks": clk, "roofline": roof,
           "e2e": {"value": c3_all_e2e / (ms_e2e * 1e-3), "unit": "V-cycles/s", "ms_per_step": ms_e2e / args.steps,
                   "h2d_bytes_per_step": w.nx * w.ny * es, "d2h_bytes_per_step": 5 * N * es,
                   "api": "mhs_solve_boundary_host + mhs_solve_interior + mhs_fields_host_async (pinned host Bz0 in; B, p, rho "
                          "out to alternating pinned host buffers, each step's device->host copy overlapping the next step's "
                          "solve; mhs_host_sync before the clock stops)",
                   "blocking": {"value": c3_all_blk / (ms_blk * 1e-3), "ms_per_step": ms_blk / args.steps,
                                "api": "the same with mhs_fields_host, which returns when the results are in host memory"}},
           "gpu_launches": nlaunch,
           "kernel_launches_by_class": by_class,
           "kernel_class_ms_per_step": dict(class_ms, note="CUDA events around every kernel class: dependent launches do not "
                                            "overlap in this pass (%.3f ms/step against %.3f)" % (ms_cls / args.steps, ms / args.steps)),
           "options": {"flags": args.flags, "fmg_cycles": args.fmg, "smoother": args.smoother}}
    S.close()
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        v, dtm, thr, nc = oracle_sample(w, 1, min_seconds=args.cpu_baseline_seconds)
        out["cpu_baseline"] = {"value": v, "unit": "V-cycles/s", "cores": thr, "kind": "oracle",
                               "sample": "%d V-cycles of the 3D interior solve at %dx%dx%d (%.1f s of CPU work); 2D solve and fields not timed"
                                         % (nc, w.nx, w.ny, w.nz, dtm)}
    if rank == 0:
        print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
