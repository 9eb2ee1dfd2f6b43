#!/usr/bin/env python
"""bench.py -- headline benchmark of the treecode BEM matvec (BASELINE.json metric) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config binding_complex]
                    [--precision fp64|mixed] [--sweep]

A step = one matvec y = A x (the hot loop of PAPER.md:169: "one evaluation of the treecode per iteration")
of the whole coupled system: density weighting, P2M, upward pass, M2P, P2P, near-field corrections and
block combination for every region.  value = direct-equivalent interactions per second
(sum_regions N_targets x N_gauss_points per matvec) with x and y resident in HBM; e2e = the
same through pygbe_matvec_host (pinned host buffers, copies inside the timed region).  The second half of
the metric, GMRES time-to-solution, is reported under "solve" (create + rhs + GMRES + energy).
L2 is flushed between timed iterations.  Multi-GPU: independent replicas of the workload, one per rank
("replicas only"), no data-path collective.  The default workload is the largest single-GPU
configuration of BASELINE.json (configs[4], the 1.08 M-panel complex of the binding-energy problem, P = 8,
fp32 kernels with fp64 accumulation); --config selects the others, --sweep prints one line per configuration
(create / matvec / solve times, energies: the table of BASELINE.md section 5).
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

METRIC = "BEM matvec interactions/s (Laplace+Yukawa), direct-equivalent"
UNIT = "interactions/s"


CONFIGS = {
    # name: (builder, create keywords, GMRES tol (fp64, mixed), description)
    "born_l3": (lambda W: W.born_problem(3), dict(K=4, P=6, theta=0.0), (1e-8, 1e-5),
                "BASELINE.json configs[0]: Born sphere, icosphere level 3 (1280 panels), K=4, direct summation (theta=0)"),
    "kirkwood_l5": (lambda W: W.kirkwood_problem(5), dict(K=4, P=6, theta=0.5), (1e-6, 1e-5),
                    "BASELINE.json configs[1]: Kirkwood sphere R=10 A, icosphere level 5 (20480 panels), K=4, P=6, theta=0.5"),
    "kirkwood_l6": (lambda W: W.kirkwood_problem(6), dict(K=4, P=6, theta=0.5), (1e-6, 1e-5),
                    "Kirkwood sphere level 6 (81920 panels), K=4, P=6, theta=0.5"),
    "protein_1000": (lambda W: W.cached("protein_1000_s105", lambda: W.protein_problem(1000, spacing=1.05)),
                     dict(K=4, P=6, theta=0.5), (1e-6, 1e-5),
                     "BASELINE.json configs[2]: synthetic protein, 1000 atoms, 41.5 k panels, K=4, P=6, theta=0.5"),
    "multisurface_3000": (lambda W: W.cached("multisurface_3000_s112", lambda: W.multisurface_problem(3000, spacing=1.12)),
                          dict(K=4, P=6, theta=0.5), (1e-6, 1e-5),
                          "BASELINE.json configs[3]: 3000 atoms, 2 cavities, Stern surface, 157 k panels, 4 regions, K=4, P=6, theta=0.5"),
    "binding_complex": (lambda W: W.cached("binding_complex_5000_500_s055",
                                           lambda: W.binding_problems(5000, 500, spacing=0.55, only=("complex",))[0]),
                        dict(K=4, P=8, theta=0.5), (1e-4, 1e-4),
                        "BASELINE.json configs[4], the complex: receptor 5000 + ligand 500 atoms at 3 A, two dielectric bodies + "
                        "one Stern surface, 1.08 M panels (4.3 M Gauss points), 3 regions, K=4, P=8, theta=0.5"),
    "binding_receptor": (lambda W: W.cached("binding_receptor_5000_500_s055",
                                            lambda: W.binding_problems(5000, 500, spacing=0.55, only=("receptor",))[1]),
                         dict(K=4, P=8, theta=0.5), (1e-4, 1e-4),
                         "BASELINE.json configs[4], the receptor alone: 5000 atoms + Stern surface, 0.86 M panels, K=4, P=8, theta=0.5"),
    "binding_ligand": (lambda W: W.cached("binding_ligand_5000_500_s055",
                                          lambda: W.binding_problems(5000, 500, spacing=0.55, only=("ligand",))[2]),
                       dict(K=4, P=8, theta=0.5), (1e-4, 1e-4),
                       "BASELINE.json configs[4], the ligand alone: 500 atoms + Stern surface, 0.23 M panels, K=4, P=8, theta=0.5"),
}
DEFAULT_CONFIG = "binding_complex"       # the largest single-GPU configuration of BASELINE.json (configs[4])


def make_problem(name):
    import workloads as W
    if name not in CONFIGS:
        raise SystemExit(f"unknown config {name}; known: {', '.join(CONFIGS)}")
    build, kw, tols, desc = CONFIGS[name]
    return build(W), dict(kw), desc


# ------------------------------------------------------------------------------------------ flop model
def m2p_nw(P):
    """W_{m,e} per moment set of the regrouped Taylor series on harmonically reduced moments (m2p.cuh, tables.cuh):
    84 at P = 6, 165 at P = 8 (unreduced: 130, 295)."""
    return sum((2 * t + 1) * ((P - t) // 2 + 1) for t in range(P + 1))


def m2p_flops(P, yukawa):
    """Algorithmic flops of one (target, cell) Taylor evaluation as the regrouped kernels do it (m2p.cuh;
    multiply-add = 2, rsqrt = exp = 1): offset and radius, the (P+1)^2 - 1 monomials d^e with ez <= 1, one FMA per W_{m,e}
    for every region in `yukawa` (a tuple of booleans: one entry, or two for twin regions evaluated in one pass), and per
    region the P + 1 radial derivatives F^(m) and their dot product with Q_m.  DESIGN.md 'Flop model'."""
    if isinstance(yukawa, bool):
        yukawa = (yukawa,)
    f = 3 + 5 + 3 + ((P + 1) * (P + 1) - 1)            # d ; r^2 ; 1/r, 1/r^2, r ; monomials
    for yk in yukawa:
        f += 2 * m2p_nw(P)                             # Q_m += W d^e
        f += (2 if yk else 0) + 1 + 5                  # [kappa r, exp] ; F0 ; F1
        f += 4 * (P - 1) + 2 * (P + 1)                 # F^(m+1) recurrence ; sum_m F^(m) Q_m
    return f


def m2p_lap_flops(P):
    """One (target, cell) evaluation of the Laplace form (k_m2p_lap): d (3), r^2 (5), rsqrt (1), 1/r^2 (1),
    a / r^2 (1), u = d a / r^2 (3), Nc - 1 Horner FMAs, times 1/r (1), accumulate (1)."""
    nc = (P + 1) * (P + 2) * (P + 3) // 6
    return 16 + 2 * (nc - 1)


P2P_FLOPS = {False: 19, True: 25}     # per (target, Gauss point) pair, Laplace / Yukawa (rsqrt, exp = 1)
P2P_FLOPS_FUSED = 30                  # Laplace + Yukawa of twin regions sharing d, r^2, 1/r, n.d


def launch_flops(rec, P, kappa):
    """Algorithmic flops of one launch of a compute-bound kernel from the record of pygbe_launch_times."""
    yA = float(kappa[rec["region"]]) > 0
    twin = rec["twin_region"] >= 0
    yB = twin and float(kappa[rec["twin_region"]]) > 0
    if rec["stage"] == "p2p":
        if twin:
            per = P2P_FLOPS_FUSED if yA != yB else (2 * P2P_FLOPS[yA] - 9)      # shared d, r^2, 1/r, n.d
        else:
            per = P2P_FLOPS[yA]
        return rec["units"] * per
    if rec["stage"] == "m2p":
        if "lap" in rec["kernel"]:
            return rec["units"] * m2p_lap_flops(P)
        return rec["units"] * m2p_flops(P, (yA, yB) if twin else yA)
    return 0


def profiled_traffic(config, precision, kernel, region):
    """dram__bytes_read.sum + dram__bytes_write.sum of one launch of `kernel` on `region`, from the newest
    profiles/*_traffic.csv (columns config, precision, kernel, region, dram_bytes, duration_ms; written from an
    `ncu --set full` capture of this command, which the *_path.md beside it names together with the commit).  None if
    there is no record for this configuration: the run itself measures no DRAM counters."""
    import csv
    import glob
    for path in sorted(glob.glob(os.path.join(ROOT, "profiles", "*_traffic.csv")), reverse=True):
        try:
            rows = list(csv.DictReader(open(path)))
        except Exception:
            continue
        for r in rows:
            if r["config"] == config and r["precision"] == precision and r["kernel"] == kernel and int(r["region"]) == region:
                note = os.path.basename(path).replace("_traffic.csv", "_path.md")
                return float(r["dram_bytes"]), "profiles/%s (capture described in profiles/%s)" % (os.path.basename(path), note)
    return None, None


def clocks_sampler(stop, out):
    q = "clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"
    while not stop.is_set():
        try:
            r = subprocess.run(["nvidia-smi", f"--query-gpu={q}", "--format=csv,noheader,nounits", "-i",
                                os.environ.get("LOCAL_RANK", "0")], capture_output=True, text=True, timeout=5)
            out.append([c.strip() for c in r.stdout.strip().split(",")])
        except Exception:
            pass
        stop.wait(0.2)


def summarize_clocks(samples):
    sm = [float(s[0]) for s in samples if len(s) >= 7 and s[0].replace(".", "").isdigit()]
    mx = [float(s[1]) for s in samples if len(s) >= 7 and s[1].replace(".", "").isdigit()]
    reasons = []
    for i, name in enumerate(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")):
        if any(len(s) >= 7 and s[3 + i].lower().startswith("active") for s in samples):
            reasons.append(name)
    return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
            "reasons": reasons, "samples": len(sm)}


# ------------------------------------------------------------------------------------- reference arm
def oracle_sample(prob, kw, seconds_target=15.0):
    """Time the oracle (as it stands, through its own OpenMP loop over rows: all host cores unless OMP_NUM_THREADS
    says otherwise) on a bounded sample of rows of the same matvec; returns (interactions/s, threads, description,
    seconds)."""
    import oracle
    o = oracle.Oracle(prob, K=kw["K"])
    rng = np.random.default_rng(42)
    x = rng.normal(size=o.n)
    # interactions of a row = Gauss points on the boundary of the row's region (row layout of include/pygbe.h)
    npts = np.zeros(prob.n_regions)
    for S in prob.surfaces:
        npts[S.region_in] += kw["K"] * S.n_panels
        npts[S.region_out] += kw["K"] * S.n_panels
    row_cost = np.concatenate([np.concatenate([np.full(S.n_panels, npts[S.region_in]), np.full(S.n_panels, npts[S.region_out])])
                               for S in prob.surfaces])
    probe = np.sort(rng.choice(o.n, min(64, o.n), replace=False))
    t = time.perf_counter(); o.matvec(x, probe); dt = time.perf_counter() - t
    nrows = int(min(o.n, max(64, 64 * seconds_target / max(dt, 1e-3))))
    rows = np.sort(rng.choice(o.n, nrows, replace=False))
    reps = 1
    if nrows == o.n:                                 # a whole matvec is cheaper than the target: repeat it
        reps = int(max(1, min(20, seconds_target / max(dt * o.n / 64, 1e-3))))
    t = time.perf_counter()
    for _ in range(reps):
        o.matvec(x, rows)
    dt = time.perf_counter() - t
    work = reps * float(row_cost[rows].sum())
    return work / dt, oracle.num_threads(), f"{reps} x {nrows} of {o.n} seeded rows of one matvec ({work:.3g} interactions, {dt:.1f} s)", dt


def oracle_single_thread(config, seconds=8.0):
    """The same sample on ONE host thread ("single-threaded and with all cores"): a child process with
    OMP_NUM_THREADS=1 running this file's reference arm, since the oracle reads its thread count at load."""
    env = dict(os.environ, OMP_NUM_THREADS="1", RANK="0", WORLD_SIZE="1")
    try:
        r = subprocess.run([sys.executable, os.path.abspath(__file__), "--impl", "reference", "--config", config, "--steps", "1",
                            "--warmup", "0", "--seconds", str(seconds)], capture_output=True, text=True, timeout=600, env=env)
        line = json.loads(r.stdout.strip().splitlines()[-1])
        return {"value": line["value"], "unit": UNIT, "cores": line["cpu_baseline"]["cores"], "kind": "oracle",
                "sample": line["cpu_baseline"]["sample"]}
    except Exception as e:                           # reported, never fatal for the GPU line
        return {"value": None, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": f"failed: {e}"}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    prob, kw, desc = make_problem(args.config)
    vals, secs = [], []
    for _ in range(args.warmup):
        oracle_sample(prob, kw, seconds_target=1.0)
    sample, cores = "", 0
    per_step = args.seconds if args.seconds > 0 else max(2.0, 60.0 / max(args.steps, 1))
    for _ in range(args.steps):
        v, cores, sample, dt = oracle_sample(prob, kw, seconds_target=per_step)
        vals.append(v); secs.append(dt)
    v = float(np.mean(vals))
    line = {"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * float(np.mean(secs)), "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": desc, "l2": "n/a (CPU)"},
            "cpu_baseline": {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


# --------------------------------------------------------------------------------------------- our arm
def max_over_ranks(v, dist, device):
    """Timing of the slowest rank (the job is as slow as its slowest replica)."""
    import torch
    t = torch.tensor([float(v)], dtype=torch.float64, device=device)
    if dist is not None and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(world, units_per_step, steps, seconds):
    """Aggregate throughput of `world` independent replicas ("replicas only": no data-path collective)."""
    return world * units_per_step * steps / seconds


def run_ours(args):
    import torch
    import paper_1309_4018_b200 as pg
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product has no CPU fallback")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    pg.lib()
    if args.sweep:
        if rank == 0:
            for name in ("born_l3", "kirkwood_l5", "protein_1000", "multisurface_3000", "binding_complex", "binding_receptor",
                         "binding_ligand"):
                for prec in ("fp64", "mixed"):
                    a = argparse.Namespace(**dict(vars(args), config=name))
                    line = measure(a, prec, pg, torch, None, 1, 0, local, full=False, brief=True)
                    print(json.dumps({"sweep": name, "precision": prec, **{k: line[k] for k in ("value", "ms_per_step", "config", "solve", "kernels", "hbm_passes")}}), flush=True)
        return
    other = "fp64" if args.precision == "mixed" else "mixed"
    line = measure(args, args.precision, pg, torch, dist, world, rank, local, full=True)
    second = measure(args, other, pg, torch, dist, world, rank, local, full=False)
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()
    if line is not None:
        keep = ("value", "ms_per_step", "dtype", "e2e", "gpu_launches", "roofline", "kernels", "hbm_passes", "solve", "actual")
        line["other_precision"] = {k: second[k] for k in keep if k in second}
        line["other_precision"]["precision"] = other
        print(json.dumps(line))


def measure(args, precision_name, pg, torch, dist, world, rank, local, full, brief=False):
    prob, kw, desc = make_problem(args.config)
    tols = CONFIGS[args.config][2]
    big = prob.n_panels > 300_000
    precision = pg.PRECISION_MIXED if precision_name == "mixed" else pg.PRECISION_FP64
    # create is timed warm, like the kernels: the first handle of a process pays the CUDA module load and the growth
    # of the memory pools (reported as create_first_ms).  A create through the binding's default path is the size
    # query (pygbe_workspace_size, a dry run of the list sizing), one torch allocation, and pygbe_create into it.
    t0 = time.perf_counter()
    pg.Handle.from_problem(prob, precision=precision, device=local, **kw).close()
    torch.cuda.synchronize()
    create_first_ms = 1e3 * (time.perf_counter() - t0)
    mem0 = torch.cuda.memory_allocated(local)
    t0 = time.perf_counter()
    h = pg.Handle.from_problem(prob, precision=precision, device=local, **kw)
    torch.cuda.synchronize()
    create_total_ms = 1e3 * (time.perf_counter() - t0)
    st = h.stats()
    n = h.n
    torch_bytes = torch.cuda.memory_allocated(local) - mem0
    rng = np.random.default_rng(7)
    x = torch.tensor(rng.normal(size=n), device="cuda")
    y = torch.empty_like(x)
    flush = torch.empty(256 * 1024 * 1024 // 4, dtype=torch.float32, device="cuda")   # 256 MB > 126 MB L2

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        h.matvec(x, y)
    # ---- timed region: K matvecs, each bracketed by its own events, L2 flushed in between
    stop, samples = threading.Event(), []
    th = threading.Thread(target=clocks_sampler, args=(stop, samples), daemon=True)
    th.start()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    launches0 = h.stats()["kernel_launches"]
    barrier()
    for a, b in ev:
        flush.zero_()
        a.record()
        h.matvec(x, y)
        b.record()
    barrier()
    launches = h.stats()["kernel_launches"] - launches0
    ms = sum(a.elapsed_time(b) for a, b in ev)
    # keep the sampler alive over a short sustained burst so that clocks under load are seen
    tend = time.perf_counter() + 1.0
    while time.perf_counter() < tend:
        h.matvec(x, y)
    torch.cuda.synchronize()
    stop.set(); th.join()
    ms = max_over_ranks(ms, dist, "cuda")
    ms_per_step = ms / args.steps
    value = whole_job_value(world, st["direct_equiv"], args.steps, ms * 1e-3)

    # ---- e2e: host buffers through pygbe_matvec_host (pinned), copies inside the timed region
    xh = torch.empty(n, dtype=torch.float64).pin_memory(); xh.copy_(x.cpu())
    yh = torch.empty(n, dtype=torch.float64).pin_memory()
    xn, yn = xh.numpy(), yh.numpy()
    for _ in range(3):
        h.matvec_host(xn, yn)
    barrier()
    e2e_s = 0.0
    for _ in range(args.steps):
        flush.zero_()
        torch.cuda.synchronize()
        t = time.perf_counter()
        h.matvec_host(xn, yn)            # synchronous: H2D copy, matvec, D2H copy, stream sync
        e2e_s += time.perf_counter() - t
    e2e = whole_job_value(world, st["direct_equiv"], args.steps, max_over_ranks(e2e_s, dist, "cuda"))

    line = None
    if rank == 0:
        # ---- per-launch timers (profiled matvecs run on one stream and are not the ones timed above)
        psteps = max(3, min(args.steps, 10))
        h.profile(True)
        for _ in range(psteps):
            flush.zero_()
            h.matvec(x, y)
        stages = h.stage_times()
        recs = h.launch_times()
        h.profile(False)
        stage_ms = {k: v[0] / psteps for k, v in stages.items()}
        peaks = pg.alu_peaks(local)
        mp = {}
        try:
            mp = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
        except Exception:
            pass
        sm_max = float(mp.get("sm_max_mhz", 1965.0))
        hbm_peak = float(mp.get("hbm_gbs", 6540.2))
        nominal = {"f64": 148 * 64 * 2 * sm_max * 1e6 / 1e12, "f32": 148 * 128 * 2 * sm_max * 1e6 / 1e12}
        dt = "f32" if precision == pg.PRECISION_MIXED else "f64"
        kernels, passes = [], []
        for r in recs:
            per_ms = r["ms"] / max(r["launches"], 1)
            base = {"kernel": r["kernel"], "stage": r["stage"], "region": r["region"], "twin_region": r["twin_region"],
                    "ms_per_launch": per_ms, "units_per_launch": r["units"]}
            if r["stage"] in ("p2p", "m2p"):
                fl = launch_flops(r, kw["P"], prob.kappa)
                tf = fl / (per_ms * 1e-3) / 1e12 if per_ms > 0 else 0.0
                kernels.append({**base, "flops_per_launch": fl, "tflops": tf, "frac": tf / nominal[dt]})
            else:
                gbs = r["bytes"] / (per_ms * 1e-3) / 1e9 if per_ms > 0 else 0.0
                passes.append({**base, "bytes_per_launch": r["bytes"], "gbs": gbs, "frac_of_hbm_peak": gbs / hbm_peak})
        dom = max(kernels, key=lambda k: k["ms_per_launch"])
        traffic, traffic_source = profiled_traffic(args.config, precision_name, dom["kernel"].replace("<P", "<%d" % kw["P"]), dom["region"])
        roofline = {"bound": "alu", "kernel": "%s, region %d%s, 1 launch/matvec" % (
                        dom["kernel"].replace("<P", "<%d" % kw["P"]), dom["region"],
                        (" + twin %d" % dom["twin_region"]) if dom["twin_region"] >= 0 else ""),
                    "achieved": dom["tflops"], "peak": nominal[dt], "unit": "TFLOP/s", "frac": dom["frac"],
                    "peak_kind": "derived: 148 SM x %d lanes x 2 x %.0f MHz (DESIGN.md 7); FMA micro-benchmark in this run: %.1f TFLOP/s"
                                 % (64 if dt == "f64" else 128, sm_max, peaks["fp64_tflops" if dt == "f64" else "fp32_tflops"]),
                    "traffic": traffic, "traffic_source": traffic_source,
                    "ms_per_launch": dom["ms_per_launch"], "flops_per_launch": dom["flops_per_launch"],
                    "units_per_launch": dom["units_per_launch"],
                    "flop_model": "DESIGN.md 7 'Flop model' (bench.py launch_flops)", "stage_ms": stage_ms,
                    "alu_peaks_measured": peaks, "hbm_peak_gbs": hbm_peak}
        if dt == "f32" and peaks.get("fp32_mix_tflops"):
            # context, not the denominator: what the FP32 pipe delivers on a register-resident FMUL + 3-register
            # FFMA mix (pygbe_alu_peaks out[3]), the practical ceiling of a mixed FMUL / FFMA stream
            roofline["frac_of_mix_ceiling"] = dom["tflops"] / peaks["fp32_mix_tflops"]
        if dt == "f32" and "lap" in dom["kernel"] and peaks.get("fp32_horner_tflops"):
            # what the bare Horner stream of this kernel (packed FFMA2, broadcast coefficient from shared memory) reaches
            # on this machine, measured in this run (pygbe_alu_peaks out[4]): the ceiling of the kernel's pattern
            roofline["frac_of_horner_ceiling"] = dom["tflops"] / peaks["fp32_horner_tflops"]
        # ---- time-to-solution (second half of the metric): create + rhs + GMRES + energy, host buffers.  The first
        # solve of a handle is reported apart on the small configs (warm-up of the cooperative launch); the large
        # ones run one solve
        tol = tols[0] if dt == "f64" else tols[1]
        solve_times = []
        for _ in range(1 if big else (2 if brief else 4)):
            t = time.perf_counter()
            xs, iters, rr, es, ec = h.solve_host(tol=tol, max_iter=3000)
            solve_times.append(1e3 * (time.perf_counter() - t))
        solve_first_ms = solve_times[0]
        solve_ms = sorted(solve_times[1:])[1] if len(solve_times) >= 4 else solve_times[-1]
        solve = {"create_ms": create_total_ms, "create_first_ms": create_first_ms,
                 "create_breakdown_ms": {"workspace_size_query": h.workspace_query_ms, "pygbe_create": st["create_ms"]},
                 "solve_ms": solve_ms, "solve_first_ms": solve_first_ms, "time_to_solution_ms": create_total_ms + solve_ms,
                 "gmres_iters": iters, "rel_resid": rr, "tol": tol, "E_solv_kJ_mol": es, "E_coul_kJ_mol": ec,
                 "ms_per_iteration": solve_ms / max(iters, 1), "preconditioner": "none (reading A16)",
                 "device_bytes": st["device_bytes"], "workspace_bytes": int(h.workspace.numel()) if h.workspace is not None else 0,
                 "torch_allocated_delta_bytes": int(torch_bytes)}
        if not brief:
            # the same with the optional block-diagonal right preconditioner (pygbe_options.precond = 1)
            t = time.perf_counter()
            h2 = pg.Handle.from_problem(prob, precision=precision, device=local, precond=1, **kw)
            torch.cuda.synchronize()
            c2 = 1e3 * (time.perf_counter() - t)
            t = time.perf_counter()
            _, it2, rr2, es2, ec2 = h2.solve_host(tol=tol, want_x=False, max_iter=3000)
            s2 = 1e3 * (time.perf_counter() - t)
            h2.close()
            solve["block_diagonal"] = {"create_ms": c2, "solve_ms": s2, "time_to_solution_ms": c2 + s2, "gmres_iters": it2,
                                       "rel_resid": rr2, "E_solv_kJ_mol": es2}
        # ---- oracle on the host cores, bounded samples: all cores and one thread
        cpu = {"value": None, "unit": UNIT, "cores": None, "kind": "oracle", "sample": None}
        if full:
            cv, cores, sample, _ = oracle_sample(prob, kw, seconds_target=15.0)
            cpu = {"value": cv, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample,
                   "single_thread": oracle_single_thread(args.config)}
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": max(args.warmup, 3), "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": dt, "data": "synthetic",
                "config": {"workload": desc, "name": args.config, "n_panels": st["n_panels"], "n_unknowns": st["n_unknowns"],
                           "n_regions": st["n_regions"], "n_charges": st["n_charges"],
                           "direct_equiv_interactions": st["direct_equiv"], "p2p_pairs": st["p2p_pairs"],
                           "m2p_evals": st["m2p_evals"], "precision": precision_name, **kw,
                           "l2": "flushed between timed iterations (256 MB write)",
                           "parallelism": "replicas only" if world > 1 else "single GPU"},
                "clocks": summarize_clocks(samples),
                "e2e": {"value": e2e, "unit": UNIT, "h2d_bytes_per_step": 8 * n, "d2h_bytes_per_step": 8 * n},
                "gpu_launches": int(launches),
                "roofline": roofline, "kernels": kernels, "hbm_passes": passes,
                "cpu_baseline": cpu,
                "solve": solve,
                "actual": {"p2p_pairs_per_s": st["p2p_pairs"] / (stage_ms["p2p"] * 1e-3) if stage_ms["p2p"] > 0 else None,
                           "m2p_evals_per_s": st["m2p_evals"] / (stage_ms["m2p"] * 1e-3) if stage_ms["m2p"] > 0 else None}}
    h.close()
    return line


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default=DEFAULT_CONFIG, choices=sorted(CONFIGS))
    ap.add_argument("--precision", default="mixed", choices=["fp64", "mixed"])
    ap.add_argument("--seconds", type=float, default=0.0, help="reference arm: CPU seconds per step (default 60 / steps)")
    ap.add_argument("--sweep", action="store_true", help="one JSON line per configuration and precision (rank 0, one GPU)")
    ap.add_argument("--probe-mma", action="store_true", help="tensor-core M2P probe (pygbe_mma_probe), P = 6 and 8; one JSON line")
    args = ap.parse_args()
    if args.probe_mma:
        import paper_1309_4018_b200 as pg
        res = {}
        for P in (6, 8):
            r = pg.mma_probe(P)
            base = r["cuda_core_k_m2p_single2"]["ms"]
            for v in r.values():
                v["ns_per_group_cell"] = 1e6 * v["ms"] / v["pairs"]
                v["time_vs_cuda_core"] = v["ms"] / base
            res["P=%d" % P] = r
        print(json.dumps({"probe": "m2p_mma", "data": "synthetic far field: 8192 groups x 32 cells, Yukawa kappa = 0.125, single set", **res}))
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
