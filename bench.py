#!/usr/bin/env python
"""bench.py -- headline benchmark of the ipole-b200 hot path (BASELINE.json metric: rays/s and full-Stokes FP64
images/s at 4096^2; FP64 roofline fraction).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload adaf4096|grid4096|...]

One "step" = one full-Stokes FP64 image of the workload (all rows of SURVEY.md 8(a): camera init, geodesics,
path storage, plasma model, coefficients, transfer, image write, sort, reduction).  N > 1: one process per GPU
(torchrun), every rank renders the same workload (rays are independent: weak scaling, no data-path collective);
`value` = rays of all ranks / max-over-ranks device time.

Prints ONE JSON line (rank 0).  See DESIGN.md section 8 for how every field is derived.
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

# ALGORITHMIC FP64 operations per geodesic step (DFMA = 2, DADD = DMUL = 1): the lean counts of the round-1 kernels,
# FROZEN as the method's work (profiles/r1_k_*.txt).  roofline.frac uses these fixed numerators over
# the live CUDA-event time, so a faster kernel can only raise it; what the shipped kernels actually execute is reported
# beside it (FLOP_EXECUTED, frac_executed).  Grid transfer: 786 per WALKED step = 390 averaged over all steps of a ray.
FLOP_PER_STEP = {"transfer_adaf": 1576.0, "transfer_grid": 390.0, "geodesic_adaf": 994.0, "geodesic_grid": 1183.0}
# executed by the kernels as shipped, per step: smsp__sass_thread_inst_executed_op_d{fma,add,mul}_pred_on summed over EVERY
# launch of a run / the steps of the run (profiles/r2_image_flops.md, made by --summarize-launches); and their FP64-pipe
# utilisation (sm__inst_executed_pipe_fp64) in a bulk launch of the ncu --set full captures profiles/r2_k_*.txt.
# k_transfer<adaf> (single kernel, --single-kernel) and the path-free / unpolarized variants: profiles/r1_k_*.txt.
FLOP_EXECUTED = {"k_stepop": 1019.0, "k_apply": 585.0, "k_transfer<adaf>": 1576.0, "k_transfer_group<grid>": 397.0,
                 "k_geodesic": 839.0, "k_geodesic<occ>": 1020.0}
# second physics workload (--edf): k_apply<true> per step, 128 quadrature nodes (profiles/r2_k_apply_edf{1,2}_adaf256.txt)
FLOP_EXECUTED.update({"k_apply<edf 1>": 11558.0, "k_apply<edf 2>": 18290.0})
# unpolarized sweep on the operator records, per (step, parameter set): ncu per-launch counters of two launches of a sweep128 call
# (1.047e12 flop over 2.981e9 pairs; 216 FP64 instructions per pair, FP64 pipe 68.9 %)
FLOP_EXECUTED["k_apply_unpol_sweep"] = 351.0
# grid sweep (gridsweep.cuh), per step of a RAY (all its steps): k_gridop once per call, k_gridapply_sweep per parameter set
# (ncu per-launch counters of a gridsweep128 call: 359.0, and 3647.6 for 64 sets)
FLOP_EXECUTED.update({"k_gridop": 359.0, "k_gridapply_sweep": 57.0})
FP64_PIPE_PCT = {"k_stepop": 72.6, "k_apply": 61.7, "k_transfer<adaf>": 58.5, "k_transfer_group<grid>": 50.6,
                 "k_geodesic": 82.5, "k_geodesic<occ>": 79.5, "k_apply<edf 1>": 75.4, "k_apply<edf 2>": 70.1}
# DRAM bytes per step of k_transfer (dram__bytes_read + write of one launch / its thread-steps, same captures)
DRAM_BYTES_PER_STEP = {"transfer_adaf": 64.2, "transfer_grid": 37.2}
DRAM_BYTES_PER_STEP_SPLIT = 192.0   # k_stepop reads 64.1 B and writes 64.0 B per step, k_apply reads 64.0 B (profiles/r2_k_*.txt)
# --unpolarized: per step of k_transfer_unpol<model> (ncu, profiles/r1_unpolarized.md)
FLOP_PER_STEP_UNPOL = {"transfer_adaf": 652.0, "transfer_grid": 76.4}   # grid: 601 per walked step, 12.7 % of the steps walked
# --path-free (PAPER.md:43 variant): per FORWARD step of k_transfer<model, 1> (RK4 push + transfer step in one kernel)
FLOP_PER_STEP_PF = {"transfer_adaf": 2559.0, "transfer_grid": 1587.0}
DRAM_BYTES_PER_STEP_PF = {"transfer_adaf": 0.1, "transfer_grid": 1.0}
# ALU roofline denominator: 148 SMs x 4 sub-partitions x 16 FP64 lanes x 2 flop x 1.965 GHz
FP64_PEAK_TFLOPS = 148 * 4 * 16 * 2 * 1.965e9 / 1e12

WORKLOADS = {
    "adaf4096": dict(kind="adaf", n=4096, config=4),
    "grid4096": dict(kind="grid", n=4096, config=4, grid=(576, 256, 256)),
    "grid1024": dict(kind="grid", n=1024, config=3, grid=(576, 256, 256), maps=True),
    "grid256": dict(kind="grid", n=256, config=2, grid=(288, 128, 128)),
    "adaf1024": dict(kind="adaf", n=1024, config=None),   # profiling size (ncu --set full replays each kernel ~40x)
    "adaf256": dict(kind="adaf", n=256, config=1),
    "adaf32": dict(kind="adaf", n=32, config=0),
    # many-small-images mode (128x128 images for model fitting): 64 parameter sets per call
    "sweep128": dict(kind="adaf", n=128, config=None, sweep=64),
    "gridsweep128": dict(kind="grid", n=128, config=None, sweep=64, grid=(288, 128, 128)),
    # small images whose GEOMETRY differs (inclination, spin): one ipole_make_images_cameras call over the union of their rays
    "cams128": dict(kind="adaf", n=128, config=None, cams=64),
    # the same for the grid model: one snapshot seen from 64 directions at three frequencies (spin and mass are the grid's)
    "gridcams128": dict(kind="grid", n=128, config=None, cams=64, grid=(288, 128, 128)),
}


def sweep_models(M):
    """Parameter sets of the model-fitting sweep: density, temperature and field scales on a seeded log-uniform draw."""
    import numpy as np
    rng = np.random.default_rng(230202733)
    return [dict(n0=1e6 * 10 ** rng.uniform(-0.5, 0.5), Th0=30.0 * 10 ** rng.uniform(-0.3, 0.3),
                 B0=30.0 * 10 ** rng.uniform(-0.3, 0.3)) for _ in range(M)]


def sweep_sets(M, desc):
    import numpy as np
    rng = np.random.default_rng(230202733)
    return [dict(M_unit=desc["M_unit"] * 10 ** rng.uniform(-0.5, 0.5), Rlow=1.0, Rhigh=10 ** rng.uniform(0.0, 2.0)) for _ in range(M)]


def run_sweep(args, g, ipole, replicas, W, wl, cam, world, rank, local, barrier, grid=None):
    """One step = one ipole_make_images_{adaf,grid} call: M full-Stokes images of one camera (geodesics shared)."""
    import torch
    M, n = wl["sweep"], wl["n"]
    is_grid = wl["kind"] == "grid"
    models = sweep_sets(M, grid[0]) if is_grid else sweep_models(M)
    make_images = g.make_images_grid if is_grid else g.make_images_adaf
    if is_grid:
        def load_one(mod):
            d = dict(grid[0]); d.update(mod); g.load_grid(d, grid[1])
    else:
        def load_one(mod):
            g.load_adaf(**mod)
    names = ["I", "Q", "U", "V"]
    out = {k: torch.empty((M, n, n), dtype=torch.float64, device="cuda") for k in names}
    for _ in range(args.warmup):
        make_images(models, out=out)
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    ev0.record()
    for _ in range(args.steps):
        make_images(models, out=out)
    ev1.record()
    barrier()
    ms = replicas.max_over_ranks(ev0.elapsed_time(ev1), "cuda")
    st = g.stats()
    # the same images by M separate calls (what a fitting loop does without the batch entry)
    single = {k: torch.empty((n, n), dtype=torch.float64, device="cuda") for k in names}
    def separate():
        for mod in models:
            load_one(mod)
            g.make_image(out=single)
    separate()
    barrier()
    ev0.record()
    for _ in range(args.steps):
        separate()
    ev1.record()
    barrier()
    ms_sep = replicas.max_over_ranks(ev0.elapsed_time(ev1), "cuda")
    clocks = sampler.stop() if rank == 0 else None
    # e2e: host buffers out (M images), parameters in
    host = {k: torch.empty((M, n, n), dtype=torch.float64).pin_memory().numpy() for k in names}
    make_images(models, out=host)
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        g.set_camera(**cam)
        make_images(models, out=host)
    torch.cuda.synchronize()
    dt = replicas.max_over_ranks(time.perf_counter() - t0, "cuda")
    if rank != 0:
        return
    rays = M * n * n
    value = replicas.job_throughput(rays * args.steps, ms * 1e-3, world)
    rt_ms, steps_rt = st["ms_transfer"], st["total_steps"] * M
    dfma_tf, _ = g.fp64_peak()
    fkey = "transfer_" + wl["kind"]
    fl_step = (FLOP_PER_STEP_UNPOL[fkey] or 0.0) if args.unpolarized else FLOP_PER_STEP[fkey]
    ach = fl_step * steps_rt / (rt_ms * 1e-3) / 1e12
    kname = "k_transfer<%s, sweep>" % wl["kind"]
    flop_note = "flop per step of the single-image kernel (the sweep runs the same arithmetic per pair)"
    if st.get("ms_stepop", 0.0) > 0.0 and wl["kind"] == "grid" and not args.unpolarized:
        flop = st["total_steps"] * (FLOP_EXECUTED["k_gridop"] + M * FLOP_EXECUTED["k_gridapply_sweep"])
        ach = flop / (rt_ms * 1e-3) / 1e12
        fl_step = flop / steps_rt
        kname = "k_gridop (once) + k_gridapply_sweep (per parameter set)"
        flop_note = ("executed flop per (step of a ray, parameter set): k_gridapply_sweep's %.0f plus k_gridop's %.0f shared by the %d sets "
                     "of a call; the single sweep kernel's frozen count is 390 per pair, so the call does %.1fx the images per FP64 operation "
                     "-- and the launches are short and latency-bound, which is what the low fraction says"
                     % (FLOP_EXECUTED["k_gridapply_sweep"], FLOP_EXECUTED["k_gridop"], M, FLOP_PER_STEP[fkey] / fl_step))
    elif st.get("ms_stepop", 0.0) > 0.0 and args.unpolarized:
        flop = st["total_steps"] * (FLOP_EXECUTED["k_stepop"] + M * FLOP_EXECUTED["k_apply_unpol_sweep"])
        ach = flop / (rt_ms * 1e-3) / 1e12
        fl_step = flop / steps_rt
        kname = "k_stepop<adaf> (once) + k_apply_unpol_sweep (per parameter set)"
        flop_note = ("executed flop per (step, parameter set): k_apply_unpol_sweep's %.0f plus k_stepop's %.0f shared by the %d sets of a "
                     "call (the single unpolarized kernel: 652 per pair)" % (FLOP_EXECUTED["k_apply_unpol_sweep"], FLOP_EXECUTED["k_stepop"], M))
    elif st.get("ms_stepop", 0.0) > 0.0:
        # analytic flow through the split kernels: k_stepop ONCE per call, k_apply once per parameter set.  The work the sets
        # share is counted once: executed flop (profiles/r2_image_flops.md) of k_stepop x steps + of k_apply x steps x M
        flop = st["total_steps"] * (FLOP_EXECUTED["k_stepop"] + M * FLOP_EXECUTED["k_apply"])
        ach = flop / (rt_ms * 1e-3) / 1e12
        fl_step = flop / steps_rt
        kname = "k_stepop<adaf> (once) + k_apply<sweep> (per parameter set)"
        flop_note = ("executed flop per (step, parameter set): k_apply's %.0f plus k_stepop's %.0f shared by the %d sets of a call; "
                     "against the single kernel's frozen 1576 per pair the call does %.2fx the images per FP64 operation"
                     % (FLOP_EXECUTED["k_apply"], FLOP_EXECUTED["k_stepop"], M, FLOP_PER_STEP[fkey] / fl_step))
    line = {"metric": "rays_per_s", "value": value, "unit": "rays/s", "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": args.workload, "image": "%dx%d" % (n, n), "models_per_call": M, "model": wl["kind"],
                       "freq_ghz": 230, "eps": cam["eps"], "full_stokes": not args.unpolarized,
                       "variant": "unpolarized, I alone (PAPER.md:74)" if args.unpolarized else "full Stokes",
                       "note": "a ray here is one (pixel, parameter set) pair; the %d geodesics are integrated once per call" % (n * n),
                       "l2": "each call streams %.2f GB of path records once per warp (>> 126 MB L2)" % (st["total_steps"] * 64 / 1e9),
                       "parallelism": "single GPU" if world == 1 else "one replica per GPU"},
            "images_per_s": world * M * args.steps / (ms * 1e-3),
            "separate_calls": {"images_per_s": world * M * args.steps / (ms_sep * 1e-3), "ms_per_%d_images" % M: ms_sep / args.steps,
                               "speedup_of_the_batch_entry": ms_sep / ms},
            "stage_ms": {"probe_sort": st["ms_probe"], "geodesic": st["ms_geodesic"], "transfer": rt_ms, "stepop": st.get("ms_stepop", 0.0),
                         "apply": st.get("ms_apply", 0.0), "total": st["ms_total"]},
            "gpu_launches": st["n_launches"] * args.steps,
            "roofline": {"bound": "alu", "kernel": kname, "peak": FP64_PEAK_TFLOPS, "unit": "TFLOP/s",
                         "peak_source": "derived: 148 SM x 64 FP64 lanes x 2 x 1.965 GHz; DFMA micro-benchmark on this GPU: %.1f" % dfma_tf,
                         "achieved": ach, "frac": ach / FP64_PEAK_TFLOPS, "flop_per_step": fl_step,
                         "flop_note": flop_note,
                         "avg_launch_ms": rt_ms, "kernel_share_of_step": rt_ms / st["ms_total"], "traffic": None},
            "e2e": {"value": replicas.job_throughput(rays * args.steps, dt, world), "unit": "rays/s",
                    "h2d_bytes_per_step": ipole.C.sizeof(ipole.Camera) + M * (ipole.C.sizeof(ipole.AdafParams) + 32),
                    "d2h_bytes_per_step": 4 * rays * 8 + M * 32},
            "clocks": clocks}
    if not args.no_cpu_baseline and world == 1:
        import numpy as np
        from oracle import ipole_ref
        cores = os.cpu_count() or 1
        r = ipole_ref.Ctx(**cam)
        if args.unpolarized:
            r.set_unpolarized(True)
        def ref_load(mod):
            if is_grid:
                d = dict(grid[0]); d.update(mod); r.load_grid(d, grid[1])
            else:
                r.load_adaf(**mod)
        pix = (np.arange(8, n, 16)[:, None] * n + np.arange(8, n, 16)[None, :]).ravel().astype(np.int64)
        t0 = time.perf_counter()
        nm = 0
        while time.perf_counter() - t0 < 10.0 and nm < M:
            ref_load(models[nm]); r.make_pixels(pix, nthreads=cores); nm += 1
        dtc = time.perf_counter() - t0
        line["cpu_baseline"] = {"value": nm * pix.size / dtc, "unit": "rays/s", "cores": cores, "kind": "oracle",
                                "sample": "%d parameter sets x %d rays (every 16th pixel of the %dx%d image), %.1f s; the oracle "
                                          "re-integrates the geodesics for every parameter set" % (nm, pix.size, n, n, dtc)}
    print(json.dumps(line), flush=True)



class ClockSampler:
    """nvidia-smi clocks / throttle reasons while the timed region runs (B200_PROFILING.md clocks line)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index = index
        self.rows = []
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        self.thread.join(timeout=2)
        sm, mx, reasons, power = [], [], set(), []
        for r in self.rows:
            try:
                sm.append(float(r[1])); mx.append(float(r[2])); power.append(float(r[3]))
            except (ValueError, IndexError):
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(power) if power else None, "samples": len(sm), "reasons": sorted(reasons)}


_GRID_CACHE = {}


def grid_inputs(shape):
    """The seeded FM-torus planes for a lattice shape, generated once per process (tens of seconds at 576x256x256)."""
    from paper_2302_02733_b200 import workloads as W
    if shape not in _GRID_CACHE:
        _GRID_CACHE.clear()
        _GRID_CACHE[shape] = W.fm_torus_grid(*shape)
    return _GRID_CACHE[shape]


def oracle_sample(workload, n_rays, nthreads, path_free=False, unpolarized=False, edf=0):
    """The CPU oracle, as it stands, on a strided sample of the workload's image.  Returns (rays, steps, seconds)."""
    import numpy as np
    from oracle import ipole_ref
    from paper_2302_02733_b200 import workloads as W
    wl = WORKLOADS[workload]
    cam = W.camera(wl["kind"], wl["n"])
    r = ipole_ref.Ctx(**cam)
    if wl["kind"] == "adaf":
        r.load_adaf(**W.ADAF)
    else:
        desc, fields = grid_inputs(tuple(wl["grid"]))
        r.load_grid(desc, fields)
    if path_free:
        r.set_path_free(True)
    if unpolarized:
        r.set_unpolarized(True)
    if edf:
        r.set_edf(edf)
    n = wl["n"]
    stride = max(1, int(round(n / max(1.0, n_rays ** 0.5))))
    ii, jj = np.meshgrid(np.arange(stride // 2, n, stride), np.arange(stride // 2, n, stride))
    pix = (jj * n + ii).ravel().astype(np.int64)
    t0 = time.perf_counter()
    r.make_pixels(pix, nthreads=nthreads)
    dt = time.perf_counter() - t0
    return pix.size, r.total_steps(), dt, stride


def run_cams(args, ipole, replicas, W, wl, world, rank, local, barrier):
    """One step = one ipole_make_images_cameras call: `cams` 128x128 images whose geometry differs (inclination and spin),
    from ONE host thread and one context, in one pass of the pipeline over the union of their rays; compared with the same
    images made one after the other by ipole_set_camera + ipole_make_image."""
    import torch
    n, nc = wl["n"], wl["cams"]
    incl = [15.0 + 150.0 * k / max(1, nc - 1) for k in range(nc)]
    grid = wl["kind"] == "grid"
    if grid:   # a grid belongs to one spacetime: its cameras vary direction and frequency
        spins = [W.camera("grid", n)["spin"]]
        freqs = [230e9, 345e9, 86e9]
        cams = [W.camera("grid", n, inclination_deg=a, freq_hz=freqs[k % 3]) for k, a in enumerate(incl)]
    else:
        spins = [0.0, 0.5, 0.9375, 0.99]
        freqs = [230e9]
        cams = [W.camera("adaf", n, inclination_deg=a, spin=spins[k % 4]) for k, a in enumerate(incl)]
    names = ["I", "Q", "U", "V"]
    g = ipole.Ipole(**cams[0])
    if grid:
        desc, fields = grid_inputs(tuple(wl["grid"]))
        g.load_grid(desc, fields)
    else:
        g.load_adaf(**W.ADAF)
    g.set_stream(torch.cuda.current_stream())
    out = {k: torch.empty((nc, n, n), dtype=torch.float64, device="cuda") for k in names}
    single = {k: torch.empty((n, n), dtype=torch.float64, device="cuda") for k in names}

    def batched():
        g.make_images_cameras(cams, out=out)

    def one_by_one():
        for cam in cams:
            g.set_camera(**cam)
            g.make_image(out=single)

    res, st = {}, None
    for name, fn in (("batched", batched), ("one_by_one", one_by_one)):
        for _ in range(args.warmup):
            fn()
        barrier()
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ev0.record()
        for _ in range(args.steps):
            fn()
        ev1.record()
        barrier()
        res[name] = replicas.max_over_ranks(ev0.elapsed_time(ev1), "cuda") * 1e-3 / args.steps
        if name == "batched":
            st = g.stats()
            if st.get("n_lanes", 1) == 2:   # per-kernel times: one more call with the batches on one stream (see measure_image)
                g.set_batch_overlap(False)
                fn(); fn()
                torch.cuda.synchronize()
                st = g.stats()
                g.set_batch_overlap(True)
    g.set_camera(**cams[0])
    host = {k: torch.empty((nc, n, n), dtype=torch.float64).pin_memory().numpy() for k in names}
    g.make_images_cameras(cams, out=host)
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        g.make_images_cameras(cams, out=host)
    torch.cuda.synchronize()
    dt = replicas.max_over_ranks(time.perf_counter() - t0, "cuda") / args.steps
    if rank != 0:
        return
    rays = nc * n * n
    fl = FLOP_PER_STEP["transfer_grid" if grid else "transfer_adaf"]
    line = {"metric": "rays_per_s", "value": world * rays / res["batched"], "unit": "rays/s", "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": res["batched"] * 1e3, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": args.workload, "image": "%dx%d" % (n, n), "cameras": nc, "inclinations_deg": [incl[0], incl[-1]],
                       "spins": spins, "model": wl["kind"], "freq_ghz": [f / 1e9 for f in freqs], "full_stokes": True,
                       "timing": "CUDA events around ipole_make_images_cameras from one host thread, one context",
                       "l2": "no flush needed: each call streams %.1f GB of path and operator records" % (st["total_steps"] * 128 / 1e9),
                       "parallelism": "single GPU"},
            "images_per_s": world * nc / res["batched"],
            "one_by_one": {"images_per_s": world * nc / res["one_by_one"], "ms_per_%d_images" % nc: res["one_by_one"] * 1e3,
                           "speedup_of_the_batch_entry": res["one_by_one"] / res["batched"]},
            "stage_ms": {"probe_sort": st["ms_probe"], "geodesic": st["ms_geodesic"], "transfer": st["ms_transfer"], "stepop": st["ms_stepop"],
                         "apply": st["ms_apply"], "total": st["ms_total"], "batches": st["n_batches"]},
            "gpu_launches": st["n_launches"] * args.steps,
            "roofline": {"bound": "alu", "kernel": "k_transfer_group<grid, cameras>" if grid else "k_stepop<adaf, cameras> + k_apply", "peak": FP64_PEAK_TFLOPS, "unit": "TFLOP/s",
                         "achieved": fl * st["total_steps"] / (st["ms_transfer"] * 1e-3) / 1e12,
                         "frac": fl * st["total_steps"] / (st["ms_transfer"] * 1e-3) / 1e12 / FP64_PEAK_TFLOPS,
                         "flop_per_step_algorithmic": fl,
                         "traffic": (DRAM_BYTES_PER_STEP["transfer_grid"] if grid else DRAM_BYTES_PER_STEP_SPLIT) * st["total_steps"] / max(1, st["n_batches"])},
            "e2e": {"value": world * rays / dt, "unit": "rays/s", "h2d_bytes_per_step": nc * ipole.C.sizeof(ipole.Camera),
                    "d2h_bytes_per_step": 4 * rays * 8 + nc * 32}}
    print(json.dumps(line), flush=True)


def run_fp32_study(args, ipole, W, wl):
    """--fp32-geodesic: the same image with the geodesics integrated in single precision
    (ipole_set_geodesic_fp32; transfer still FP64) beside the FP64 image: stage times and per-pixel differences.  A study
    line, not a bench value: `value` is the FP32-geodesic image's rays/s."""
    import torch
    n = wl["n"]
    cam = W.camera("adaf", n)
    g = ipole.Ipole(**cam); g.set_stream(torch.cuda.current_stream()); g.load_adaf(**W.ADAF)
    ref = {k: torch.empty((n, n), dtype=torch.float64, device="cuda") for k in "IQUV"}
    out = {k: torch.empty((n, n), dtype=torch.float64, device="cuda") for k in "IQUV"}
    for _ in range(args.warmup + args.steps):
        g.make_image(out=ref)
    torch.cuda.synchronize(); s64 = g.stats(); ns64, nt64 = g.ray_info()
    g.set_geodesic_fp32(True)
    for _ in range(args.warmup + args.steps):
        g.make_image(out=out)
    torch.cuda.synchronize(); s32 = g.stats(); ns32, nt32 = g.ray_info()
    I = ref["I"]; peak = float(I.max())
    rel = ((out["I"] - I).abs() / (I.abs() + 1e-300)).flatten()
    lit = (I > 1e-6 * peak).flatten()
    pol = torch.maximum(torch.maximum((out["Q"] - ref["Q"]).abs(), (out["U"] - ref["U"]).abs()), (out["V"] - ref["V"]).abs()).flatten() / peak
    sub = rel[lit][:: max(1, int(lit.sum()) // 2000000)]
    line = {"metric": "rays_per_s", "value": n * n / (s32["ms_total"] * 1e-3), "unit": "rays/s", "n_gpus": 1, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": s32["ms_total"], "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32 geodesics + f64 transfer (study)", "data": "synthetic",
            "config": {"workload": args.workload, "image": "%dx%d" % (n, n), "model": "adaf", "variant": "FP32 study, not a product path"},
            "fp32_study": {"ms_geodesic_f64": s64["ms_geodesic"], "ms_geodesic_f32": s32["ms_geodesic"],
                           "ms_image_f64": s64["ms_total"], "ms_image_f32": s32["ms_total"],
                           "geodesic_speedup": s64["ms_geodesic"] / s32["ms_geodesic"], "image_speedup": s64["ms_total"] / s32["ms_total"],
                           "rel_dI_median": float(sub.median()), "rel_dI_p99": float(torch.quantile(sub, 0.99)),
                           "rel_dI_max": float(rel[lit].max()), "dI_over_peak_max": float(((out["I"] - I).abs() / peak).max()),
                           "dQUV_over_peak_max": float(pol.max()),
                           "flux_rel": [abs(a / b - 1) if b else 0.0 for a, b in zip(s32["flux_jy"], s64["flux_jy"])],
                           "rays_with_other_step_count": float((ns64 != ns32).mean()), "rays_with_other_turn_count": float((nt64 != nt32).mean()),
                           "note": "differences are FP32-geodesic image minus the FP64 image of this library (which matches the oracle "
                                   "to <= 1e-9 per pixel, tests/test_gpu_parity.py); pixels brighter than 1e-6 of the peak"},
            "gpu_launches": s32["n_launches"], "roofline": None, "e2e": None}
    print(json.dumps(line), flush=True)


def run_adaptive(args, g, replicas, wl, cam, world, rank, local, barrier):
    """One step = one ipole_make_image_adaptive call; the full image of the same workload is made once for the error."""
    import torch
    n = wl["n"]
    names = ["I", "Q", "U", "V"]
    full = g.make_image()
    st_full = g.stats()
    peak = float(full["I"].max())
    rel, ab = 0.02, 1e-3 * peak
    out = {k: torch.empty((n, n), dtype=torch.float64, device="cuda") for k in names}
    for _ in range(args.warmup):
        g.make_image_adaptive(args.adaptive, rel, ab, out=out)
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    ev0.record()
    for _ in range(args.steps):
        res, info = g.make_image_adaptive(args.adaptive, rel, ab, out=out)
    ev1.record()
    barrier()
    ms = replicas.max_over_ranks(ev0.elapsed_time(ev1), "cuda")
    clocks = sampler.stop() if rank == 0 else None
    host = {k: torch.empty((n, n), dtype=torch.float64).pin_memory().numpy() for k in names}
    g.make_image_adaptive(args.adaptive, rel, ab, out=host)
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        g.set_camera(**cam)
        g.make_image_adaptive(args.adaptive, rel, ab, out=host)
    torch.cuda.synchronize()
    dt = replicas.max_over_ranks(time.perf_counter() - t0, "cuda")
    if rank != 0:
        return
    err = (out["I"] - full["I"]).abs() / peak
    pol = torch.maximum(torch.maximum((out["Q"] - full["Q"]).abs(), (out["U"] - full["U"]).abs()), (out["V"] - full["V"]).abs()) / peak
    pix = n * n
    line = {"metric": "rays_per_s", "value": replicas.job_throughput(pix * args.steps, ms * 1e-3, world), "unit": "rays/s",
            "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": args.workload, "image": "%dx%d" % (n, n), "model": wl["kind"], "freq_ghz": 230, "eps": cam["eps"],
                       "full_stokes": True, "variant": "adaptive ray tracing (PAPER.md:70): %d lattice levels, rel_tol %.3g, "
                                                        "abs_tol 1e-3 of the brightest pixel" % (args.adaptive, rel),
                       "note": "value counts image PIXELS delivered per second; the rays actually followed are in `adaptive`",
                       "l2": "no flush needed: every level streams its own path buffer", "parallelism": "single GPU"},
            "images_per_s": world * args.steps / (ms * 1e-3),
            "adaptive": {"rays_followed": info["n_traced"], "fraction_of_pixels": info["n_traced"] / pix,
                         "per_level": info["n_traced_level"], "rays_followed_per_s": info["n_traced"] * args.steps / (ms * 1e-3),
                         "geodesic_steps": info["total_steps"], "speedup_vs_full_image": st_full["ms_total"] / (ms / args.steps),
                         "full_image_ms": st_full["ms_total"],
                         "error_vs_full_image": {"I_max_over_peak": float(err.max()), "I_p99_over_peak": float(torch.quantile(err.flatten()[:: max(1, pix // 1000000)], 0.99)),
                                                 "QUV_max_over_peak": float(pol.max()),
                                                 "total_flux_rel": abs(float(out["I"].sum()) / float(full["I"].sum()) - 1)}},
            "gpu_launches": info["n_launches"] * args.steps,
            "roofline": {"bound": "alu", "kernel": "k_transfer<%s>" % wl["kind"], "peak": FP64_PEAK_TFLOPS, "unit": "TFLOP/s",
                         "achieved": None, "frac": None, "traffic": None,
                         "note": "the per-ray kernels are those of the full image (see the default bench line); this line measures the ray saving"},
            "e2e": {"value": replicas.job_throughput(pix * args.steps, dt, world), "unit": "rays/s",
                    "h2d_bytes_per_step": 160, "d2h_bytes_per_step": 4 * pix * 8 + pix},
            "clocks": clocks}
    print(json.dumps(line), flush=True)


def measure_image(args, name, ipole, replicas, W, world, rank, local, barrier):
    """Time `args.steps` full-Stokes images of workload `name` through ipole_make_image (device outputs), then the same
    through host buffers (e2e), the roofline of the transfer stage, and the oracle on a strided sample.  Returns the
    JSON line as a dict (rank 0; None elsewhere)."""
    import torch
    wl = WORKLOADS[name]
    cam = W.camera(wl["kind"], wl["n"])
    g = ipole.Ipole(**cam)
    g.set_stream(torch.cuda.current_stream())
    if args.path_free:
        g.set_path_free(True)
    if args.unpolarized:
        g.set_unpolarized(True)
    if args.single_kernel:
        g.set_transfer_split(False)
    if args.edf:
        g.set_edf(args.edf)
    grid_bytes = 0
    if wl["kind"] == "adaf":
        g.load_adaf(**W.ADAF)
    else:
        desc, fields = grid_inputs(tuple(wl["grid"]))
        g.load_grid(desc, fields)
        grid_bytes = fields.nbytes
        del fields
    maps = bool(wl.get("maps"))
    names = ["I", "Q", "U", "V"] + (["tau", "tauF"] if maps else [])
    out = {k: torch.empty((wl["n"], wl["n"]), dtype=torch.float64, device="cuda") for k in names}
    rays = wl["n"] * wl["n"]

    for _ in range(args.warmup):
        g.make_image(maps=maps, out=out)
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    ev0.record()
    host_s = 0.0
    for _ in range(args.steps):
        th = time.perf_counter()
        g.make_image(maps=maps, out=out)
        host_s += time.perf_counter() - th      # the call alone: with a reused plan it only enqueues (ipole_set_plan_reuse)
    ev1.record()
    barrier()
    ms = ev0.elapsed_time(ev1)
    st = g.stats()  # of the last timed image (event times are per image)
    st_live = st
    st_plan = st
    host_idle = None
    if st.get("n_lanes", 1) == 2 or st.get("plan_reused", 0):
        # The timed images ran with consecutive batches side by side on two streams (ipole_set_batch_overlap): the event
        # spans of concurrent kernels overlap, so the per-kernel times come from one more image with the lanes off.  The
        # first image after the switch plans afresh (probe pass: its time is the probe_sort entry), the second reuses
        # that plan like the timed ones.
        g.set_batch_overlap(False)
        g.make_image(maps=maps, out=out)
        torch.cuda.synchronize()
        st_plan = g.stats()
        th = time.perf_counter()
        g.make_image(maps=maps, out=out)
        host_idle = time.perf_counter() - th      # a reused-plan call into an empty launch queue
        torch.cuda.synchronize()
        st = g.stats()
        g.set_batch_overlap(True)
    # one image planned afresh with everything else as timed: what the first call for a camera costs
    planning = None
    if st_live.get("plan_reused", 0) and not (args.path_free or args.edf):
        g.set_plan_reuse(False)
        tp = time.perf_counter()
        g.make_image(maps=maps, out=out)
        host_plan = time.perf_counter() - tp
        torch.cuda.synchronize()
        sp = g.stats()
        planning = {"ms_total": sp["ms_total"], "ms_probe": sp["ms_probe"], "host_call_ms": host_plan * 1e3, "gpu_launches": sp["n_launches"]}
        g.set_plan_reuse(True)
    clocks = sampler.stop() if rank == 0 else None
    ms = replicas.max_over_ranks(ms, "cuda")
    value = replicas.job_throughput(rays * args.steps, ms * 1e-3, world)

    # ---- e2e: the C-ABI call with HOST buffers (parameters in, image out), copies inside the timed region ----
    e2e = None
    if not args.no_e2e:
        host = {k: torch.empty((wl["n"], wl["n"]), dtype=torch.float64).pin_memory() for k in names}
        hnp = {k: v.numpy() for k, v in host.items()}
        h2d = 0
        def one_e2e():
            nonlocal h2d
            g.set_camera(**cam)                       # parameters travel host -> device every step
            h2d = ipole.C.sizeof(ipole.Camera)
            if wl["kind"] == "adaf":
                g.load_adaf(**W.ADAF); h2d += ipole.C.sizeof(ipole.AdafParams)
            g.make_image_host(maps=maps, out=hnp)     # synchronises: outputs are host pointers
        one_e2e()
        barrier()
        t0 = time.perf_counter()
        for _ in range(args.steps):
            one_e2e()
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        dt = replicas.max_over_ranks(dt, "cuda")
        e2e = {"value": replicas.job_throughput(rays * args.steps, dt, world), "unit": "rays/s", "h2d_bytes_per_step": h2d,
               "d2h_bytes_per_step": len(names) * rays * 8,
               "note": "inputs of this workload are parameters only (analytic model)" if wl["kind"] == "adaf" else
                       "grid planes (%d bytes) are loaded once by ipole_load_model_grid, outside the step" % grid_bytes}
        del host, hnp
    if rank != 0:
        g.close()
        return None

    # ---- roofline of the transfer stage (67 % of the image), live CUDA-event time of the last timed image ----
    key = "transfer_" + wl["kind"]
    pf = args.path_free
    split = st["ms_stepop"] > 0.0
    fl_rt = FLOP_PER_STEP_PF[key] if pf else FLOP_PER_STEP[key]
    if args.edf:   # no round-1 count exists for this workload: its algorithmic count IS the executed one (k_stepop + k_apply<edf>)
        fl_rt = FLOP_EXECUTED["k_stepop"] + FLOP_EXECUTED["k_apply<edf %d>" % args.edf]
    if args.unpolarized:
        fl_rt = FLOP_PER_STEP_UNPOL[key] or 0.0
    # steps the bulk transfer kernels walk: the long rays (>= path_cap steps each) run on the side stream, outside rt_ms
    rt_steps = st["total_steps_forward"] if pf else st["total_steps"] - st["n_long"] * st["path_cap"]
    dram_rt = DRAM_BYTES_PER_STEP_PF[key] if pf else (DRAM_BYTES_PER_STEP_SPLIT if split else DRAM_BYTES_PER_STEP[key])
    dfma_tf, _ = g.fp64_peak()
    n_rt = max(1, st["n_batches"])          # bulk launches; the long-ray passes run beside them on a side stream
    rt_ms = st["ms_transfer"]
    if args.unpolarized:
        kname = "k_transfer_unpol<%s>" % wl["kind"]
    elif split:
        kname = "k_stepop<%s> + k_apply (split transfer)" % wl["kind"]
    else:
        kname = "k_transfer_group<grid>" if (wl["kind"] == "grid" and not pf) else "k_transfer<%s%s>" % (wl["kind"], ", path-free" if pf else "")
    roof = {"bound": "alu", "kernel": kname, "peak": FP64_PEAK_TFLOPS, "unit": "TFLOP/s",
            "peak_source": "derived: 148 SM x 64 FP64 lanes x 2 x 1.965 GHz; DFMA micro-benchmark on this GPU: %.1f" % dfma_tf,
            "launches": n_rt * (2 if split else 1), "avg_launch_ms": rt_ms / n_rt, "kernel_share_of_step": rt_ms / st["ms_total"],
            "steps_per_launch": rt_steps / n_rt,
            "traffic": dram_rt * rt_steps / n_rt,
            "traffic_note": "ncu dram__bytes_read+write per step of the stage (profiles/), scaled by the steps of a batch; "
                            + ("algorithmic: 64 B read and 32-48 B written per RAY, nothing per step" if pf else
                               "algorithmic: 64 B path record read + 64 B operator record written and read per step" if split else
                               "algorithmic: 64 B per step (one path record read)")}
    ach = fl_rt * rt_steps / (rt_ms * 1e-3) / 1e12
    roof.update(achieved=ach, frac=ach / FP64_PEAK_TFLOPS, flop_per_step_algorithmic=fl_rt,
                flop_note="frac = frozen algorithmic flop per step (round-1 lean count, DESIGN.md section 7) x steps / live "
                          "CUDA-event time / peak; frac_executed uses what the shipped kernels execute (ncu); "
                          "fp64_pipe_pct is sm__inst_executed_pipe_fp64 of the ncu captures under profiles/, not live")
    if not (pf or args.unpolarized):
        if args.edf:
            parts = {"k_stepop": st["ms_stepop"], "k_apply<edf %d>" % args.edf: st["ms_apply"]}
        elif split:
            parts = {"k_stepop": st["ms_stepop"], "k_apply": st["ms_apply"]}
        else:
            parts = {("k_transfer_group<grid>" if wl["kind"] == "grid" else "k_transfer<%s>" % wl["kind"]): rt_ms}
        roof["kernels"] = {k: {"ms": v, "flop_per_step_executed": FLOP_EXECUTED[k], "fp64_pipe_pct": FP64_PIPE_PCT[k],
                               "tflops_executed": FLOP_EXECUTED[k] * rt_steps / (v * 1e-3) / 1e12,
                               "frac_executed": FLOP_EXECUTED[k] * rt_steps / (v * 1e-3) / 1e12 / FP64_PEAK_TFLOPS}
                           for k, v in parts.items() if v > 0}
        fx = sum(FLOP_EXECUTED[k] for k in parts)
        roof["flop_per_step_executed"] = fx
        roof["frac_executed"] = fx * rt_steps / (rt_ms * 1e-3) / 1e12 / FP64_PEAK_TFLOPS
        roof["fp64_pipe_pct"] = sum(FP64_PIPE_PCT[k] * v for k, v in parts.items()) / max(1e-9, sum(parts.values()))
    # the whole step against the same roofline: the algorithmic FP64 operations of both stages over the image time
    gkey = "geodesic_" + wl["kind"]
    fl_step = fl_rt * rt_steps + FLOP_PER_STEP[gkey] * st["total_steps"]
    gk = "k_geodesic<occ>" if wl["kind"] == "grid" else "k_geodesic"
    roof["whole_step"] = {"achieved": fl_step / (st_live["ms_total"] * 1e-3) / 1e12,
                          "frac": fl_step / (st_live["ms_total"] * 1e-3) / 1e12 / FP64_PEAK_TFLOPS,
                          "geodesic_tflops": FLOP_PER_STEP[gkey] * st["total_steps"] / (st["ms_geodesic"] * 1e-3) / 1e12,
                          "geodesic_frac": FLOP_PER_STEP[gkey] * st["total_steps"] / (st["ms_geodesic"] * 1e-3) / 1e12 / FP64_PEAK_TFLOPS,
                          "geodesic_fp64_pipe_pct": FP64_PIPE_PCT[gk]}
    path_bytes = 0.0 if pf else (256.0 if split else 128.0)
    roof["hbm_path_gbs"] = path_bytes * st["total_steps"] / ((st["ms_geodesic"] + st["ms_transfer"]) * 1e-3) / 1e9
    # The roofline object describes the DOMINANT kernel.  Stored path: the geodesic kernel is one launch per batch like the
    # transfer stage; where it takes the larger share of the image (the grid model: k_geodesic<occ>) it becomes the
    # top-level entry and the transfer stage moves to roofline.other_stage, else the other way round.
    if not (pf or args.unpolarized or args.edf):
        gms = st["ms_geodesic"]
        gach = FLOP_PER_STEP[gkey] * st["total_steps"] / (gms * 1e-3) / 1e12
        geo = {"bound": "alu", "kernel": "k_geodesic<true> (h != 1, stencil-occupancy test)" if wl["kind"] == "grid" else "k_geodesic<false>",
               "peak": FP64_PEAK_TFLOPS, "unit": "TFLOP/s", "launches": n_rt, "avg_launch_ms": gms / n_rt,
               "kernel_share_of_step": gms / st["ms_total"], "steps_per_launch": st["total_steps"] / n_rt,
               "traffic": 64.0 * st["total_steps"] / n_rt,
               "traffic_note": "ncu dram__bytes_write per step (64.0-64.1 B: one path record, profiles/r2_k_geodesic_*.txt) x steps of a batch; algorithmic: the same 64 B",
               "achieved": gach, "frac": gach / FP64_PEAK_TFLOPS, "flop_per_step_algorithmic": FLOP_PER_STEP[gkey],
               "flop_per_step_executed": FLOP_EXECUTED[gk],
               "frac_executed": FLOP_EXECUTED[gk] * st["total_steps"] / (gms * 1e-3) / 1e12 / FP64_PEAK_TFLOPS,
               "fp64_pipe_pct": FP64_PIPE_PCT[gk]}
        if gms > rt_ms:
            for k in ("peak_source", "flop_note", "whole_step", "hbm_path_gbs"):
                geo[k] = roof.pop(k)
            geo["other_stage"] = roof
            roof = geo
        else:
            roof["other_stage"] = geo

    line = {"metric": "rays_per_s", "value": value, "unit": "rays/s", "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": name, "configs_index": wl["config"], "image": "%dx%d" % (wl["n"], wl["n"]),
                       "model": wl["kind"], "freq_ghz": 230, "eps": cam["eps"], "maps": maps,
                       "variant": "unpolarized, I alone (PAPER.md:74), stored path" if args.unpolarized else
                                  "path-free bidirectional (PAPER.md:43)" if pf else
                                  "stored path, split transfer, j and alpha integrated over the eDF at every step (PAPER.md:78; kind %d)" % args.edf if args.edf else
                                  "stored path, split transfer (k_stepop + k_apply)" if split else "stored path, single transfer kernel",
                       "full_stokes": not args.unpolarized,
                       "l2": ("no flush needed: nothing is re-read; per image %.2f GB of end points and outputs stream once"
                              % (rays * (64.0 + 8.0 * len(names)) / 1e9)) if pf else
                             "no flush needed: every batch streams %.1f GB of path and operator records (>> 126 MB L2)"
                             % (path_bytes / 2 * st["total_steps"] / max(1, st["n_batches"]) / 1e9),
                       "parallelism": "rays sharded: one replica per GPU" if world > 1 else "single GPU"},
            "images_per_s": value / rays, "steps_per_s": world * st["total_steps"] * args.steps / (ms * 1e-3),
            "mean_steps_per_ray": st["total_steps"] / rays, "forward_steps": st["total_steps_forward"],
            "stage_ms": {"probe_sort": st_plan["ms_probe"], "geodesic": st["ms_geodesic"], "transfer": st["ms_transfer"],
                         "stepop": st["ms_stepop"], "apply": st["ms_apply"],
                         "long_rays_side_stream": st["ms_long"], "total": st["ms_total"], "batches": st["n_batches"], "path_cap": st["path_cap"],
                         "long_rays": st["n_long"], "retried_rays": st["n_retry"],
                         "lanes": st_live.get("n_lanes", 1), "total_timed_image": st_live["ms_total"], "batches_timed_image": st_live["n_batches"],
                         "note": ("the timed images alternate their batches between two streams (kernels of consecutive batches side by side: "
                                  "total_timed_image); the per-kernel times here and in roofline are of one more image with the lanes off (total)")
                                 if st_live.get("n_lanes", 1) == 2 else "one stream"},
            "flux_jy": st["flux_jy"], "lp": st["lp"], "cp": st["cp"], "ring_rays": st["n_ring"],
            "gpu_launches": st_live["n_launches"] * args.steps, "roofline": roof, "e2e": e2e, "clocks": clocks,
            "plan": {"reused": bool(st_live.get("plan_reused", 0)), "host_ms_per_call": host_s * 1e3 / args.steps,
                     "host_ms_per_call_idle_queue": None if host_idle is None else host_idle * 1e3,
                     "planning_call": planning,
                     "note": "the timed images are scheduled from the plan of the call before them (ipole_set_plan_reuse: same camera, no "
                             "probe pass, no host-device synchronisation; the call returns after host_ms_per_call while the GPU works for "
                             "ms_per_step -- in this back-to-back loop that includes waiting for room in the driver's launch queue when "
                             "several images of some 400 launches each are pending; host_ms_per_call_idle_queue is one such call after a "
                             "synchronise); planning_call = one image planned afresh (probe pass, read-backs, blocking), as the first "
                             "call for a camera is; stage_ms.probe_sort is that call's probe time and is not part of a reused image"},
            "paper_context": {"note": "paper Table 1, other model/hardware (A100): context only",
                              "a100_semianalytic_4096_rays_per_s": 127583, "a100_grmhd_4096_rays_per_s": 188720}}
    g.close()
    del out
    torch.cuda.empty_cache()

    if not args.no_cpu_baseline and world == 1:
        cores = os.cpu_count() or 1
        n, steps, dt, stride = oracle_sample(name, args.cpu_baseline_rays if not args.edf else min(args.cpu_baseline_rays, 256), cores,
                                             path_free=pf, unpolarized=args.unpolarized, edf=args.edf)
        line["cpu_baseline"] = {"value": n / dt, "unit": "rays/s", "cores": cores, "kind": "oracle",
                                "sample": "%d rays: every %d-th pixel in x and y of the %dx%d image, %.1f s"
                                          % (n, stride, wl["n"], wl["n"], dt),
                                "steps_per_s": steps / dt}
    return line

def reference_line(args, name, cores):
    """The oracle, as it stands, on a strided lattice of workload `name`: `args.steps` timed steps of `args.ref_rays` rays."""
    wl = WORKLOADS[name]
    n_rays = args.ref_rays
    for _ in range(args.warmup):
        oracle_sample(name, min(n_rays, 256), cores)
    rays = steps = 0
    dt = 0.0
    stride = 0
    for _ in range(args.steps):
        a, b, c, stride = oracle_sample(name, n_rays, cores)
        rays += a; steps += b; dt += c
    val = rays / dt
    return {"impl": "reference", "metric": "rays_per_s", "value": val, "unit": "rays/s", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": name, "configs_index": wl["config"], "image": "%dx%d" % (wl["n"], wl["n"]),
                       "model": wl["kind"], "freq_ghz": 230, "eps": 0.01, "maps": bool(wl.get("maps")), "full_stokes": True,
                       "variant": "CPU oracle (oracle/), one ray per work item, %d host threads" % cores,
                       "step": "oracle on every %d-th pixel in x and y (%d rays) of the image" % (stride, rays // args.steps)},
            "cpu_baseline": {"value": val, "unit": "rays/s", "cores": cores, "kind": "oracle",
                             "sample": "%d rays per step, strided lattice of the %dx%d image" % (rays // args.steps, wl["n"], wl["n"])},
            "e2e": {"value": val, "unit": "rays/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "steps_per_s": steps / dt, "gpu_launches": 0}


def run_reference(args):
    """--impl reference: the oracle on the box's host cores (rank 0 only).  Builds and loads the oracle alone: the
    product library is neither compiled nor opened in this arm."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import __graft_entry__ as ge
    ge.build_oracle()
    cores = os.cpu_count() or 1
    line = reference_line(args, args.workload, cores)
    if args.workload == "adaf4096" and not args.no_second_workload:   # the other half of configs[4], as in our arm
        other = reference_line(args, "grid4096", cores)
        for k in ("impl", "metric", "unit", "n_gpus", "steps", "warmup", "higher_is_better", "scaling", "vs_baseline", "dtype", "data"):
            other.pop(k, None)
        line["workloads"] = {"grid4096": other}
    print(json.dumps(line), flush=True)


NCU_KEYS = ["gpu__time_duration.sum", "launch__grid_size", "launch__block_size", "launch__registers_per_thread",
            "sm__warps_active.avg.pct_of_peak_sustained_active", "smsp__thread_inst_executed_per_inst_executed.ratio",
            "smsp__sass_average_branch_targets_threads_uniform.pct", "sm__inst_executed_pipe_fp64.avg.pct_of_peak_sustained_active",
            "smsp__issue_active.avg.pct_of_peak_sustained_active", "sm__inst_executed_pipe_alu.avg.pct_of_peak_sustained_active",
            "sm__inst_executed_pipe_lsu.avg.pct_of_peak_sustained_active", "l1tex__data_pipe_lsu_wavefronts.avg.pct_of_peak_sustained_elapsed",
            "smsp__inst_executed.sum", "dram__bytes_read.sum", "dram__bytes_write.sum",
            "gpu__dram_throughput.avg.pct_of_peak_sustained_elapsed", "l1tex__t_sector_hit_rate.pct", "lts__t_sector_hit_rate.pct",
            "sass__inst_executed_local_loads", "sass__inst_executed_local_stores", "sm__cycles_elapsed.avg"]


def summarize_ncu(args):
    """--summarize-ncu REPORT: the text summaries under profiles/ (no GPU needed: reads an .ncu-rep with the ncu CLI).
    Quoted counters come straight from `ncu -i REPORT --page raw --csv`; the lines after the blank line are DERIVED here:
    FP64 thread instructions = per_cycle_elapsed counters x sm__cycles_elapsed, flop = 2 DFMA + DADD + DMUL, and, with
    --ncu-steps-from read|write, per-step figures with steps = DRAM bytes read|written / --ncu-bytes-per-step."""
    import csv
    import io
    import re
    raw = subprocess.run(["ncu", "-i", args.summarize_ncu, "--page", "raw", "--csv"], capture_output=True, text=True, check=True).stdout
    rows = list(csv.reader(io.StringIO(raw)))
    hdr, units = rows[0], rows[1]
    mult = {"Gbyte": 1e9, "Mbyte": 1e6, "Kbyte": 1e3, "byte": 1.0}
    tmul = {"s": 1e3, "ms": 1.0, "us": 1e-3, "ns": 1e-6}   # -> ms (ncu picks the unit per report)
    for r in rows[2:]:
        d = dict(zip(hdr, r))
        if args.ncu_kernel and not re.search(args.ncu_kernel, d["Kernel Name"]):
            continue
        num = lambda k: float(d[k].replace(",", ""))
        un = lambda k: units[hdr.index(k)]
        print("%-78s %s" % ("Kernel Name", d["Kernel Name"]))
        for k in NCU_KEYS:
            if k in d:
                print("%-78s %s %s" % (k, d[k], un(k)))
        cyc = num("sm__cycles_elapsed.avg")
        ops = {k: num("smsp__sass_thread_inst_executed_op_%s_pred_on.sum.per_cycle_elapsed" % k) * cyc for k in ("dfma", "dadd", "dmul")}
        flop = 2 * ops["dfma"] + ops["dadd"] + ops["dmul"]
        ms = num("gpu__time_duration.sum") * tmul.get(un("gpu__time_duration.sum"), 1.0)
        print()
        print("FP64 thread instructions: DFMA %.4e  DADD %.4e  DMUL %.4e   flop (DFMA=2) %.4e" % (ops["dfma"], ops["dadd"], ops["dmul"], flop))
        tf = flop / (ms * 1e-3) / 1e12
        print("achieved %.2f TFLOP/s = %.3f of %.2f TFLOP/s (148 SM x 64 lanes x 2 x 1.965 GHz); FMA share of FP64 instructions %.2f"
              % (tf, tf / FP64_PEAK_TFLOPS, FP64_PEAK_TFLOPS, ops["dfma"] / sum(ops.values())))
        st = {k: float(v.replace(",", "")) for k, v in d.items()
              if k.startswith("smsp__average_warps_issue_stalled") and k.endswith("_per_issue_active.ratio") and v}
        print("warp stall cycles per issued instruction: " + "  ".join(
            "%s %.2f" % (k.replace("smsp__average_warps_issue_stalled_", "").replace("_per_issue_active.ratio", ""), v)
            for k, v in sorted(st.items(), key=lambda x: -x[1])[:9]))
        if args.ncu_steps_from:
            key = "dram__bytes_read.sum" if args.ncu_steps_from == "read" else "dram__bytes_write.sum"
            steps = num(key) * mult[un(key)] / args.ncu_bytes_per_step
            traffic = (num("dram__bytes_read.sum") * mult[un("dram__bytes_read.sum")] + num("dram__bytes_write.sum") * mult[un("dram__bytes_write.sum")])
            print("steps of this launch (DRAM bytes %s / %g): %.4e" % ("read" if args.ncu_steps_from == "read" else "written", args.ncu_bytes_per_step, steps))
            print("=> %.0f flop per step, %.0f FP64 instructions per step, %.0f warp instructions x threads per step, %.1f B of DRAM traffic per step"
                  % (flop / steps, sum(ops.values()) / steps, num("smsp__inst_executed.sum") * num("smsp__thread_inst_executed_per_inst_executed.ratio") / steps,
                     traffic / steps))
        print()


LAUNCH_METRICS = ("gpu__time_duration.sum,dram__bytes_read.sum,dram__bytes_write.sum,"
                  "smsp__sass_thread_inst_executed_op_dfma_pred_on.sum,smsp__sass_thread_inst_executed_op_dadd_pred_on.sum,"
                  "smsp__sass_thread_inst_executed_op_dmul_pred_on.sum,sm__inst_executed_pipe_fp64.avg.pct_of_peak_sustained_active,"
                  "smsp__thread_inst_executed_per_inst_executed.ratio")


def summarize_launches(args):
    """--summarize-launches CSV: totals per kernel over EVERY launch of a run, from the log of
    `ncu --metrics LAUNCH_METRICS --clock-control none --csv --log-file CSV python bench.py ...` (no GPU needed).
    Steps of the run = DRAM bytes written by the k_geodesic launches / 64 (one path record per step; the probe launches
    write none), so "per step" is an average over all steps of all images of the run, whatever a kernel does with them."""
    import csv
    import collections
    import re
    rows = [r for r in csv.reader(l for l in open(args.summarize_launches) if l.startswith('"'))]
    hdr = rows[0]
    ix = {h: i for i, h in enumerate(hdr)}
    mult = {"Gbyte": 1e9, "Mbyte": 1e6, "Kbyte": 1e3, "byte": 1.0, "s": 1e3, "ms": 1.0, "us": 1e-3, "ns": 1e-6, "msecond": 1.0,
            "usecond": 1e-3, "nsecond": 1e-6, "second": 1e3}
    launches = collections.OrderedDict()
    for r in rows[1:]:
        key = r[ix["ID"]]
        d = launches.setdefault(key, {"name": re.sub(r"\(.*", "", r[ix["Kernel Name"]])})
        v = float(r[ix["Metric Value"]].replace(",", ""))
        d[r[ix["Metric Name"]]] = v * mult.get(r[ix["Metric Unit"]], 1.0)
    tot = collections.OrderedDict()
    for d in launches.values():
        t = tot.setdefault(d["name"], collections.Counter())
        ms = d.get("gpu__time_duration.sum", 0.0)
        t["launches"] += 1
        t["ms"] += ms
        t["read"] += d.get("dram__bytes_read.sum", 0.0)
        t["write"] += d.get("dram__bytes_write.sum", 0.0)
        for k in ("dfma", "dadd", "dmul"):
            t[k] += d.get("smsp__sass_thread_inst_executed_op_%s_pred_on.sum" % k, 0.0)
        t["pipe_ms"] += d.get("sm__inst_executed_pipe_fp64.avg.pct_of_peak_sustained_active", 0.0) * ms
        t["lanes_ms"] += d.get("smsp__thread_inst_executed_per_inst_executed.ratio", 0.0) * ms
    steps = max(1.0, sum(t["write"] for n, t in tot.items() if "k_geodesic" in n) / 64.0)   # (1: a log without the byte counters)
    all_ms = sum(t["ms"] for t in tot.values())
    print("steps of the run (bytes written by k_geodesic / 64): %.4e; kernel time under ncu %.1f ms" % (steps, all_ms))
    print("%-34s %8s %10s %7s %10s %10s %8s %7s %9s %9s" % ("kernel", "launches", "ms (ncu)", "share", "flop/step", "FP64/step", "pipe %", "lanes", "B rd/step", "B wr/step"))
    for n, t in tot.items():
        flop = 2 * t["dfma"] + t["dadd"] + t["dmul"]
        print("%-34s %8d %10.2f %6.1f%% %10.1f %10.1f %8.1f %7.2f %9.1f %9.1f"
              % (n[-34:], t["launches"], t["ms"], 100 * t["ms"] / all_ms, flop / steps, (t["dfma"] + t["dadd"] + t["dmul"]) / steps,
                 t["pipe_ms"] / max(t["ms"], 1e-9), t["lanes_ms"] / max(t["ms"], 1e-9), t["read"] / steps, t["write"] / steps))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=2)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="adaf4096", choices=sorted(WORKLOADS))
    ap.add_argument("--ref-rays", type=int, default=4096, help="rays per step of the --impl reference arm")
    ap.add_argument("--cpu-baseline-rays", type=int, default=16384)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--adaptive", type=int, default=0, metavar="LEVELS",
                    help="adaptive ray tracing (PAPER.md:70) with this many lattice levels, rel_tol 0.02, abs_tol 1e-3 of the peak")
    ap.add_argument("--unpolarized", action="store_true", help="I alone (PAPER.md:74 'nonpolarized images')")
    ap.add_argument("--single-kernel", action="store_true",
                    help="transfer in the single per-ray kernel k_transfer instead of k_stepop + k_apply (ipole_set_transfer_split 0)")
    ap.add_argument("--edf", type=int, default=0, choices=[0, 1, 2],
                    help="second physics workload (PAPER.md:78): j, alpha integrated numerically over a Maxwell-Juettner (1) or "
                         "kappa (2) electron distribution at every step (ipole_set_edf); analytic-flow workloads only")
    ap.add_argument("--fp32-geodesic", action="store_true",
                    help="FP32 study (PAPER.md:70): geodesics in single precision, compared with the FP64 image; analytic-flow workloads")
    ap.add_argument("--no-second-workload", action="store_true",
                    help="default run only: skip the grid4096 half of configs[4] that is otherwise timed after adaf4096")
    ap.add_argument("--path-free", action="store_true",
                    help="the paper's own GPU design (PAPER.md:43): no stored path, forward re-integration")
    ap.add_argument("--summarize-ncu", metavar="REPORT", help="print the text summary of an .ncu-rep (profiles/*.txt); no GPU needed")
    ap.add_argument("--summarize-launches", metavar="CSV", help="per-kernel totals of an ncu --metrics launch log (see summarize_launches); no GPU needed")
    ap.add_argument("--ncu-kernel", default=None, help="--summarize-ncu: only kernels whose name matches this regex")
    ap.add_argument("--ncu-steps-from", choices=["read", "write"], default=None)
    ap.add_argument("--ncu-bytes-per-step", type=float, default=64.0)
    args = ap.parse_args()
    if args.summarize_ncu:
        return summarize_ncu(args)
    if args.summarize_launches:
        return summarize_launches(args)
    if args.impl == "reference":
        return run_reference(args)

    import numpy as np
    import torch
    import torch.distributed as dist
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    if rank == 0:
        import __graft_entry__ as ge
        ge.build()
    if world > 1:
        dist.barrier()
    from paper_2302_02733_b200 import ipole, replicas, workloads as W

    wl = WORKLOADS[args.workload]

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def finish():
        if world > 1:
            dist.destroy_process_group()

    if wl.get("cams"):
        run_cams(args, ipole, replicas, W, wl, world, rank, local, barrier)
        return finish()
    if args.fp32_geodesic:
        if rank == 0:
            run_fp32_study(args, ipole, W, wl)
        return finish()
    if wl.get("sweep") or args.adaptive:
        cam = W.camera(wl["kind"], wl["n"])
        g = ipole.Ipole(**cam)
        g.set_stream(torch.cuda.current_stream())
        if args.unpolarized:
            g.set_unpolarized(True)
        grid = None
        if wl["kind"] == "adaf":
            g.load_adaf(**W.ADAF)
        else:
            grid = grid_inputs(tuple(wl["grid"]))
            g.load_grid(*grid)
        if wl.get("sweep"):
            run_sweep(args, g, ipole, replicas, W, wl, cam, world, rank, local, barrier, grid=grid)
        else:
            run_adaptive(args, g, replicas, wl, cam, world, rank, local, barrier)
        return finish()

    line = measure_image(args, args.workload, ipole, replicas, W, world, rank, local, barrier)
    # The default run covers BOTH halves of BASELINE.json configs[4]: the analytic ADAF image is the top-level value,
    # the GRMHD-like grid image of the same size is timed in the same process and reported under "workloads".
    plain = not (args.path_free or args.unpolarized or args.single_kernel or args.edf)
    if args.workload == "adaf4096" and plain and not args.no_second_workload:
        other = measure_image(args, "grid4096", ipole, replicas, W, world, rank, local, barrier)
        if rank == 0:
            for k in ("metric", "unit", "n_gpus", "steps", "warmup", "higher_is_better", "scaling", "vs_baseline", "dtype", "data", "paper_context"):
                other.pop(k, None)
            line["workloads"] = {"grid4096": other}
            line["gpu_launches"] += other["gpu_launches"]
    if rank == 0:
        print(json.dumps(line), flush=True)
    finish()


if __name__ == "__main__":
    main()
