#!/usr/bin/env python
"""bench.py -- ms per projection solve on the headline workload (BASELINE.json configs[2]:
256x256x128 volume, 1.5 mm voxels, K = 3, detector 512x384 @ 0.776 mm, 360 projections at 1 deg,
irregular breathing at 1.5x amplitude, Poisson noise at 1e5 photons per ray; all synthetic, seeded).

One step = one whole per-projection solve: initial evaluation and fit, 10
iterations of {residual, fused adjoint gradient, Armijo backtracking with one
warp + projection per trial, Eq. 4 fit}, closing cost, tumour localisation.  Consecutive steps
solve consecutive projections of the rotation (1 degree, 1/6 s apart) and each starts from the
previous frame's coefficients.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--config C2]
    python bench.py --frames-study | --pca-study     (SURVEY 8(f).2 / 8(f).3 measurements; their own JSON line)
    python bench.py --field-storage 1                (u_k stored in half; not the headline)

N > 1 (under torchrun): replicas only -- every rank holds the model and solves its own contiguous
block of K projections; no data-path collective; scaling is weak.
--impl reference times the CPU oracle (fp64, OpenMP on the host cores) on the same workload.
Prints ONE JSON line on rank 0.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from workloads import get_config                                   # noqa: E402
from workloads.build import build_workload                         # noqa: E402
from workloads.motion import dvf_grid                              # noqa: E402
from workloads.noise import add_noise                              # noqa: E402
from workloads.phantom import voxelise                             # noqa: E402

METRIC = "ms_per_projection_solve"
FIRST_FRAME = 60      # where in the rotation the timed block starts (any frame is representative)
PAPER_MS = None       # the paper's 240 ms is for another volume/detector/machine: context only


def log(*a):
    print(*a, file=sys.stderr, flush=True)


# ----------------------------------------------------------------------------- inputs (CPU, seeded)

_G = {}


def _gt_worker(idx):
    cfg, spec, frames = _G["cfg"], _G["spec"], _G["frames"]
    fr = frames[idx]
    return idx, voxelise(cfg, dvf_grid(cfg, spec, fr.phase, fr.amplitude)).astype(np.float32)


def ground_truth_volumes(wl, indices):
    """The phantom deformed by the test DVF of each frame (workloads recipe), in parallel on the host
    cores.  Must run before CUDA is initialised (fork)."""
    import multiprocessing as mp
    _G.update(cfg=wl.cfg, spec=wl.spec, frames=wl.frames)
    uniq = sorted(set(indices))
    n_proc = max(1, min(len(uniq), (os.cpu_count() or 2) - 1, 12))
    if n_proc == 1:
        return dict(_gt_worker(i) for i in uniq)
    with mp.get_context("fork").Pool(n_proc) as pool:
        return dict(pool.map(_gt_worker, uniq))


def solver_iterations(cfg) -> int:
    return cfg.iterations


def field_bytes_per_voxel(cfg, field_storage=0):
    """12 (K + 1) bytes of float fields per voxel; with field_storage = 1 the u_k planes
    are halves (6 K bytes instead of 12 K)."""
    return 12 * (cfg.K + 1) if field_storage == 0 else 12 + 6 * cfg.K


def algorithmic_bytes(cfg, field_storage=0):
    """what the dense method must move per launch, every voxel's fields counted,
    f0 gathers counted once."""
    V, npix = cfg.V, cfg.npix
    fields = field_bytes_per_voxel(cfg, field_storage)
    return {"warp": (fields + 4 + 4) * V,
            "project": 4 * V + 4 * npix,
            "gradient": (fields + 4) * V + 4 * npix}


RECORD_BYTES = 48       # one gradient record: packed voxel coordinates, three fractions, eight taps of f0 (stream.cuh GradRecord)


def moved_bytes(cfg, field_storage, tiles_loaded, vox_per_tile, records=None, n_tiles=0):
    """What one launch really had to move, from the tiles the timed launches loaded (counted inside the
    kernels, pcamm_tile_counts; reading B8: tiles that can only see zeros / constant cells are skipped).
    A loaded tile costs its fields and its f0 gathers (4 B per voxel, counted once); the warp kernel
    writes every voxel of the volume (skipped tiles as zeros), the gradient kernel reads the residual.
    With gradient records (the default for one solve) the warp kernel also writes 48 B per voxel with
    a non-constant cell and a count per sub-tile (8 per tile); the gradient reads those, the voxel's 3 K values of
    u (12 K bytes, from the copy that holds them side by side) per record, and the residual."""
    fields = field_bytes_per_voxel(cfg, field_storage)
    out = {"warp": tiles_loaded["warp"] * vox_per_tile * (fields + 4) + 4 * cfg.V,
           "gradient": tiles_loaded["gradient"] * vox_per_tile * (fields + 4) + 4 * cfg.npix}
    if records and records["gathered"] > 0:
        out["warp"] += RECORD_BYTES * records["written"] + 4 * 8 * n_tiles
        out["gradient"] = (RECORD_BYTES + 12 * cfg.K) * records["gathered"] + 4 * 8 * n_tiles + 4 * cfg.npix
    return out


def measured_peak_gbs():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", f"--id={gpu_index}", f"--query-gpu={self.Q}",
                                       "--format=csv,noheader,nounits", "-lms", "200"],
                                      stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except Exception:
            self.p = None

    def stop(self):
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        time.sleep(0.25)
        self.p.terminate()
        try:
            out, _ = self.p.communicate(timeout=5)
        except Exception:
            self.p.kill()
            out = ""
        sm, smax, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in out.splitlines():
            f = [x.strip() for x in line.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); smax.append(float(f[1]))
            except ValueError:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(smax) if smax else None,
                "reasons": sorted(reasons), "samples": len(sm)}


# ----------------------------------------------------------------------------- the two arms

def oracle_geometry(cfg):
    import oracle
    return oracle.Geometry(cfg.nx, cfg.ny, cfg.nz, cfg.hx, cfg.hy, cfg.hz, cfg.K, cfg.nu, cfg.nv, cfg.pu, cfg.pv,
                           cfg.sad, cfg.sdd)


def time_oracle_solves(wl, gts, frame_ids, iterations, threads=None):
    """The oracle as it stands (fp64 C++, OpenMP over rays / voxels) on the host cores: one full
    solve per frame, projections simulated by the oracle's own projector.  Returns seconds per
    solve (list) and the thread count."""
    import oracle
    cfg = wl.cfg
    g = oracle_geometry(cfg)
    nthr = threads or oracle.max_threads()
    oracle.set_threads(nthr)
    w = np.zeros(cfg.K)
    secs = []
    for fid in frame_ids:
        fr = wl.frames[fid]
        y = add_noise(oracle.project(g, gts[fid], fr.angle_rad), cfg.noise, seed=fid)
        t0 = time.perf_counter()
        res = oracle.solve(g, wl.f0, wl.model.mean, wl.model.eig, y, fr.angle_rad, w,
                           oracle.Opts(max_iter=iterations, batched_linesearch=int(cfg.batched_linesearch)),
                           want_volume=False)
        oracle.invert(g, wl.model.mean, wl.model.eig, res["w"], wl.landmarks)
        secs.append(time.perf_counter() - t0)
        w = res["w"]
    return secs, nthr


def run_reference(args, cfg, rank, world):
    if rank != 0:
        return
    wl = build_workload(cfg)
    n = args.steps + args.warmup
    ids = [(FIRST_FRAME + i) % len(wl.frames) for i in range(n)]
    # bounded sample: the block's first frames only, one full solve each, cycled over the steps
    n_distinct = min(n, 2)
    gts = ground_truth_volumes(wl, ids[:n_distinct])
    it = solver_iterations(cfg)
    cyc = [ids[i % n_distinct] for i in range(n)]
    if args.projector == 1:
        import oracle
        oracle.set_projector(oracle.RAY_MARCHING, (args.ray_step_vox or 0.5) * min(cfg.hx, cfg.hy, cfg.hz))
    secs, nthr = time_oracle_solves(wl, gts, cyc, it)
    timed = secs[args.warmup:]
    ms = 1e3 * float(np.mean(timed))
    fan = 1 if cfg.batched_linesearch else int(args.fan)
    line = {"impl": "reference", "metric": METRIC, "value": ms, "unit": "ms", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms, "ms_per_step_median": 1e3 * float(np.median(timed)),
            "higher_is_better": False,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": dict(full_config(cfg, it, fan, args.field_storage, max(int(args.in_flight), 1)), **projector_config(args)),
            "cpu_baseline": {"value": ms, "unit": "ms", "cores": nthr, "kind": "oracle",
                             "sample": f"full {it}-iteration oracle solves, {n_distinct} distinct projections "
                                       f"cycled over {n} steps, OpenMP on {nthr} threads"},
            "e2e": {"value": ms, "unit": "ms", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def projector_config(args):
    """Extra config key of the runs that use the ray-marching variant of P: none for the
    headline configuration (Siddon)."""
    if args.projector == 0:
        return {}
    return {"projector": f"fixed-step trilinear ray marching, nominal step {args.ray_step_vox or 0.5} x the smallest voxel "
                         "edge (DESIGN.md reading C1; NOT the headline configuration, which is Siddon's exact path)"}


def full_config(cfg, iterations, fan, field_storage, in_flight):
    """The config object of the bench line (identical in both arms)."""
    return dict(config_dict(cfg, iterations, fan, field_storage), in_flight=in_flight,
                field_storage="float32" if field_storage == 0 else
                "u_k stored as float16 with a power-of-two scale per field, x-bar float32, arithmetic float32 "
                "(SURVEY 8(f).4; NOT the headline configuration)")


def config_dict(cfg, iterations, fan=1, field_storage=0):
    return {"workload": f"{cfg.name}: volume {cfg.nx}x{cfg.ny}x{cfg.nz} @ {cfg.hx} mm, K={cfg.K}, detector "
                        f"{cfg.nu}x{cfg.nv} @ {cfg.pu} mm, consecutive projections 1 deg / (1/6) s apart from frame "
                        f"{FIRST_FRAME}, {cfg.noise} noise, {'irregular' if cfg.irregular else 'regular'} breathing "
                        f"x{cfg.amplitude}",
            "iterations": iterations, "warm_start": "previous frame's w (PAPER.md:L141)",
            "line_search": "Armijo backtracking, all 8 candidate steps per pass" if cfg.batched_linesearch else
                           ("sequential Armijo backtracking" if fan <= 1 else
                            f"Armijo backtracking, {fan} candidate steps evaluated per pass: the accepted steps are those of "
                            "sequential backtracking, bit for bit (DESIGN.md reading B7)"),
            "l2": "inputs larger than L2: every pass streams the (K+1) vector fields "
                  f"({(12 * (cfg.K + 1) if field_storage == 0 else 12 + 6 * cfg.K) * cfg.V / 2**20:.0f} MiB) through a 126 MB L2",
            "parallelism": "replicas"}


def run_ours(args, cfg, rank, local_rank, world):
    from paper_1004_0014_b200 import replicas
    it = solver_iterations(cfg)
    n = args.steps + args.warmup
    # ---- inputs on the CPU first (the worker pool forks before CUDA is initialised)
    t0 = time.perf_counter()
    wl = build_workload(cfg)
    B = max(int(args.in_flight), 1)
    if B == 1:
        ids = replicas.frame_block(rank, world, n, FIRST_FRAME, len(wl.frames))
    else:
        # B solves in flight: gantry angles and breathing states drawn from the test trajectory
        # (seeded, BASELINE.json configs[4]); a pool of 8 distinct frames, re-noised per use
        pool = np.random.default_rng(4 + rank).choice(len(wl.frames), size=min(8, len(wl.frames)), replace=False)
        ids = [int(pool[i % len(pool)]) for i in range(min(n, 2) * B)]
    gts = ground_truth_volumes(wl, ids)
    log(f"[rank {rank}] inputs built in {time.perf_counter() - t0:.1f} s")

    import torch
    import paper_1004_0014_b200 as pc
    for kv in args.tune:
        name, _, value = kv.partition("=")
        pc.tune(name, int(value))
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    dist = replicas.init_process_group("nccl")
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).to(dev)
    fan = 1 if cfg.batched_linesearch else int(args.fan)     # pcamm_opts.batched_linesearch (1 = all 8 at once)
    C = 8 if cfg.batched_linesearch else max(fan, 1)
    m = pc.Model(nx=cfg.nx, ny=cfg.ny, nz=cfg.nz, hx=cfg.hx, hy=cfg.hy, hz=cfg.hz, K=cfg.K, nu=cfg.nu, nv=cfg.nv,
                 pu=cfg.pu, pv=cfg.pv, f0=t(wl.f0), mean_dvf=t(wl.model.mean), eig_dvf=t(wl.model.eig),
                 landmarks_mm=wl.landmarks, sad=cfg.sad, sdd=cfg.sdd, max_candidates=C, max_batch=B,
                 field_storage=args.field_storage, projector=args.projector, ray_step_vox=args.ray_step_vox)
    # measured projections: the scanner is simulated with the library's own projector applied to
    # the ground-truth volume, plus seeded noise (the CPU arm simulates its own with the oracle)
    ys_host, ys_dev = [], []
    p_true = {}
    for j, fid in enumerate(ids):
        fr = wl.frames[fid]
        if fid not in p_true:
            p_true[fid] = m.project(t(gts[fid]), fr.angle_rad).cpu().numpy()
        y = add_noise(p_true[fid], cfg.noise, seed=fid + 1000 * (j // max(len(p_true), 1)) if B > 1 else fid)
        ys_host.append(torch.from_numpy(y).pin_memory())
        ys_dev.append(t(y))
    angles = [float(wl.frames[fid].angle_rad) for fid in ids]
    opts = pc.Opts(max_iter=it, batched_linesearch=fan if fan > 1 or cfg.batched_linesearch else 0, loop_mode=args.loop_mode)
    if B > 1:   # one stacked [B][nv][nu] tensor per distinct step
        n_distinct = len(ids) // B
        yb_dev = [torch.stack(ys_dev[j * B:(j + 1) * B]) for j in range(n_distinct)]
        yb_host = [torch.stack([h for h in ys_host[j * B:(j + 1) * B]]).pin_memory() for j in range(n_distinct)]
        ab = [np.array(angles[j * B:(j + 1) * B], np.float32) for j in range(n_distinct)]
        stage = torch.empty_like(yb_dev[0])
        w_zero = np.zeros((B, cfg.K), np.float32)

    tumour_mm = {}          # frame index in the block -> localised tumour position (device-resident pass)
    step_events = []        # one CUDA event behind every step of the device-resident pass

    def run_block(first, count, w, host, events=None):
        for i in range(first, first + count):
            if B > 1:
                j = i % n_distinct
                if host:
                    stage.copy_(yb_host[j], non_blocking=True)
                    r = m.reconstruct_batch(stage, ab[j], w_zero, opts)[-1]
                else:
                    r = m.reconstruct_batch(yb_dev[j], ab[j], w_zero, opts)[-1]
            elif host:
                r = m.reconstruct(ys_host[i].numpy(), angles[i], w, opts, host_y=True)
                w = r.w
            else:
                r = m.reconstruct(ys_dev[i], angles[i], w, opts)
                if r.landmarks is not None and len(r.landmarks):
                    tumour_mm[i] = np.array(r.landmarks[0], np.float64)
                w = r.w
            if events is not None:
                ev = torch.cuda.Event(enable_timing=True)
                ev.record()
                events.append(ev)
        return w, r

    # ---- device-resident timing: y already in HBM
    w = np.zeros(cfg.K, np.float32)
    w, _ = run_block(0, args.warmup, w, host=False)
    w_after_warmup = w.copy()
    torch.cuda.synchronize()
    replicas.barrier(dist)
    sampler = ClockSampler(local_rank) if rank == 0 else None
    pc.launch_count(reset=True)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    w, last = run_block(args.warmup, args.steps, w, host=False, events=step_events)
    e1.record()
    torch.cuda.synchronize()
    marks = [e0] + step_events
    step_ms = [marks[i].elapsed_time(marks[i + 1]) for i in range(len(step_events))]
    launches = pc.launch_count(reset=True)
    replicas.barrier(dist)
    clocks = sampler.stop() if sampler else None
    elapsed_ms = replicas.max_over_ranks(dist, e0.elapsed_time(e1), dev)
    launches = int(replicas.sum_over_ranks(dist, launches, dev))

    # ---- end to end: y in pinned host memory, copied inside the call; results read back inside it
    run_block(max(args.warmup - 1, 0), 1, w_after_warmup, host=True)
    torch.cuda.synchronize()
    replicas.barrier(dist)
    t0 = time.perf_counter()
    run_block(args.warmup, args.steps, w_after_warmup, host=True)
    torch.cuda.synchronize()
    e2e_ms = replicas.max_over_ranks(dist, 1e3 * (time.perf_counter() - t0), dev)
    h2d = B * (cfg.npix * 4 + 56) + 128           # y + the call's option block (CallOpts, SolveIn)
    d2h = B * (272 + 24 * len(wl.landmarks)) + 24  # SolveState + landmark positions (double) + LoopFlags

    if rank != 0:
        return
    ms_per_solve = elapsed_ms / (args.steps * world * B)

    # ---- per-kernel device times on the last frame's state (CUDA events inside the library, on the
    #      stream the kernels are launched on), and the launch mix of one traced solve
    i_last = (n - 1) if B == 1 else 0
    tr = m.reconstruct(ys_dev[i_last], angles[i_last], w_after_warmup if B == 1 else np.zeros(cfg.K, np.float32),
                       opts, trace=True)
    width = 8 if cfg.batched_linesearch else max(fan, 1)
    # line-search passes (each one warp + one projection launch over `width` candidates), candidates evaluated
    passes = int(np.sum(tr.backtracks // width + 1)) if tr.backtracks is not None else it
    trials = int(np.sum(np.minimum(width * (tr.backtracks // width + 1), 8))) if tr.backtracks is not None else it
    m.eval(ys_dev[i_last], angles[i_last], tr.w, tr.a, tr.b, want_proj=False)
    # the warp and projection kernels are timed over as many candidate steps as a line-search pass
    # evaluates (nearby coefficient vectors: the candidates of a pass differ by one step)
    m.time_slots(np.stack([tr.w * (1.0 + 0.02 * c) for c in range(width)]))
    for which in (0, 1, 2):
        m.time_kernel(which, 3)
    REPS = 20
    kt, tiles_loaded, records = {}, {}, {"written": 0.0, "gathered": 0.0}
    for which, name in ((0, "warp"), (1, "project"), (2, "gradient")):
        m.tile_counts(reset=True)
        kt[name] = m.time_kernel(which, REPS)
        tc = m.tile_counts(reset=True)               # tiles the timed launches loaded, counted in the kernels
        tiles_loaded[name] = tc[0 if which == 0 else 1] / REPS
        if which == 0:
            records["written"] = tc[5] / REPS        # gradient records, all candidates of the launch
        if which == 2:
            records["gathered"] = tc[4] / REPS       # those of the accepted candidate
    n_tiles, vox_per_tile = tc[2], tc[3]
    by_records = records["gathered"] > 0
    nl = {"warp": passes + 1, "project": passes + 1, "gradient": tr.iters}
    ab = algorithmic_bytes(cfg, args.field_storage)
    peak, peak_src = measured_peak_gbs()
    # per launch over `width` candidates: the fields once, the f0 gathers, the volume and the projection per candidate
    ab["warp"] += (width - 1) * 8 * cfg.V
    ab["project"] *= width
    if n_tiles:
        mv = moved_bytes(cfg, args.field_storage, tiles_loaded, vox_per_tile, records, n_tiles)
        mv["warp"] += (width - 1) * (tiles_loaded["warp"] * vox_per_tile * 4 + 4 * cfg.V)
    else:                                            # generic kernels (shapes TMA cannot describe): every tile
        mv = {"warp": ab["warp"], "gradient": ab["gradient"]}
    mv["project"] = ab["project"]
    per_kernel = {}
    for k in kt:
        sec = kt[k] * 1e-3
        per_kernel[k] = {"bound": "hbm", "ms": kt[k], "launches_per_solve": nl[k],
                         "candidates_per_launch": 1 if k == "gradient" else width,
                         "moved_bytes": mv[k], "achieved": mv[k] / sec / 1e9, "peak": peak, "unit": "GB/s",
                         "frac": mv[k] / sec / 1e9 / peak,
                         "dense_algorithmic_bytes": ab[k], "speedup_vs_dense_bytes": ab[k] / sec / 1e9 / peak}
        if k != "project" and n_tiles:
            per_kernel[k]["tiles_loaded_per_launch"] = tiles_loaded[k]
            per_kernel[k]["tiles_total"] = n_tiles
    if by_records:
        per_kernel["warp"]["gradient_records_written_per_launch"] = records["written"]
        per_kernel["gradient"].update({
            "kernel": "k_grad_gather", "records_per_launch": records["gathered"],
            "records_per_voxel": records["gathered"] / cfg.V,
            "note": "a gather over the records the warp kernel left for the voxels with G_j != 0 (DESIGN.md section 5b): "
                    "latency-bound scattered loads, not a stream; moved_bytes counts 48 B per record, "
                    "12 K B of u per record, the counts and the residual"})
    # the projector's volume was just written and is L2-resident: it is not an HBM kernel.
    # What it does per launch: one pass over (detector column, slab, level) and one look-up per z crossing.
    per_kernel["project"].update({
        "note": "L2-resident input: bound by issue and shared-memory latency, not by HBM (DESIGN.md section 5a); "
                "frac = SURVEY 8(d) bytes (4 V + 4 Npix) / time / HBM peak, as BASELINE.json asks",
        "rays_per_s": width * cfg.npix / (kt["project"] * 1e-3)})
    dom = max(kt, key=lambda k: kt[k] * nl[k])
    wp_gbs = (mv["warp"] + mv["project"]) / ((kt["warp"] + kt["project"]) * 1e-3) / 1e9
    d = per_kernel[dom]
    roofline = {"kernel": dom, "bound": d["bound"], "achieved": d["achieved"], "peak": d["peak"], "unit": d["unit"],
                "frac": d["frac"], "traffic": None,
                "note": "achieved = bytes the launch had to move / CUDA-event time of the launch (pcamm_time_kernel, on the "
                        "launching stream): fields and f0 of the tiles the kernel loaded (counted in the kernel for the same "
                        "launches), the volume written, the residual read.  speedup_vs_dense_bytes puts SURVEY 8(a)'s dense "
                        "bytes (every voxel's fields) over the same time: the kernels skip, exactly, tiles that can only "
                        "see zeros / constant cells of f0 (DESIGN.md reading B8).  traffic (ncu DRAM bytes): profiles/",
                "peak_source": peak_src,
                "per_kernel": per_kernel,
                "warp_plus_project": {"gbs": wp_gbs, "frac": wp_gbs / peak, "frac_of_nominal_8000": wp_gbs / 8000.0,
                                      "dense_gbs": (ab["warp"] + ab["project"]) / ((kt["warp"] + kt["project"]) * 1e-3) / 1e9},
                "kernel_share_of_step": {k: kt[k] * nl[k] / (elapsed_ms / args.steps / B) for k in kt}}

    # ---- the oracle on this box's host cores (a baseline, not the target): one full solve of the same
    #      workload on all cores, and a short one on a single core
    cpu = None
    if not args.no_cpu_baseline:
        tc0 = time.perf_counter()
        if args.projector == 1:
            import oracle
            oracle.set_projector(oracle.RAY_MARCHING, (args.ray_step_vox or 0.5) * min(cfg.hx, cfg.hy, cfg.hz))
        secs, nthr = time_oracle_solves(wl, gts, [ids[args.warmup]], it)
        cpu = {"value": 1e3 * secs[0], "unit": "ms", "cores": nthr, "kind": "oracle",
               "sample": f"1 projection (frame {ids[args.warmup]}), full {it}-iteration solve from w = 0, "
                         f"OpenMP on {nthr} threads; {time.perf_counter() - tc0:.0f} s including its simulated y"}
        it1 = min(it, args.cpu_single_iters)
        if it1 > 0:
            secs1, _ = time_oracle_solves(wl, gts, [ids[args.warmup]], it1, threads=1)
            cpu["single_thread"] = {"value": 1e3 * secs1[0], "unit": "ms", "cores": 1, "iterations": it1,
                                    "ms_per_iteration": 1e3 * secs1[0] / it1,
                                    "sample": f"the same projection, {it1}-iteration solve from w = 0 on one thread "
                                              f"(bounded: a full {it}-iteration solve takes about {it / it1:.0f}x as long)"}

    # ---- accuracy context (PAPER.md:L119 3D localisation error; not a parity value): the tumour
    #      position of every timed solve against the fixed point of the analytic test DVF
    accuracy = None
    if B == 1 and tumour_mm:
        from workloads.motion import true_tumour_position
        errs = [float(np.linalg.norm(tumour_mm[i] - true_tumour_position(cfg, wl.spec, wl.frames[ids[i]], wl.landmarks[0])))
                for i in sorted(tumour_mm) if i >= args.warmup]
        if errs:
            accuracy = {"tumour_error_mm_mean": float(np.mean(errs)), "tumour_error_mm_max": float(np.max(errs)),
                        "n": len(errs), "note": "synthetic phantom, context only (the paper reports 0.8 +- 0.5 mm on NCAT, L135)"}

    line = {"metric": METRIC, "value": ms_per_solve, "unit": "ms", "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": elapsed_ms / args.steps,
            "ms_per_step_median": float(np.median(step_ms)) if step_ms else None, "higher_is_better": False,
            "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": dict(full_config(cfg, it, fan, args.field_storage, B), **projector_config(args)),
            "projections_per_s": 1e3 * args.steps * world * B / elapsed_ms,
            "clocks": clocks,
            "e2e": {"value": e2e_ms / (args.steps * world * B), "unit": "ms", "h2d_bytes_per_step": h2d,
                    "d2h_bytes_per_step": d2h},
            "gpu_launches": launches, "roofline": roofline, "cpu_baseline": cpu,
            "last_solve": {"iters": tr.iters, "line_search_passes": passes, "candidates_evaluated": trials,
                           "status": tr.status, "J0": tr.J0, "J": tr.J},
            "accuracy": accuracy,
            "context": {"paper_ms_per_projection_tesla_c1060": 240.0}}
    print(json.dumps(line), flush=True)


def run_frames_study(args, cfg, rank, local_rank):
    """--frames-study: the frame stream (pcamm_frames_*) over the
    same consecutive projections under each start predictor, stopping on the gradient norm
     instead of after a fixed 10 iterations.  Prints one JSON line (not the bench
    contract's line): iterations, candidate evaluations, ms per solve and 6 Hz headroom per
    predictor.  grad_tol, unless given, is the median ||g|| the paper's fixed 10 iterations reach
    on the warm-up frames started from the previous frame's w."""
    if rank != 0:
        return
    n = args.steps + args.warmup
    wl = build_workload(cfg)
    ids = list(range(FIRST_FRAME, FIRST_FRAME + n))
    gts = ground_truth_volumes(wl, ids)
    import torch
    import paper_1004_0014_b200 as pc
    from workloads.motion import true_tumour_position
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).to(dev)
    m = pc.Model(nx=cfg.nx, ny=cfg.ny, nz=cfg.nz, hx=cfg.hx, hy=cfg.hy, hz=cfg.hz, K=cfg.K, nu=cfg.nu, nv=cfg.nv,
                 pu=cfg.pu, pv=cfg.pv, f0=t(wl.f0), mean_dvf=t(wl.model.mean), eig_dvf=t(wl.model.eig),
                 landmarks_mm=wl.landmarks, sad=cfg.sad, sdd=cfg.sdd)
    frames = [wl.frames[i] for i in ids]
    ys = [t(add_noise(m.project(t(gts[fr.index]), fr.angle_rad).cpu().numpy(), cfg.noise, seed=fr.index)) for fr in frames]
    it = solver_iterations(cfg)
    tol = args.grad_tol
    if tol is None:
        fs = pc.Frames(m, order=0)
        gn = []
        for fr, y in zip(frames[:max(args.warmup, 3)], ys):
            r = fs.push(y, fr.angle_rad, fr.time_s, pc.Opts(max_iter=it), trace=True)
            gn.append(float(r.gnorm_trace[-1]))
        tol = float(np.median(gn[1:])) if len(gn) > 1 else gn[0]
    opts = pc.Opts(max_iter=args.study_max_iter, grad_tol=tol)
    per = {}
    for order, name in ((-1, "none (w = 0 every frame)"), (0, "previous frame (L141)"), (1, "linear"), (2, "quadratic")):
        fs = pc.Frames(m, order=order)
        for fr, y in zip(frames[:args.warmup], ys):
            fs.push(y, fr.angle_rad, fr.time_s, opts)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        out = [fs.push(y, fr.angle_rad, fr.time_s, opts, trace=True) for fr, y in zip(frames[args.warmup:], ys[args.warmup:])]
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / len(out)
        errs = [float(np.linalg.norm(np.array(r.landmarks[0], np.float64) -
                                     true_tumour_position(cfg, wl.spec, fr, wl.landmarks[0])))
                for r, fr in zip(out, frames[args.warmup:])]
        per[str(order)] = {"predictor": name, "ms_per_solve": ms, "mean_iters": float(np.mean([r.iters for r in out])),
                           "mean_candidate_evaluations": float(np.mean([int(np.sum(r.backtracks + 1)) for r in out])),
                           "stopped_on_grad_tol": int(sum(r.status == pc.S_GRADTOL for r in out)),
                           "mean_J": float(np.mean([r.J for r in out])), "tumour_error_mm_mean": float(np.mean(errs)),
                           "headroom_at_6_hz": (1000.0 / 6.0) / ms}
    print(json.dumps({"study": "frames", "config": config_dict(cfg, args.study_max_iter), "frames": len(frames) - args.warmup,
                      "warmup": args.warmup, "grad_tol": tol, "max_iter": args.study_max_iter, "per_order": per}), flush=True)


TL_KINDS = ("ysums", "begin", "view_tables", "warp", "project", "ctl_after_project", "resid", "gradient", "ctl_grad",
            "iter_end", "final", "invert")


def run_timeline(args, cfg, rank, local_rank):
    """--timeline: the kernels of one solve of the timed workload, as the device saw them: start (first
    block in) and end (last block out) of every kernel on the global timer, recorded inside the kernels
    (pcamm_tune "timeline"; nsys is not installed in this image).  Prints one JSON line (not the bench
    contract's): per kernel kind the count, the summed duration and the summed gap to the previous
    kernel's end; with --timeline-out FILE also the event list as text."""
    if rank != 0:
        return
    n = args.warmup + 1
    wl = build_workload(cfg)
    ids = list(range(FIRST_FRAME, FIRST_FRAME + n))
    gts = ground_truth_volumes(wl, ids)
    import torch
    import paper_1004_0014_b200 as pc
    for kv in args.tune:
        name, _, value = kv.partition("=")
        pc.tune(name, int(value))
    pc.tune("timeline", 1)
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).to(dev)
    m = pc.Model(nx=cfg.nx, ny=cfg.ny, nz=cfg.nz, hx=cfg.hx, hy=cfg.hy, hz=cfg.hz, K=cfg.K, nu=cfg.nu, nv=cfg.nv,
                 pu=cfg.pu, pv=cfg.pv, f0=t(wl.f0), mean_dvf=t(wl.model.mean), eig_dvf=t(wl.model.eig),
                 landmarks_mm=wl.landmarks, sad=cfg.sad, sdd=cfg.sdd,
                 max_candidates=8 if cfg.batched_linesearch else max(int(args.fan), 1))
    fan = 1 if cfg.batched_linesearch else int(args.fan)
    opts = pc.Opts(max_iter=solver_iterations(cfg), batched_linesearch=1 if cfg.batched_linesearch else (fan if fan > 1 else 0))
    w = np.zeros(cfg.K, np.float32)
    for i, fid in enumerate(ids):
        fr = wl.frames[fid]
        y = t(add_noise(m.project(t(gts[fid]), fr.angle_rad).cpu().numpy(), cfg.noise, seed=fid))
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        r = m.reconstruct(y, fr.angle_rad, w, opts)
        e1.record()
        torch.cuda.synchronize()
        w = r.w
    kind, t0, t1 = m.timeline()
    per = {}
    prev_end = None
    for k, a, b in zip(kind, t0, t1):
        d = per.setdefault(TL_KINDS[k], {"count": 0, "busy_us": 0.0, "gap_before_us": 0.0})
        d["count"] += 1
        d["busy_us"] += float(b - a)
        if prev_end is not None:
            d["gap_before_us"] += float(a - prev_end)
        prev_end = b
    busy = sum(d["busy_us"] for d in per.values())
    span = float(t1[-1] - t0[0]) if len(t0) else 0.0
    if args.timeline_out:
        with open(args.timeline_out, "w") as f:
            f.write("# kernel timeline of one solve (us on the device's global timer, relative to the first kernel's start)\n")
            f.write("# index kind start end duration gap_before\n")
            pe = None
            for i, (k, a, b) in enumerate(zip(kind, t0, t1)):
                f.write(f"{i:4d} {TL_KINDS[k]:18s} {a:10.2f} {b:10.2f} {b - a:8.2f} {0.0 if pe is None else a - pe:8.2f}\n")
                pe = b
    print(json.dumps({"study": "timeline", "config": config_dict(cfg, solver_iterations(cfg), fan), "kernels": int(len(kind)),
                      "span_us": span, "busy_us": busy, "busy_frac": busy / span if span else None,
                      "solve_ms_cuda_events_with_timeline_on": e0.elapsed_time(e1),
                      "per_kind": per, "iters": int(r.iters)}), flush=True)


def run_pca_study(args, cfg, rank, local_rank):
    """--pca-study: pcamm_pca_fit on the config's nine training
    DVFs: device time of its two streaming passes (CUDA events on the launching stream, inside the
    library) against their algorithmic bytes, the whole call's wall time, and the distance of the
    fitted fields from the input recipe's own PCA (context).  One JSON line, not the bench contract's."""
    if rank != 0:
        return
    from workloads.motion import motion_spec, training_dvfs
    from workloads.pca import fit_pca
    t0 = time.perf_counter()
    dvfs = np.ascontiguousarray(training_dvfs(cfg, motion_spec(cfg)), dtype=np.float32)
    log(f"training DVFs {dvfs.shape} built in {time.perf_counter() - t0:.1f} s")
    import torch
    import paper_1004_0014_b200 as pc
    torch.cuda.set_device(local_rank)
    d = torch.from_numpy(dvfs).to(torch.device("cuda", local_rank))
    N, n = dvfs.shape[0], dvfs[0].size
    for _ in range(max(args.warmup, 1)):
        pc.pca_fit(d, cfg.K)
    ms1, ms2, wall = [], [], []
    for _ in range(args.steps):
        pm = []
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        mean, eig, lam, coeffs = pc.pca_fit(d, cfg.K, pass_ms=pm)
        wall.append(1e3 * (time.perf_counter() - t0))
        ms1.append(pm[0]); ms2.append(pm[1])
    peak, peak_src = measured_peak_gbs()
    b1, b2 = 4 * N * n, 4 * N * n + 4 * (cfg.K + 1) * n
    m1, m2 = float(np.median(ms1)), float(np.median(ms2))
    t0 = time.perf_counter()
    ref = fit_pca(dvfs, cfg.K)
    host_s = time.perf_counter() - t0
    e = eig.cpu().numpy().astype(np.float64)
    print(json.dumps({"study": "pca", "workload": f"{cfg.name}: {N} training DVFs of 3 x {cfg.nx}x{cfg.ny}x{cfg.nz} floats, K={cfg.K}",
                      "reps": args.steps,
                      "scatter_matrix_pass": {"ms": m1, "algorithmic_bytes": b1, "achieved_gbs": b1 / m1 / 1e6, "frac": b1 / m1 / 1e6 / peak},
                      "fields_pass": {"ms": m2, "algorithmic_bytes": b2, "achieved_gbs": b2 / m2 / 1e6, "frac": b2 / m2 / 1e6 / peak},
                      "peak_gbs": peak, "peak_source": peak_src, "call_wall_ms": float(np.median(wall)),
                      "eigenvalues": [float(x) for x in lam[:N]],
                      "context": {"input_recipe_pca_numpy_float64_s": host_s,
                                  "eig_l2_distance_from_recipe": [float(np.linalg.norm(e[k] - ref.eig[k].astype(np.float64)))
                                                                  for k in range(cfg.K)],
                                  "mean_max_abs_distance_mm": float(np.abs(mean.cpu().numpy() - ref.mean).max())}}),
          flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="C2")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--fan", type=int, default=None,
                    help="candidate steps evaluated per line-search pass (pcamm_opts.batched_linesearch): the "
                         "accepted step is the same for every width, bit for bit; 1 = sequential backtracking.  "
                         "Default: 2 for one solve in flight on volumes up to C2's size (a pass then shares the field "
                         "stream and the launches between its candidates), else 1 (larger volumes, and --in-flight > 1 "
                         "where the solves in flight share them already: a second candidate per pass then only adds "
                         "candidates that are evaluated and thrown away)")
    ap.add_argument("--cpu-single-iters", type=int, default=1,
                    help="iterations of the single-thread oracle leg (0: skip it)")
    ap.add_argument("--in-flight", type=int, default=1,
                    help="B > 1: every step advances B independent projection solves in lock step "
                         "(pcamm_reconstruct_batch; BASELINE.json configs[4] sweeps 1, 4, 16, 64), each from w = 0")
    ap.add_argument("--loop-mode", type=int, default=0, choices=[0, 1],
                    help="0: the solve is one CUDA graph with device-side while-loops (default, the timed "
                         "configuration); 1: same kernels launched from the host (for per-launch ncu lists)")
    ap.add_argument("--frames-study", action="store_true",
                    help="instead of the bench line: iterations and ms per solve of the frame stream under each "
                         "start predictor (pcamm_frames_*), stopping on ||g|| <= --grad-tol")
    ap.add_argument("--field-storage", type=int, default=0, choices=[0, 1],
                    help="pcamm_geometry.field_storage: 0 float32 fields (the headline configuration), 1 u_k in half")
    ap.add_argument("--pca-study", action="store_true",
                    help="instead of the bench line: pcamm_pca_fit on the config's training DVFs (device time of its "
                         "two passes against their algorithmic bytes)")
    ap.add_argument("--tune", action="append", default=[], metavar="NAME=VALUE",
                    help="pcamm_tune measurement knob, set before the model is created (repeatable)")
    ap.add_argument("--projector", type=int, default=0, choices=[0, 1],
                    help="pcamm_geometry.projector: 0 Siddon's exact path (the headline configuration), 1 fixed-step "
                         "trilinear ray marching (SURVEY 8(f) row 1)")
    ap.add_argument("--ray-step-vox", type=float, default=0.0, help="projector 1: nominal step in voxels (0 = 0.5)")
    ap.add_argument("--timeline", action="store_true",
                    help="instead of the bench line: the kernel timeline of one solve, recorded inside the kernels")
    ap.add_argument("--timeline-out", default=None, help="with --timeline: write the event list to this text file")
    ap.add_argument("--grad-tol", type=float, default=None)
    ap.add_argument("--study-max-iter", type=int, default=30)
    args = ap.parse_args()
    args.warmup = max(args.warmup, 0)
    from paper_1004_0014_b200.replicas import env_rank_world
    rank, local_rank, world = env_rank_world()
    cfg = get_config(args.config)
    if args.fan is None:
        # measured: two candidates per pass win up to C2's size for one solve in flight (C1 0.95 against 1.06 ms,
        # C2 2.55 against 2.68), one candidate wins beyond (C4: 8.45 against 9.11) and for solves in flight
        args.fan = 2 if max(int(args.in_flight), 1) == 1 and cfg.V <= (1 << 23) else 1
    if args.frames_study:
        run_frames_study(args, cfg, rank, local_rank)
    elif args.pca_study:
        run_pca_study(args, cfg, rank, local_rank)
    elif args.timeline:
        run_timeline(args, cfg, rank, local_rank)
    elif args.impl == "reference":
        run_reference(args, cfg, rank, world)
    else:
        run_ours(args, cfg, rank, local_rank, world)


if __name__ == "__main__":
    main()
