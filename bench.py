#!/usr/bin/env python
"""bench.py - throughput of the DrivingVoxels hot path (steps 1-5 behind include/dvx.h) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 3] [--impl reference]

One "step" = one pass of the whole hot path over one synthetic frame: dvx_render (projection + binning, key
generation + radix sort, ray-OBB schedule, compositing) followed by dvx_backward (replay + atomics + SH post-pass).
Workload at N=1: BASELINE.json configs[2] ("PandaSet-shaped frame", 1920x1080, 4 M + 10x50 k voxels, SH degree 3,
K = 8), the configuration the metric is quoted on.  Prints ONE JSON line.
The path does not shard (BASELINE.json north_star: one GPU, no collectives): --gpus N runs N independent replicas.
"""
import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "fwd+bwd megapixels/s at 1920x1080 (1 B200)"
UNIT = "MP/s"
SMI_QUERY = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
             "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=30)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=3, help="BASELINE.json config number 1..5 (default 3 = the headline workload)")
    ap.add_argument("--impl", default="dvx", choices=["dvx", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true", help="skip the oracle timing leg (profiling runs)")
    ap.add_argument("--cpu-tiles", type=int, default=0, help="tiles in the CPU-oracle sample (0 = pick for about 10-30 s)")
    ap.add_argument("--fwd-only", action="store_true", help="profiling aid: time dvx_render alone")
    ap.add_argument("--k-samples", type=int, default=0, help="report-only variant: override K (samples per voxel segment)")
    ap.add_argument("--activation", type=int, default=-1, help="report-only variant: density activation (0 exp, 1 exp-linear, R5)")
    ap.add_argument("--opaque", action="store_true", help="report-only variant 3b: config 3 with raw += 8 on leaves holding a LiDAR return")
    ap.add_argument("--no-records", action="store_true",
                    help="A/B aid: DVX_FLAG_NO_RECORDS (the backward walks the tile lists again instead of replaying hit records)")
    ap.add_argument("--no-extra", action="store_true", help="skip the extra workloads (configs 4 and 5) reported beside the headline")
    ap.add_argument("--profiler-range", action="store_true",
                    help="bracket the first timed region with cudaProfilerStart/Stop (use with ncu --profile-from-start off)")
    return ap.parse_args()


def workload_name(n):
    return {1: "config1_tiny_128x96", 2: "config2_small_960x540", 3: "config3_pandaset_shaped_1920x1080_4M+10x50k_sh3_K8",
            4: "config4_crowded_1920x1080_500k+40x25k_sh3_K8", 5: "config5_training_batch_6x1920x1080_8M+20x50k_sh3_K8"}[n]


# ----------------------------------------------------------------------------------------------- clocks
class ClockSampler:
    """nvidia-smi sampled every 50 ms DURING the timed region (B200_PROFILING.md clocks line)."""

    def __init__(self, index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), "--query-gpu=" + SMI_QUERY, "--format=csv,noheader,nounits",
                                       "-lms", "50"], stdout=self.f, stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def stop(self):
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.p.kill()
        self.f.flush()
        rows = [r.split(",") for r in open(self.f.name).read().strip().splitlines() if r.strip()]
        os.unlink(self.f.name)
        sm, smax, reasons, power = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in rows:
            try:
                sm.append(float(r[1])); smax.append(float(r[2])); power.append(float(r[3]))
            except (ValueError, IndexError):
                continue
            for name, val in zip(names, r[5:9]):
                if val.strip().lower() == "active":
                    reasons.add(name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(smax)), "reasons": sorted(reasons),
                "samples": len(sm), "power_w_max": max(power)}


def config_dict(args, scene, world):
    """The `config` object of the JSON line: the same keys from both arms (the driver compares them)."""
    return {"workload": workload_name(args.config) + ("_opaque3b" if args.opaque else "") + ("_K%d" % args.k_samples if args.k_samples else "") + ("_act%d" % args.activation if args.activation >= 0 else ""),
            "cameras": len(scene.cameras), "k_samples": scene.k_samples, "sh_degree": scene.static.sh_degree,
            "voxels": int(sum(t.n_voxels for t in scene.octrees)), "actors": len(scene.actors),
            "l2_policy": "inputs larger than L2 (voxel records + gradient buffers >> 126 MB)", "replicas": world,
            "passes": "fwd" if args.fwd_only else "fwd+bwd"}


# ----------------------------------------------------------------------------------------------- CPU oracle leg
def oracle_sample(scene, n_tiles_sample, backward, seed=7):
    """Times the oracle (tile-culled mode, validated bit-identical to brute force by pin P13), as it stands, on a seeded
    sample of whole 16x16 tiles of camera 0.  Returns dict(seconds_binning, seconds_sample, pixels, mp_s_full_frame)."""
    from oracle import oracle as O
    cam = scene.cameras[0]
    H, W = cam.height, cam.width
    tw, th = (W + 15) // 16, (H + 15) // 16
    rng = np.random.default_rng(seed)
    tiles = rng.choice(tw * th, size=min(n_tiles_sample, tw * th), replace=False)
    mask = np.zeros((H, W), dtype=np.uint8)
    for t in tiles:
        ty, tx = divmod(int(t), tw)
        mask[ty * 16:(ty + 1) * 16, tx * 16:(tx + 1) * 16] = 1
    gin = scene.image_grads(rgb_std=1e-2) if backward else None
    t0 = time.perf_counter()
    O.render(scene, mode=1, mask=np.zeros((H, W), dtype=np.uint8))       # binning of the whole frame, no pixel rendered
    t_bin = time.perf_counter() - t0
    t0 = time.perf_counter()
    O.render(scene, mode=1, mask=mask, grads_in=gin)
    t_all = time.perf_counter() - t0
    npx = int(mask.sum())
    t_px = max(t_all - t_bin, 1e-9)
    full = t_bin + t_px * (W * H / npx)
    return {"seconds_binning": t_bin, "seconds_sample": t_all, "pixels": npx, "tiles": int(len(tiles)),
            "mp_s_full_frame": W * H / full / 1e6, "threads": O.num_threads()}


def pick_cpu_tiles(scene, backward):
    """Sizes the sample for roughly 15 s of CPU work from a 4-tile probe."""
    probe = oracle_sample(scene, 4, backward, seed=11)
    per_tile = max((probe["seconds_sample"] - probe["seconds_binning"]) / 4, 1e-3)
    return int(min(max(15.0 / per_tile, 8), 8160))


def run_reference(args, scene):
    """--impl reference: the oracle as it stands on the host cores, each step a bounded sample of the workload.
    `ms_per_step` is the wall time one step really took (so steps x ms_per_step is what the driver's clock saw); the
    full-frame time the metric needs is extrapolated from it (binning + per-pixel time x W*H) under its own key."""
    n_tiles = args.cpu_tiles or max(4, pick_cpu_tiles(scene, True) // max(args.steps + args.warmup, 1))
    vals, wall = [], []
    for it in range(args.warmup + args.steps):
        t0 = time.perf_counter()
        r = oracle_sample(scene, n_tiles, True, seed=100 + it)
        if it >= args.warmup:
            vals.append(r)
            wall.append(time.perf_counter() - t0)
    mp = float(np.mean([r["mp_s_full_frame"] for r in vals]))
    cam = scene.cameras[0]
    sample = "%d seeded 16x16 tiles (%d px) of camera 0 per step, fwd+bwd, tile-culled oracle; full-frame time = binning + per-pixel time x W*H" % (
        vals[0]["tiles"], vals[0]["pixels"])
    line = {"impl": "reference", "metric": METRIC, "value": mp, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": float(np.mean(wall)) * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": config_dict(args, scene, args.gpus),
            "full_frame_ms_extrapolated": cam.width * cam.height / (mp * 1e6) * 1e3,
            "cpu_baseline": {"value": mp, "unit": UNIT, "cores": vals[0]["threads"], "kind": "oracle", "sample": sample},
            "e2e": {"value": mp, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}, "gpu_launches": 0}
    print(json.dumps(line))


# ----------------------------------------------------------------------------------------------- replicas
def max_over_ranks(ms, device=None):
    """Replicas only: the job time is the slowest replica's.  all_reduce(MAX) over the default
    process group (nccl on the GPU box, gloo in the CPU test); identity for a single process."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(ms)
    t = torch.tensor([float(ms)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_value(px_per_step_per_replica, world, ms_per_step):
    """Whole-job MP/s of `world` independent replicas that each finish a step of px pixels in ms_per_step (max over ranks)."""
    return world * px_per_step_per_replica / (ms_per_step * 1e-3) / 1e6


# ----------------------------------------------------------------------------------------------- GPU arm
def measured_peaks():
    """Roofline denominators: MEASURED_PEAKS.json (driver-written) or the fallback B200_PROFILING.md states."""
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        d = json.load(open(path))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json)", d
    except (OSError, ValueError, KeyError):
        return 6650.0, "fallback (B200_PROFILING.md)", {}


def algorithmic_bytes(scene, W, H, cnt, touched):
    """bytes the method must move, from the run's own counters.  cnt: v_vis (per frame), pairs_eff."""
    n_sh = scene.static.n_sh
    rec = 8 + 32 + 12 * n_sh                    # key + 8 corner densities + SH coefficients of one voxel record
    px = W * H
    b = {}
    b["min_fwd"] = cnt["v_vis"] * rec + 20 * px
    b["min_fwdbwd"] = b["min_fwd"] + 12 * px + touched * (2 * 32 + 2 * 12 * n_sh)
    # per kernel (what a tile-sort rasterizer of this method streams): id + per-frame voxel record + corners
    b["composite_fwd"] = cnt["pairs_eff"] * (4 + 32 + 32) + 20 * px + 24 * px
    b["composite_bwd"] = cnt["pairs_eff"] * (4 + 32 + 32) + px * (12 + 24) + touched * (2 * 32 + 2 * 16)
    return b


def _bits_for(n):
    b = 1
    while (1 << b) < n:
        b += 1
    return b


def sort_throughput(ctx, n_pairs, scene, W, H, reps=5):
    """Step 2's radix sort alone (dvx_sort_pairs: the same kernels dvx_render runs), on as many seeded random pairs as one
    frame produces, with the frame's key width (tile | octant | combined rank of all octrees).  Mpairs/s, CUDA events, median of reps."""
    import torch
    n_tiles = ((W + 15) // 16) * ((H + 15) // 16)
    key_bits = _bits_for(sum(t.n_voxels for t in scene.octrees)) + _bits_for(n_tiles * 8)   # combined rank | tile, octant
    n = max(int(n_pairs), 1)
    g = torch.Generator(device="cuda").manual_seed(1)
    base = torch.randint(0, 1 << min(key_bits, 62), (n,), dtype=torch.int64, device="cuda", generator=g)
    vals0 = torch.arange(n, dtype=torch.int32, device="cuda")
    times = []
    for _ in range(reps + 1):
        keys, vals = base.clone(), vals0.clone()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        ctx.check(ctx.lib.dvx_sort_pairs(ctx.h, keys.data_ptr(), vals.data_ptr(), n, key_bits))
        e1.record()
        torch.cuda.synchronize()
        times.append(e0.elapsed_time(e1))
    assert bool((keys[1:] >= keys[:-1]).all())
    ms = float(np.median(times[1:]))
    return {"pairs": n, "key_bits": key_bits, "passes": (key_bits + 7) // 8, "ms": ms, "mpairs_per_s": n / ms / 1e3,
            "gb_per_s_moved": n * 12 * 2 * ((key_bits + 7) // 8) / ms / 1e6}


def optimizer_step_stats(ctx, dev, grads, peak, reps=5):
    """Widening row N2, reported beside the headline (not part of `value`): the optimizer step that follows the
    rasterizer's backward - dvx_grid_adam_step on the corner densities of every octree and dvx_adam_step on their SH
    coefficients, all octrees in one launch each (dvx_*_step_n) - timed with CUDA events (median of reps) against its algorithmic bytes:
      grid Adam : per grid point 4 (CSR offset) + 12 read + 12 written (density, m, v), per corner slot 4 (slot index)
                  + 4 (gradient read) + 4 (gradient zeroed) + 4 (corner record written)  = 28 G + 16 * 8V
                  (two kernels: the per-point update, then the per-voxel rewrite of the corner and gradient records,
                  which also reads the 4-byte point index of every slot: + 4 * 8V of real traffic, not counted)
      SH Adam   : 32 bytes per coefficient (g, p, m, v read; p, m, v, g = 0 written)"""
    import torch
    hp = dict(lr=0.01, beta1=0.9, beta2=0.99, eps=1e-15)
    grids, build_ms = [], 0.0
    for t in dev.trees:
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        grids.append(ctx.grid(t.code))
        e1.record()
        torch.cuda.synchronize()
        build_ms += e0.elapsed_time(e1)
    state = []
    for t, g in zip(dev.trees, grids):
        d = torch.zeros(g.n_points, device=ctx.device)
        if t.n_voxels:
            d[g.point_of().reshape(-1).long()] = t.geo.reshape(-1)   # the scene's corner record is consistent on shared corners
        state.append((d, torch.zeros_like(d), torch.zeros_like(d), torch.zeros_like(t.sh), torch.zeros_like(t.sh)))
    G_total = sum(g.n_points for g in grids)
    V_total = sum(t.n_voxels for t in dev.trees)
    n_sh = sum(t.sh.numel() for t in dev.trees)
    t_grid, t_sh = [], []
    for r in range(reps + 1):
        for (dgeo, dsh) in grads:  # the kernels zero the gradients: refill so that every repetition does the same work
            dgeo.fill_(1e-3); dsh.fill_(1e-3)
        e = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
        torch.cuda.synchronize()
        e[0].record()
        ctx.grid_adam_step_n([(g, d, m, v, dgeo, t.geo) for t, g, (d, m, v, ms, vs), (dgeo, dsh) in
                              zip(dev.trees, grids, state, grads)], step=r + 1, **hp)
        e[1].record()
        ctx.adam_step_n([(t.sh, ms, vs, dsh) for t, (d, m, v, ms, vs), (dgeo, dsh) in zip(dev.trees, state, grads)],
                        step=r + 1, **hp)
        e[2].record()
        torch.cuda.synchronize()
        t_grid.append(e[0].elapsed_time(e[1])); t_sh.append(e[1].elapsed_time(e[2]))
    ms_grid, ms_sh = float(np.median(t_grid[1:])), float(np.median(t_sh[1:]))
    b_grid, b_sh = 28 * G_total + 16 * 8 * V_total, 32 * n_sh
    for g in grids:
        g.close()
    return {"grid_points": G_total, "corner_slots": 8 * V_total, "sh_coefficients": n_sh, "grid_build_ms": build_ms,
            "grid_adam": {"ms": ms_grid, "bytes": b_grid, "gb_per_s": b_grid / ms_grid / 1e6, "hbm_frac": b_grid / ms_grid / 1e6 / peak},
            "sh_adam": {"ms": ms_sh, "bytes": b_sh, "gb_per_s": b_sh / ms_sh / 1e6, "hbm_frac": b_sh / ms_sh / 1e6 / peak},
            "launches": 3 * ((len(dev.trees) + 31) // 32)}


def feature_stats(ctx, dev, scene, peak, n_ch=64, reps=5):
    """Widening row N3, reported beside the headline (not part of `value`): camera 0's compositing weights exported as a
    CSR matrix (one replay of the tile kernel), then the feature render F = W feat and the fuser num += W^T img for C = 64
    channels, CUDA events, median of reps.  Bytes: `dram_floor` = every datum once (8 nnz CSR + 4C per touched voxel row +
    4C per pixel); `gathered` = what the SMs pull through L1/L2 (8 nnz + 4C nnz + 4C per pixel)."""
    import torch
    cam = scene.cameras[0]
    H, W = cam.height, cam.width
    _, _, _, fr = dev.render(0, save=True)   # warm call: first-use allocations of the CSR arrays go through the caching allocator
    fr.weights()
    fr.release()
    _, _, _, fr = dev.render(0, save=True)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record()
    nnz, rows, vox, w = fr.weights()
    e1.record()
    torch.cuda.synchronize()
    export_ms = e0.elapsed_time(e1)
    v_total = sum(t.n_voxels for t in dev.trees)
    g = torch.Generator(device="cuda").manual_seed(3)
    feat = torch.rand((v_total, n_ch), device="cuda", generator=g) * 2 - 1
    img = torch.rand((H, W, n_ch), device="cuda", generator=g) * 2 - 1
    num = torch.zeros((v_total, n_ch), device="cuda")
    wsum = torch.zeros(v_total, device="cuda")
    touched = int(torch.unique(vox).numel()) if nnz else 0
    t_r, t_f = [], []
    for _ in range(reps + 1):
        e = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
        e[0].record()
        fr.render_features(feat, H, W)
        e[1].record()
        fr.fuse_features(img, num, wsum)
        e[2].record()
        torch.cuda.synchronize()
        t_r.append(e[0].elapsed_time(e[1])); t_f.append(e[1].elapsed_time(e[2]))
    fr.release()
    ms_r, ms_f = float(np.median(t_r[1:])), float(np.median(t_f[1:]))
    floor = 8 * nnz + 4 * n_ch * touched + 4 * n_ch * H * W
    gathered = 8 * nnz + 4 * n_ch * nnz + 4 * n_ch * H * W

    def leg(ms, extra=0):
        return {"ms": ms, "mp_per_s": H * W / ms / 1e3, "dram_floor_gb_per_s": (floor + extra) / ms / 1e6,
                "dram_floor_hbm_frac": (floor + extra) / ms / 1e6 / peak, "gathered_gb_per_s": gathered / ms / 1e6}
    return {"channels": n_ch, "nnz": nnz, "touched_voxels": touched, "weights_export_ms": export_ms,
            "bytes": {"dram_floor": floor, "gathered": gathered},
            "render": leg(ms_r), "fuse": leg(ms_f, 4 * n_ch * touched), "launches": 1 + 2 * (reps + 1) + 3}


def structure_stats(ctx, dev, scene, n_points=2_000_000):
    """Widening row N4, reported beside the headline (not part of `value`): the LiDAR-guided structure operations on the
    static octree with a seeded synthetic cloud (points scattered around the centres of randomly chosen leaves, sigma = 2
    minimum voxel sizes): cloud binning, one proximity-subdivision round (threshold 1.5 s), grid tables + Eq. 1 prior on the
    result, pruning at v < -9.5.  One-off operations, search- and fp64-bound: times and rates only, no roofline claim."""
    import torch
    t = dev.trees[0]
    tree = scene.octrees[0]
    if t.n_voxels == 0:
        return None
    code = t.code
    level = (code >> 48) & 31
    lmax = int(level.max())
    side = float(tree.side)
    s_min = side / (1 << lmax)
    g = torch.Generator(device="cuda").manual_seed(11)
    pick = torch.randint(0, t.n_voxels, (n_points,), device="cuda", generator=g)
    # leaf centres from the code (input generation only: 3-bit groups -> lattice coordinates)
    c = code[pick]
    xyz = torch.zeros((n_points, 3), dtype=torch.float64, device="cuda")
    for m in range(16):
        grp = (c >> (45 - 3 * m)) & 7
        for a, sh in enumerate((2, 1, 0)):
            xyz[:, a] += ((grp >> sh) & 1).double() * (1 << (15 - m))
    size = (1 << (16 - ((c >> 48) & 31))).double()
    centre = torch.tensor([float(x) for x in tree.center], dtype=torch.float64, device="cuda")
    pos = centre - 0.5 * side + (xyz + 0.5 * size[:, None]) * (side / 65536.0)
    pts = (pos + torch.randn((n_points, 3), dtype=torch.float64, device="cuda", generator=g) * (2.0 * s_min)).float().contiguous()

    def timed(fn):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record()
        r = fn()
        e1.record()
        torch.cuda.synchronize()
        return r, e0.elapsed_time(e1)
    thr = 1.5 * s_min
    cloud, ms_cloud = timed(lambda: ctx.cloud(pts, thr))
    (new, split), ms_sub = timed(lambda: ctx.subdivide_near(cloud, code, tree.center, side, thr, min(lmax + 1, 16)))
    new = new.contiguous()
    grid, ms_grid = timed(lambda: ctx.grid(new))
    s2 = 0.5 * s_min
    cloud2, ms_cloud2 = timed(lambda: ctx.cloud(pts, 3.1 * s2))
    dens, ms_prior = timed(lambda: ctx.density_prior(cloud2, new, tree.center, side, grid, s2))
    geo = torch.empty((new.shape[0], 8), device="cuda")
    grid.gather(dens, geo)
    (kept, idx), ms_prune = timed(lambda: ctx.prune(new, geo, -9.5))
    out = {"points": n_points, "leaves_in": t.n_voxels, "leaves_split": int(split.sum().item()), "leaves_out": int(new.shape[0]),
           "grid_points": grid.n_points, "leaves_after_prune": int(kept.shape[0]),
           "cloud_build_ms": ms_cloud, "subdivide_round_ms": ms_sub, "mleaves_per_s": t.n_voxels / ms_sub / 1e3,
           "grid_tables_ms": ms_grid, "density_prior_ms": ms_prior, "mpoints_per_s": grid.n_points / ms_prior / 1e3,
           "prune_ms": ms_prune}
    for o in (cloud, cloud2, grid):
        o.close()
    return out


def time_workload(ctx, dvx, cfg, steps, warmup):
    """fwd+bwd step time of another BASELINE.json config on this context: every camera of the scene rendered and
    back-propagated into one gradient set, inputs resident in HBM, CUDA events around `steps` steps after `warmup`."""
    import torch
    import dvx_scenes
    scene = dvx_scenes.make_config(cfg)
    dev = dvx.SceneOnDevice(ctx, scene)
    grads = dev.zero_grads()
    n_cams = len(scene.cameras)
    cam0 = scene.cameras[0]
    g_dev = [torch.from_numpy(scene.image_grads(c, rgb_std=1e-2)["rgb"]).to(ctx.device) for c in range(n_cams)]
    out = (torch.empty((cam0.height, cam0.width, 3), device=ctx.device), torch.empty((cam0.height, cam0.width), device=ctx.device),
           torch.empty((cam0.height, cam0.width), device=ctx.device))

    outs = [tuple(torch.empty_like(t) for t in out) for _ in range(n_cams)] if n_cams > 1 else None

    def step():
        if n_cams > 1:   # the batched entry points: one host round trip, steps 1-2 and the SH post-pass on the second stream
            _, frames = dev.render_batch(save=True, outs=outs)
            ctx.backward_batch(frames, g_dev, grads)
            for fr in frames:
                fr.release()
            return
        _, _, _, fr = dev.render(0, save=True, out=out)
        fr.backward(g_dev[0], grads=grads)
        fr.release()
    for _ in range(warmup):
        step()
    ctx.stage_ms_collect()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record()
    for _ in range(steps):
        step()
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / steps
    sums, _ = ctx.stage_ms_collect()
    px = n_cams * cam0.width * cam0.height
    res = {"ms_per_step": ms, "value": px / ms / 1e3, "unit": UNIT, "cameras": n_cams, "steps": steps, "warmup": warmup,
           "api": "dvx_render_batch + dvx_backward_batch" if n_cams > 1 else "dvx_render + dvx_backward",
           "voxels": int(sum(t.n_voxels for t in scene.octrees)), "actors": len(scene.actors),
           "stage_ms": {k: v / steps for k, v in sums.items()}}
    for t in dev.trees:
        t.close()
    del dev, grads, g_dev, out
    ctx.trim()
    return res


def run_dvx(args):
    import torch
    import torch.distributed as dist
    import dvx_scenes
    import paper_2606_23031_b200 as dvx

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: libdvx has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    scene = make_scene(args)
    ctx = dvx.Context(local)
    dev = dvx.SceneOnDevice(ctx, scene)
    n_cams = len(scene.cameras)
    cam0 = scene.cameras[0]
    W, H = cam0.width, cam0.height
    px_step = n_cams * W * H
    grads = dev.zero_grads()
    g_dev = [torch.from_numpy(scene.image_grads(c, rgb_std=1e-2)["rgb"]).to(ctx.device) for c in range(n_cams)]
    g_host = [g.cpu().pin_memory() for g in g_dev]
    out_dev = (torch.empty((H, W, 3), dtype=torch.float32, device=ctx.device), torch.empty((H, W), dtype=torch.float32, device=ctx.device),
               torch.empty((H, W), dtype=torch.float32, device=ctx.device))
    out_host = tuple(t.cpu().pin_memory() for t in out_dev)

    outs_b = [tuple(torch.empty_like(t) for t in out_dev) for _ in range(n_cams)] if n_cams > 1 else None

    def step(host=False, bwd=True):
        if n_cams > 1 and not host and not args.no_records:   # config 5: the batched entry points
            _, frames = dev.render_batch(save=bwd, outs=outs_b)
            if bwd:
                ctx.backward_batch(frames, g_dev, grads)
                for fr in frames:
                    fr.release()
            return
        for c in range(n_cams):
            _, _, _, fr = dev.render(c, save=bwd, out=out_host if host else out_dev, host=host,
                                     flags=dvx.FLAG_NO_RECORDS if args.no_records else 0)
            if bwd:
                fr.backward(g_host[c] if host else g_dev[c], grads=grads, host=host)
                fr.release()

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def timed(n, **kw):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        e0.record()
        for _ in range(n):
            step(**kw)
        if kw.get("host"):
            ctx.host_io_wait()   # the timed stream waits for the last frames' copy-outs: they are inside the timed region
        e1.record()
        barrier()
        return max_over_ranks(e0.elapsed_time(e1), ctx.device)

    # ---- untimed: counters of this workload (one frame per camera, counting build of the kernels)
    cnt = {"v_vis": 0, "pairs": 0, "pairs_eff": 0, "q_test": 0, "q_hit": 0}
    for c in range(n_cams):
        _, _, _, fr = dev.render(c, save=True, flags=dvx.FLAG_COUNTERS)
        for k, v in fr.counters().items():
            cnt[k] += v
        fr.release()
    if cnt["pairs_eff"] == 0:
        cnt["pairs_eff"] = cnt["pairs"]
    for _ in range(args.warmup):
        step(bwd=not args.fwd_only)
    torch.cuda.synchronize()
    touched = int(sum(int((g[0] != 0).any(dim=1).sum().item()) for g in grads))
    # fraction of rays that reached T < t_stop (camera 0), hits per ray; step 0 uncached; the caller's gradient zeroing
    frac_term = float((out_dev[2] > 1.0 - scene.t_stop).float().mean().item()) if scene.t_stop > 0 else 0.0
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t = scene.octrees[0]
    e0.record()
    tmp = ctx.octree(dev.trees[0].code, dev.trees[0].geo, dev.trees[0].sh, t.center, t.side, t.sh_degree)  # 8 sorts of V keys
    e1.record()
    torch.cuda.synchronize()
    step0_ms = e0.elapsed_time(e1)
    tmp.close()
    e0.record()
    for ga, gb in grads:
        ga.zero_(); gb.zero_()
    e1.record()
    torch.cuda.synchronize()
    grad_zero_ms = e0.elapsed_time(e1)
    for _ in range(2):  # refill the gradient buffers so that the timed steps accumulate into touched memory as before
        step(bwd=not args.fwd_only)
    torch.cuda.synchronize()

    # ---- timed region 1: device-resident inputs
    ctx.stage_ms_collect()                       # drop the stage times of the warm-up frames
    l0 = ctx.lib.dvx_launch_count()
    sampler = ClockSampler(local) if rank == 0 else None
    if args.profiler_range:
        torch.cuda.synchronize()
        torch.cuda.cudart().cudaProfilerStart()
    ms_total = timed(args.steps, bwd=not args.fwd_only)
    if args.profiler_range:
        torch.cuda.cudart().cudaProfilerStop()
    launches = int(ctx.lib.dvx_launch_count() - l0)
    sums, n_frames = ctx.stage_ms_collect()      # CUDA-event stage times of exactly the timed steps (on the ctx stream)
    stage = {k: v / args.steps for k, v in sums.items()}
    # ---- forward only (reported beside the headline)
    for _ in range(2):
        step(bwd=False)
    ms_fwd = timed(args.steps, bwd=False)
    # ---- timed region 2: end to end through the host-buffer entry points (pinned host <-> device copies inside)
    for _ in range(2):
        step(host=True, bwd=not args.fwd_only)
    ms_e2e = timed(args.steps, host=True, bwd=not args.fwd_only)
    clocks = sampler.stop() if sampler else None
    sort_stats = sort_throughput(ctx, cnt["pairs"] // n_cams, scene, W, H) if rank == 0 else None
    # the widening rows and the extra workloads are single-process reports: with replicas the other ranks would sit in the
    # process-group teardown while rank 0 measures them
    solo = rank == 0 and world == 1 and not args.fwd_only
    feat_stats = feature_stats(ctx, dev, scene, measured_peaks()[0]) if solo else None
    struct_stats = structure_stats(ctx, dev, scene) if solo else None
    opt_stats = optimizer_step_stats(ctx, dev, grads, measured_peaks()[0]) if solo else None
    rec_stats = None
    if rank == 0 and not args.fwd_only and not args.no_records:   # what the hit records of one frame take (camera 0)
        _, _, _, fr = dev.render(0, save=True)
        rec_stats = fr.record_stats()
        rec_stats["bytes_per_hit"] = rec_stats["bytes_used"] / max(cnt["q_hit"] / n_cams, 1)
        fr.release()
    extra = None
    if rank == 0 and world == 1 and args.config == 3 and not (args.no_extra or args.fwd_only or args.opaque or args.k_samples or args.no_records or args.activation >= 0):
        extra = {}
        for cfg_x in (4, 5):   # BASELINE.json configs[3] (crowded) and configs[4] (6-camera training batch), device-resident
            extra[workload_name(cfg_x)] = time_workload(ctx, dvx, cfg_x, steps=max(3, min(args.steps, 10)), warmup=3)

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    ms_step = ms_total / args.steps
    value = aggregate_value(px_step, world, ms_step)
    fwd_value = aggregate_value(px_step, world, ms_fwd / args.steps)
    e2e_value = aggregate_value(px_step, world, ms_e2e / args.steps)
    peak, peak_src, peaks = measured_peaks()
    ab = algorithmic_bytes(scene, W, H, {k: v / 1 for k, v in cnt.items()}, touched)
    # ---- rooflines.  [NS] names the HBM roofline; the compositing kernels are bound by instruction issue,
    # so both are reported: HBM for the dominant kernel (the one with the largest share of the step in THIS run), and the issue
    # rate against the FMA / issue peak measured a moment ago by dvx_microbench_fma on this device.
    kernels = {"composite_fwd": stage.get("composite", 0.0)}
    if not args.fwd_only:
        kernels["composite_bwd"] = stage.get("backward_composite", 0.0)
    dom = max(kernels, key=kernels.get)
    dom_ms = kernels[dom]
    dom_bytes = ab[dom]
    achieved = dom_bytes / (dom_ms * 1e-3) / 1e9 if dom_ms > 0 else 0.0
    prof = {}
    try:  # ncu --set full capture of the two compositing kernels (profiles/traffic.json names its commit and source hash)
        prof = json.load(open(os.path.join(ROOT, "profiles", "traffic.json")))
    except (OSError, ValueError):
        pass
    src = os.path.join(ROOT, "paper_2606_23031_b200", "csrc", "dvx_composite_tile.cu")
    try:
        import hashlib
        src_sha = hashlib.sha256(open(src, "rb").read()).hexdigest()
    except OSError:
        src_sha = None
    stale = (not prof) or prof.get("source_sha256") != src_sha or prof.get("workload") != workload_name(args.config)
    pk = prof.get("kernels", {})
    hbm_floor_ms = ab["min_fwdbwd" if not args.fwd_only else "min_fwd"] / peak / 1e6
    hbm_frac_step = hbm_floor_ms / ms_step
    mb = ctx.microbench_fma()
    issue_peak = mb["warp_instr_per_s"]
    issue = {"peak_warp_instr_per_s": issue_peak, "peak_lane_fma_per_s": mb["lane_fma_per_s"],
             "peak_source": "dvx_microbench_fma in this run (%.3f ms, 16 FFMA chains per thread on every warp slot)" % mb["ms"],
             "nominal_warp_instr_per_s": 148 * 4 * ((clocks or {}).get("sm_mhz") or peaks.get("sm_max_mhz") or 1965.0) * 1e6,
             "kernels": {}}
    issue_floor_ms = None
    if pk and not stale:
        issue_floor_ms = 0.0
        for k, ms_k in kernels.items():
            if k in pk and ms_k > 0:
                wi = pk[k]["warp_instructions"]
                floor = wi / issue_peak * 1e3
                issue_floor_ms += floor
                issue["kernels"][k] = {"warp_instructions": wi, "ms": ms_k, "achieved_warp_instr_per_s": wi / (ms_k * 1e-3),
                                       "frac": wi / (ms_k * 1e-3) / issue_peak, "issue_floor_ms": floor}
    binding = max(hbm_floor_ms, issue_floor_ms or 0.0)
    rec_bytes = 0 if (args.fwd_only or args.no_records) else 44 * cnt["q_hit"] / n_cams
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
        "data": "synthetic", "config": config_dict(args, scene, world),
        "fwd_value": fwd_value, "fwd_ms": ms_fwd / args.steps,
        "hbm_roofline_frac_step": hbm_frac_step,       # the [NS] definition: B_min / peak / step time (target 0.5: NOT met)
        "hbm_floor_ms": hbm_floor_ms, "issue_floor_ms": issue_floor_ms,
        # the larger of the two floors over the step time; None when no fresh ncu instruction count exists for this workload
        "frac_of_binding_floor": binding / ms_step if (ms_step > 0 and issue_floor_ms is not None) else None,
        "stage_ms": stage,
        "counters": dict(cnt, touched_voxels=touched, hits_per_ray=cnt["q_hit"] / px_step, frac_rays_terminated=frac_term),
        "records": rec_stats,
        "step0_uncached_ms_static_octree": step0_ms, "grad_zero_ms_excluded": grad_zero_ms,
        "algorithmic_bytes": ab,
        "roofline": {"bound": "hbm", "kernel": dom, "achieved": achieved, "peak": peak, "unit": "GB/s",
                     "frac": achieved / peak if peak else None,
                     # the same kernel with the hit records it streams counted as well (this design's own traffic, 44 B per
                     # composited hit in each direction; not part of SURVEY 8(d)'s algorithmic bytes)
                     "achieved_with_records": (dom_bytes + rec_bytes) / (dom_ms * 1e-3) / 1e9 if dom_ms > 0 else 0.0,
                     "frac_with_records": (dom_bytes + rec_bytes) / (dom_ms * 1e-3) / 1e9 / peak if (dom_ms > 0 and peak) else None,
                     "traffic": (pk.get(dom) or {}).get("dram_bytes"), "traffic_commit": prof.get("commit"),
                     "traffic_note": "traffic above the algorithmic bytes is the hit-record stream (44 B per composited hit, written by "
                                     "the forward, read by the backward instead of re-walking the tile lists; DESIGN.md section 6), not re-reads",
                     "traffic_stale": bool(stale), "peak_source": peak_src, "bytes_per_launch": dom_bytes, "ms_per_launch": dom_ms,
                     "all_kernels_ms": kernels,
                     # both compositing kernels (the forward writes the hit records, the backward reads them)
                     "per_kernel": {k: {"ms": ms_k, "algorithmic_bytes": ab[k],
                                        "achieved": ab[k] / (ms_k * 1e-3) / 1e9 if ms_k > 0 else 0.0,
                                        "frac": ab[k] / (ms_k * 1e-3) / 1e9 / peak if (ms_k > 0 and peak) else None,
                                        "frac_with_records": (ab[k] + rec_bytes) / (ms_k * 1e-3) / 1e9 / peak if (ms_k > 0 and peak) else None,
                                        "traffic": (pk.get(k) or {}).get("dram_bytes")} for k, ms_k in kernels.items()}},
        "issue_roofline": dict(issue, bound="alu", unit="warp-instr/s", profile_commit=prof.get("commit"), profile_stale=bool(stale)),
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": (0 if args.fwd_only else 12 * px_step),
                "d2h_bytes_per_step": 20 * px_step, "ms_per_step": ms_e2e / args.steps},
        "sort": sort_stats, "n2_optimizer_step": opt_stats, "n3_features": feat_stats, "n4_structure": struct_stats,
        "extra_workloads": extra,
        "gpu_launches": launches, "clocks": clocks,
    }
    if not args.no_cpu_baseline and world == 1:
        n_tiles = args.cpu_tiles or pick_cpu_tiles(scene, True)
        r = oracle_sample(scene, n_tiles, True)
        line["cpu_baseline"] = {"value": r["mp_s_full_frame"], "unit": UNIT, "cores": r["threads"], "kind": "oracle",
                                "sample": "%d seeded 16x16 tiles (%d px) of camera 0, fwd+bwd, tile-culled oracle (pin P13); "
                                          "full-frame time = whole-frame binning (%.1f s) + per-pixel time x W*H" % (
                                              r["tiles"], r["pixels"], r["seconds_binning"])}
    else:
        line["cpu_baseline"] = None
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def make_scene(args):
    import dvx_scenes
    scene = dvx_scenes.make_config(args.config, **({"opaque": True} if args.opaque and args.config == 3 else {}))
    if args.k_samples:
        scene.k_samples = args.k_samples
    if args.activation >= 0:
        scene.activation = args.activation
    return scene


def main():
    args = parse_args()
    if args.impl == "reference":
        if int(os.environ.get("RANK", "0")) != 0:
            return
        import dvx_scenes
        run_reference(args, make_scene(args))
        return
    run_dvx(args)


if __name__ == "__main__":
    main()
