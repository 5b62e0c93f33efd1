"""The five BASELINE.json workloads as concrete, seeded synthetic inputs (recipe: DESIGN.md §4).

``make_config(n)`` returns a ``Scene``.  Seed of config n is 1000+n.  Shapes follow PandaSet
(1920x1080 front camera, 64-beam LiDAR, 80-sweep sequences, car/truck boxes; PAPER.md:131,
:299-307); the records themselves are synthetic and stand in for the dataset.
Inputs only - no rendering arithmetic lives here.
"""
import numpy as np
from . import rng, lidar, octree

CAR = (4.5, 2.0, 1.6)
TRUCK = (10.0, 2.5, 3.5)


class Camera:
    def __init__(self, width, height, fx, fy, cx, cy, c2w, near=0.05, far=1.0e9):
        self.width, self.height = int(width), int(height)
        self.fx, self.fy, self.cx, self.cy = float(fx), float(fy), float(cx), float(cy)
        self.c2w = np.asarray(c2w, dtype=np.float32).reshape(12)
        self.near, self.far = float(near), float(far)


class Scene:
    def __init__(self, name, seed, static, actors, poses, box_half, cameras, k_samples=8, activation=0, t_stop=1e-4):
        self.name, self.seed = name, seed
        self.static, self.actors = static, actors
        self.poses = np.ascontiguousarray(poses, dtype=np.float32).reshape(len(actors), 12)
        self.box_half = np.ascontiguousarray(box_half, dtype=np.float32).reshape(len(actors), 3)
        self.cameras = cameras
        self.k_samples, self.activation, self.t_stop = k_samples, activation, t_stop

    @property
    def octrees(self):
        return [self.static] + list(self.actors)

    def image_grads(self, cam_index=0, rgb_std=1e-2, depth_std=0.0, alpha_std=0.0):
        """Seeded incoming gradients dL/dRGB ~ N(0,std) (and optionally depth / alpha)."""
        cam = self.cameras[cam_index]
        n = cam.width * cam.height
        out = {}
        for key, std, stream, ch in (("rgb", rgb_std, 900, 3), ("depth", depth_std, 901, 1), ("alpha", alpha_std, 902, 1)):
            if std > 0:
                idx = np.arange(n * ch, dtype=np.uint64) + np.uint64(cam_index) * np.uint64(1 << 40)
                g = (std * rng.normal(self.seed, stream, idx)).astype(np.float32)
                out[key] = g.reshape(cam.height, cam.width, 3) if ch == 3 else g.reshape(cam.height, cam.width)
            else:
                out[key] = None
        return out


def look_yaw(position, yaw):
    """c2w = [R_c | o_c]: camera x right, y down, z forward; forward = (cos yaw, sin yaw, 0) (reading R10)."""
    c, s = np.cos(yaw), np.sin(yaw)
    R = np.array([[s, 0.0, c], [-c, 0.0, s], [0.0, -1.0, 0.0]])  # columns: right, down, forward
    return np.concatenate([R, np.asarray(position, dtype=np.float64).reshape(3, 1)], 1)


def pose_yaw(position, yaw):
    c, s = np.cos(yaw), np.sin(yaw)
    R = np.array([[c, -s, 0.0], [s, c, 0.0], [0.0, 0.0, 1.0]])
    return np.concatenate([R, np.asarray(position, dtype=np.float64).reshape(3, 1)], 1)


def _actors(seed, specs, sh_degree, mu, sigma):
    """specs: list of (dims, target voxels, (x, y), yaw).  Box centre sits at z = half height."""
    actors, poses, halves = [], [], []
    for n, (dims, target, xy, yaw) in enumerate(specs):
        code, side = octree.actor_leaves(dims, target)
        actors.append(octree.make_octree(code, (0.0, 0.0, 0.0), side, sh_degree, seed, n + 1, mu, sigma))
        poses.append(pose_yaw((xy[0], xy[1], 0.5 * dims[2]), yaw))
        halves.append(0.5 * np.asarray(dims))
    return actors, np.array(poses), np.array(halves)


def _lane_tracks(seed, n, dims_list, lanes, x_lo, x_hi, stream=401):
    """Constant-velocity style placements: each actor gets a lane and an x so that boxes stay disjoint."""
    placed, out = [], []
    for n_i in range(n):
        dims = dims_list[n_i]
        lane = lanes[n_i % len(lanes)]
        for attempt in range(1000):
            u = rng.uniform(seed, stream, np.uint64(n_i * 1000 + attempt))
            x = x_lo + (x_hi - x_lo) * float(u)
            if all(not (l == lane and abs(x - px) < 0.5 * (dims[0] + pd[0]) + 1.0) for (l, px, pd) in placed):
                break
        else:
            raise RuntimeError("could not place actor")
        placed.append((lane, x, dims))
        yaw0 = 0.0 if lane < 0 or abs(lane) > 6 else np.pi  # oncoming traffic on the left lanes
        yaw = yaw0 + 0.1 * (float(rng.uniform(seed, stream + 1, np.uint64(n_i))) - 0.5)
        out.append(((x, lane), yaw))
    return out


def config1():
    seed = 1001
    sensor = (-24.0, 0.0)
    boxes = lidar.make_boxes(seed, 4, (-10.0, 25.0), (4.0, 14.0), (3.0, 8.0), (2.0, 6.0))
    pts = lidar.sweep(seed, 0, sensor, 2048, boxes, None)
    code = octree.uniform_leaves_from_cloud(pts, (0, 0, 0), 64.0, 6, 4096)
    static = octree.make_octree(code, (0, 0, 0), 64.0, 0, seed, 0, -1.0, 1.0)
    yaw = -np.pi + 2 * np.pi * float(rng.uniform(seed, 501, np.uint64(0)))
    x = -24.0 + 5.0 + 15.0 * float(rng.uniform(seed, 502, np.uint64(0)))
    y = -3.0 + 6.0 * float(rng.uniform(seed, 503, np.uint64(0)))
    actors, poses, halves = _actors(seed, [(CAR, 512, (x, y), yaw)], 0, -1.0, 1.0)
    cam = Camera(128, 96, 100.0, 100.0, 64.0, 48.0, look_yaw((-24.0, 0.0, 1.6), 0.0))
    return Scene("config1_tiny", seed, static, actors, poses, halves, [cam])


def _static_from_cloud(seed, n_sweeps, n_az, side, l_min, l_max, target, sh_degree, mu, sigma):
    boxes = lidar.make_boxes(seed, 120, (-40.0, 200.0), (12.0, 60.0), (6.0, 25.0), (4.0, 25.0))
    poles = lidar.make_poles(seed, 80, (-40.0, 200.0), (5.0, 9.0))
    pts, path = lidar.cloud(seed, n_sweeps, n_az, 0.0, boxes, poles)
    dist = lidar.dist_to_path(pts, path)
    code, flag, _ = octree.adaptive_leaves_from_cloud(pts, dist, (0, 0, 0), side, l_min, l_max, target)
    return octree.make_octree(code, (0, 0, 0), side, sh_degree, seed, 0, mu, sigma, has_return=flag)


def config2(sh_degree=1, seed=1002):
    static = _static_from_cloud(seed, 20, 1563, 400.0, 8, 12, 500_000, sh_degree, -2.0, 1.5)
    cam_x = 0.8 * 10
    tracks = _lane_tracks(seed, 3, [CAR] * 3, (-1.75, 1.75, -5.25), cam_x + 10.0, cam_x + 40.0)
    actors, poses, halves = _actors(seed, [(CAR, 20_000, xy, yaw) for xy, yaw in tracks], sh_degree, -2.0, 1.5)
    cam = Camera(960, 540, 985.0, 985.0, 480.0, 270.0, look_yaw((cam_x, 0.0, 1.6), 0.0))
    return Scene("config2_small", seed, static, actors, poses, halves, [cam])


def config3(opaque=False):
    seed = 1003
    static = _static_from_cloud(seed, 80, 1563, 512.0, 10, 16, 4_000_000, 3, -2.0, 1.5)
    if opaque:  # variant 3b (report-only): opaque surfaces where the LiDAR returned
        static.geo[static.has_return] += np.float32(8.0)
    cam_x = 0.8 * 40
    dims = [CAR] * 7 + [TRUCK] * 3
    tracks = _lane_tracks(seed, 10, dims, (-1.75, 1.75, -5.25, 5.25, 8.75, -8.75), cam_x + 8.0, cam_x + 80.0)
    actors, poses, halves = _actors(seed, [(d, 50_000, xy, yaw) for d, (xy, yaw) in zip(dims, tracks)], 3, -2.0, 1.5)
    cam = Camera(1920, 1080, 1970.0, 1970.0, 960.0, 540.0, look_yaw((cam_x, 0.0, 1.6), 0.0))
    return Scene("config3_pandaset_shaped" + ("_opaque" if opaque else ""), seed, static, actors, poses, halves, [cam])


def config4():
    seed = 1004
    static = config2(sh_degree=3, seed=1002).static  # the config-2 static scene, SH degree 3
    specs = []
    for row_y in (3.5, -8.75):  # two parked rows of 8, pitch 5.5 m from x = 4 m
        for n in range(8):
            specs.append((CAR, 25_000, (4.0 + 5.5 * n + 2.25, row_y), 0.0))
    for n in range(24):  # oncoming traffic within 60 m
        lane = -1.75 if n % 2 == 0 else -5.25
        specs.append((CAR, 25_000, (3.0 + 4.9 * (n // 2) + 2.25 + (1.3 if n % 2 else 0.0), lane), np.pi))
    jitter = [0.1 * (float(rng.uniform(seed, 402, np.uint64(n))) - 0.5) for n in range(len(specs))]
    specs = [(d, t, xy, yaw + 0.3 * j) for (d, t, xy, yaw), j in zip(specs, jitter)]
    actors, poses, halves = _actors(seed, specs, 3, -2.0, 1.5)
    cam = Camera(1920, 1080, 1970.0, 1970.0, 960.0, 540.0, look_yaw((0.0, 1.0, 1.4), np.deg2rad(5.0)))
    return Scene("config4_crowded", seed, static, actors, poses, halves, [cam])


def config5():
    seed = 1005
    static = _static_from_cloud(seed, 80, 3126, 512.0, 10, 16, 8_000_000, 3, -2.0, 1.5)
    cam_x = 0.8 * 40
    dims = [CAR] * 14 + [TRUCK] * 6
    tracks = _lane_tracks(seed, 20, dims, (-1.75, 1.75, -5.25, 5.25, 8.75, -8.75), cam_x - 60.0, cam_x + 80.0)
    actors, poses, halves = _actors(seed, [(d, 50_000, xy, yaw) for d, (xy, yaw) in zip(dims, tracks)], 3, -2.0, 1.5)
    cams = [Camera(1920, 1080, 1970.0, 1970.0, 960.0, 540.0, look_yaw((cam_x, 0.0, 1.6), np.deg2rad(a)))
            for a in (0.0, 45.0, -45.0, 90.0, -90.0, 180.0)]
    return Scene("config5_training_batch", seed, static, actors, poses, halves, cams)


def make_config(n, **kw):
    return {1: config1, 2: config2, 3: config3, 4: config4, 5: config5}[n](**kw)


def tiny_random_scene(seed, n_static=30, n_actor=8, sh_degree=1, width=16, height=12, colour_floor=False):
    """A very small random adaptive scene for finite-difference and invariance checks."""
    def random_leaves(stream, n_target, max_level):
        leaves = [(0, 0, 0, 0)]
        step = 0
        while len(leaves) < n_target:
            pick = int(rng.hash_u64(seed, stream, np.uint64(step)) % np.uint64(len(leaves)))
            step += 1
            i, j, k, l = leaves[pick]
            if l >= max_level:
                continue
            leaves.pop(pick)
            leaves += [(2 * i + a, 2 * j + b, 2 * k + c, l + 1) for a in (0, 1) for b in (0, 1) for c in (0, 1)]
        # drop a third of them so the tree is sparse; keep level >= 1
        keep = [v for n, v in enumerate(leaves) if v[3] >= 1 and rng.uniform(seed, stream + 1, np.uint64(n)) > 0.33]
        a = np.array(keep, dtype=np.int64)
        return octree.sort_morton(octree.encode(a[:, 0], a[:, 1], a[:, 2], a[:, 3]))

    static = octree.make_octree(random_leaves(601, n_static, 3), (1.0, 0.5, -0.25), 8.0, sh_degree, seed, 0, -1.0, 1.0)
    dims = (2.0, 1.0, 1.5)
    act = octree.make_octree(random_leaves(611, n_actor, 2), (0, 0, 0), 2.4, sh_degree, seed, 1, 0.0, 1.0)
    if colour_floor:  # keep colours away from the clamp at 0
        for t in (static, act):
            t.sh[:, 0, :] = np.abs(t.sh[:, 0, :]) + np.float32(0.3 / octree.C0)
    yaw = 0.7
    pose = pose_yaw((1.5, 0.3, 0.2), yaw)
    Rz = pose[:, :3]
    tilt = 0.4
    Rx = np.array([[1, 0, 0], [0, np.cos(tilt), -np.sin(tilt)], [0, np.sin(tilt), np.cos(tilt)]])
    pose = np.concatenate([Rz @ Rx, pose[:, 3:]], 1)
    cam = Camera(width, height, 0.9 * width, 0.9 * width, 0.5 * width + 0.25, 0.5 * height - 0.25,
                 look_yaw((-6.0, 0.4, 0.3), 0.05), near=0.05, far=1e9)
    return Scene("tiny_random_%d" % seed, seed, static, [act], [pose], [0.5 * np.asarray(dims)], [cam], t_stop=0.0)
