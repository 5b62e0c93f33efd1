"""Seeded LiDAR-like point clouds over analytic primitives (ground plane, boxes, poles).

A 64-beam spinning sensor (elevations evenly spaced in [-25 deg, +15 deg]) at 1.8 m above an
ego pose that advances 0.8 m per sweep along +x; every beam returns its nearest hit within
200 m.  Stands in for PandaSet's 360-degree LiDAR; no dataset record
is reproduced.  Inputs only - no rendering arithmetic.
"""
import numpy as np
from . import rng

N_BEAMS = 64
SENSOR_HEIGHT = 1.8
MAX_RANGE = 200.0
POLE_RADIUS = 0.15
POLE_HEIGHT = 6.0


def make_boxes(seed, n, x_range, absy_range, foot_range, height_range, stream=101):
    """Axis-aligned box "buildings": rows of (x0, x1, y0, y1, h)."""
    idx = np.arange(n, dtype=np.uint64)
    u = [rng.uniform(seed, stream + s, idx) for s in range(6)]
    cx = x_range[0] + (x_range[1] - x_range[0]) * u[0]
    ay = absy_range[0] + (absy_range[1] - absy_range[0]) * u[1]
    sign = np.where(u[2] < 0.5, -1.0, 1.0)
    fx = foot_range[0] + (foot_range[1] - foot_range[0]) * u[3]
    fy = foot_range[0] + (foot_range[1] - foot_range[0]) * u[4]
    h = height_range[0] + (height_range[1] - height_range[0]) * u[5]
    # near edge of the footprint sits at |y| = ay, so nothing straddles the ego path
    y_near = sign * ay
    y_far = sign * (ay + fy)
    return np.stack([cx - 0.5 * fx, cx + 0.5 * fx, np.minimum(y_near, y_far), np.maximum(y_near, y_far), h], 1)


def make_poles(seed, n, x_range, absy_range, stream=201):
    idx = np.arange(n, dtype=np.uint64)
    px = x_range[0] + (x_range[1] - x_range[0]) * rng.uniform(seed, stream, idx)
    ay = absy_range[0] + (absy_range[1] - absy_range[0]) * rng.uniform(seed, stream + 1, idx)
    sign = np.where(rng.uniform(seed, stream + 2, idx) < 0.5, -1.0, 1.0)
    return np.stack([px, sign * ay], 1)


def sweep(seed, sweep_index, sensor_xy, n_azimuth, boxes, poles):
    """One revolution: returns the (n,3) hit points."""
    a = np.arange(n_azimuth, dtype=np.uint64)
    jitter = rng.uniform(seed, 301, np.uint64(sweep_index) * np.uint64(1 << 20) + a)
    az = 2.0 * np.pi * (a.astype(np.float64) + jitter) / n_azimuth
    ca, sa = np.cos(az), np.sin(az)
    elev = np.deg2rad(np.linspace(-25.0, 15.0, N_BEAMS))
    te, ce = np.tan(elev), np.cos(elev)
    sx, sy = float(sensor_xy[0]), float(sensor_xy[1])
    rho_max = MAX_RANGE * ce  # horizontal range limit per beam
    best = np.broadcast_to(rho_max[None, :], (n_azimuth, N_BEAMS)).copy()
    hit = np.zeros((n_azimuth, N_BEAMS), dtype=bool)
    # ground z = 0
    down = te < 0
    rho_g = np.where(down, SENSOR_HEIGHT / np.where(down, -te, 1.0), np.inf)
    g_ok = rho_g < rho_max
    best[:, g_ok] = rho_g[g_ok][None, :]
    hit[:, g_ok] = True
    with np.errstate(divide="ignore", invalid="ignore"):
        if boxes is not None and len(boxes):
            inv_c, inv_s = 1.0 / ca[:, None], 1.0 / sa[:, None]
            tx0, tx1 = (boxes[None, :, 0] - sx) * inv_c, (boxes[None, :, 1] - sx) * inv_c
            ty0, ty1 = (boxes[None, :, 2] - sy) * inv_s, (boxes[None, :, 3] - sy) * inv_s
            r_in = np.maximum(np.minimum(tx0, tx1), np.minimum(ty0, ty1))
            r_out = np.minimum(np.maximum(tx0, tx1), np.maximum(ty0, ty1))
            ai, bi = np.nonzero((r_out > r_in) & (r_in > 0))
            if ai.size:
                rin, rout, h = r_in[ai, bi][:, None], r_out[ai, bi][:, None], boxes[bi, 4][:, None]
                z_in = SENSOR_HEIGHT + rin * te[None, :]
                side = (z_in >= 0) & (z_in <= h)
                rho_top = np.where(te[None, :] < 0, (h - SENSOR_HEIGHT) / np.where(te < 0, te, -1.0)[None, :], np.inf)
                top = (z_in > h) & (rho_top > rin) & (rho_top <= rout)
                rho = np.where(side, rin, np.where(top, rho_top, np.inf))
                pa, pb = np.nonzero(np.isfinite(rho))
                np.minimum.at(best, (ai[pa], pb), rho[pa, pb])
                hit[ai[pa], pb] = True
        if poles is not None and len(poles):
            ox, oy = poles[None, :, 0] - sx, poles[None, :, 1] - sy
            along = ox * ca[:, None] + oy * sa[:, None]
            perp2 = ox * ox + oy * oy - along * along
            disc = POLE_RADIUS * POLE_RADIUS - perp2
            ai, bi = np.nonzero((disc > 0) & (along > POLE_RADIUS))
            if ai.size:
                rin = (along[ai, bi] - np.sqrt(disc[ai, bi]))[:, None]
                z_in = SENSOR_HEIGHT + rin * te[None, :]
                ok = (z_in >= 0) & (z_in <= POLE_HEIGHT)
                pa, pb = np.nonzero(ok)
                np.minimum.at(best, (ai[pa], pb), np.broadcast_to(rin, ok.shape)[pa, pb])
                hit[ai[pa], pb] = True
    hit &= best < rho_max[None, :]
    ai, bi = np.nonzero(hit)
    rho = best[ai, bi]
    return np.stack([sx + rho * ca[ai], sy + rho * sa[ai], SENSOR_HEIGHT + rho * te[bi]], 1)


def cloud(seed, n_sweeps, n_azimuth, x_start, boxes, poles, step=0.8):
    """All sweeps; returns points (n,3) and the ego path segment (x_start, x_end)."""
    pts = [sweep(seed, s, (x_start + step * s, 0.0), n_azimuth, boxes, poles) for s in range(n_sweeps)]
    return np.concatenate(pts, 0), (x_start, x_start + step * (n_sweeps - 1))


def dist_to_path(points, path):
    """Horizontal distance of each point to the ego trajectory segment (y = 0, x in path)."""
    dx = points[:, 0] - np.clip(points[:, 0], path[0], path[1])
    return np.sqrt(dx * dx + points[:, 1] * points[:, 1])
