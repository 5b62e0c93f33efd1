"""CPU oracle of widening row N2: shared grid-point corner densities + the optimizer step.

TEST INFRASTRUCTURE ONLY (same rule as oracle.py): only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this module; it never imports the CUDA package.

What the paper fixes: every leaf voxel carries "discrete raw volume densities (v_geo) at its eight corners", which "are
optimized during training", "following SVRaster".  It is silent on whether coincident corners of
neighbouring voxels are one parameter, and it never names the optimizer.  Readings:
  R23  coincident corners are ONE parameter (a "grid point"), identified by the corner's integer coordinate on the
       level-16 lattice of the octree, hanging nodes included (a fine voxel's corner in the middle of a coarse
       neighbour's face is its own grid point).  Grid points are numbered in ascending order of the 51-bit Morton key
       of that coordinate (x most significant within a 3-bit group, like the voxel code).
  R24  the optimizer is Adam (Kingma & Ba 2015, Algorithm 1) with bias correction, one step per call.

Pins: tests/test_oracle_grid_pins.py P16-P21 (closed-form counts, a hand count, brute force with exact fractions,
adjointness + torch autograd, torch.optim.Adam in float64).  R23 and R24 are readings the paper does not fix:
PARITY UNPINNED against the authors' implementation for the choice of parameterisation and optimizer.

Plain numpy, int64/uint64 for the tables and float64 for the arithmetic.  No blocking, no fusion: each function is
the definition written out.
"""
import numpy as np

MAX_LEVEL = 16


def decode(code):
    """code (include/dvx.h, R14a) -> (level, X, Y, Z): the voxel's level and the level-16 lattice coordinate of its
    minimum corner.  Group m (bits 45-3m..47-3m) = 4 x_m + 2 y_m + z_m holds bit (l-1-m) of the cell coordinate, i.e.
    bit (15-m) of the lattice coordinate; groups m >= l are zero."""
    code = np.asarray(code, dtype=np.uint64)
    level = ((code >> np.uint64(48)) & np.uint64(31)).astype(np.int64)
    X = np.zeros(code.shape, dtype=np.int64)
    Y = np.zeros(code.shape, dtype=np.int64)
    Z = np.zeros(code.shape, dtype=np.int64)
    for m in range(MAX_LEVEL):
        g = ((code >> np.uint64(45 - 3 * m)) & np.uint64(7)).astype(np.int64)
        X |= ((g >> 2) & 1) << (15 - m)
        Y |= ((g >> 1) & 1) << (15 - m)
        Z |= (g & 1) << (15 - m)
    return level, X, Y, Z


def corner_coords(code):
    """[V,8,3] int64 lattice coordinates of the 8 corners; corner c = 4 b_x + 2 b_y + b_z (R7)."""
    level, X, Y, Z = decode(code)
    size = np.int64(1) << (MAX_LEVEL - level)
    out = np.empty(level.shape + (8, 3), dtype=np.int64)
    for c in range(8):
        out[..., c, 0] = X + ((c >> 2) & 1) * size
        out[..., c, 1] = Y + ((c >> 1) & 1) * size
        out[..., c, 2] = Z + (c & 1) * size
    return out


def morton51(xyz):
    """17-bit coordinates (0..65536) -> 51-bit key, bit b of x at 3b+2, of y at 3b+1, of z at 3b (R23)."""
    xyz = np.asarray(xyz, dtype=np.int64)
    key = np.zeros(xyz.shape[:-1], dtype=np.uint64)
    for b in range(MAX_LEVEL + 1):
        for a in range(3):
            bit = ((xyz[..., a] >> b) & 1).astype(np.uint64)
            key |= bit << np.uint64(3 * b + 2 - a)
    return key


def grid_tables(code):
    """R23.  Returns (point_of [V,8] uint32, offsets [G+1] uint32, slots [8V] uint32, keys [G] uint64):
    point_of[v,c] = grid point of corner c of voxel v; slots[offsets[p]:offsets[p+1]] = the corner slots 8v+c that are
    grid point p, ascending; keys[p] = the point's Morton key (ascending in p)."""
    code = np.asarray(code, dtype=np.uint64)
    V = code.shape[0]
    if V == 0:
        return (np.zeros((0, 8), np.uint32), np.zeros(1, np.uint32), np.zeros(0, np.uint32), np.zeros(0, np.uint64))
    keys = morton51(corner_coords(code)).reshape(-1)            # [8V], slot 8v+c
    uniq, inverse = np.unique(keys, return_inverse=True)       # uniq ascending
    point_of = inverse.astype(np.uint32).reshape(V, 8)
    slots = np.argsort(inverse, kind="stable").astype(np.uint32)
    counts = np.bincount(inverse, minlength=uniq.shape[0])
    offsets = np.concatenate([[0], np.cumsum(counts)]).astype(np.uint32)
    return point_of, offsets, slots, uniq


def grid_gather(density, point_of):
    """geo[v,c] = density[point_of[v,c]]  (the [V,8] corner record the rasterizer reads)."""
    return np.asarray(density)[np.asarray(point_of, dtype=np.int64)]


def grid_reduce(dgeo, point_of, n_points):
    """dL/ddensity[p] = sum of dL/dgeo over the corner slots that are p (chain rule through grid_gather)."""
    out = np.zeros(n_points, dtype=np.float64)
    np.add.at(out, np.asarray(point_of, dtype=np.int64).reshape(-1), np.asarray(dgeo, dtype=np.float64).reshape(-1))
    return out


def adam_step(p, m, v, g, lr, beta1, beta2, eps, t):
    """R24: Kingma & Ba 2015, Algorithm 1, step t >= 1.  Returns (p, m, v) after the step, float64.
        m <- b1 m + (1-b1) g;  v <- b2 v + (1-b2) g^2;  mhat = m/(1-b1^t);  vhat = v/(1-b2^t)
        p <- p - lr mhat / (sqrt(vhat) + eps)"""
    p = np.asarray(p, dtype=np.float64)
    m = np.asarray(m, dtype=np.float64)
    v = np.asarray(v, dtype=np.float64)
    g = np.asarray(g, dtype=np.float64)
    m = beta1 * m + (1.0 - beta1) * g
    v = beta2 * v + (1.0 - beta2) * g * g
    mhat = m / (1.0 - beta1 ** t)
    vhat = v / (1.0 - beta2 ** t)
    p = p - lr * mhat / (np.sqrt(vhat) + eps)
    return p, m, v


def grid_adam_step(density, m, v, dgeo, point_of, lr, beta1, beta2, eps, t):
    """One optimizer step of the corner densities of one octree: reduce the [V,8] corner gradients to grid points,
    Adam on the grid points, and the refreshed [V,8] corner record.  Returns (density, m, v, geo)."""
    g = grid_reduce(dgeo, point_of, np.asarray(density).shape[0])
    density, m, v = adam_step(density, m, v, g, lr, beta1, beta2, eps, t)
    return density, m, v, grid_gather(density, point_of)
