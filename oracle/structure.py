"""CPU oracle of widening row N4: LiDAR-guided structure operations of the static octree.

TEST INFRASTRUCTURE ONLY (same rule as oracle.py): only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this module; it never imports the CUDA package.

What the paper fixes ("LiDAR-guided structural initialization pipeline"):
  step 2  "voxels closer than a distance threshold to a LiDAR point are subdivided", in rounds, "until the minimum voxel
          sizes falls below 30 cm";
  step 3  Eq. 1: for each grid corner, d = Euclidean distance to the nearest LiDAR point,
          v_init = v_far + (v_close - v_far) exp(-2 d^2 / s^2),  s = minimum voxel size, v_close = -2, v_far = -10.
Readings:
  R26  "closer than a distance threshold": the Euclidean distance from the point to the voxel's closed box (0 inside) is
       <= the threshold.  One round replaces every such leaf below the maximum level by its 8 children and keeps the
       others; the output lists kept leaves and children in the input order (children in octant order 4x+2y+z).
  R27  Eq. 1 is evaluated per grid point of reading R23 (a corner shared by several voxels has one density); an empty
       cloud gives v_far everywhere.
  R28  pruning (PAPER.md:63 "adaptive pruning", :379 "eliminate residual low-density voxels"): a leaf is removed when the
       largest of its 8 raw corner densities is below a threshold; the survivors keep their order.

Plain numpy in float64; the nearest neighbour is scipy's cKDTree (a library primitive serving as one step), pinned
against brute force in tests/test_oracle_structure_pins.py.  R26-R28 are readings: PARITY UNPINNED against the authors'
implementation; Eq. 1 itself is the paper's formula written out.
"""
import numpy as np
from scipy.spatial import cKDTree

from . import grid as _grid

MAX_LEVEL = 16
V_CLOSE, V_FAR = -2.0, -10.0


def lattice_to_frame(xyz, center, side):
    """Level-16 lattice coordinates -> positions in the octree's frame: the root cube is centre +- side/2."""
    return np.asarray(center, dtype=np.float64) - 0.5 * float(side) + np.asarray(xyz, dtype=np.float64) * (float(side) / 65536.0)


def grid_point_positions(code, center, side):
    """[G,3] positions of the grid points of reading R23, in grid-point order."""
    code = np.asarray(code, dtype=np.uint64)
    coords = _grid.corner_coords(code).reshape(-1, 3)
    point_of = _grid.grid_tables(code)[0].reshape(-1).astype(np.int64)
    n_points = int(point_of.max()) + 1 if point_of.size else 0
    xyz = np.zeros((n_points, 3), dtype=np.int64)
    xyz[point_of] = coords          # all slots of a point carry the same coordinate
    return lattice_to_frame(xyz, center, side)


def nearest_distance(points, queries):
    """Distance from every query to its nearest point; +inf when there are no points."""
    points = np.asarray(points, dtype=np.float64).reshape(-1, 3)
    queries = np.asarray(queries, dtype=np.float64).reshape(-1, 3)
    if points.shape[0] == 0:
        return np.full(queries.shape[0], np.inf)
    return cKDTree(points).query(queries, k=1)[0]


def density_prior(code, center, side, points, s_min, v_close=V_CLOSE, v_far=V_FAR):
    """Eq. 1 per grid point (R27): v_far + (v_close - v_far) exp(-2 d^2 / s^2)."""
    d = nearest_distance(points, grid_point_positions(code, center, side))
    return v_far + (v_close - v_far) * np.exp(-2.0 * d * d / (float(s_min) ** 2))


def voxel_boxes(code, center, side):
    """(lo [V,3], hi [V,3]) of the leaves in the octree's frame."""
    level, X, Y, Z = _grid.decode(code)
    size = (np.int64(1) << (MAX_LEVEL - level))
    lo = np.stack([X, Y, Z], axis=1)
    hi = lo + size[:, None]
    return lattice_to_frame(lo, center, side), lattice_to_frame(hi, center, side)


def near_mask(code, center, side, points, threshold):
    """R26: leaf v is near when some point lies within `threshold` of its closed box."""
    lo, hi = voxel_boxes(code, center, side)
    points = np.asarray(points, dtype=np.float64).reshape(-1, 3)
    out = np.zeros(lo.shape[0], dtype=bool)
    if points.shape[0] == 0:
        return out
    tree = cKDTree(points)
    # candidates: points within the ball that contains the inflated box, then the exact point-box distance
    c = 0.5 * (lo + hi)
    r = 0.5 * np.linalg.norm(hi - lo, axis=1) + threshold
    for v in range(lo.shape[0]):
        idx = tree.query_ball_point(c[v], r[v] * (1 + 1e-12))
        if not idx:
            continue
        p = points[idx]
        gap = np.maximum(np.maximum(lo[v] - p, p - hi[v]), 0.0)
        out[v] = bool((np.sqrt((gap * gap).sum(axis=1)) <= threshold).any())
    return out


def children(code):
    """The 8 children of each leaf, [V,8] codes in octant order 4x+2y+z (R14a: the child's 3-bit group follows the parent's
    path, the level field goes up by one)."""
    code = np.asarray(code, dtype=np.uint64)
    level = (code >> np.uint64(48)) & np.uint64(31)
    path = code & np.uint64((1 << 48) - 1)
    shift = (np.uint64(45) - np.uint64(3) * level)
    out = np.empty(code.shape + (8,), dtype=np.uint64)
    for o in range(8):
        out[..., o] = ((level + np.uint64(1)) << np.uint64(48)) | path | (np.uint64(o) << shift)
    return out


def subdivide_near(code, center, side, points, threshold, max_level=MAX_LEVEL):
    """One round of proximity-based subdivision (R26).  Returns (new codes, split mask of the input leaves)."""
    code = np.asarray(code, dtype=np.uint64)
    level = ((code >> np.uint64(48)) & np.uint64(31)).astype(np.int64)
    split = near_mask(code, center, side, points, threshold) & (level < max_level)
    kids = children(code)
    out = []
    for v in range(code.shape[0]):
        if split[v]:
            out.extend(kids[v].tolist())
        else:
            out.append(int(code[v]))
    return np.array(out, dtype=np.uint64), split


def prune(code, geo, threshold):
    """R28: keep the leaves whose largest raw corner density is >= threshold.  Returns (codes, kept indices)."""
    geo = np.asarray(geo, dtype=np.float64).reshape(-1, 8)
    keep = np.nonzero(geo.max(axis=1) >= threshold)[0]
    return np.asarray(code, dtype=np.uint64)[keep], keep.astype(np.uint32)


def subdivide_fill(split, geo, sh):
    """Parameters of the leaves after one subdivision round (reading R29): a kept leaf keeps its corner densities and SH
    coefficients; child o = 4 ox + 2 oy + oz of a split leaf occupies the half-cube [o_a / 2, (o_a + 1) / 2] of its parent
    along every axis, and its corner c = 4 bx + 2 by + bz takes the parent's trilinear raw density at u = (o + b) / 2, so the
    continuous density field ('raw volume densities at its eight corners', trilinear inside) is unchanged by
    the split; the SH coefficients are copied.  Output order = subdivide_near's.  float64."""
    split = np.asarray(split).astype(bool)
    geo = np.asarray(geo, dtype=np.float64).reshape(split.shape[0], 8)
    sh = np.asarray(sh, dtype=np.float64)
    out_geo, out_sh = [], []
    for v in range(split.shape[0]):
        if not split[v]:
            out_geo.append(geo[v]); out_sh.append(sh[v])
            continue
        for o in range(8):
            child = np.zeros(8)
            for c in range(8):
                u = [(((o >> (2 - a)) & 1) + ((c >> (2 - a)) & 1)) / 2.0 for a in range(3)]
                val = 0.0
                for pc in range(8):   # the parent's trilinear interpolant, corner pc = 4 bx + 2 by + bz (R7)
                    w = 1.0
                    for a in range(3):
                        w *= u[a] if (pc >> (2 - a)) & 1 else 1.0 - u[a]
                    val += w * geo[v, pc]
                child[c] = val
            out_geo.append(child); out_sh.append(sh[v])
    n = len(out_geo)
    return np.array(out_geo).reshape(n, 8), np.array(out_sh).reshape((n,) + sh.shape[1:])
