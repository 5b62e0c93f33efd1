"""Leaf-octree containers and generators (seeded, synthetic).

Voxel key format (reading R14a / SURVEY.md §8(c)): ``code`` is a uint64 with
bits 48-52 = level l in [1,16] and bits 0-47 = Morton path left-aligned: 3-bit group m in
[0,l) sits at bits [45-3m, 47-3m] and equals 4*x_m + 2*y_m + z_m, where x_m is bit l-1-m of
the integer cell coordinate i (likewise y_m of j, z_m of k).  Groups m >= l are zero.

This file builds inputs only; it contains no rendering arithmetic.
"""
import numpy as np
from . import rng

MAX_LEVEL = 16


def _spread3(x):
    """Put bit b of the (<=16-bit) integers ``x`` at bit 3b of a uint64."""
    x = np.asarray(x, dtype=np.uint64) & np.uint64(0xFFFF)
    x = (x | (x << np.uint64(32))) & np.uint64(0x1F00000000FFFF)
    x = (x | (x << np.uint64(16))) & np.uint64(0x1F0000FF0000FF)
    x = (x | (x << np.uint64(8))) & np.uint64(0x100F00F00F00F00F)
    x = (x | (x << np.uint64(4))) & np.uint64(0x10C30C30C30C30C3)
    x = (x | (x << np.uint64(2))) & np.uint64(0x1249249249249249)
    return x


def _compact3(x):
    x = np.asarray(x, dtype=np.uint64) & np.uint64(0x1249249249249249)
    x = (x | (x >> np.uint64(2))) & np.uint64(0x10C30C30C30C30C3)
    x = (x | (x >> np.uint64(4))) & np.uint64(0x100F00F00F00F00F)
    x = (x | (x >> np.uint64(8))) & np.uint64(0x1F0000FF0000FF)
    x = (x | (x >> np.uint64(16))) & np.uint64(0x1F00000000FFFF)
    x = (x | (x >> np.uint64(32))) & np.uint64(0xFFFF)
    return x


def morton_path(i, j, k):
    """Plain (not left-aligned) Morton number with x as the most significant bit of a group."""
    return (_spread3(i) << np.uint64(2)) | (_spread3(j) << np.uint64(1)) | _spread3(k)


def encode(i, j, k, level):
    """Cell coordinates at ``level`` -> 64-bit voxel code."""
    level = np.asarray(level, dtype=np.uint64)
    path = morton_path(i, j, k) << (np.uint64(3) * (np.uint64(MAX_LEVEL) - level))
    return path | (level << np.uint64(48))


def decode(code):
    """64-bit voxel code -> (i, j, k, level) as int64 arrays."""
    code = np.asarray(code, dtype=np.uint64)
    level = (code >> np.uint64(48)) & np.uint64(31)
    path = (code & np.uint64((1 << 48) - 1)) >> (np.uint64(3) * (np.uint64(MAX_LEVEL) - level))
    i = _compact3(path >> np.uint64(2))
    j = _compact3(path >> np.uint64(1))
    k = _compact3(path)
    return i.astype(np.int64), j.astype(np.int64), k.astype(np.int64), level.astype(np.int64)


def sort_morton(code):
    """Order leaves by their left-aligned 48-bit path (prefix-free, so the order is total)."""
    code = np.asarray(code, dtype=np.uint64)
    return code[np.argsort(code & np.uint64((1 << 48) - 1), kind="stable")]


class Octree:
    """One leaf-only octree: ``code[V]`` u64, ``geo[V,8]`` f32, ``sh[V,C,3]`` f32."""

    def __init__(self, code, geo, sh, center, side, sh_degree, has_return=None):
        self.code = np.ascontiguousarray(code, dtype=np.uint64)
        self.geo = np.ascontiguousarray(geo, dtype=np.float32)
        self.sh = np.ascontiguousarray(sh, dtype=np.float32)
        self.center = np.asarray(center, dtype=np.float32)
        self.side = np.float32(side)
        self.sh_degree = int(sh_degree)
        self.has_return = has_return

    @property
    def n_voxels(self):
        return int(self.code.shape[0])

    @property
    def n_sh(self):
        return (self.sh_degree + 1) ** 2


C0 = 0.28209479177387814  # Y_0 of the real SH basis (reading R8); only used to map a base colour to k_0


def corner_densities(code, seed, tree_index, mu, sigma):
    """raw(o,X,Y,Z) = mu + sigma * normal(hash(stream=16o+1, (X*65537+Y)*65537+Z)).

    (X,Y,Z) is the corner's integer coordinate at level-16 resolution, so neighbouring voxels
    agree on shared corners.  Corner c = 4*bx + 2*by + bz (reading R7).
    """
    i, j, k, level = decode(code)
    size = (np.int64(1) << (MAX_LEVEL - level))
    geo = np.empty((code.shape[0], 8), dtype=np.float32)
    for c in range(8):
        bx, by, bz = (c >> 2) & 1, (c >> 1) & 1, c & 1
        X = ((i + bx) * size).astype(np.uint64)
        Y = ((j + by) * size).astype(np.uint64)
        Z = ((k + bz) * size).astype(np.uint64)
        idx = (X * np.uint64(65537) + Y) * np.uint64(65537) + Z
        geo[:, c] = mu + sigma * rng.normal(seed, 16 * tree_index + 1, idx)
    return geo


def sh_coefficients(n_voxels, sh_degree, seed, tree_index):
    """k_0 = (U(0,1) - 1/2)/c0 per channel; higher coefficients U(-0.1, 0.1)."""
    n_sh = (sh_degree + 1) ** 2
    n = n_voxels * n_sh * 3
    u = rng.uniform_chunked(seed, 16 * tree_index + 2, n, 0.0, 1.0, dtype=np.float32).reshape(n_voxels, n_sh, 3)
    sh = (u - np.float32(0.5)) * np.float32(0.2)
    sh[:, 0, :] = (u[:, 0, :] - np.float32(0.5)) / np.float32(C0)
    return sh


def make_octree(code, center, side, sh_degree, seed, tree_index, mu, sigma, has_return=None):
    code = np.asarray(code, dtype=np.uint64)
    geo = corner_densities(code, seed, tree_index, mu, sigma)
    sh = sh_coefficients(code.shape[0], sh_degree, seed, tree_index)
    return Octree(code, geo, sh, center, side, sh_degree, has_return)


# ----------------------------------------------------------------------------------------------
# static octree from a LiDAR-like cloud (imitates PAPER.md:83-87 proximity subdivision)
# ----------------------------------------------------------------------------------------------

def point_cells(points, center, side, level=MAX_LEVEL):
    """Integer cell coordinates of the points inside the cube (and the mask of those inside)."""
    lo = np.asarray(center, dtype=np.float64) - 0.5 * float(side)
    g = (points - lo) * ((1 << level) / float(side))
    inside = np.all((g >= 0) & (g < (1 << level)), axis=1)
    return np.floor(g[inside]).astype(np.int64), inside


def adaptive_leaves_from_cloud(points, dist, center, side, l_min, l_max, target, tol=0.01):
    """Leaves of the adaptive octree described in SURVEY.md §8(d) "Static octree from the cloud".

    Each point gets a target level l*(p) = clamp(ceil(log2(side/(r0*max(dist,0.5 m)))), l_min, l_max);
    a node at level l is split iff it contains a point with l* > l; leaves = occupied l_min cells
    that are not split + all children of split nodes that are not themselves split.  r0 is found
    by bisection so that the leaf count hits ``target`` within ``tol``.
    Returns (codes in Morton order, has_return flags, r0).
    """
    cells, inside = point_cells(points, center, side)
    g = np.log2(float(side) / np.maximum(dist[inside], 0.5))
    m16 = morton_path(cells[:, 0], cells[:, 1], cells[:, 2])
    order = np.argsort(m16, kind="stable")
    m16 = m16[order]
    g = g[order]
    # per level: the distinct occupied cells and the largest g inside each
    cell_ids, gmax = {}, {}
    for l in range(l_min, l_max + 1):
        cid = m16 >> np.uint64(3 * (MAX_LEVEL - l))
        first = np.concatenate([[True], cid[1:] != cid[:-1]])
        starts = np.nonzero(first)[0]
        cell_ids[l] = cid[starts]
        gmax[l] = np.maximum.reduceat(g, starts)

    def split_masks(log2_r0):
        return {l: np.clip(np.ceil(gmax[l] - log2_r0), l_min, l_max) > l for l in range(l_min, l_max)}

    def count(log2_r0):
        sm = split_masks(log2_r0)
        return cell_ids[l_min].shape[0] + 7 * sum(int(m.sum()) for m in sm.values())

    lo, hi = -12.0, 4.0  # log2 r0 ; count decreases as r0 grows
    if count(lo) < target:
        log2_r0 = lo
    else:
        for _ in range(60):
            mid = 0.5 * (lo + hi)
            c = count(mid)
            if abs(c - target) <= tol * target:
                break
            if c > target:
                lo = mid
            else:
                hi = mid
        log2_r0 = mid
    sm = split_masks(log2_r0)
    codes, flags = [], []
    # level l_min: occupied, unsplit cells (all contain a return)
    keep = ~sm[l_min]
    ids = cell_ids[l_min][keep]
    codes.append((ids << np.uint64(3 * (MAX_LEVEL - l_min))) | (np.uint64(l_min) << np.uint64(48)))
    flags.append(np.ones(ids.shape[0], dtype=bool))
    for l in range(l_min, l_max):
        split_ids = cell_ids[l][sm[l]]
        children = (split_ids[:, None] << np.uint64(3)) | np.arange(8, dtype=np.uint64)[None, :]
        children = children.reshape(-1)
        if l + 1 < l_max:
            child_split = cell_ids[l + 1][sm[l + 1]]
            children = children[~np.isin(children, child_split, assume_unique=True)]
        occupied = np.isin(children, cell_ids[l + 1], assume_unique=True)
        codes.append((children << np.uint64(3 * (MAX_LEVEL - l - 1))) | (np.uint64(l + 1) << np.uint64(48)))
        flags.append(occupied)
    code = np.concatenate(codes)
    flag = np.concatenate(flags)
    order = np.argsort(code & np.uint64((1 << 48) - 1), kind="stable")
    return code[order], flag[order], float(2.0 ** log2_r0)


def uniform_leaves_from_cloud(points, center, side, level, target):
    """Config 1: the ``target`` occupied cells at ``level`` with most points (ties: Morton order).

    If fewer cells are occupied, the set is grown by 6-neighbour dilation in Morton order."""
    cells, _ = point_cells(points, center, side, level)
    m = morton_path(cells[:, 0], cells[:, 1], cells[:, 2])
    ids, counts = np.unique(m, return_counts=True)
    order = np.lexsort((ids, -counts))
    chosen = ids[order[:target]]
    n = 1 << level
    while chosen.shape[0] < target:
        path = chosen
        i = _compact3(path >> np.uint64(2)).astype(np.int64)
        j = _compact3(path >> np.uint64(1)).astype(np.int64)
        k = _compact3(path).astype(np.int64)
        nb = []
        for d in ((1, 0, 0), (-1, 0, 0), (0, 1, 0), (0, -1, 0), (0, 0, 1), (0, 0, -1)):
            a, b, c = i + d[0], j + d[1], k + d[2]
            ok = (a >= 0) & (a < n) & (b >= 0) & (b < n) & (c >= 0) & (c < n)
            nb.append(morton_path(a[ok], b[ok], c[ok]))
        new = np.setdiff1d(np.unique(np.concatenate(nb)), chosen)
        if new.shape[0] == 0:
            break
        chosen = np.concatenate([chosen, new[: target - chosen.shape[0]]])
    chosen = np.sort(chosen)
    return (chosen << np.uint64(3 * (MAX_LEVEL - level))) | (np.uint64(level) << np.uint64(48))


# ----------------------------------------------------------------------------------------------
# actor octree (cube = largest box dimension x 1.2, centred on the local origin)
# ----------------------------------------------------------------------------------------------

def actor_leaves(box_dims, target):
    """Leaves of an actor octree with about ``target`` voxels (SURVEY.md §8(d) "Actor octree")."""
    box_dims = np.asarray(box_dims, dtype=np.float64)
    side = 1.2 * float(box_dims.max())
    half = 0.5 * box_dims

    def cells_hitting_box(level):
        n = 1 << level
        s = side / n
        rng_axes = []
        for a in range(3):
            lo = int(np.floor((-half[a] + 0.5 * side) / s + 1e-9))
            hi = int(np.ceil((half[a] + 0.5 * side) / s - 1e-9)) - 1
            rng_axes.append(np.arange(max(lo, 0), min(hi, n - 1) + 1))
        return rng_axes, s

    level = 1
    while level < MAX_LEVEL:
        ax, _ = cells_hitting_box(level + 1)
        if len(ax[0]) * len(ax[1]) * len(ax[2]) > target:
            break
        level += 1
    ax, s = cells_hitting_box(level)
    I, J, K = np.meshgrid(ax[0], ax[1], ax[2], indexing="ij")
    I, J, K = I.ravel(), J.ravel(), K.ravel()
    path = morton_path(I, J, K)
    order = np.argsort(path)
    I, J, K, path = I[order], J[order], K[order], path[order]
    # a cell touches the box surface iff it is not strictly inside the box
    lo = np.stack([I, J, K], 1) * s - 0.5 * side
    inside = np.all((lo > -half) & (lo + s < half), axis=1)
    leaves = [(path, level)]
    count = path.shape[0]
    cand = np.concatenate([np.nonzero(~inside)[0], np.nonzero(inside)[0]])  # surface first, Morton order within
    n_split = max(0, min(cand.shape[0], (target - count) // 7))
    if n_split > 0 and level < MAX_LEVEL:
        split = np.sort(cand[:n_split])
        keep = np.ones(path.shape[0], dtype=bool)
        keep[split] = False
        children = ((path[split][:, None] << np.uint64(3)) | np.arange(8, dtype=np.uint64)[None, :]).reshape(-1)
        leaves = [(path[keep], level), (children, level + 1)]
    code = np.concatenate([(p << np.uint64(3 * (MAX_LEVEL - l))) | (np.uint64(l) << np.uint64(48)) for p, l in leaves])
    return sort_morton(code), side
