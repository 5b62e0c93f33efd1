"""Small scene builders used by the pin tests (inputs only)."""
import numpy as np
import dvx_scenes as S

NOTES = []   # one line per parity test (pixels compared, threshold-ambiguous pixels used); conftest prints them at the end


def note(line):
    NOTES.append(line)
    print(line)

from dvx_scenes.octree import Octree, encode, sort_morton, C0


def tree_from_cells(cells, geo=None, sh=None, center=(0, 0, 0), side=4.0, sh_degree=0, dtype=np.float64):
    """cells: list of (i,j,k,level); geo [V,8] or scalar; sh [V,C,3] or None (colour 1)."""
    a = np.array(cells, dtype=np.int64).reshape(-1, 4)
    code = encode(a[:, 0], a[:, 1], a[:, 2], a[:, 3]) if len(a) else np.zeros(0, dtype=np.uint64)
    V, nsh = len(a), (sh_degree + 1) ** 2
    g = np.zeros((V, 8), dtype=dtype)
    if geo is not None:
        g[...] = np.asarray(geo, dtype=dtype).reshape(-1, 8) if np.ndim(geo) else geo
    k = np.zeros((V, nsh, 3), dtype=dtype)
    if sh is None:
        if V:
            k[:, 0, :] = 0.5 / C0  # colour == 1
    else:
        k[...] = sh
    return _raw(code, g, k, center, side, sh_degree)


def _raw(code, geo, sh, center, side, sh_degree):
    t = Octree.__new__(Octree)
    t.code = np.ascontiguousarray(code, dtype=np.uint64)
    t.geo = np.ascontiguousarray(geo)
    t.sh = np.ascontiguousarray(sh)
    t.center = np.asarray(center, dtype=np.float64)
    t.side = float(side)
    t.sh_degree = int(sh_degree)
    t.has_return = None
    return t


def empty_tree(sh_degree=0, side=4.0):
    return tree_from_cells([], center=(0, 0, 0), side=side, sh_degree=sh_degree)


def scene(static, actors=(), poses=(), halves=(), cam=None, **kw):
    s = S.Scene("custom", 1, static, list(actors), np.zeros((len(actors), 12)), np.zeros((len(actors), 3)), [cam], **kw)
    # keep double precision for poses / boxes in custom scenes
    s.poses = np.ascontiguousarray(poses, dtype=np.float64).reshape(len(actors), 12)
    s.box_half = np.ascontiguousarray(halves, dtype=np.float64).reshape(len(actors), 3)
    return s


def axis_camera(position=(-5.0, 1.0, 1.0), width=9, height=7, f=20.0, yaw=0.0, near=0.05, far=1e9):
    """Pinhole looking along +x (yaw 0) whose centre pixel ray is exactly the optical axis."""
    cam = S.Camera(width, height, f, f, width // 2 + 0.5, height // 2 + 0.5, S.look_yaw(position, yaw), near, far)
    cam.c2w = np.asarray(S.look_yaw(position, yaw), dtype=np.float64).reshape(12)
    return cam
