"""Pins of oracle/structure.py (widening row N4: LiDAR-guided structure operations) against things other than itself.

P27 Eq. 1 closed forms: one LiDAR point on a corner / at distance s / far away; an empty cloud gives v_far
P28 the k-d tree nearest distance against brute force
P29 the near mask against brute-force point-box distances, and the inclusive threshold on an exactly representable case
P30 a subdivision round: the children tile the parent exactly (decoded with the scene module's decoder, not the
    oracle's), n_out = n + 7 splits, order kept, the maximum level is honoured, the leaves still tile the same volume
P31 pruning keeps exactly the leaves with a corner at or above the threshold, in order
"""
import math

import numpy as np

import dvx_scenes as S
from dvx_scenes import octree as so
from oracle import structure as T


def test_p27_eq1_closed_forms():
    # one level-2 leaf of a 4 m cube centred at the origin: cell (1,2,3) -> box [-1,0]x[0,1]x[1,2]
    code = so.encode(np.array([1]), np.array([2]), np.array([3]), 2)
    center, side, s = (0.0, 0.0, 0.0), 4.0, 0.5
    pos = T.grid_point_positions(code, center, side)
    want = sorted([(-1.0 + bx, 0.0 + by, 1.0 + bz) for bx in (0, 1) for by in (0, 1) for bz in (0, 1)])
    assert sorted(map(tuple, pos.tolist())) == want
    p = np.array([[-1.0, 0.0, 1.0]])                       # on the minimum corner
    dens = T.density_prior(code, center, side, p, s)
    for q, v in zip(pos, dens):
        d2 = float(((q - p[0]) ** 2).sum())                # 0, 1, 2 or 3 m^2
        assert abs(v - (-10.0 + 8.0 * math.exp(-2.0 * d2 / 0.25))) < 1e-12
    assert abs(dens.max() - (-2.0)) < 1e-12                # d = 0 -> v_close
    # a point at distance exactly s from one corner along x, further from all others
    p = np.array([[-1.5, 0.0, 1.0]])
    dens = T.density_prior(code, center, side, p, s)
    assert abs(dens.max() - (-10.0 + 8.0 * math.exp(-2.0))) < 1e-12
    assert np.allclose(T.density_prior(code, center, side, np.array([[100.0, 100.0, 100.0]]), s), -10.0, atol=1e-12)
    assert np.array_equal(T.density_prior(code, center, side, np.zeros((0, 3)), s), np.full(8, -10.0))


def test_p28_nearest_distance_brute_force():
    rs = np.random.RandomState(0)
    pts, q = rs.randn(300, 3) * 3, rs.randn(200, 3) * 4
    brute = np.sqrt(((q[:, None, :] - pts[None, :, :]) ** 2).sum(-1)).min(axis=1)
    np.testing.assert_allclose(T.nearest_distance(pts, q), brute, rtol=1e-13, atol=1e-13)


def _brute_near(code, center, side, pts, thr):
    i, j, k, level = so.decode(code)
    out = np.zeros(code.shape[0], bool)
    for v in range(code.shape[0]):
        n = 1 << int(level[v])
        lo = np.array(center) - side / 2 + np.array([i[v], j[v], k[v]]) * (side / n)
        hi = lo + side / n
        gap = np.maximum(np.maximum(lo - pts, pts - hi), 0.0)
        out[v] = bool((np.sqrt((gap ** 2).sum(1)) <= thr).any())
    return out


def test_p29_near_mask_brute_force_and_inclusive_threshold():
    sc = S.tiny_random_scene(6, n_static=60)
    tree = sc.static
    rs = np.random.RandomState(1)
    c, side = np.asarray(tree.center, dtype=np.float64), float(tree.side)
    pts = c + (rs.rand(40, 3) - 0.5) * side * 1.2
    for thr in (0.0, 0.05 * side, 0.3 * side):
        assert np.array_equal(T.near_mask(tree.code, c, side, pts, thr), _brute_near(tree.code, c, side, pts, thr))
    # box [0,2]^3 (cell (1,1,1), level 1, 4 m cube): a point 0.5 above the top face
    code = so.encode(np.array([1]), np.array([1]), np.array([1]), 1)
    p = np.array([[1.0, 1.0, 2.5]])
    assert T.near_mask(code, (0, 0, 0), 4.0, p, 0.5)[0] and not T.near_mask(code, (0, 0, 0), 4.0, p, 0.4999)[0]
    assert T.near_mask(code, (0, 0, 0), 4.0, np.array([[0.5, 1.5, 0.1]]), 0.0)[0]        # inside: distance 0
    assert not T.near_mask(code, (0, 0, 0), 4.0, np.zeros((0, 3)), 1.0)[0]


def _volume(code):
    level = so.decode(code)[3]
    return float((8.0 ** (-level.astype(np.float64))).sum())


def test_p30_subdivision_round():
    sc = S.tiny_random_scene(8, n_static=50)
    tree = sc.static
    c, side = np.asarray(tree.center, dtype=np.float64), float(tree.side)
    rs = np.random.RandomState(2)
    pts = c + (rs.rand(25, 3) - 0.5) * side
    new, split = T.subdivide_near(tree.code, c, side, pts, 0.02 * side)
    assert 0 < split.sum() < tree.code.shape[0]
    assert new.shape[0] == tree.code.shape[0] + 7 * int(split.sum())
    assert abs(_volume(new) - _volume(tree.code)) < 1e-12          # the leaves tile the same volume
    assert np.unique(new).shape[0] == new.shape[0]
    # children of a split leaf, decoded independently: the 8 octants of the parent cell, in order 4x+2y+z
    at = 0
    i, j, k, level = so.decode(tree.code)
    for v in range(tree.code.shape[0]):
        if not split[v]:
            assert new[at] == tree.code[v]
            at += 1
            continue
        ci, cj, ck, cl = so.decode(new[at:at + 8])
        for o in range(8):
            assert (ci[o], cj[o], ck[o], cl[o]) == (2 * i[v] + (o >> 2), 2 * j[v] + ((o >> 1) & 1), 2 * k[v] + (o & 1), level[v] + 1)
        at += 8
    assert at == new.shape[0]
    # nothing splits beyond the maximum level
    deep = so.encode(np.array([5]), np.array([6]), np.array([7]), 16)
    i16, j16, k16, _ = so.decode(deep)
    p = np.array([c - side / 2 + (np.array([i16[0], j16[0], k16[0]]) + 0.5) * side / 65536])
    out, sp = T.subdivide_near(deep, c, side, p, 1.0)
    assert not sp[0] and np.array_equal(out, deep)
    out, sp = T.subdivide_near(so.encode(np.array([0]), np.array([0]), np.array([0]), 3), c, side, c[None] - side / 2, 0.0, max_level=3)
    assert not sp[0]


def test_p31_prune():
    code = np.arange(6, dtype=np.uint64) + np.uint64(1 << 48)
    geo = np.full((6, 8), -10.0)
    geo[1, 3] = -3.0
    geo[4, 7] = -5.0
    geo[5, 0] = -5.0000001
    kept, idx = T.prune(code, geo, -5.0)
    assert idx.tolist() == [1, 4] and kept.tolist() == code[[1, 4]].tolist()
    kept, idx = T.prune(code, geo, -20.0)
    assert idx.tolist() == list(range(6))


# ---------------------------------------------------------------- P35 parameters of new children (reading R29)
def test_p35_subdivide_fill_is_the_parents_trilinear_field():
    """R29: a child's corners sample the parent's trilinear density, so (a) the child corner that coincides with a parent
    corner keeps its value, an edge midpoint is the mean of 2 parent corners, a face centre of 4, the cube centre of 8
    (written out by hand); (b) the continuous field is unchanged: rendering the parent and rendering its 8 children agree
    up to the quadrature, whose error falls 4 x when K doubles (P2) and vanishes for large K - and exactly for a density
    that is linear along the ray, where the midpoint rule on a half segment ... is NOT exact either, so only convergence is
    asserted; (c) a constant voxel splits into constant children (P8's case) bit for bit; (d) SH rows are copied."""
    import math
    import dvx_scenes as S
    from oracle import oracle as O
    from helpers import tree_from_cells, scene, axis_camera
    rs = np.random.RandomState(4)
    geo = rs.normal(-0.5, 1.0, size=(2, 8))
    sh = rs.normal(size=(2, 4, 3))
    g2, s2 = T.subdivide_fill([True, False], geo, sh)
    assert g2.shape == (9, 8) and s2.shape == (9, 4, 3)
    assert np.array_equal(g2[8], geo[1]) and np.array_equal(s2[8], sh[1])          # the kept leaf, last in order
    assert all(np.array_equal(s2[o], sh[0]) for o in range(8))                       # SH copied
    p = geo[0]
    for o in range(8):
        assert g2[o, o] == p[o]                                                      # the shared corner
        assert abs(g2[o, 7 - o] - p.mean()) < 1e-15                                  # the parent's centre
    # child 0 = (0,0,0): its corner 4 (bx=1) is the midpoint of the parent's edge 0-4, corner 6 (bx=by=1) the centre of the
    # face bz=0 (parent corners 0, 2, 4, 6), corner 1 (bz=1) the midpoint of edge 0-1
    assert abs(g2[0, 4] - 0.5 * (p[0] + p[4])) < 1e-15 and abs(g2[0, 1] - 0.5 * (p[0] + p[1])) < 1e-15
    assert abs(g2[0, 6] - 0.25 * (p[0] + p[2] + p[4] + p[6])) < 1e-15
    # child 5 = (1,0,1): its corner 2 (by=1) sits at u = (1/2, 1/2, 1/2)+... -> u = (0.5, 0.5, 0.5)? no: o=(1,0,1), b=(0,1,0) -> u=(.5,.5,.5)
    assert abs(g2[5, 2] - p.mean()) < 1e-15
    const, _ = T.subdivide_fill([True], np.full((1, 8), -0.75), np.zeros((1, 1, 3)))   # exactly representable: sums are exact
    assert np.array_equal(const, np.full((8, 8), -0.75))
    # (b) the field is unchanged: parent voxel [0,2]^3 of a 4 m cube vs its 8 children with the filled corners
    cam = axis_camera(width=5, height=5, f=6.0)
    kids = [(2 + ((o >> 2) & 1), 2 + ((o >> 1) & 1), 2 + (o & 1), 2) for o in range(8)]
    err = {}
    for K in (8, 16, 64):
        A = O.render(scene(tree_from_cells([(1, 1, 1, 1)], geo=geo[:1]), cam=cam, k_samples=K))
        B = O.render(scene(tree_from_cells(kids, geo=g2[:8]), cam=cam, k_samples=K))
        assert A["alpha"].max() > 0.3
        err[K] = np.abs(A["alpha"] - B["alpha"]).max()
    assert err[64] < 2e-5 and 3.0 < err[8] / err[16] < 5.0, err
