"""Pins of the oracle's feature pass O12 (widening row N3, reading R25) against things other than itself.

P22 two slabs, closed form: F = a1 f1 + (1-a1) a2 f2 with a_i = 1 - exp(-sigma_i chord), per channel
P23 a constant feature renders to alpha = 1 - T_final (the weights telescope), every pixel of a random scene
P24 with SH degree 0 the per-voxel colour is a feature: the feature image equals the (separately pinned) RGB render,
    actors included (pins the (octree, voxel) indexing of the feature tables and the weights themselves)
P25 fuse is the transpose of render: <render(f), G> = <f, fuse(G)>; wsum = fuse of a ones channel; fusing a constant
    image gives num/wsum = that constant for every voxel seen
P26 linearity in the features, and the mask is respected
"""
import math

import numpy as np

import dvx_scenes as S
from dvx_scenes.octree import C0
from oracle import oracle as O
from helpers import axis_camera, scene, tree_from_cells


def test_p22_two_slabs_closed_form():
    # cells (0,1,1) and (1,1,1) at level 1 of a 4 m cube: slabs -2<=x<=0 and 0<=x<=2, camera on the axis looking down +x
    v1, v2 = -0.3, 0.4
    f1, f2 = np.array([1.0, -2.0, 0.5, 7.0]), np.array([0.25, 3.0, -1.0, 0.0])
    cam = axis_camera(width=7, height=1, f=30.0)
    cam.cy = 0.5
    tree = tree_from_cells([(0, 1, 1, 1), (1, 1, 1, 1)], geo=np.array([[v1] * 8, [v2] * 8]))
    sc = scene(tree, cam=cam)
    r = O.render_features(sc, feats=[np.stack([f1, f2])])
    for u in range(7):
        x = (u + 0.5 - cam.cx) / cam.fx
        chord = 2 * math.sqrt(1 + x * x)
        a1, a2 = 1 - math.exp(-math.exp(v1) * chord), 1 - math.exp(-math.exp(v2) * chord)
        want = a1 * f1 + (1 - a1) * a2 * f2
        assert np.abs(r["features"][0, u] - want).max() < 1e-12
        assert abs(r["alpha"][0, u] - (1 - (1 - a1) * (1 - a2))) < 1e-12


def test_p23_constant_feature_is_alpha():
    for seed in (2, 7):
        sc = S.tiny_random_scene(seed)
        ref = O.render(sc)
        r = O.render_features(sc, feats=[np.full((t.n_voxels, 3), 2.5) for t in sc.octrees])
        assert np.abs(r["features"] - 2.5 * ref["alpha"][..., None]).max() < 1e-13
        assert np.array_equal(r["alpha"], ref["alpha"])


def test_p24_degree0_colour_as_feature_equals_rgb():
    sc = S.tiny_random_scene(4, sh_degree=0)
    assert len(sc.actors) >= 1
    ref = O.render(sc)
    feats = [np.maximum(0.0, C0 * t.sh[:, 0, :].astype(np.float64) + 0.5) for t in sc.octrees]   # R8 at degree 0
    r = O.render_features(sc, feats=feats)
    assert ref["rgb"].max() > 0.05
    assert np.abs(r["features"] - ref["rgb"]).max() < 1e-13


def test_p25_fuse_is_the_transpose():
    sc = S.tiny_random_scene(9)
    rs = np.random.RandomState(3)
    C = 6
    feats = [rs.randn(t.n_voxels, C) for t in sc.octrees]
    H, W = sc.cameras[0].height, sc.cameras[0].width
    G = rs.randn(H, W, C)
    F = O.render_features(sc, feats=feats)["features"]
    fu = O.render_features(sc, img=G)
    lhs = float((F * G).sum())
    rhs = float(sum((f * n).sum() for f, n in zip(feats, fu["num"])))
    assert abs(lhs - rhs) < 1e-11 * max(1.0, abs(lhs))
    ones = O.render_features(sc, img=np.ones((H, W, 1)))
    for a, b in zip(ones["num"], fu["wsum"]):
        np.testing.assert_allclose(a[:, 0], b, rtol=1e-13, atol=1e-15)
    const = O.render_features(sc, img=np.broadcast_to(np.array([0.5, -3.0]), (H, W, 2)).copy())
    seen = 0
    for n, w in zip(const["num"], const["wsum"]):
        m = w > 1e-12
        seen += int(m.sum())
        np.testing.assert_allclose(n[m] / w[m, None], np.broadcast_to([0.5, -3.0], (int(m.sum()), 2)), rtol=1e-12)
    assert seen > 5
    # both passes in one call give the same results
    both = O.render_features(sc, feats=feats, img=G)
    assert np.array_equal(both["features"], F) and all(np.allclose(a, b, rtol=1e-13, atol=1e-15) for a, b in zip(both["num"], fu["num"]))


def test_p26_linearity_and_mask():
    sc = S.tiny_random_scene(12)
    rs = np.random.RandomState(5)
    fa = [rs.randn(t.n_voxels, 4) for t in sc.octrees]
    fb = [rs.randn(t.n_voxels, 4) for t in sc.octrees]
    Fa = O.render_features(sc, feats=fa)["features"]
    Fb = O.render_features(sc, feats=fb)["features"]
    Fc = O.render_features(sc, feats=[2.0 * a - 3.0 * b for a, b in zip(fa, fb)])["features"]
    np.testing.assert_allclose(Fc, 2.0 * Fa - 3.0 * Fb, rtol=1e-12, atol=1e-13)
    H, W = Fa.shape[:2]
    mask = np.zeros((H, W), np.uint8)
    mask[::2, 1::3] = 1
    Fm = O.render_features(sc, feats=fa, mask=mask)["features"]
    assert np.array_equal(Fm[mask == 1], Fa[mask == 1]) and not Fm[mask == 0].any()
    # culled candidates == brute force (P13) for the feature pass too
    Fq = O.render_features(sc, feats=fa, mode=1)["features"]
    assert np.array_equal(Fq, Fa)
