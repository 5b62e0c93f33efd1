"""Pins of the CPU oracle against what the paper and the mathematics fix (no GPU, no CUDA code).

P-numbers follow DESIGN.md §3 / SURVEY.md §8(c).  Each check is chosen so that a plausible mistake in
oracle/dvx_oracle.c (dropped term, wrong sign or index, transposed operand) fails at least one.
"""
import math
import os
import numpy as np
import pytest

import dvx_scenes as S
from dvx_scenes.octree import C0, decode, encode
from oracle import oracle as O
from helpers import tree_from_cells, empty_tree, scene, axis_camera

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


# ---------------------------------------------------------------- P1 closed-form transmittance
@pytest.mark.parametrize("K", [1, 3, 8])
@pytest.mark.parametrize("v", [-2.0, 0.3])
def test_p1_single_constant_voxel(K, v):
    """BASELINE.json north_star: 'closed-form transmittance for a single voxel of constant density'.
    Voxel = cell (1,1,1) at level 1 of a 4 m cube -> [0,2]^3; camera at (-5,1,1) looking down +x.
    A ray at horizontal angle theta crosses the slab 0<=x<=2 with chord 2/cos(theta) (elementary geometry),
    entering at distance 5/cos(theta)."""
    cam = axis_camera(width=9, height=1, f=40.0)
    cam.cy = 0.5  # single row through the optical axis
    sc = scene(tree_from_cells([(1, 1, 1, 1)], geo=v), cam=cam, k_samples=K)
    r = O.render(sc)
    for u in range(9):
        x = (u + 0.5 - cam.cx) / cam.fx
        sec = math.sqrt(1 + x * x)
        chord, a = 2 * sec, 5 * sec
        alpha = 1 - math.exp(-math.exp(v) * chord)
        assert abs(r["alpha"][0, u] - alpha) < 1e-12
        assert np.abs(r["rgb"][0, u] - alpha).max() < 1e-12  # colour == 1
        assert abs(r["depth"][0, u] - alpha * (a + chord / 2)) < 1e-11


def test_p1_explinear_activation():
    """R5 option 1: exp-linear is the identity above theta=1.1 and C1-continuous there."""
    cam = axis_camera(width=1, height=1)
    for v, sigma in ((2.0, 2.0), (1.1, 1.1), (0.0, math.exp(0.0 / 1.1 - 1 + math.log(1.1)))):
        sc = scene(tree_from_cells([(1, 1, 1, 1)], geo=v), cam=cam, activation=1)
        assert abs(O.render(sc)["alpha"][0, 0] - (1 - math.exp(-sigma * 2))) < 1e-12


# ---------------------------------------------------------------- P2 quadrature order
def test_p2_midpoint_rule_order():
    """raw linear along the ray: int exp(p+q t) dt closed form; midpoint rule error falls 4x when K doubles (R6)."""
    p0, q0 = -1.0, 1.5  # raw = p0 + q0 * u_x
    geo = np.array([[p0 + q0 * ((c >> 2) & 1) for c in range(8)]])
    cam = axis_camera(width=1, height=1)
    exact = 2.0 * (math.exp(p0 + q0) - math.exp(p0)) / q0  # int_0^2 exp(p0 + q0 x/2) dx
    err = {}
    for K in (8, 16):
        sc = scene(tree_from_cells([(1, 1, 1, 1)], geo=geo), cam=cam, k_samples=K)
        tau = -math.log(1 - O.render(sc)["alpha"][0, 0])
        err[K] = abs(tau - exact)
    assert 3.9 < err[8] / err[16] < 4.1
    assert err[8] < 2e-3 * exact


def test_p2_corner_order_each_axis():
    """Corner index c = 4 bx + 2 by + bz (R7): a density ramp along one axis only changes the integral of a ray
    travelling along that axis in the closed-form way; rays along the other axes see a constant."""
    p0, q0 = -0.5, 1.0
    for axis, bit in ((0, 4), (1, 2), (2, 1)):
        geo = np.array([[p0 + q0 * (1 if (c & bit) else 0) for c in range(8)]])
        tree = tree_from_cells([(1, 1, 1, 1)], geo=geo)
        # camera looking along +x through the voxel centre line y=z=1: u_y = u_z = 1/2
        cam = axis_camera(width=1, height=1)
        tau = -math.log(1 - O.render(scene(tree, cam=cam, k_samples=64))["alpha"][0, 0])
        if axis == 0:
            expect = 2.0 * (math.exp(p0 + q0) - math.exp(p0)) / q0
            assert abs(tau - expect) < 1e-3 * expect
        else:
            assert abs(tau - 2.0 * math.exp(p0 + 0.5 * q0)) < 1e-12
    # ... and looking along +y (yaw 90 deg) the y-ramp is the one that integrates in closed form
    geo = np.array([[p0 + q0 * (1 if (c & 2) else 0) for c in range(8)]])
    cam = axis_camera(position=(1.0, -5.0, 1.0), width=1, height=1, yaw=math.pi / 2)
    tau = -math.log(1 - O.render(scene(tree_from_cells([(1, 1, 1, 1)], geo=geo), cam=cam, k_samples=64))["alpha"][0, 0])
    expect = 2.0 * (math.exp(p0 + q0) - math.exp(p0)) / q0
    assert abs(tau - expect) < 1e-3 * expect


# ---------------------------------------------------------------- P3 Morton order == depth order
def _random_leaves(rs, n_target, max_level):
    leaves = [(0, 0, 0, 0)]
    while len(leaves) < n_target:
        i, j, k, l = leaves.pop(rs.integers(len(leaves)))
        if l >= max_level:
            leaves.append((i, j, k, l))
            continue
        leaves += [(2 * i + a, 2 * j + b, 2 * k + c, l + 1) for a in (0, 1) for b in (0, 1) for c in (0, 1)]
    return [v for v in leaves if v[3] >= 1 and rs.random() > 0.3]


def test_p3_morton_order_matches_true_depth_order():
    """north_star: 'agreement between Morton order and true depth order on tiny random octrees'."""
    rs = np.random.default_rng(123)
    checked = 0
    for trial in range(12):
        cells = _random_leaves(rs, int(rs.integers(50, 300)), 5)
        tree = tree_from_cells(cells, geo=-1.0, center=(0.3, -0.2, 0.1), side=6.0)
        yaw = rs.uniform(-math.pi, math.pi)
        pos = (-8 * math.cos(yaw) + 0.3, -8 * math.sin(yaw) - 0.2, rs.uniform(-2.5, 2.5))
        cam = S.Camera(24, 24, 30.0, 30.0, 12.0, 12.0, S.look_yaw(pos, yaw))
        sc = scene(tree, cam=cam, t_stop=0.0)
        for _ in range(20):
            u, v = int(rs.integers(24)), int(rs.integers(24))
            o, d = O.ray(sc, u, v)
            q = 4 * (d[0] < 0) + 2 * (d[1] < 0) + (d[2] < 0)
            _, vox, a, b = O.ray_segments(sc, u, v)
            keep = (b - a) > 1e-9
            keys = O.order_key(tree.code[vox[keep]], q)
            assert np.all(keys[1:] > keys[:-1])
            checked += int(keep.sum())
    assert checked > 500


def test_p3_order_key_layout():
    """R14a/R14b bit layout: x is the most significant bit of each 3-bit group, groups left-aligned at bit 45."""
    c = encode(np.array([1]), np.array([0]), np.array([0]), np.array([1]))[0]
    assert c == (1 << 48) | (4 << 45)
    c = encode(np.array([2]), np.array([1]), np.array([3]), np.array([2]))[0]  # i=10b j=01b k=11b
    assert c == (2 << 48) | (0b101 << 45) | (0b011 << 42)
    assert O.order_key([c], 0)[0] == (c & ((1 << 48) - 1))
    assert O.order_key([c], 5)[0] == (c & ((1 << 48) - 1)) ^ int("101" * 16, 2)
    i, j, k, l = decode(np.array([c]))
    assert (i[0], j[0], k[0], l[0]) == (2, 1, 3, 2)


# ---------------------------------------------------------------- P4 world-frame rewrites
def _rot_z90_tree(t):
    """Rewrite an octree (centre 0) under p' = Rz(90deg) p: (x,y,z)->(-y,x,z).  SH degree <= 1."""
    i, j, k, l = decode(t.code)
    n = (1 << l)
    code = encode(n - 1 - j, i, k, l)
    geo = np.empty_like(t.geo)
    for c in range(8):
        bx, by, bz = (c >> 2) & 1, (c >> 1) & 1, c & 1
        geo[:, 4 * (1 - by) + 2 * bx + bz] = t.geo[:, c]
    sh = t.sh.copy()
    if t.sh_degree >= 1:  # colour term = -c1 (k3,k1,-k2).dir ; the vector rotates with the frame
        sh[:, 1] = t.sh[:, 3]
        sh[:, 3] = -t.sh[:, 1]
    from helpers import _raw
    return _raw(code, geo, sh, (0, 0, 0), t.side, t.sh_degree)


def test_p4_yaw90_rewrite():
    """north_star: 'invariance when a whole actor octree plus its pose is rewritten'.  An actor under yaw psi+90deg
    equals the actor with integer coordinates / corner order / degree-1 SH rotated, under yaw psi."""
    s0 = S.tiny_random_scene(11, sh_degree=1)
    act = s0.actors[0]
    psi = 0.35
    t = np.array([1.5, 0.3, 0.2])
    half = np.array([1.0, 0.5, 0.75])
    A = scene(s0.static, [act], [S.pose_yaw(t, psi + math.pi / 2)], [half], cam=s0.cameras[0], t_stop=0.0)
    B = scene(s0.static, [_rot_z90_tree(act)], [S.pose_yaw(t, psi)], [half[[1, 0, 2]]], cam=s0.cameras[0], t_stop=0.0)
    ra, rb = O.render(A), O.render(B)
    assert ra["alpha"].max() > 0.1
    for k in ("rgb", "depth", "alpha"):
        assert np.abs(ra[k] - rb[k]).max() < 1e-10
    # the actor must be visible for this to mean anything
    C = scene(s0.static, [], [], [], cam=s0.cameras[0], t_stop=0.0)
    assert np.abs(O.render(C)["rgb"] - ra["rgb"]).max() > 1e-3


def test_p4_static_as_actor_and_rigid_motion():
    s0 = S.tiny_random_scene(5, sh_degree=1)
    cam = s0.cameras[0]
    st = s0.static
    from helpers import _raw
    st0 = _raw(st.code, st.geo, st.sh, (0, 0, 0), st.side, st.sh_degree)  # centred so a centred box covers it
    big = [st.side, st.side, st.side]
    ident = np.concatenate([np.eye(3), np.zeros((3, 1))], 1)
    A = scene(st0, [], [], [], cam=cam, t_stop=0.0)
    B = scene(empty_tree(1), [st0], [ident], [big], cam=cam, t_stop=0.0)
    ra, rb = O.render(A), O.render(B)
    for k in ("rgb", "depth", "alpha"):
        assert np.abs(ra[k] - rb[k]).max() < 1e-10
    # (d) one rigid motion G applied to the camera and to every pose
    th, ax = 0.9, np.array([0.3, -0.5, 0.8]) / np.linalg.norm([0.3, -0.5, 0.8])
    Kx = np.array([[0, -ax[2], ax[1]], [ax[2], 0, -ax[0]], [-ax[1], ax[0], 0]])
    G = np.eye(3) + math.sin(th) * Kx + (1 - math.cos(th)) * Kx @ Kx
    g = np.array([0.7, -1.1, 2.0])
    P1 = np.asarray(s0.poses[0], dtype=np.float64).reshape(3, 4)
    P2 = S.pose_yaw((-1.0, -2.0, 0.5), -0.4)
    acts, halves = [s0.actors[0], st0], [s0.box_half[0], [1.0, 1.0, 1.0]]
    c2w = np.asarray(cam.c2w, dtype=np.float64).reshape(3, 4)

    def moved(P):
        return np.concatenate([G @ P[:, :3], (G @ P[:, 3] + g)[:, None]], 1)

    A = scene(empty_tree(1), acts, [P1, P2], halves, cam=cam, t_stop=0.0)
    cam2 = S.Camera(cam.width, cam.height, cam.fx, cam.fy, cam.cx, cam.cy, cam.c2w, cam.near, cam.far)
    cam2.c2w = moved(c2w).reshape(12)
    cam.c2w = c2w.reshape(12)
    B = scene(empty_tree(1), acts, [moved(P1), moved(P2)], halves, cam=cam2, t_stop=0.0)
    ra, rb = O.render(A), O.render(B)
    assert ra["alpha"].max() > 0.1
    for k in ("rgb", "depth", "alpha"):
        assert np.abs(ra[k] - rb[k]).max() < 1e-10


# ---------------------------------------------------------------- P5 empty actor boxes
def test_p5_empty_actor_box_leaves_static_unchanged():
    """north_star: 'an empty actor box leaves the static render unchanged' (where it masks no static voxel)."""
    s0 = S.tiny_random_scene(3, sh_degree=1)
    cam = s0.cameras[0]
    base = O.render(scene(s0.static, [], [], [], cam=cam))
    behind = S.pose_yaw((-20.0, 0.0, 0.0), 0.3)        # behind the camera
    outside = S.pose_yaw((0.0, 60.0, 0.0), 0.3)         # outside the frustum
    free = S.pose_yaw((-5.0, 0.4, 0.3), 0.5)            # in front, in free space before the static cube
    for pose in (behind, outside, free):
        r = O.render(scene(s0.static, [empty_tree(1)], [pose], [[0.2, 0.2, 0.2]], cam=cam))
        for k in ("rgb", "depth", "alpha"):
            assert np.array_equal(r[k], base[k])
    # the free-space box really is crossed by rays (the schedule splits)
    o, d = O.ray(scene(s0.static, cam=cam), cam.width // 2, cam.height // 2)
    assert any(O.ray_box(free, [0.2, 0.2, 0.2], *O.ray(scene(s0.static, cam=cam), u, v)) is not None
               for u in range(cam.width) for v in range(cam.height))


# ---------------------------------------------------------------- P6 finite differences
def test_p6_finite_difference_gradients():
    """north_star: 'finite-difference gradients on tiny scenes'.  Loss = random linear functional of RGB, depth, alpha."""
    s = S.tiny_random_scene(7, sh_degree=1, colour_floor=True)
    for t in s.octrees:
        t.geo = t.geo.astype(np.float64)
        t.sh = t.sh.astype(np.float64)
    g = s.image_grads(0, 1.0, 0.3, 1.0)
    r = O.render(s, grads_in=g)
    assert r["alpha"].max() > 0.3

    def loss():
        q = O.render(s)
        return (q["rgb"] * g["rgb"]).sum() + (q["depth"] * g["depth"]).sum() + (q["alpha"] * g["alpha"]).sum()

    h = 1e-5
    worst, n_nonzero = 0.0, 0
    for n, t in enumerate(s.octrees):
        for arr, ana in ((t.geo, r["dgeo"][n]), (t.sh, r["dsh"][n])):
            flat, aflat = arr.reshape(-1), ana.reshape(-1)
            scale = max(np.abs(aflat).max(), 1e-12)
            for idx in range(flat.shape[0]):
                keep = flat[idx]
                flat[idx] = keep + h; lp = loss()
                flat[idx] = keep - h; lm = loss()
                flat[idx] = keep
                fd = (lp - lm) / (2 * h)
                worst = max(worst, abs(fd - aflat[idx]) / scale)
                n_nonzero += abs(aflat[idx]) > 1e-9 * scale
    assert n_nonzero > 100
    assert worst < 1e-6


def test_p6_clamped_colour_has_zero_gradient():
    cam = axis_camera(width=1, height=1)
    sh = np.zeros((1, 1, 3)); sh[0, 0] = [(-0.7) / C0, 0.2 / C0, 0.0]  # red channel clamps at 0
    sc = scene(tree_from_cells([(1, 1, 1, 1)], geo=0.0, sh=sh), cam=cam)
    r = O.render(sc, grads_in={"rgb": np.ones((1, 1, 3))})
    assert r["rgb"][0, 0, 0] == 0.0 and r["dsh"][0][0, 0, 0] == 0.0 and r["dsh"][0][0, 0, 1] != 0.0


# ---------------------------------------------------------------- P7 partition of unity
def test_p7_partition_of_unity(config1):
    s = config1
    for t in s.octrees:
        t = t
    import copy
    s2 = copy.deepcopy(s)
    for t in s2.octrees:
        t.sh[:] = 0
        t.sh[:, 0, :] = np.float32(0.5 / C0)
    r = O.render(s2, mode=1)
    one = 0.5 + C0 * float(np.float32(0.5 / C0))
    assert np.abs(r["rgb"] - one * r["alpha"][..., None]).max() < 1e-12
    assert r["alpha"].min() >= 0 and r["alpha"].max() < 1
    assert np.all(r["depth"] >= 0)


# ---------------------------------------------------------------- P8 subdivision invariance
def test_p8_subdivision_invariance_constant_density():
    cam = axis_camera(width=9, height=7, f=12.0)
    A = scene(tree_from_cells([(1, 1, 1, 1)], geo=-0.7), cam=cam)
    kids = [(2 + a, 2 + b, 2 + c, 2) for a in (0, 1) for b in (0, 1) for c in (0, 1)]
    B = scene(tree_from_cells(kids, geo=-0.7), cam=cam)
    ra, rb = O.render(A), O.render(B)
    assert ra["alpha"].max() > 0.5
    assert np.abs(ra["alpha"] - rb["alpha"]).max() < 1e-12
    assert np.abs(ra["rgb"] - rb["rgb"]).max() < 1e-12


# ---------------------------------------------------------------- P9 ray-box against dense sampling
def test_p9_ray_box_dense_sampling():
    rs = np.random.default_rng(9)
    n_hit = 0
    for trial in range(60):
        yaw = rs.uniform(-math.pi, math.pi)
        pose = S.pose_yaw(rs.uniform(-2, 2, 3), yaw)
        half = rs.uniform(0.3, 2.0, 3)
        o = rs.uniform(-4, 4, 3) if trial % 3 else pose[:, 3] + 0.1 * half  # some origins inside the box
        d = rs.normal(size=3)
        if trial % 5 == 0:
            d = pose[:, :3] @ np.array([1.0, 0.0, 0.0])  # parallel to two slabs (d_local has exact or near zeros)
        d /= np.linalg.norm(d)
        ts = np.linspace(0.0, 12.0, 100001)
        p = o[None] + ts[:, None] * d[None]
        pl = (p - pose[:, 3][None]) @ pose[:, :3]
        inside = np.all(np.abs(pl) <= half[None], axis=1) & (ts >= 0.05)
        res = O.ray_box(pose, half, o, d, near=0.05, far=1e9)
        if inside.sum() < 3:
            assert res is None or res[1] - res[0] < 3 * 12.0 / 100000
            continue
        n_hit += 1
        assert res is not None
        assert abs(res[0] - ts[inside][0]) < 2 * 12.0 / 100000
        assert abs(res[1] - ts[inside][-1]) < 2 * 12.0 / 100000
    assert n_hit > 15


# ---------------------------------------------------------------- P10 two slabs across octrees
def test_p10_two_slab_closed_form_across_octrees():
    """Static voxel [0,2]^3 (sigma1, colour c1) and one actor voxel (sigma2, colour c2) on the optical axis;
    C = c1 (1-e^{-s1 l1}) + e^{-s1 l1} c2 (1-e^{-s2 l2}), roles swapped when the pose moves the actor in front."""
    cam = axis_camera(width=1, height=1)
    v1, v2, c1, c2 = -0.5, 0.2, 0.8, 0.3
    sh1 = np.full((1, 1, 3), (c1 - 0.5) / C0); sh2 = np.full((1, 1, 3), (c2 - 0.5) / C0)
    st = tree_from_cells([(1, 1, 1, 1)], geo=v1, sh=sh1)
    # actor: 1 m cube octree, a single level-1 cell (1,1,1) -> local [0,0.5]^3 ; box half 0.6 covers it
    act = tree_from_cells([(1, 1, 1, 1)], geo=v2, sh=sh2, side=1.0)
    s1, s2, l1, l2 = math.exp(v1), math.exp(v2), 2.0, 0.5
    for x_act, actor_first in ((4.0, False), (-3.0, True)):
        pose = S.pose_yaw((x_act, 1.0 - 0.25, 1.0 - 0.25), 0.0)  # centre line of the actor voxel on the axis y=z=1
        r = O.render(scene(st, [act], [pose], [[0.6, 0.6, 0.6]], cam=cam))
        e1, e2 = math.exp(-s1 * l1), math.exp(-s2 * l2)
        expect = c2 * (1 - e2) + e2 * c1 * (1 - e1) if actor_first else c1 * (1 - e1) + e1 * c2 * (1 - e2)
        assert abs(r["rgb"][0, 0, 0] - expect) < 1e-12
        assert abs(r["alpha"][0, 0] - (1 - e1 * e2)) < 1e-12
        a_act = x_act + 5.0  # actor voxel starts at world x = x_act
        d1, d2 = (1 - e1) * 6.0, (1 - e2) * (a_act + 0.25)
        expect_d = d2 + e2 * d1 if actor_first else d1 + e1 * d2
        assert abs(r["depth"][0, 0] - expect_d) < 1e-11


def test_p10_overlapping_boxes_rule_r2():
    """R2: a box entered later is clipped to start where the earlier one ended; ties by lower index."""
    cam = axis_camera(width=1, height=1)
    act = tree_from_cells([(0, 0, 0, 1), (1, 0, 0, 1), (0, 1, 0, 1), (1, 1, 0, 1), (0, 0, 1, 1), (1, 0, 1, 1), (0, 1, 1, 1), (1, 1, 1, 1)],
                          geo=0.0, side=2.0)  # a full 2 m cube of sigma=1
    pa, pb = S.pose_yaw((0.0, 1.0, 1.0), 0.0), S.pose_yaw((1.0, 1.0, 1.0), 0.0)  # boxes [-1,1] and [0,2] in x overlap on [0,1]
    r = O.render(scene(empty_tree(), [act, act], [pa, pb], [[1, 1, 1], [1, 1, 1]], cam=cam))
    assert abs(r["alpha"][0, 0] - (1 - math.exp(-3.0))) < 1e-12  # union length 3, never double-counted


# ---------------------------------------------------------------- P11 masking and clipping
def test_p11_empty_box_masks_static_content():
    """R1 / Alg. 1 l.4-7: the static stream is skipped on [tau_in, tau_out]; voxels are clipped, not dropped."""
    cam = axis_camera(width=1, height=1)
    v = -0.3
    st = tree_from_cells([(1, 1, 1, 1)], geo=v)
    pose = S.pose_yaw((1.0, 1.0, 1.0), 0.0)
    r = O.render(scene(st, [empty_tree()], [pose], [[0.4, 0.3, 0.3]], cam=cam))
    s = math.exp(v)
    assert abs(r["alpha"][0, 0] - (1 - math.exp(-s * (2.0 - 0.8)))) < 1e-12
    # depth: two pieces [5,5.6] and [6.4,7]
    e = math.exp(-s * 0.6)
    expect = (1 - e) * 5.3 + e * (1 - e) * 6.7
    assert abs(r["depth"][0, 0] - expect) < 1e-11


# ---------------------------------------------------------------- P12 SH basis
def test_p12_sh_orthonormal():
    n_t, n_p = 24, 48
    x, w = np.polynomial.legendre.leggauss(n_t)
    G = np.zeros((16, 16))
    for ct, wt in zip(x, w):
        st = math.sqrt(1 - ct * ct)
        for ip in range(n_p):
            ph = 2 * math.pi * (ip + 0.5) / n_p
            Y = O.sh_basis([st * math.cos(ph), st * math.sin(ph), ct])
            G += wt * (2 * math.pi / n_p) * np.outer(Y, Y)
    assert np.abs(G - np.eye(16)).max() < 1e-12


def test_p12_sh_values_golden():
    """Values of the basis at two directions, computed once from the closed-form associated-Legendre definition
    (tests/golden/make_sh_golden.py, which does not call the oracle)."""
    rows = np.loadtxt(os.path.join(GOLDEN, "sh_basis.txt"))
    for row in rows:
        Y = O.sh_basis(row[:3])
        assert np.abs(Y - row[3:]).max() < 1e-13


# ---------------------------------------------------------------- P13 tile-culled == brute force
def test_p13_culled_equals_brute_config1(config1):
    a, b = O.render(config1, mode=0), O.render(config1, mode=1)
    for k in ("rgb", "depth", "alpha", "n_used"):
        assert np.array_equal(a[k], b[k])
    assert a["alpha"].max() > 0.9 and a["n_used"].max() > 10


@pytest.mark.slow
def test_p13_culled_equals_brute_config2_sampled():
    s = S.make_config(2)
    cam = s.cameras[0]
    rs = np.random.default_rng(2)
    mask = np.zeros((cam.height, cam.width), dtype=np.uint8)
    mask.reshape(-1)[rs.choice(cam.height * cam.width, 192, replace=False)] = 1
    # include near-ground pixels (voxels crossing the near plane) and actor pixels
    mask[-1, ::97] = 1
    a, b = O.render(s, mode=0, mask=mask), O.render(s, mode=1, mask=mask)
    m = mask.astype(bool)
    for k in ("rgb", "depth", "alpha", "n_used"):
        assert np.array_equal(a[k][m], b[k][m])


# ---------------------------------------------------------------- P14 sky composite (Eq. 2; reading R21)
def _sky_tex(h, w, seed=5):
    rs = np.random.RandomState(seed)
    return rs.uniform(0.0, 1.0, size=(h, w, 3))


def test_p14_constant_sky_and_partition_of_unity():
    """Eq. 2 with a constant map: C = C_voxels + T_final c_sky exactly, wherever the ray points; empty scene: C = c_sky."""
    s = S.tiny_random_scene(3, sh_degree=1)
    c_sky = np.array([0.2, 0.5, 0.9])
    tex = np.broadcast_to(c_sky, (6, 12, 3)).copy()
    base, with_sky = O.render(s), O.render(s, sky=tex)
    assert np.abs(with_sky["rgb"] - (base["rgb"] + (1.0 - base["alpha"])[..., None] * c_sky)).max() < 1e-14
    assert np.array_equal(with_sky["alpha"], base["alpha"]) and np.array_equal(with_sky["depth"], base["depth"])
    empty = scene(empty_tree(), cam=s.cameras[0])
    assert np.abs(O.render(empty, sky=tex)["rgb"] - c_sky).max() < 1e-15


def test_p14_single_voxel_closed_form_with_sky():
    """P1 + Eq. 2: one constant-density voxel of colour c in front of a constant sky: C = alpha c + (1 - alpha) c_sky."""
    cam = axis_camera(width=1, height=1)
    v, c = -0.4, 0.7
    st = tree_from_cells([(1, 1, 1, 1)], geo=v, sh=np.full((1, 1, 3), (c - 0.5) / C0))
    tex = np.broadcast_to(np.array([0.1, 0.3, 0.6]), (4, 8, 3)).copy()
    r = O.render(scene(st, cam=cam), sky=tex)
    alpha = 1.0 - math.exp(-math.exp(v) * 2.0)
    assert np.abs(r["rgb"][0, 0] - (alpha * c + (1 - alpha) * tex[0, 0])).max() < 1e-13


def test_p14_bilinear_footprint_geometry():
    """The footprint is a bilinear one (4 texels, weights in [0,1] summing to 1), it reproduces maps that are linear in the
    texel coordinates, the azimuth wraps, and rotating the direction by one texel of azimuth shifts the sample by one
    column; known directions land where R21 says: +x -> column W/2, horizon -> row H/2, zenith -> row 0."""
    W, H = 16, 8
    rs = np.random.RandomState(1)
    for _ in range(200):
        d = rs.normal(size=3); d /= np.linalg.norm(d)
        idx, wt = O.sky_footprint(W, H, d)
        assert abs(wt.sum() - 1) < 1e-14 and wt.min() >= 0 and wt.max() <= 1
        jj, ii = idx // W, idx % W
        assert jj[0] == jj[1] and jj[2] == jj[3] and ii[0] == ii[2] and ii[1] == ii[3]
        assert ii[1] == (ii[0] + 1) % W and jj[2] in (jj[0], jj[0] + 1)
        # one texel of azimuth = rotation by 2 pi / W about z
        a = 2 * math.pi / W
        d2 = np.array([math.cos(a) * d[0] - math.sin(a) * d[1], math.sin(a) * d[0] + math.cos(a) * d[1], d[2]])
        idx2, wt2 = O.sky_footprint(W, H, d2)
        assert np.array_equal(idx2 // W, jj) and np.array_equal(idx2 % W, (ii + 1) % W) and np.abs(wt2 - wt).max() < 1e-9
    idx, wt = O.sky_footprint(W, H, (1.0, 0.0, 0.0))       # phi = 0, theta = pi/2: between columns W/2-1, W/2 and rows H/2-1, H/2
    assert sorted(idx.tolist()) == sorted([(H // 2 - 1) * W + W // 2 - 1, (H // 2 - 1) * W + W // 2, (H // 2) * W + W // 2 - 1,
                                           (H // 2) * W + W // 2]) and np.abs(wt - 0.25).max() < 1e-12
    idx, wt = O.sky_footprint(W, H, (0.0, 0.0, 1.0))       # zenith: clamped to row 0
    assert set((idx // W)[wt > 0].tolist()) == {0}
    idx, wt = O.sky_footprint(W, H, (0.0, 0.0, -1.0))      # nadir: row H-1
    assert set((idx // W)[wt > 0].tolist()) == {H - 1}
    # reproduces a map linear in the row index (away from the clamp): value = t = theta / pi * H - 1/2
    d = np.array([0.3, -0.4, 0.2]); d /= np.linalg.norm(d)
    idx, wt = O.sky_footprint(W, H, d)
    assert abs((wt * (idx // W)).sum() - (math.acos(d[2]) / math.pi * H - 0.5)) < 1e-12


def test_p14_finite_difference_gradients_with_sky():
    """O9 + O10: analytic gradients of the texture, the corner densities and the SH coefficients with the sky on."""
    s = S.tiny_random_scene(9, sh_degree=1, colour_floor=True)
    for t in s.octrees:
        t.geo = t.geo.astype(np.float64)
        t.sh = t.sh.astype(np.float64)
    tex = _sky_tex(5, 9)
    g = s.image_grads(0, 1.0, 0.3, 1.0)
    r = O.render(s, grads_in=g, sky=tex)

    def loss():
        q = O.render(s, sky=tex)
        return (q["rgb"] * g["rgb"]).sum() + (q["depth"] * g["depth"]).sum() + (q["alpha"] * g["alpha"]).sum()

    h = 1e-5
    checks = [(tex, r["dsky"])] + [(t.geo, r["dgeo"][n]) for n, t in enumerate(s.octrees)]
    for arr, ana in checks:
        flat, aflat = arr.reshape(-1), ana.reshape(-1)
        scale = max(np.abs(aflat).max(), 1e-12)
        assert np.count_nonzero(aflat) > 10
        for idx in range(0, flat.shape[0], 3):
            keep = flat[idx]
            flat[idx] = keep + h; lp = loss()
            flat[idx] = keep - h; lm = loss()
            flat[idx] = keep
            assert abs((lp - lm) / (2 * h) - aflat[idx]) / scale < 1e-6


# ---------------------------------------------------------------- P15 normal map (state tuple S; reading R22)
def _ramp_geo(axis, lo=0.0, hi=1.0):
    """8 corner values, corner c = 4 bx + 2 by + bz, raw density = lo on the face b_axis = 0 and hi on b_axis = 1."""
    return np.array([hi if (c >> (2 - axis)) & 1 else lo for c in range(8)], dtype=np.float64)


@pytest.mark.parametrize("axis", [0, 1, 2])
def test_p15_linear_density_gives_axis_normal(axis):
    """A voxel whose raw density rises linearly along one axis has the normal -e_axis; N = alpha n (one voxel)."""
    cam = axis_camera(width=3, height=3)
    st = tree_from_cells([(1, 1, 1, 1)], geo=_ramp_geo(axis, -1.0, 0.5).reshape(1, 8))
    r = O.render(scene(st, cam=cam), normals=True)
    n = np.zeros(3); n[axis] = -1.0
    assert r["alpha"][1, 1] > 0.3
    assert np.abs(r["normal"] - r["alpha"][..., None] * n).max() < 1e-14
    # falling density flips it; a constant voxel has no normal at all
    st2 = tree_from_cells([(1, 1, 1, 1)], geo=_ramp_geo(axis, 0.5, -1.0).reshape(1, 8))
    r2 = O.render(scene(st2, cam=cam), normals=True)
    assert np.abs(r2["normal"] + r2["alpha"][..., None] * n).max() < 1e-14
    r3 = O.render(scene(tree_from_cells([(1, 1, 1, 1)], geo=0.2), cam=cam), normals=True)
    assert np.abs(r3["normal"]).max() == 0.0


def test_p15_actor_normal_is_rotated_into_the_world_frame():
    cam = axis_camera(width=3, height=3)
    act = tree_from_cells([(1, 1, 1, 1)], geo=_ramp_geo(0, -1.0, 0.5).reshape(1, 8), side=1.0)
    for yaw in (0.0, 0.7, math.pi / 2, -2.0):
        pose = S.pose_yaw((0.0, 1.0, 1.0), yaw)
        r = O.render(scene(empty_tree(), [act], [pose], [[0.6, 0.6, 0.6]], cam=cam), normals=True)
        n = np.array([-math.cos(yaw), -math.sin(yaw), 0.0])
        assert r["alpha"].max() > 0.1
        assert np.abs(r["normal"] - r["alpha"][..., None] * n).max() < 1e-14


def test_p15_rigid_motion_rotates_the_normal_map_and_bound():
    """One rigid motion G applied to the camera and to every pose (P4 (d)): N' = G_R N; and |N| <= alpha everywhere."""
    s0 = S.tiny_random_scene(5, sh_degree=1)
    cam = s0.cameras[0]
    from helpers import _raw
    st = s0.static
    st0 = _raw(st.code, st.geo, st.sh, (0, 0, 0), st.side, st.sh_degree)
    th, ax = 0.9, np.array([0.3, -0.5, 0.8]) / np.linalg.norm([0.3, -0.5, 0.8])
    Kx = np.array([[0, -ax[2], ax[1]], [ax[2], 0, -ax[0]], [-ax[1], ax[0], 0]])
    G = np.eye(3) + math.sin(th) * Kx + (1 - math.cos(th)) * Kx @ Kx
    g = np.array([0.7, -1.1, 2.0])
    P1 = np.asarray(s0.poses[0], dtype=np.float64).reshape(3, 4)
    P2 = S.pose_yaw((-1.0, -2.0, 0.5), -0.4)
    acts, halves = [s0.actors[0], st0], [s0.box_half[0], [1.0, 1.0, 1.0]]
    c2w = np.asarray(cam.c2w, dtype=np.float64).reshape(3, 4)
    moved = lambda P: np.concatenate([G @ P[:, :3], (G @ P[:, 3] + g)[:, None]], 1)
    cam.c2w = c2w.reshape(12)
    A = scene(empty_tree(1), acts, [P1, P2], halves, cam=cam, t_stop=0.0)
    cam2 = S.Camera(cam.width, cam.height, cam.fx, cam.fy, cam.cx, cam.cy, cam.c2w, cam.near, cam.far)
    cam2.c2w = moved(c2w).reshape(12)
    B = scene(empty_tree(1), acts, [moved(P1), moved(P2)], halves, cam=cam2, t_stop=0.0)
    ra, rb = O.render(A, normals=True), O.render(B, normals=True)
    assert np.abs(ra["normal"]).max() > 0.05
    assert np.abs(ra["normal"] @ G.T - rb["normal"]).max() < 1e-10
    assert (np.linalg.norm(ra["normal"], axis=-1) <= ra["alpha"] * (1 + 1e-6) + 1e-12).all()  # poses are fp32-rounded rotations


def test_p15_finite_difference_gradients_with_normals():
    s = S.tiny_random_scene(13, sh_degree=1, colour_floor=True)
    for t in s.octrees:
        t.geo = t.geo.astype(np.float64)
        t.sh = t.sh.astype(np.float64)
    g = s.image_grads(0, 1.0, 0.3, 1.0)
    rs = np.random.RandomState(2)
    g["normal"] = rs.normal(size=g["rgb"].shape)
    r = O.render(s, grads_in=g)

    def loss():
        q = O.render(s, normals=True)
        return ((q["rgb"] * g["rgb"]).sum() + (q["depth"] * g["depth"]).sum() + (q["alpha"] * g["alpha"]).sum()
                + (q["normal"] * g["normal"]).sum())

    h = 1e-6
    for n, t in enumerate(s.octrees):
        flat, aflat = t.geo.reshape(-1), r["dgeo"][n].reshape(-1)
        scale = max(np.abs(aflat).max(), 1e-12)
        assert np.count_nonzero(aflat) > 20
        for idx in range(flat.shape[0]):
            keep = flat[idx]
            flat[idx] = keep + h; lp = loss()
            flat[idx] = keep - h; lm = loss()
            flat[idx] = keep
            assert abs((lp - lm) / (2 * h) - aflat[idx]) / scale < 2e-6, (n, idx)


# ---------------------------------------------------------------- P32 early termination (Alg. 1 l.8-9; R3)
def _two_slab_scene(v1, t_stop, v2=0.2, c1=0.8, c2=0.3):
    """P10's geometry: static voxel [0,2]^3 (chord 2 on the optical axis, entered at tau = 5) in front of one actor voxel
    (chord 0.5, entered at tau = 9)."""
    cam = axis_camera(width=1, height=1)
    sh1 = np.full((1, 1, 3), (c1 - 0.5) / C0); sh2 = np.full((1, 1, 3), (c2 - 0.5) / C0)
    st = tree_from_cells([(1, 1, 1, 1)], geo=v1, sh=sh1)
    act = tree_from_cells([(1, 1, 1, 1)], geo=v2, sh=sh2, side=1.0)
    pose = S.pose_yaw((4.0, 0.75, 0.75), 0.0)
    return scene(st, [act], [pose], [[0.6, 0.6, 0.6]], cam=cam, t_stop=t_stop)


def test_p32_early_termination_after_the_crossing_voxel():
    """north_star (4) 'early termination at T < 1e-4', Alg. 1 l.8-9, reading R3: T is tested AFTER each
    voxel, the voxel that crosses the threshold is composited, everything behind it is not.  t_stop = 0.05:
      T1 = 0.04 -> the second slab must be ABSENT  (alpha = 1 - T1, C = c1 (1 - T1), n_used = 1);
      T1 = 0.06 -> the second slab must be PRESENT (closed form of P10, n_used = 2).
    Fails under: no termination at all (first case), a threshold compared against alpha or against tau instead of T
    (second case: alpha1 = 0.94, tau1 = 2.8), termination that drops the crossing voxel as 3DGS-style rasterizers do
    (test_p32_crossing_voxel_is_included), `<=` instead of `<` (test_p32_threshold_is_strict)."""
    c1, c2, v2, l2 = 0.8, 0.3, 0.2, 0.5
    e2 = math.exp(-math.exp(v2) * l2)
    for T1, second in ((0.04, False), (0.06, True)):
        v1 = math.log(-math.log(T1) / 2.0)          # sigma1 * 2 = -ln T1
        r = O.render(_two_slab_scene(v1, 0.05))
        if second:
            assert r["n_used"][0, 0] == 2
            assert abs(r["alpha"][0, 0] - (1 - T1 * e2)) < 1e-12
            assert abs(r["rgb"][0, 0, 0] - (c1 * (1 - T1) + T1 * c2 * (1 - e2))) < 1e-12
            assert abs(r["depth"][0, 0] - ((1 - T1) * 6.0 + T1 * (1 - e2) * 9.25)) < 1e-11
        else:
            assert r["n_used"][0, 0] == 1
            assert abs(r["alpha"][0, 0] - (1 - T1)) < 1e-12
            assert abs(r["rgb"][0, 0, 0] - c1 * (1 - T1)) < 1e-12
            assert abs(r["depth"][0, 0] - (1 - T1) * 6.0) < 1e-11
        # t_stop = 0 disables the test: both slabs, whatever T1
        r0 = O.render(_two_slab_scene(v1, 0.0))
        assert r0["n_used"][0, 0] == 2 and abs(r0["alpha"][0, 0] - (1 - T1 * e2)) < 1e-12


def test_p32_crossing_voxel_is_included():
    """One slab whose own transmittance (0.01) is already below t_stop = 0.05: it is composited in full (R3).  A renderer
    that tests T * exp(-tau) BEFORE blending and skips the voxel returns alpha = 0 here."""
    T1 = 0.01
    cam = axis_camera(width=1, height=1)
    sc = scene(tree_from_cells([(1, 1, 1, 1)], geo=math.log(-math.log(T1) / 2.0)), cam=cam, t_stop=0.05)
    r = O.render(sc)
    assert r["n_used"][0, 0] == 1
    assert abs(r["alpha"][0, 0] - 0.99) < 1e-12 and abs(r["depth"][0, 0] - 0.99 * 6.0) < 1e-11


def test_p32_threshold_is_strict():
    """'T < eps_stop' (Alg. 1 l.8): with t_stop EXACTLY the transmittance after the first slab the ray goes
    on.  T1 is taken from a t_stop = 0 render of the first slab alone; for T1 in [1/2, 1] both 1 - T1 and 1 - (1 - T1)
    are exact in binary floating point (Sterbenz), so 1 - alpha is the T the oracle holds, bit for bit."""
    v1 = math.log(-math.log(0.6) / 2.0)
    cam = axis_camera(width=1, height=1)
    alone = O.render(scene(tree_from_cells([(1, 1, 1, 1)], geo=v1), cam=cam, t_stop=0.0))
    T1 = 1.0 - alone["alpha"][0, 0]
    assert 0.5 < T1 < 0.7
    assert O.render(_two_slab_scene(v1, T1))["n_used"][0, 0] == 2              # T1 < T1 is false: continue
    assert O.render(_two_slab_scene(v1, np.nextafter(T1, 1.0)))["n_used"][0, 0] == 1


# ---------------------------------------------------------------- P33 exp-linear derivative and the truncated tape
def _fd_check(s, g, opt, h, tol, stride=1):
    """Central differences of the loss <g, render> against the analytic gradients, every `stride`-th parameter; every
    perturbed render must composite exactly the sub-segments the base render did (n_used unchanged)."""
    r = O.render(s, grads_in=g, **opt)

    def loss():
        q = O.render(s, **opt)
        assert np.array_equal(q["n_used"], r["n_used"]), "perturbation moved a ray across the termination threshold"
        return (q["rgb"] * g["rgb"]).sum() + (q["depth"] * g["depth"]).sum() + (q["alpha"] * g["alpha"]).sum()

    worst, n_nonzero = 0.0, 0
    for n, t in enumerate(s.octrees):
        for arr, ana in ((t.geo, r["dgeo"][n]), (t.sh, r["dsh"][n])):
            flat, aflat = arr.reshape(-1), ana.reshape(-1)
            scale = max(np.abs(aflat).max(), 1e-12)
            for idx in range(0, flat.shape[0], stride):
                keep = flat[idx]
                flat[idx] = keep + h; lp = loss()
                flat[idx] = keep - h; lm = loss()
                flat[idx] = keep
                worst = max(worst, abs((lp - lm) / (2 * h) - aflat[idx]) / scale)
                n_nonzero += abs(aflat[idx]) > 1e-9 * scale
    assert worst < tol, worst
    return r, n_nonzero


def _fd_scene(seed, gain, shift):
    s = S.tiny_random_scene(seed, sh_degree=1, colour_floor=True)
    for t in s.octrees:
        t.geo = t.geo.astype(np.float64) * gain + shift
        t.sh = t.sh.astype(np.float64)
    return s


def test_p33_finite_differences_exp_linear_activation():
    """R5 option 1 (PAPER.md:107 'exponential-linear density activation'): act(x) = x above theta = 1.1, exp(x/theta - 1 +
    ln theta) below; its derivative is 1 above and act/theta below.  P6's loop with activation = 1 on raw densities spread
    over both branches.  Fails when dact forgets the 1/theta factor, uses the wrong branch, or returns act itself."""
    s = _fd_scene(7, 1.5, 1.8)
    raw = np.concatenate([t.geo.reshape(-1) for t in s.octrees])
    assert (raw > 1.3).mean() > 0.2 and (raw < 0.9).mean() > 0.2      # both branches of the activation are exercised
    g = s.image_grads(0, 1.0, 0.3, 1.0)
    r, n_nonzero = _fd_check(s, g, dict(activation=1, t_stop=0.0), 1e-5, 1e-6)
    assert n_nonzero > 100 and r["alpha"].max() > 0.5


@pytest.mark.parametrize("activation", [0, 1])
def test_p33_finite_differences_of_the_truncated_tape(activation):
    """O9 with early termination ON (the configured case, t_stop = 1e-4): the gradient of what was composited is the
    gradient of the image as long as no ray changes its stopping voxel.  Dense scene (raw shifted up) so that many rays
    terminate early; voxels behind the stopping point must get exactly zero gradient from those rays."""
    s = _fd_scene(7, 1.0, 3.2)
    g = s.image_grads(0, 1.0, 0.3, 1.0)
    full = O.render(s, t_stop=0.0, activation=activation)
    r, n_nonzero = _fd_check(s, g, dict(activation=activation, t_stop=1e-4), 1e-6, 2e-6)
    stopped = (r["n_used"] < full["n_used"])
    assert stopped.sum() >= 10, stopped.sum()                       # the truncation really fires
    assert (r["alpha"][stopped] > 1 - 1e-4).all() and n_nonzero > 60


# ---------------------------------------------------------------- P34 the T1 reference list (orc_tile_hit_list)
def _p34_scene():
    """One 16x16 tile, camera at (-5,0,0) looking down +x with the optical axis on the pixel corner (8,8): the four pixel
    quadrants are the four ray octants q = 2 (d_y<0) + (d_z<0) in {0,1,2,3} (d_x > 0 always).  Static 4 m cube centred at
    the origin, leaves given in scrambled order (ids = positions in this list):
       id 0  L1 (1,1,1)   x in [0,2],   y,z in [0,2]            seen by q = 0 only
       id 1  L2 (1,1,1)   x in [-1,0],  y,z in [-1,0]           q = 3
       id 2  L1 (0,1,0)   x in [-2,0],  y in [0,2], z in [-2,0] q = 1
       id 3  L2 (0,3,3)   x in [-2,-1], y,z in [1,2]            q = 0
       id 4  L2 (0,0,0)   x in [-2,-1], y,z in [-2,-1]          q = 3
       id 5  L1 (1,0,0)   x in [0,2],   y,z in [-2,0]           q = 3, but masked by the box except a 1.4e-5 m sliver
       id 6  L2 (1,3,2)   x in [-1,0],  y in [1,2], z in [0,1]  q = 0
       id 7  L2 (0,2,2)   x in [-2,-1], y,z in [0,1]            q = 0
       id 8  L1 (0,0,1)   x in [-2,0],  y in [-2,0], z in [0,2] q = 2
       id 9  L2 (0,1,1)   x in [-2,-1], y,z in [-1,0]           q = 3
       id 10 L2 (1,2,2)   x in [-1,0],  y,z in [0,1]            q = 0
    Actor: 4 m cube, box half 1.5, pose = translation (1.5 + 1.4e-5, -1.5, -1.5): world box x in [1.4e-5, 3.000014],
    y,z in [-3,0].  Leaves  id 0  L3 (0,3,3): local x in [-2,-1.5] -> OUTSIDE the box (R18), on the path of ray (14,14);
                            id 1  L3 (1,3,3): local x in [-1.5,-1], y,z in [-0.5,0] -> inside, world x in [0,0.5], y,z in [-2,-1.5]."""
    cells = [(1, 1, 1, 1), (1, 1, 1, 2), (0, 1, 0, 1), (0, 3, 3, 2), (0, 0, 0, 2), (1, 0, 0, 1), (1, 3, 2, 2), (0, 2, 2, 2),
             (0, 0, 1, 1), (0, 1, 1, 2), (1, 2, 2, 2)]
    st = tree_from_cells(cells, geo=-1.0, center=(0, 0, 0), side=4.0)
    act = tree_from_cells([(0, 3, 3, 3), (1, 3, 3, 3)], geo=-1.0, center=(0, 0, 0), side=4.0)
    cam = S.Camera(16, 16, 16.0, 16.0, 8.0, 8.0, S.look_yaw((-5.0, 0.0, 0.0), 0.0))
    cam.c2w = np.asarray(S.look_yaw((-5.0, 0.0, 0.0), 0.0), dtype=np.float64).reshape(12)
    pose = S.pose_yaw((1.5 + 1.4e-5, -1.5, -1.5), 0.0)
    return scene(st, [act], [pose], [[1.5, 1.5, 1.5]], cam=cam, t_stop=0.0), cells


def test_p34_tile_hit_list_hand_case():
    """T1's reference: per (tile, octree, octant) the voxels hit by a pixel of that octant with a sub-segment
    longer than 1e-5 s_l, sorted by the R14b key.  Expected lists written out by hand (see _p34_scene):
      q = 0: plain Morton order                 -> L2 (0,2,2), (0,3,3), (1,2,2), (1,3,2), then L1 (1,1,1)  = ids 7, 3, 10, 6, 0
      q = 3: y and z bits flipped in every group -> L2 (0,1,1) [group 011 -> 000], (0,0,0) [000 -> 011], (1,1,1) [111 -> 100]
                                                   = ids 9, 4, 1   (plain Morton order would give 4, 9, 1)
      id 5 is absent from q = 3: its only pieces are 1.4e-5..1.7e-5 m long, below 1e-5 * 2 m but above an absolute 1e-5.
    Fails under: a wrong octant formula (bit order), a missing or unscaled length cut, the static intervals used for the
    actor (its outside-the-box leaf would appear), an unsorted or plain-Morton-sorted list."""
    sc, cells = _p34_scene()
    want0 = {0: [7, 3, 10, 6, 0], 1: [2], 2: [8], 3: [9, 4, 1]}
    for q in range(8):
        assert O.tile_hit_list(sc, 0, 0, 0, q).tolist() == want0.get(q, []), q
        assert O.tile_hit_list(sc, 0, 0, 1, q).tolist() == ([1] if q == 3 else []), q
    # without the box, id 5 and the actor-masked part come back: the sliver cut is what removed it
    sc2 = scene(sc.static, cam=sc.cameras[0], t_stop=0.0)
    assert O.tile_hit_list(sc2, 0, 0, 0, 3).tolist() == [9, 4, 1, 5]


def test_p34_tile_hit_list_against_dense_ray_sampling():
    """The same lists from a method that shares nothing with the slab test: 40 000 points along every ray of the tile,
    point-in-box membership, masked where the point is inside the actor box (static) or outside it (actor)."""
    sc, cells = _p34_scene()
    cam = sc.cameras[0]
    ts = np.linspace(0.05, 12.0, 40001)
    dt = ts[1] - ts[0]
    hit = {(tree, q): {} for tree in (0, 1) for q in range(8)}
    bx_lo, bx_hi = np.array([1.4e-5, -3.0, -3.0]), np.array([3.0 + 1.4e-5, 0.0, 0.0])
    a_cells = [(0, 3, 3, 3), (1, 3, 3, 3)]
    for v in range(16):
        for u in range(16):
            dc = np.array([(u + 0.5 - 8.0) / 16.0, (v + 0.5 - 8.0) / 16.0, 1.0])
            d = np.array([dc[2], -dc[0], -dc[1]]) / np.linalg.norm(dc)      # R10: x right = -y_world, y down = -z_world
            q = 4 * (d[0] < 0) + 2 * (d[1] < 0) + (d[2] < 0)
            p = np.array([-5.0, 0.0, 0.0])[None] + ts[:, None] * d[None]
            in_box = np.all((p >= bx_lo) & (p <= bx_hi), axis=1)
            for tree, cl, origin in ((0, cells, np.array([-2.0, -2.0, -2.0])),
                                     (1, a_cells, np.array([-2.0, -2.0, -2.0]) + np.array([1.5 + 1.4e-5, -1.5, -1.5]))):
                for n, (i, j, k, l) in enumerate(cl):
                    s_l = 4.0 / (1 << l)
                    lo = origin + np.array([i, j, k]) * s_l
                    inside = np.all((p >= lo) & (p <= lo + s_l), axis=1) & (in_box if tree else ~in_box)
                    if inside.sum() * dt > 10 * dt:     # far above the sampling step, far above the 1e-5 s_l cut
                        hit[(tree, q)][n] = True
    for tree in (0, 1):
        codes = sc.octrees[tree].code
        for q in range(8):
            ids = sorted(hit[(tree, q)], key=lambda n: int(O.order_key([codes[n]], q)[0]))
            assert O.tile_hit_list(sc, 0, 0, tree, q).tolist() == ids, (tree, q)
