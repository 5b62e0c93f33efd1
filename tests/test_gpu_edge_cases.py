"""GPU-vs-oracle parity on the degenerate and edge cases of the method (through the C ABI, brute-force oracle, every pixel
and every gradient entry): other K / activation / t_stop than the configured ones, axis-parallel rays (R20), a static voxel
cut into two pieces by a box (R1), overlapping boxes (R2), the camera inside a box (R11), empty octrees and actor lists,
ragged and single-pixel images (R15)."""
import numpy as np
import pytest

import dvx_scenes as S
from oracle import oracle as O
from helpers import tree_from_cells, empty_tree, scene, axis_camera
from dvx_scenes.octree import C0

pytestmark = pytest.mark.gpu

RGB_TOL, DEPTH_REL, GRAD_REL, GRAD_ABS = 2e-4, 1e-4, 1e-3, 1e-6


@pytest.fixture(scope="module")
def ctx():
    import paper_2606_23031_b200 as dvx
    c = dvx.Context(0)
    yield c
    c.close()


def _round_to_f32(sc):
    """The library takes fp32 inputs: make every input exactly fp32-representable so both sides see the same numbers."""
    for t in sc.octrees:
        t.geo = np.ascontiguousarray(t.geo, dtype=np.float32)
        t.sh = np.ascontiguousarray(t.sh, dtype=np.float32)
        t.center = np.asarray(t.center, dtype=np.float32).astype(np.float64)
        t.side = float(np.float32(t.side))
    sc.poses = np.ascontiguousarray(sc.poses, dtype=np.float32)
    sc.box_half = np.ascontiguousarray(sc.box_half, dtype=np.float32)
    for cam in sc.cameras:
        cam.c2w = np.asarray(cam.c2w, dtype=np.float32).reshape(12)
        for k in ("fx", "fy", "cx", "cy", "near", "far"):
            setattr(cam, k, float(np.float32(getattr(cam, k))))
    return sc


def _compare(ctx, sc, backward=True, **opt):
    import paper_2606_23031_b200 as dvx
    import torch
    _round_to_f32(sc)
    for k, v in opt.items():
        setattr(sc, k, v)
    cam = sc.cameras[0]
    gin = sc.image_grads(rgb_std=1e-2, depth_std=1e-3, alpha_std=1e-2) if backward else None
    ref = O.render(sc, mode=0, grads_in=gin)
    dev = dvx.SceneOnDevice(ctx, sc)
    for flags in (0, dvx.FLAG_NAIVE):
        rgb, depth, alpha, frame = dev.render(flags=flags)
        torch.cuda.synchronize()
        r, d, a = (x.cpu().numpy().astype(np.float64) for x in (rgb, depth, alpha))
        assert np.abs(r - ref["rgb"]).max() <= RGB_TOL, (flags, np.abs(r - ref["rgb"]).max())
        assert np.abs(a - ref["alpha"]).max() <= RGB_TOL, (flags, np.abs(a - ref["alpha"]).max())
        e_d = (np.abs(d - ref["depth"]) / np.maximum(np.abs(ref["depth"]), 1.0)).max()
        assert e_d <= DEPTH_REL, (flags, e_d)
        if backward:
            g = [None if gin[k] is None else torch.from_numpy(gin[k]).cuda() for k in ("rgb", "depth", "alpha")]
            grads = frame.backward(g[0], g[1], g[2])
            torch.cuda.synchronize()
            for t in range(len(sc.octrees)):
                for got, want, name in ((grads[t][0], ref["dgeo"][t], "dgeo"), (grads[t][1], ref["dsh"][t], "dsh")):
                    err = np.abs(got.cpu().numpy().astype(np.float64) - want)
                    bound = GRAD_REL * np.abs(want) + GRAD_ABS
                    assert (err <= bound).all(), "%s[%d] flags %d: worst excess %g" % (name, t, flags, (err - bound).max())
        frame.release()
    for t in dev.trees:
        t.close()
    return ref


@pytest.mark.parametrize("seed,K,act,t_stop", [(3, 8, 0, 0.0), (5, 1, 0, 1e-4), (7, 3, 0, 1e-4), (11, 5, 1, 0.0), (13, 8, 1, 1e-4),
                                               (17, 2, 0, 0.05)])
def test_random_tiny_scenes_other_options(ctx, seed, K, act, t_stop):
    """K != 8 and the exp-linear activation take the generic quadrature path of the kernels; a large t_stop makes most rays
    terminate early (R3)."""
    sc = S.tiny_random_scene(seed, sh_degree=1, width=24, height=20)
    _compare(ctx, sc, k_samples=K, activation=act, t_stop=t_stop)


def _cube8(geo, side=2.0, sh=None):
    cells = [(i, j, k, 1) for i in (0, 1) for j in (0, 1) for k in (0, 1)]
    return tree_from_cells(cells, geo=geo, side=side, sh=sh)


def test_axis_parallel_rays_and_two_slabs(ctx):
    """The centre pixel's ray is exactly the +x axis (two zero direction components, R20); static + actor voxel on the axis."""
    cam = axis_camera(width=9, height=7)
    sh1 = np.full((1, 1, 3), (0.8 - 0.5) / C0); sh2 = np.full((1, 1, 3), (0.3 - 0.5) / C0)
    st = tree_from_cells([(1, 1, 1, 1)], geo=-0.5, sh=sh1)
    act = tree_from_cells([(1, 1, 1, 1)], geo=0.25, sh=sh2, side=1.0)
    for x_act in (4.0, -3.0):
        pose = S.pose_yaw((x_act, 0.75, 0.75), 0.0)
        ref = _compare(ctx, scene(st, [act], [pose], [[0.625, 0.625, 0.625]], cam=cam))
        assert ref["alpha"][3, 4] > 0.5


def test_box_inside_a_voxel_gives_two_pieces(ctx):
    """R1: one large static voxel, an empty actor box strictly inside it: the voxel is composited as two clipped pieces."""
    cam = axis_camera(width=9, height=7)
    st = tree_from_cells([(1, 1, 1, 1)], geo=-0.25)
    pose = S.pose_yaw((1.0, 1.0, 1.0), 0.0)
    ref = _compare(ctx, scene(st, [empty_tree()], [pose], [[0.375, 0.25, 0.25]], cam=cam))
    assert ref["n_used"][3, 4] == 2


def test_overlapping_boxes_rule_r2(ctx):
    cam = axis_camera(width=9, height=7)
    act = _cube8(0.0)
    pa, pb = S.pose_yaw((0.0, 1.0, 1.0), 0.0), S.pose_yaw((1.0, 1.0, 1.0), 0.0)   # boxes overlap on x in [0,1]
    st = tree_from_cells([(0, 0, 0, 1), (1, 1, 1, 1)], geo=-1.0, side=8.0)
    _compare(ctx, scene(st, [act, act], [pa, pb], [[1, 1, 1], [1, 1, 1]], cam=cam))


def test_camera_inside_an_actor_box(ctx):
    """R11: everything is clipped at `near`; tau_in of the enclosing box is negative."""
    cam = axis_camera(position=(0.25, 1.0, 1.0), width=9, height=7)
    act = _cube8(np.linspace(-1.0, 0.5, 64).reshape(8, 8))
    pose = S.pose_yaw((0.5, 1.0, 1.0), 0.3)
    st = tree_from_cells([(1, 1, 1, 1), (1, 0, 1, 1)], geo=-0.5, side=16.0, center=(4.0, 0.0, 0.0))
    _compare(ctx, scene(st, [act], [pose], [[1, 1, 1]], cam=cam))


@pytest.mark.parametrize("w,h", [(1, 1), (17, 33), (40, 16)])
def test_ragged_and_single_pixel_images(ctx, w, h):
    sc = S.tiny_random_scene(23, sh_degree=1, width=w, height=h)
    _compare(ctx, sc)


def test_no_actors_and_empty_trees(ctx):
    sc = S.tiny_random_scene(29, sh_degree=1, width=16, height=12)
    only_static = scene(sc.static, [], [], [], cam=sc.cameras[0], t_stop=0.0)
    _compare(ctx, only_static)
    empty_static = scene(empty_tree(sh_degree=1, side=8.0), sc.actors, sc.poses, sc.box_half, cam=sc.cameras[0], t_stop=0.0)
    _compare(ctx, empty_static)
    empty_actor = scene(sc.static, [empty_tree(sh_degree=1)], sc.poses, sc.box_half, cam=sc.cameras[0], t_stop=0.0)
    _compare(ctx, empty_actor)


def test_sh_degrees_0_2_3(ctx):
    for deg in (0, 2, 3):
        _compare(ctx, S.tiny_random_scene(31 + deg, sh_degree=deg, width=16, height=12))


def _sky_map(h, w, seed):
    idx = np.arange(h * w * 3, dtype=np.uint64)
    return S.rng.uniform(seed, 950, idx).astype(np.float32).reshape(h, w, 3)


@pytest.mark.parametrize("seed,hw", [(41, (16, 32)), (43, (5, 9)), (47, (1, 1))])
def test_sky_composite_eq2(ctx, seed, hw):
    """Eq. 2 (reading R21): C = C_voxels + T_final C_sky through both kernels, and the backward's texture,
    density and SH gradients, against the oracle; depth and alpha must not change when the sky is switched on."""
    import paper_2606_23031_b200 as dvx
    import torch
    sc = _round_to_f32(S.tiny_random_scene(seed, sh_degree=1, width=40, height=24))
    tex = _sky_map(hw[0], hw[1], seed)
    gin = sc.image_grads(rgb_std=1e-2, depth_std=1e-3, alpha_std=1e-2)
    ref = O.render(sc, mode=0, grads_in=gin, sky=tex)
    assert np.abs(ref["dsky"]).max() > 0
    dev = dvx.SceneOnDevice(ctx, sc)
    tex_d = torch.from_numpy(tex).cuda()
    for flags in (0, dvx.FLAG_NAIVE):
        dsky = torch.zeros_like(tex_d)
        rgb, depth, alpha, frame = dev.render(flags=flags, sky=tex_d, dsky=dsky)
        rgb0, depth0, alpha0, _ = dev.render(flags=flags, save=False)
        torch.cuda.synchronize()
        assert torch.equal(depth, depth0) and torch.equal(alpha, alpha0)
        assert np.abs(rgb.cpu().numpy() - ref["rgb"]).max() <= RGB_TOL
        assert np.abs(alpha.cpu().numpy() - ref["alpha"]).max() <= RGB_TOL
        g = [torch.from_numpy(gin[k]).cuda() for k in ("rgb", "depth", "alpha")]
        grads = frame.backward(g[0], g[1], g[2])
        torch.cuda.synchronize()
        pairs = [(dsky, ref["dsky"], "dsky")]
        for t in range(len(sc.octrees)):
            pairs += [(grads[t][0], ref["dgeo"][t], "dgeo[%d]" % t), (grads[t][1], ref["dsh"][t], "dsh[%d]" % t)]
        for got, want, name in pairs:
            err = np.abs(got.cpu().numpy().astype(np.float64) - want)
            bound = GRAD_REL * np.abs(want) + GRAD_ABS
            assert (err <= bound).all(), "%s flags %d: worst excess %g" % (name, flags, (err - bound).max())
        frame.release()


def test_sky_on_config1_and_empty_scene(ctx, config1):
    """An empty scene renders the sky map itself (T_final = 1); config 1 with a sky at full tile coverage."""
    import paper_2606_23031_b200 as dvx
    import torch
    tex = _sky_map(32, 64, 3)
    tex_d = torch.from_numpy(tex).cuda()
    sc = config1
    dev = dvx.SceneOnDevice(ctx, sc)
    rgb, _, _, _ = dev.render(save=False, sky=tex_d)
    torch.cuda.synchronize()
    assert np.abs(rgb.cpu().numpy() - O.render(sc, mode=0, sky=tex)["rgb"]).max() <= RGB_TOL
    empty = ctx.octree(torch.zeros(0, dtype=torch.int64, device="cuda"), torch.zeros((0, 8), device="cuda"),
                       torch.zeros((0, 1, 3), device="cuda"), (0, 0, 0), 1.0, 0)
    r, d, a, _ = ctx.render(dev.cams[0], empty, save=False, sky=tex_d)
    torch.cuda.synchronize()
    es = scene(empty_tree(), cam=sc.cameras[0])
    assert np.abs(r.cpu().numpy() - O.render(es, sky=tex)["rgb"]).max() <= 1e-5 and float(a.abs().max()) == 0.0


@pytest.mark.parametrize("seed,t_stop", [(51, 0.0), (53, 1e-4), (57, 0.05)])
def test_normal_map_o11(ctx, seed, t_stop):
    """O11 / R22: N = sum T alpha n (world frame) and its backward (through the weights and through the voxel normals),
    every pixel and every gradient entry against the oracle; the other outputs must not change when normals are on."""
    import paper_2606_23031_b200 as dvx
    import torch
    sc = _round_to_f32(S.tiny_random_scene(seed, sh_degree=1, width=40, height=24))
    sc.t_stop = t_stop
    gin = sc.image_grads(rgb_std=1e-2, depth_std=1e-3, alpha_std=1e-2)
    idx = np.arange(40 * 24 * 3, dtype=np.uint64)
    gin["normal"] = (1e-2 * S.rng.normal(seed, 960, idx)).astype(np.float32).reshape(24, 40, 3)
    ref = O.render(sc, mode=0, grads_in=gin)
    assert np.abs(ref["normal"]).max() > 0.05
    dev = dvx.SceneOnDevice(ctx, sc)
    rgb, depth, alpha, normal, frame = dev.render(normals=True)
    rgb0, depth0, alpha0, _ = dev.render(save=False)
    torch.cuda.synchronize()
    assert torch.equal(rgb, rgb0) and torch.equal(depth, depth0) and torch.equal(alpha, alpha0)
    assert np.abs(normal.cpu().numpy() - ref["normal"]).max() <= RGB_TOL
    assert np.abs(rgb.cpu().numpy() - ref["rgb"]).max() <= RGB_TOL
    g = {k: torch.from_numpy(v).cuda() for k, v in gin.items()}
    grads = frame.backward(g["rgb"], g["depth"], g["alpha"], dL_dnormal=g["normal"])
    torch.cuda.synchronize()
    for t in range(len(sc.octrees)):
        for got, want, name in ((grads[t][0], ref["dgeo"][t], "dgeo"), (grads[t][1], ref["dsh"][t], "dsh")):
            err = np.abs(got.cpu().numpy().astype(np.float64) - want)
            bound = GRAD_REL * np.abs(want) + GRAD_ABS
            assert (err <= bound).all(), "%s[%d]: worst excess %g" % (name, t, (err - bound).max())
    # a frame rendered without normals refuses a normal gradient
    _, _, _, f2 = dev.render()
    with pytest.raises(dvx.DvxError):
        f2.backward(g["rgb"], dL_dnormal=g["normal"])
    f2.release()
    frame.release()


def test_normal_map_on_config1_with_sky(ctx, config1):
    import paper_2606_23031_b200 as dvx
    import torch
    sc = config1
    tex = _sky_map(8, 16, 5)
    ref = O.render(sc, mode=0, sky=tex, normals=True)
    dev = dvx.SceneOnDevice(ctx, sc)
    rgb, depth, alpha, normal, _ = dev.render(save=False, normals=True, sky=torch.from_numpy(tex).cuda())
    torch.cuda.synchronize()
    assert np.abs(normal.cpu().numpy() - ref["normal"]).max() <= RGB_TOL
    assert np.abs(rgb.cpu().numpy() - ref["rgb"]).max() <= RGB_TOL


def test_refresh_structure_and_max_actors(ctx):
    """dvx_octree_refresh_structure after the leaf set changed = a freshly created handle; 64 actors (DVX_MAX_ACTORS) render
    like the oracle, 65 are refused."""
    import ctypes as C
    import paper_2606_23031_b200 as dvx
    import torch
    sc = _round_to_f32(S.tiny_random_scene(61, sh_degree=1, width=24, height=16))
    other = _round_to_f32(S.tiny_random_scene(67, sh_degree=1, width=24, height=16))
    dev = dvx.SceneOnDevice(ctx, sc)
    # swap the static tree's arrays for those of another scene through refresh_structure
    t0, new = dev.trees[0], other.static
    code = torch.from_numpy(np.ascontiguousarray(new.code).view(np.int64)).cuda()
    geo = torch.from_numpy(np.ascontiguousarray(new.geo, dtype=np.float32)).cuda()
    sh = torch.from_numpy(np.ascontiguousarray(new.sh, dtype=np.float32)).cuda()
    desc = dvx.binding.OctreeDesc(new.n_voxels, new.sh_degree, (C.c_float * 3)(*[float(x) for x in new.center]), float(new.side),
                                  code.data_ptr(), geo.data_ptr(), sh.data_ptr())
    ctx.check(ctx.lib.dvx_octree_refresh_structure(ctx.h, t0.h, C.byref(desc)))
    t0.code, t0.geo, t0.sh, t0.n_voxels = code, geo, sh, new.n_voxels
    rgb, depth, alpha, _ = dev.render(save=False)
    torch.cuda.synchronize()
    mixed = scene(new, sc.actors, sc.poses, sc.box_half, cam=sc.cameras[0], t_stop=sc.t_stop)
    ref = O.render(mixed, mode=0)
    assert np.abs(rgb.cpu().numpy() - ref["rgb"]).max() <= RGB_TOL and np.abs(alpha.cpu().numpy() - ref["alpha"]).max() <= RGB_TOL
    # 64 actors: one single-voxel actor replicated on a grid in front of the camera
    act = tree_from_cells([(0, 0, 0, 1), (1, 1, 1, 1)], geo=np.linspace(-1, 1, 16).reshape(2, 8), side=0.5)
    poses, halves = [], []
    for n in range(64):
        poses.append(S.pose_yaw((1.0 + 0.7 * (n // 8), -2.5 + 0.7 * (n % 8), 0.2 * ((n * 7) % 5)), 0.1 * n))
        halves.append([0.25, 0.25, 0.25])
    many = _round_to_f32(scene(sc.static, [act] * 64, poses, halves, cam=sc.cameras[0], t_stop=0.0))
    dev2 = dvx.SceneOnDevice(ctx, many)
    rgb, depth, alpha, _ = dev2.render(save=False)
    torch.cuda.synchronize()
    ref = O.render(many, mode=0)
    assert np.abs(rgb.cpu().numpy() - ref["rgb"]).max() <= RGB_TOL
    assert (np.abs(depth.cpu().numpy() - ref["depth"]) / np.maximum(np.abs(ref["depth"]), 1.0)).max() <= DEPTH_REL
    with pytest.raises(dvx.DvxError) as e:
        ctx.render(dev2.cams[0], dev2.trees[0], dev2.trees[1:] + [dev2.trees[1]], np.concatenate([dev2.poses, dev2.poses[:1]]),
                   np.concatenate([dev2.box_half, dev2.box_half[:1]]))
    assert e.value.status == -1


def test_unaligned_gradient_buffers_are_rejected_and_trim_frees_the_cache(ctx):
    """red.global.add.v4.f32 and the float4 read-modify-writes of the SH / normal post-passes fault on gradient
    pointers that are not 16-byte aligned -> DVX_ERR_INVALID_ARG instead.  dvx_trim returns the scratch cache to the
    allocator; the next frame renders the same image."""
    import paper_2606_23031_b200 as dvx
    import torch
    sc = S.tiny_random_scene(3, sh_degree=1, width=40, height=24)
    dev = dvx.SceneOnDevice(ctx, sc)
    rgb0, _, _, fr = dev.render()
    g = torch.from_numpy(sc.image_grads(0, 1e-2)["rgb"]).cuda()
    good = dev.zero_grads()
    for which in (0, 1):
        bad = [list(x) for x in good]
        t = dev.trees[0]
        shape = (t.n_voxels, 8) if which == 0 else (t.n_voxels, t.n_sh, 3)
        numel = int(np.prod(shape))
        bad[0][which] = torch.zeros(numel + 1, device="cuda")[1:].view(shape)      # 4 bytes off a 16-byte boundary
        assert bad[0][which].data_ptr() % 16 == 4
        with pytest.raises(dvx.DvxError) as e:
            fr.backward(g, grads=[tuple(x) for x in bad])
        assert e.value.status == -1
    fr.backward(g, grads=good)
    torch.cuda.synchronize()
    assert float(good[0][0].abs().max()) > 0
    fr.release()
    freed = ctx.trim()
    assert freed > 0 and ctx.trim() == 0
    rgb1, _, _, fr = dev.render()
    torch.cuda.synchronize()
    assert torch.equal(rgb0, rgb1)
    fr.release()
