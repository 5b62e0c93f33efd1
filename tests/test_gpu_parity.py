"""GPU-vs-oracle parity through the C ABI (tolerances of BASELINE.json north_star, R16)."""
import numpy as np
import pytest

import dvx_scenes as S
from oracle import oracle as O
from helpers import note

pytestmark = pytest.mark.gpu

RGB_TOL = 2e-4      # fp32 RGB / alpha: max abs error
DEPTH_REL = 1e-4    # depth: |dD| <= 1e-4 * max(|D_ref|, 1 m, 1 % of the pixel's mean hit distance)   (R16)
GRAD_REL, GRAD_ABS = 1e-3, 1e-6


@pytest.fixture(scope="module")
def ctx():
    import paper_2606_23031_b200 as dvx
    c = dvx.Context(0)
    yield c
    c.close()


def _pixel_errors(rgb, depth, alpha, ref):
    e_rgb = np.abs(rgb - ref["rgb"]).max(-1) / RGB_TOL
    e_a = np.abs(alpha - ref["alpha"]) / RGB_TOL
    # R16: D = sum_j T_j alpha_j mid_j is a weight-times-distance sum, so an error d_w of a weight (tolerance 2e-4 through
    # alpha) enters D as d_w x distance.  The depth tolerance is relative, 1e-4, to the larger of |D_ref|, 1 m and 1 % of the
    # pixel's mean hit distance D_ref / alpha_ref: that caps the weight error D may carry at 1e-6, 200 x below alpha's own
    # tolerance.  (Without the last term a lone 1.8 mm graze of a level-8 voxel 166 m away, alpha = 1.1e-3, D_ref = 0.18 m,
    # sits at 1.08e-4 m: the chord is exact to 12 fp32 ulps of the 1.56 m voxel edge, 6e-7 in alpha, x 166 m in D.)
    mean_dist = np.where(ref["alpha"] > 0, ref["depth"] / np.maximum(ref["alpha"], 1e-300), 0.0)
    e_d = np.abs(depth - ref["depth"]) / np.maximum(np.maximum(np.abs(ref["depth"]), 1.0), 0.01 * mean_dist) / DEPTH_REL
    return np.maximum(np.maximum(e_rgb, e_a), e_d)   # > 1 = out of tolerance


def _check_images(rgb, depth, alpha, ref, mask=None, scene=None, bad_out=None):
    """Every compared pixel must be within the tolerances of R16.  A pixel may instead be *threshold-ambiguous* (DESIGN.md
    section 3): its transmittance passes within fp32 rounding of t_stop, so stopping one voxel earlier or later are both
    valid; that is established with the oracle alone (its own result changes under t_stop (1 +- 2e-3)) and the GPU result must
    then match one of the two oracle outcomes.  Returns the number of such pixels (at most 1e-4 of the sample)."""
    rgb, depth, alpha = rgb.cpu().numpy().astype(np.float64), depth.cpu().numpy().astype(np.float64), alpha.cpu().numpy().astype(np.float64)
    m = np.ones(depth.shape, bool) if mask is None else mask.astype(bool)
    err = _pixel_errors(rgb, depth, alpha, ref) * m
    bad = err > 1.0
    n_bad = int(bad.sum())
    if bad_out is not None:
        bad_out.append(bad)
    if n_bad == 0:
        return 0
    v, u = np.unravel_index(np.argmax(err), err.shape)
    detail = "worst pixel (%d,%d): %.2f x tolerance; %d pixels out" % (u, v, err[v, u], n_bad)
    assert scene is not None and n_bad <= max(1, int(1e-4 * m.sum())), detail
    lo = O.render(scene, mode=1, mask=bad.astype(np.uint8), t_stop=scene.t_stop * (1 - 2e-3))
    hi = O.render(scene, mode=1, mask=bad.astype(np.uint8), t_stop=scene.t_stop * (1 + 2e-3))
    ambiguous = bad & (lo["n_used"] != hi["n_used"])
    assert np.array_equal(ambiguous, bad), "not a termination-threshold effect: " + detail
    e2 = np.minimum(_pixel_errors(rgb, depth, alpha, lo), _pixel_errors(rgb, depth, alpha, hi))
    assert (e2[bad] <= 1.0).all(), "threshold-ambiguous pixel matches neither outcome: " + detail
    return n_bad


def _check_grads(got, ref, what):
    got = got.cpu().numpy().astype(np.float64)
    err = np.abs(got - ref)
    bound = GRAD_REL * np.abs(ref) + GRAD_ABS
    worst = (err - bound).max() if err.size else 0.0
    assert worst <= 0, "%s: %d entries out of tolerance, worst excess %g (|ref| max %g)" % (what, int((err > bound).sum()), worst, np.abs(ref).max())
    nref = np.linalg.norm(ref)
    return np.linalg.norm(got - ref) / nref if nref > 0 else 0.0


def test_sort_pairs_matches_numpy(ctx):
    import torch
    rng = np.random.default_rng(7)
    for n, bits in ((1, 8), (33, 13), (4096, 20), (4097, 33), (100003, 46), (1 << 20, 64)):
        keys = rng.integers(0, 1 << min(bits, 63), size=n, dtype=np.uint64)
        if bits == 64:
            keys |= rng.integers(0, 2, size=n, dtype=np.uint64) << np.uint64(63)
        keys[: n // 3] = keys[n // 3: 2 * (n // 3)]  # duplicates: stability is visible in the values
        vals = np.arange(n, dtype=np.uint32)
        k = torch.from_numpy(keys.view(np.int64)).cuda()
        v = torch.from_numpy(vals.view(np.int32)).cuda()
        ctx.check(ctx.lib.dvx_sort_pairs(ctx.h, k.data_ptr(), v.data_ptr(), n, bits))
        torch.cuda.synchronize()
        order = np.argsort(keys, kind="stable")
        assert np.array_equal(k.cpu().numpy().view(np.uint64), keys[order])
        assert np.array_equal(v.cpu().numpy().view(np.uint32), vals[order])


def test_t2_t3_config1_images_and_gradients(ctx, config1):
    """Config 1: every pixel and every gradient entry against the pure brute-force oracle."""
    import paper_2606_23031_b200 as dvx
    import torch
    sc = config1
    gin = sc.image_grads(rgb_std=1e-2, depth_std=1e-3, alpha_std=1e-2)
    ref = O.render(sc, mode=0, grads_in=gin)
    dev = dvx.SceneOnDevice(ctx, sc)
    for flags in (dvx.FLAG_NAIVE, 0, dvx.FLAG_NO_RECORDS):   # debug walker; tile kernel + record replay; tile kernel + list walk
        rgb, depth, alpha, frame = dev.render(flags=flags)
        torch.cuda.synchronize()
        _check_images(rgb, depth, alpha, ref, scene=sc)
        g = [torch.from_numpy(gin[k]).cuda() for k in ("rgb", "depth", "alpha")]
        grads = frame.backward(g[0], g[1], g[2])
        torch.cuda.synchronize()
        for t in range(len(sc.octrees)):
            _check_grads(grads[t][0], ref["dgeo"][t], "dgeo[%d]" % t)
            _check_grads(grads[t][1], ref["dsh"][t], "dsh[%d]" % t)
        # accumulate semantics (R17): a second backward into the same buffers doubles them
        frame.backward(g[0], g[1], g[2], grads=grads)
        torch.cuda.synchronize()
        _check_grads(grads[0][0] * 0.5, ref["dgeo"][0], "dgeo[0] accumulated")
        frame.release()


def test_t1_config1_tile_order(ctx, config1):
    """Per-tile sorted voxel order, bit-exact: the oracle's hit list H (sorted by the R14b key) must be a subsequence of
    the library's list, and the library's list must itself ascend in the key."""
    import paper_2606_23031_b200 as dvx
    sc = config1
    dev = dvx.SceneOnDevice(ctx, sc)
    _, _, _, frame = dev.render()
    cam = sc.cameras[0]
    tw, th = (cam.width + 15) // 16, (cam.height + 15) // 16
    n_checked = 0
    for ty in range(th):
        for tx in range(tw):
            for tree in range(len(sc.octrees)):
                for q in range(8):
                    got = frame.tile_list(ty * tw + tx, tree, q)
                    if len(got):
                        keys = O.order_key(sc.octrees[tree].code[got], q)
                        assert np.all(keys[1:] > keys[:-1]), "list not strictly ascending in the R14b key"
                    want = O.tile_hit_list(sc, tx, ty, tree, q)
                    if len(want) == 0:
                        continue
                    pos = {int(v): i for i, v in enumerate(got)}
                    idx = [pos.get(int(v), -1) for v in want]
                    assert min(idx) >= 0, "tile (%d,%d) tree %d octant %d: hit voxel missing from the list" % (tx, ty, tree, q)
                    assert all(a < b for a, b in zip(idx, idx[1:]))
                    n_checked += len(want)
    assert n_checked > 1000
    frame.release()


# ----------------------------------------------------------------------------------------------- larger configs
def _tile_mask(cam, n_tiles, seed):
    tw, th = (cam.width + 15) // 16, (cam.height + 15) // 16
    rng = np.random.default_rng(seed)
    tiles = rng.choice(tw * th, size=min(n_tiles, tw * th), replace=False)
    mask = np.zeros((cam.height, cam.width), dtype=np.uint8)
    for t in tiles:
        ty, tx = divmod(int(t), tw)
        mask[ty * 16:(ty + 1) * 16, tx * 16:(tx + 1) * 16] = 1
    return mask, tiles


def _sampled_parity(ctx, sc, n_tiles, seed, backward):
    """Full-size launch (the configuration bench.py times) against the oracle in its tile-culled mode (pin P13), pixel by
    pixel: the whole frame when n_tiles is None, else seeded whole tiles.  Gradients: dL/dimage is
    zeroed outside the compared pixels on both sides, so every gradient entry is compared."""
    import paper_2606_23031_b200 as dvx
    import torch
    cam = sc.cameras[0]
    mask = np.ones((cam.height, cam.width), dtype=np.uint8) if n_tiles is None else _tile_mask(cam, n_tiles, seed)[0]
    gin = None
    if backward:
        gin = sc.image_grads(rgb_std=1e-2)
        gin["rgb"] = gin["rgb"] * mask[:, :, None].astype(np.float32)
    ref = O.render(sc, mode=1, mask=mask, grads_in=gin)
    dev = dvx.SceneOnDevice(ctx, sc)
    errs = 0
    for flags in ((0, dvx.FLAG_NO_RECORDS) if backward else (0,)):   # backward from the hit records, then by the list walk
        rgb, depth, alpha, frame = dev.render(flags=flags)
        torch.cuda.synchronize()
        bad = []
        errs = _check_images(rgb, depth, alpha, ref, mask, scene=sc, bad_out=bad)
        if backward and errs:
            # a threshold-ambiguous pixel composites one voxel more or fewer than the oracle: its gradient is the gradient of
            # the OTHER valid outcome, so it is taken out of the gradient comparison on both sides
            keep = (~bad[0]).astype(np.float32)
            gin["rgb"] = gin["rgb"] * keep[:, :, None]
            ref = O.render(sc, mode=1, mask=mask, grads_in=gin)
        if backward:
            if flags == 0:
                st = frame.record_stats()
                if st["overflowed"]:   # the context's history came from a lighter workload: this frame would fall back
                    frame.release()    # to the list walk (covered below); its count sizes the pool of the next one
                    rgb, depth, alpha, frame = dev.render(flags=flags)
                    st = frame.record_stats()
                assert st["bytes_used"] > 0 and not st["overflowed"], st
            grads = frame.backward(torch.from_numpy(gin["rgb"]).cuda())
            torch.cuda.synchronize()
            for t in range(len(sc.octrees)):
                _check_grads(grads[t][0], ref["dgeo"][t], "dgeo[%d] flags %d" % (t, flags))
                _check_grads(grads[t][1], ref["dsh"][t], "dsh[%d] flags %d" % (t, flags))
            del grads
        frame.release()
    for t in dev.trees:
        t.close()
    note("%s: %d pixels compared, %d threshold-ambiguous (DESIGN.md section 3), hits per ray %.1f%s" % (
        sc.name, int(mask.sum()), errs, float(ref["n_used"][mask.astype(bool)].mean()),
        ", all gradient entries by record replay and by list walk" if backward else ""))
    return errs


def _boxes_crossed(sc, cam_index=0, stride=1):
    """How many actor boxes each pixel's ray crosses (plain numpy slab test; selects stress tiles, nothing is compared with it)."""
    cam = sc.cameras[cam_index]
    c2w = np.asarray(cam.c2w, dtype=np.float64).reshape(3, 4)
    us, vs = np.arange(0, cam.width, stride), np.arange(0, cam.height, stride)
    x = (us[None, :] + 0.5 - cam.cx) / cam.fx + 0 * vs[:, None]
    y = (vs[:, None] + 0.5 - cam.cy) / cam.fy + 0 * us[None, :]
    d = np.stack([x, y, np.ones_like(x)], -1)
    d = (d / np.linalg.norm(d, axis=-1, keepdims=True)) @ c2w[:, :3].T
    count = np.zeros(x.shape, dtype=np.int32)
    for pose, half in zip(np.asarray(sc.poses, np.float64).reshape(-1, 3, 4), np.asarray(sc.box_half, np.float64)):
        ol = (c2w[:, 3] - pose[:, 3]) @ pose[:, :3]
        dl = d @ pose[:, :3]
        with np.errstate(divide="ignore", invalid="ignore"):
            t1, t2 = (-half - ol) / dl, (half - ol) / dl
        lo, hi = np.minimum(t1, t2).max(-1), np.maximum(t1, t2).min(-1)
        count += (hi > np.maximum(lo, cam.near))
    return count


def test_t2_config2_forward_full_frame(ctx):
    _sampled_parity(ctx, S.make_config(2), None, 21, backward=False)


def test_t2_t3_config3_fwd_bwd_full_frame(ctx, config3):
    """The headline workload, every pixel and every gradient entry (4.5 M voxels x (8 + 48) values)."""
    _sampled_parity(ctx, config3, None, 31, backward=True)


def test_t2_t3_config4_crowded_fwd_bwd_full_frame(ctx):
    """The occlusion stress case, every pixel and every gradient entry; the frame must really contain rays through >= 6
    boxes (what config 4 exists for)."""
    sc = S.make_config(4)
    crossed = _boxes_crossed(sc, stride=2)
    assert crossed.max() >= 6 and (crossed >= 1).mean() > 0.3, (crossed.max(), (crossed >= 1).mean())
    _sampled_parity(ctx, sc, None, 41, backward=True)


def test_config3_exp_linear_activation_sampled_tiles(ctx, config3):
    """R5 option 1 (PAPER.md:107 'exponential-linear density activation') at the headline size through its K = 8
    specialisation: 48 seeded tiles of config 3, forward and every gradient entry, by record replay and by list walk."""
    sc = config3
    keep = sc.activation
    sc.activation = 1
    try:
        _sampled_parity(ctx, sc, 48, 35, backward=True)
    finally:
        sc.activation = keep


def test_t1_config4_tile_order_where_boxes_stack(ctx):
    """T1 on 16 tiles of config 4 chosen where rays cross the most boxes (each holds a pixel crossing >= 6): the list of every
    (tile, octree, octant) bucket ascends in the R14b key and contains the oracle's hit list as a subsequence, bit-exact."""
    import paper_2606_23031_b200 as dvx
    sc = S.make_config(4)
    cam = sc.cameras[0]
    crossed = _boxes_crossed(sc)
    tw, th = (cam.width + 15) // 16, (cam.height + 15) // 16
    pad = np.zeros((th * 16, tw * 16), dtype=np.int32)
    pad[:cam.height, :cam.width] = crossed
    per_tile = pad.reshape(th, 16, tw, 16).max(axis=(1, 3)).reshape(-1)
    order = np.argsort(-per_tile, kind="stable")
    rng = np.random.default_rng(43)
    pool = order[per_tile[order] >= 6]
    assert len(pool) >= 16, "config 4 must hold at least 16 tiles with a ray through >= 6 boxes (has %d)" % len(pool)
    tiles = rng.choice(pool, size=16, replace=False)
    dev = dvx.SceneOnDevice(ctx, sc)
    _, _, _, frame = dev.render()
    n_checked, n_lists = 0, 0
    for tile in tiles:
        ty, tx = divmod(int(tile), tw)
        for tree in range(len(sc.octrees)):
            for q in range(8):
                got = frame.tile_list(int(tile), tree, q)
                if len(got) == 0:
                    continue
                keys = O.order_key(sc.octrees[tree].code[got], q)
                assert np.all(keys[1:] > keys[:-1])
                want = O.tile_hit_list(sc, tx, ty, tree, q)
                pos = {int(v): i for i, v in enumerate(got)}
                idx = [pos.get(int(v), -1) for v in want]
                assert len(idx) == 0 or min(idx) >= 0, "hit voxel missing from the tile list"
                assert all(a < b for a, b in zip(idx, idx[1:]))
                n_checked += len(want)
                n_lists += len(want) > 0
    assert n_checked > 2000 and n_lists >= 16 * 6, (n_checked, n_lists)   # several actor lists per tile, not only the static one
    frame.release()
    for t in dev.trees:
        t.close()


def test_config5_two_cameras_full_size_one_gradient_set(ctx):
    """BASELINE.json configs[4] at its own size: 8 M + 20 x 50 k voxels, two of the six surround cameras (front and left),
    full 1920x1080 frames, forward + backward accumulating into ONE dgeo / dsh set (R17; PAPER.md:117-119 'jointly
    optimize ... end-to-end'); every pixel and every gradient entry against the tile-culled oracle."""
    import paper_2606_23031_b200 as dvx
    import torch
    sc = S.make_config(5)
    dev = dvx.SceneOnDevice(ctx, sc)
    grads = dev.zero_grads()
    ref_dgeo = [np.zeros((t.n_voxels, 8)) for t in sc.octrees]
    ref_dsh = [np.zeros((t.n_voxels, t.n_sh, 3)) for t in sc.octrees]
    ambiguous = 0
    for c in (0, 2):
        gin = sc.image_grads(c, rgb_std=1e-2)
        ref = O.render(sc, cam_index=c, mode=1, grads_in=gin)
        rgb, depth, alpha, frame = dev.render(c)
        torch.cuda.synchronize()
        # threshold-ambiguous pixels are decided with the oracle for this camera
        sc_c = S.Scene(sc.name, sc.seed, sc.static, sc.actors, sc.poses, sc.box_half, [sc.cameras[c]], sc.k_samples, sc.activation, sc.t_stop)
        bad = []
        n_amb = _check_images(rgb, depth, alpha, ref, scene=sc_c, bad_out=bad)
        if n_amb:   # see _sampled_parity: such a pixel is taken out of the gradient comparison on both sides
            gin["rgb"] = gin["rgb"] * (~bad[0]).astype(np.float32)[:, :, None]
            ref = O.render(sc, cam_index=c, mode=1, grads_in=gin)
        ambiguous += n_amb
        frame.backward(torch.from_numpy(gin["rgb"]).cuda(), grads=grads)
        frame.release()
        for t in range(len(sc.octrees)):
            ref_dgeo[t] += ref["dgeo"][t]
            ref_dsh[t] += ref["dsh"][t]
        del ref
    torch.cuda.synchronize()
    note("config 5 (8 M + 20 x 50 k voxels), cameras 0 and 2, full frames into one gradient set: %d threshold-ambiguous pixels" % ambiguous)
    for t in range(len(sc.octrees)):
        _check_grads(grads[t][0], ref_dgeo[t], "dgeo[%d] over 2 cameras" % t)
        _check_grads(grads[t][1], ref_dsh[t], "dsh[%d] over 2 cameras" % t)
    for t in dev.trees:
        t.close()


def test_normals_and_sky_config3_sampled_tiles(ctx, config3):
    """Rows N1 at the headline size: the NRM instantiations of the tile kernel and of the replay kernel, the 14-value run
    reduction, normal_backward_kernel and the sky epilogue / prologue on config 3 (near-plane crossers, level-16 voxels,
    actors), 64 seeded tiles, forward (RGB with sky, depth, alpha, N) and backward (dgeo, dsh, dsky: every entry), with
    gradients of RGB and N (PAPER.md:297 state tuple S = (C, D, N, T), Eq. 2 :111; O10, O11)."""
    import paper_2606_23031_b200 as dvx
    import torch
    sc = config3
    cam = sc.cameras[0]
    mask, _ = _tile_mask(cam, 64, 33)
    rs = np.random.RandomState(8)
    tex = rs.uniform(0.0, 1.0, size=(32, 64, 3)).astype(np.float32)
    gin = sc.image_grads(rgb_std=1e-2)
    m3 = mask[:, :, None].astype(np.float32)
    gin["rgb"] = gin["rgb"] * m3
    idx = np.arange(cam.width * cam.height * 3, dtype=np.uint64)
    gin["normal"] = (1e-2 * S.rng.normal(sc.seed, 960, idx)).astype(np.float32).reshape(cam.height, cam.width, 3) * m3
    ref = O.render(sc, mode=1, mask=mask, grads_in=gin, sky=tex)
    mb = mask.astype(bool)
    assert np.abs(ref["normal"][mb]).max() > 0.05 and ref["dsky"].any()
    dev = dvx.SceneOnDevice(ctx, sc)
    sky = torch.from_numpy(tex).cuda()
    for flags in (0, dvx.FLAG_NO_RECORDS):
        dsky = torch.zeros_like(sky)
        rgb, depth, alpha, normal, frame = dev.render(normals=True, sky=sky, dsky=dsky, flags=flags)
        torch.cuda.synchronize()
        bad = []
        n_amb = _check_images(rgb, depth, alpha, ref, mask, scene=None, bad_out=bad)   # no ambiguity allowance here
        assert n_amb == 0
        assert np.abs(normal.cpu().numpy() - ref["normal"])[mb].max() <= RGB_TOL
        grads = frame.backward(torch.from_numpy(gin["rgb"]).cuda(), dL_dnormal=torch.from_numpy(gin["normal"]).cuda())
        torch.cuda.synchronize()
        for t in range(len(sc.octrees)):
            _check_grads(grads[t][0], ref["dgeo"][t], "dgeo[%d] normals+sky flags %d" % (t, flags))
            _check_grads(grads[t][1], ref["dsh"][t], "dsh[%d] normals+sky flags %d" % (t, flags))
        _check_grads(dsky, ref["dsky"], "dsky flags %d" % flags)
        del grads
        frame.release()
    note("config 3 normals + sky: %d pixels of 64 tiles, forward and backward, replay and list walk" % int(mask.sum()))
    for t in dev.trees:
        t.close()


def test_t1_config2_tile_order_sampled(ctx):
    """T1 on seeded tiles of config 2 (brute-force hit lists are slow: 12 tiles)."""
    import paper_2606_23031_b200 as dvx
    sc = S.make_config(2)
    dev = dvx.SceneOnDevice(ctx, sc)
    _, _, _, frame = dev.render()
    cam = sc.cameras[0]
    tw = (cam.width + 15) // 16
    _, tiles = _tile_mask(cam, 12, 51)
    n_checked = 0
    for tile in tiles:
        ty, tx = divmod(int(tile), tw)
        for tree in range(len(sc.octrees)):
            for q in range(8):
                got = frame.tile_list(int(tile), tree, q)
                if len(got) == 0:
                    continue
                keys = O.order_key(sc.octrees[tree].code[got], q)
                assert np.all(keys[1:] > keys[:-1])
                want = O.tile_hit_list(sc, tx, ty, tree, q)
                pos = {int(v): i for i, v in enumerate(got)}
                idx = [pos.get(int(v), -1) for v in want]
                assert len(idx) == 0 or min(idx) >= 0, "hit voxel missing from the tile list"
                assert all(a < b for a, b in zip(idx, idx[1:]))
                n_checked += len(want)
    assert n_checked > 100
    frame.release()


def test_t4_api_errors_and_inference_path(ctx, config1):
    import ctypes as C
    import paper_2606_23031_b200 as dvx
    import torch
    sc = config1
    dev = dvx.SceneOnDevice(ctx, sc)
    # saved = NULL path renders the same image and keeps nothing
    rgb0, d0, a0, fr = dev.render(save=True)
    rgb1, d1, a1, none = dev.render(save=False)
    torch.cuda.synchronize()
    assert none is None and torch.equal(rgb0, rgb1) and torch.equal(d0, d1) and torch.equal(a0, a1)
    # host-buffer entry points give the same bits
    rgbh, dh, ah, frh = dev.render(save=True, host=True)
    torch.cuda.synchronize()
    assert torch.equal(rgbh, rgb0.cpu()) and torch.equal(dh, d0.cpu()) and torch.equal(ah, a0.cpu())
    gin = sc.image_grads(rgb_std=1e-2)
    g_dev = torch.from_numpy(gin["rgb"]).cuda()
    ga = fr.backward(g_dev)
    gb = frh.backward(torch.from_numpy(gin["rgb"]).pin_memory(), host=True)
    torch.cuda.synchronize()
    ref = ga[0][0].abs().max().item()
    assert (ga[0][0] - gb[0][0]).abs().max().item() <= 1e-5 * ref + 1e-7   # float-atomic order is free (R17)
    fr.release(); frh.release()
    # invalid arguments -> DVX_ERR_INVALID_ARG, never a crash
    for kw in (dict(k_samples=0), dict(k_samples=9), dict(activation=2), dict(t_stop=-1.0)):
        with pytest.raises(dvx.DvxError) as e:
            dev.render(**kw)
        assert e.value.status == -1
    bad_pose = dev.poses.copy(); bad_pose[0, 0] *= 1.5
    with pytest.raises(dvx.DvxError) as e:
        ctx.render(dev.cams[0], dev.trees[0], dev.trees[1:], bad_pose, dev.box_half)
    assert e.value.status == -1
    cam = dvx.camera_from(sc.cameras[0]); cam.fx = 0.0
    with pytest.raises(dvx.DvxError):
        ctx.render(cam, dev.trees[0], dev.trees[1:], dev.poses, dev.box_half)
    # bad octrees -> DVX_ERR_BAD_OCTREE (duplicate leaf; nested leaf; bits below the level)
    t = sc.static
    code = t.code.copy(); code[1] = code[0]
    for bad in (code, np.concatenate([t.code[:4], [np.uint64((np.uint64(5) << np.uint64(48)) | (t.code[0] & np.uint64(0xFFFFFFFFFFFF) & ~np.uint64((1 << 33) - 1)))]]).astype(np.uint64)):
        n = len(bad)
        with pytest.raises(dvx.DvxError) as e:
            ctx.octree(torch.from_numpy(bad.view(np.int64)).cuda(), torch.zeros((n, 8), device="cuda"),
                       torch.zeros((n, 1, 3), device="cuda"), t.center, t.side, 0)
        assert e.value.status == -2, e.value
    # empty actor list and empty octree are legal
    empty = ctx.octree(torch.zeros(0, dtype=torch.int64, device="cuda"), torch.zeros((0, 8), device="cuda"),
                       torch.zeros((0, 1, 3), device="cuda"), (0, 0, 0), 1.0, 0)
    r, d, a, f2 = ctx.render(dev.cams[0], empty)
    torch.cuda.synchronize()
    assert float(a.abs().max()) == 0.0 and float(r.abs().max()) == 0.0
    f2.release()


def test_t1_config3_tile_order_sampled(ctx, config3):
    """T1 at the headline size: 4 seeded tiles of config 3 (the brute-force hit list costs ~10 s per tile and list)."""
    import paper_2606_23031_b200 as dvx
    sc = config3
    dev = dvx.SceneOnDevice(ctx, sc)
    _, _, _, frame = dev.render()
    cam = sc.cameras[0]
    tw = (cam.width + 15) // 16
    _, tiles = _tile_mask(cam, 4, 61)
    n_checked = 0
    for tile in tiles:
        ty, tx = divmod(int(tile), tw)
        for tree in range(len(sc.octrees)):
            for q in range(8):
                got = frame.tile_list(int(tile), tree, q)
                if len(got) == 0:
                    continue
                keys = O.order_key(sc.octrees[tree].code[got], q)
                assert np.all(keys[1:] > keys[:-1])
                want = O.tile_hit_list(sc, tx, ty, tree, q)
                pos = {int(v): i for i, v in enumerate(got)}
                idx = [pos.get(int(v), -1) for v in want]
                assert len(idx) == 0 or min(idx) >= 0, "hit voxel missing from the tile list"
                assert all(a < b for a, b in zip(idx, idx[1:]))
                n_checked += len(want)
    assert n_checked > 50
    frame.release()
    for t in dev.trees:
        t.close()


def test_multi_camera_accumulation_config5_semantics(ctx):
    """Config 5's contract at a size the oracle handles: several cameras at one ego pose render the same octrees and
    accumulate into ONE set of gradient buffers (R17); compared on seeded tiles of every camera, all gradient entries."""
    import paper_2606_23031_b200 as dvx
    import torch
    sc = S.make_config(2)
    cam0 = sc.cameras[0]
    pos = np.asarray(cam0.c2w).reshape(3, 4)[:, 3]
    sc.cameras = [S.Camera(cam0.width, cam0.height, cam0.fx, cam0.fy, cam0.cx, cam0.cy, S.look_yaw(pos, np.deg2rad(a)))
                  for a in (0.0, 45.0, -90.0)]
    dev = dvx.SceneOnDevice(ctx, sc)
    grads = dev.zero_grads()
    ref_dgeo = [np.zeros((t.n_voxels, 8)) for t in sc.octrees]
    ref_dsh = [np.zeros((t.n_voxels, t.n_sh, 3)) for t in sc.octrees]
    for c in range(len(sc.cameras)):
        mask, _ = _tile_mask(sc.cameras[c], 48, 71 + c)
        gin = sc.image_grads(c, rgb_std=1e-2)
        gin["rgb"] = gin["rgb"] * mask[:, :, None].astype(np.float32)
        ref = O.render(sc, cam_index=c, mode=1, mask=mask, grads_in=gin)
        rgb, depth, alpha, frame = dev.render(c)
        torch.cuda.synchronize()
        _check_images(rgb, depth, alpha, ref, mask, scene=None)
        frame.backward(torch.from_numpy(gin["rgb"]).cuda(), grads=grads)
        frame.release()
        for t in range(len(sc.octrees)):
            ref_dgeo[t] += ref["dgeo"][t]
            ref_dsh[t] += ref["dsh"][t]
    torch.cuda.synchronize()
    for t in range(len(sc.octrees)):
        _check_grads(grads[t][0], ref_dgeo[t], "dgeo[%d] over 3 cameras" % t)
        _check_grads(grads[t][1], ref_dsh[t], "dsh[%d] over 3 cameras" % t)


def test_key_generation_ahead_of_the_pair_count_is_repeated_when_it_did_not_fit(config1):
    """Step 2's key generation is enqueued before the host knows the frame's pair count, with a capacity taken from the
    context's recent frames (include/dvx.h, "one host round trip").  A context that has only seen a tiny scene guesses far too
    small for config 2: the frame must repeat the key generation at the true size and come out bit-identical to the same
    frame rendered by a context with no history (which sizes from the count) and by one with the right history."""
    import paper_2606_23031_b200 as dvx
    import torch
    big = S.make_config(2)
    fresh = dvx.Context(0)
    dev_f = dvx.SceneOnDevice(fresh, big)
    ref = dev_f.render()                       # no history: sized from the count
    ref2 = dev_f.render()                      # history = this frame: the guess fits
    torch.cuda.synchronize()
    pairs_ref = ref[3].counters()["pairs"]
    lists_ref = [ref[3].tile_list(t, 0, q) for t in (5, 700, 1500) for q in range(8)]
    small_ctx = dvx.Context(0)
    dev_s = dvx.SceneOnDevice(small_ctx, config1)
    for _ in range(3):
        dev_s.render()[3].release()            # history: a few thousand pairs
    pairs_small = dev_s.render()
    n_small = pairs_small[3].counters()["pairs"]
    pairs_small[3].release()
    dev_b = dvx.SceneOnDevice(small_ctx, big)
    got = dev_b.render()                       # the guess (1.25 x a few thousand) cannot hold config 2's pairs
    torch.cuda.synchronize()
    assert pairs_ref > 8 * (n_small + n_small // 4 + 4096), (pairs_ref, n_small)
    assert got[3].counters()["pairs"] == pairs_ref
    for a, b, c in zip(ref[:3], ref2[:3], got[:3]):
        assert torch.equal(a, b) and torch.equal(a, c)
    lists_got = [got[3].tile_list(t, 0, q) for t in (5, 700, 1500) for q in range(8)]
    assert sum(len(x) for x in lists_ref) > 0
    for a, b in zip(lists_ref, lists_got):
        assert np.array_equal(a, b)
    for fr in (ref[3], ref2[3], got[3]):
        fr.release()
    fresh.close()
    small_ctx.close()


@pytest.mark.parametrize("cfg", [2, 4])
def test_forward_is_bit_deterministic(ctx, cfg):
    """The forward has no atomics: two renders of the same frame must agree bit for bit (a data race between the phases of
    the tile kernel, or an unstable sort, would show up here), and the backward twice must agree to float-atomic noise."""
    import paper_2606_23031_b200 as dvx
    import torch
    sc = S.make_config(cfg)
    dev = dvx.SceneOnDevice(ctx, sc)
    a = dev.render(normals=True)
    b = dev.render(normals=True)
    torch.cuda.synchronize()
    for x, y in zip(a[:4], b[:4]):
        assert torch.equal(x, y)
    cam = sc.cameras[0]
    tw = (cam.width + 15) // 16
    for tile in (0, tw * 20 + 31, tw * 33 + 7):
        for tree in range(min(len(sc.octrees), 3)):
            for q in range(8):
                assert np.array_equal(a[4].tile_list(tile, tree, q), b[4].tile_list(tile, tree, q))
    g = torch.from_numpy(sc.image_grads(rgb_std=1e-2)["rgb"]).cuda()
    ga, gb = a[4].backward(g), b[4].backward(g)
    torch.cuda.synchronize()
    for t in range(len(sc.octrees)):
        ref = ga[t][0].abs().max().item()
        assert (ga[t][0] - gb[t][0]).abs().max().item() <= 1e-5 * ref + 1e-9
    a[4].release(); b[4].release()
    for t in dev.trees:
        t.close()


def test_render_batch_and_backward_batch_match_the_sequential_calls(ctx):
    """dvx_render_batch / dvx_backward_batch (include/dvx.h; config 5's schedule: one host round trip for all cameras, step 2
    and the SH post-pass on the second stream) against one dvx_render / dvx_backward per camera: images bit-identical, the
    shared gradient set equal up to float summation order; twice in a row (the scratch cache is shared by both streams)."""
    import paper_2606_23031_b200 as dvx
    import torch
    sc = S.make_config(2)
    cam0 = sc.cameras[0]
    pos = np.asarray(cam0.c2w).reshape(3, 4)[:, 3]
    sc.cameras = [S.Camera(cam0.width, cam0.height, cam0.fx, cam0.fy, cam0.cx, cam0.cy, S.look_yaw(pos, np.deg2rad(a)))
                  for a in (0.0, 45.0, -90.0, 180.0)]
    dev = dvx.SceneOnDevice(ctx, sc)
    g = [torch.from_numpy(sc.image_grads(c, rgb_std=1e-2)["rgb"]).cuda() for c in range(len(sc.cameras))]
    seq_imgs, seq_grads = [], dev.zero_grads()
    for c in range(len(sc.cameras)):
        rgb, depth, alpha, fr = dev.render(c)
        seq_imgs.append((rgb.clone(), depth.clone(), alpha.clone()))
        fr.backward(g[c], grads=seq_grads)
        fr.release()
    torch.cuda.synchronize()
    for rep in range(2):
        grads = dev.zero_grads()
        outs, frames = dev.render_batch()
        ctx.backward_batch(frames, g, grads)
        for fr in frames:
            fr.release()
        torch.cuda.synchronize()
        for c in range(len(sc.cameras)):
            for a, b in zip(outs[c], seq_imgs[c]):
                assert torch.equal(a, b), "camera %d, repetition %d" % (c, rep)
        for t in range(len(sc.octrees)):
            for k in (0, 1):
                scale = seq_grads[t][k].abs().max().item()
                assert (grads[t][k] - seq_grads[t][k]).abs().max().item() <= 2e-5 * scale + 1e-9, (t, k, rep)
    # inference: nothing saved
    outs2, none = dev.render_batch(save=False)
    torch.cuda.synchronize()
    assert none is None and all(torch.equal(a[0], b[0]) for a, b in zip(outs2, seq_imgs))
    for t in dev.trees:
        t.close()
