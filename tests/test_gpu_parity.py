"""GPU-vs-oracle parity through the C ABI (tolerances of BASELINE.json north_star, R16)."""
import numpy as np
import pytest

import dvx_scenes as S
from oracle import oracle as O

pytestmark = pytest.mark.gpu

RGB_TOL = 2e-4      # fp32 RGB / alpha: max abs error
DEPTH_REL = 1e-4    # depth: |dD| <= 1e-4 * max(|D_ref|, 1 m)
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
    e_d = np.abs(depth - ref["depth"]) / np.maximum(np.abs(ref["depth"]), 1.0) / DEPTH_REL
    return np.maximum(np.maximum(e_rgb, e_a), e_d)   # > 1 = out of tolerance


def _check_images(rgb, depth, alpha, ref, mask=None, scene=None):
    """Every compared pixel must be within the tolerances of R16.  A pixel may instead be *threshold-ambiguous* (DESIGN.md
    section 3): its transmittance passes within fp32 rounding of t_stop, so stopping one voxel earlier or later are both
    valid; that is established with the oracle alone (its own result changes under t_stop (1 +- 2e-3)) and the GPU result must
    then match one of the two oracle outcomes.  Returns the number of such pixels (at most 1e-4 of the sample)."""
    rgb, depth, alpha = rgb.cpu().numpy().astype(np.float64), depth.cpu().numpy().astype(np.float64), alpha.cpu().numpy().astype(np.float64)
    m = np.ones(depth.shape, bool) if mask is None else mask.astype(bool)
    err = _pixel_errors(rgb, depth, alpha, ref) * m
    bad = err > 1.0
    n_bad = int(bad.sum())
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
    """Full-size launch (the configuration bench.py times); compared on seeded whole tiles the oracle (tile-culled mode,
    pin P13) renders pixel by pixel.  Gradients: dL/dimage is zeroed outside the sample on both sides, so every gradient
    entry is compared."""
    import paper_2606_23031_b200 as dvx
    import torch
    cam = sc.cameras[0]
    mask, _ = _tile_mask(cam, n_tiles, seed)
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
        errs = _check_images(rgb, depth, alpha, ref, mask, scene=sc)
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
    return errs


def test_t2_config2_forward_sampled_tiles(ctx):
    _sampled_parity(ctx, S.make_config(2), 192, 21, backward=False)


def test_t2_t3_config3_fwd_bwd_sampled_tiles(ctx, config3):
    _sampled_parity(ctx, config3, 96, 31, backward=True)


def test_t2_t3_config4_crowded_fwd_bwd_sampled_tiles(ctx):
    sc = S.make_config(4)
    # sample tiles where boxes overlap the rays: restrict the draw to the lower-middle band where the traffic is
    _sampled_parity(ctx, sc, 96, 41, backward=True)


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
