"""Row N3 through the C ABI against the oracle's feature pass O12: compositing weights, feature render
(F = W feat) and feature fusion (num += W^T img), config 1 in full and config 3 on sampled tiles at full size."""
import numpy as np
import pytest

import dvx_scenes as S
from oracle import oracle as O

pytestmark = pytest.mark.gpu

FEAT_TOL = 2e-4      # features in [-1, 1]: the RGB tolerance of R16
FUSE_REL, FUSE_ABS = 1e-3, 1e-6   # like the gradients (float atomics, many terms)


@pytest.fixture(scope="module")
def ctx():
    import paper_2606_23031_b200 as dvx
    c = dvx.Context(0)
    yield c
    c.close()


def _features(scene, n_ch, seed):
    rs = np.random.RandomState(seed)
    return [rs.uniform(-1.0, 1.0, size=(t.n_voxels, n_ch)).astype(np.float32) for t in scene.octrees]


def _cat(arrs):
    import torch
    return torch.from_numpy(np.ascontiguousarray(np.concatenate(arrs, axis=0))).cuda()


def _tile_mask(cam, n_tiles, seed):
    tw, th = (cam.width + 15) // 16, (cam.height + 15) // 16
    rng = np.random.default_rng(seed)
    tiles = rng.choice(tw * th, size=min(n_tiles, tw * th), replace=False)
    mask = np.zeros((cam.height, cam.width), dtype=np.uint8)
    for t in tiles:
        ty, tx = divmod(int(t), tw)
        mask[ty * 16:(ty + 1) * 16, tx * 16:(tx + 1) * 16] = 1
    return mask


def _check_fuse(got, ref, scale, what):
    got = got.astype(np.float64)
    err = np.abs(got - ref)
    bound = FUSE_REL * np.abs(ref) + FUSE_ABS * scale
    assert (err <= bound).all(), "%s: %d entries out, worst excess %g" % (what, int((err > bound).sum()), (err - bound).max())


def test_weights_rows_sum_to_alpha(ctx, config1):
    import torch
    import paper_2606_23031_b200 as dvx
    dev = dvx.SceneOnDevice(ctx, config1)
    rgb, depth, alpha, frame = dev.render()
    nnz, rows, vox, w = frame.weights()
    torch.cuda.synchronize()
    H, W = alpha.shape
    rows = rows[:H * W + 1].cpu().numpy().astype(np.int64)
    assert rows[0] == 0 and rows[-1] == nnz and (np.diff(rows) >= 0).all()
    ref = O.render(config1, mode=0)
    # composited sub-segments per ray: equal except where a grazing hit of ~zero length (weight ~0) is decided differently
    # in fp32 and fp64 - what is unique is the sum of the weights, checked below
    d = np.abs(np.diff(rows).reshape(H, W) - ref["n_used"].astype(np.int64))
    from helpers import note
    note("config 1 weight rows: n_used differs from the oracle on %.5f of the pixels (largest difference %d)" % (float((d != 0).mean()), int(d.max())))
    # observed 2.6 % on B200 (config 1 is an axis-aligned uniform 1 m grid seen from a camera standing on its lattice planes:
    # zero-length grazing hits are common); bound = twice the observation
    assert (d != 0).mean() <= 0.052, (int(d.max()), float((d != 0).mean()))
    v_total = sum(t.n_voxels for t in config1.octrees)
    assert int(vox.max()) < v_total and float(w.min()) >= 0.0
    sums = np.add.reduceat(np.concatenate([w.cpu().numpy().astype(np.float64), [0.0]]), np.minimum(rows[:-1], nnz))
    sums[np.diff(rows) == 0] = 0.0
    assert np.abs(sums.reshape(H, W) - ref["alpha"]).max() <= 2e-4           # the weights telescope to 1 - T_final
    # a second call returns the cached matrix
    nnz2, rows2, vox2, w2 = frame.weights()
    assert nnz2 == nnz and w2.data_ptr() == w.data_ptr()
    frame.release()


@pytest.mark.parametrize("n_ch", [1, 5, 8, 64, 132, 512])
def test_feature_render_config1_all_pixels(ctx, config1, n_ch):
    import torch
    import paper_2606_23031_b200 as dvx
    sc = config1
    feats = _features(sc, n_ch, 100 + n_ch)
    dev = dvx.SceneOnDevice(ctx, sc)
    rgb, depth, alpha, frame = dev.render()
    H, W = alpha.shape
    F = frame.render_features(_cat(feats), H, W)
    torch.cuda.synchronize()
    ref = O.render_features(sc, feats=feats, mode=0)
    assert np.abs(ref["features"]).max() > 0.1
    err = np.abs(F.cpu().numpy().astype(np.float64) - ref["features"]).max()
    assert err <= FEAT_TOL, err
    frame.release()


@pytest.mark.parametrize("n_ch", [3, 16, 64])
def test_feature_fuse_config1(ctx, config1, n_ch):
    import torch
    import paper_2606_23031_b200 as dvx
    sc = config1
    cam = sc.cameras[0]
    rs = np.random.RandomState(n_ch)
    img = rs.uniform(-1.0, 1.0, size=(cam.height, cam.width, n_ch)).astype(np.float32)
    dev = dvx.SceneOnDevice(ctx, sc)
    _, _, _, frame = dev.render()
    v_total = sum(t.n_voxels for t in sc.octrees)
    num = torch.zeros((v_total, n_ch), device="cuda")
    wsum = torch.zeros(v_total, device="cuda")
    frame.fuse_features(torch.from_numpy(img).cuda(), num, wsum)
    torch.cuda.synchronize()
    ref = O.render_features(sc, img=img, mode=0)
    ref_num, ref_w = np.concatenate(ref["num"], axis=0), np.concatenate(ref["wsum"])
    assert ref_w.max() > 1.0
    _check_fuse(wsum.cpu().numpy(), ref_w, ref_w.max(), "wsum")
    _check_fuse(num.cpu().numpy(), ref_num, ref_w.max(), "num")
    # accumulate semantics; wsum optional
    frame.fuse_features(torch.from_numpy(img).cuda(), num, None)
    torch.cuda.synchronize()
    _check_fuse(num.cpu().numpy() * 0.5, ref_num, ref_w.max(), "num accumulated")
    _check_fuse(wsum.cpu().numpy(), ref_w, ref_w.max(), "wsum untouched")
    # fuse is the transpose of render, on the device alone
    feats = _features(sc, n_ch, 7)
    F = frame.render_features(_cat(feats), cam.height, cam.width)
    num1 = torch.zeros((v_total, n_ch), device="cuda")
    frame.fuse_features(torch.from_numpy(img).cuda(), num1)
    lhs = float((F.double() * torch.from_numpy(img).cuda().double()).sum())
    rhs = float((_cat(feats).double() * num1.double()).sum())
    assert abs(lhs - rhs) <= 1e-4 * max(1.0, abs(lhs))
    frame.release()


def test_feature_render_and_fuse_config3_sampled_tiles(ctx, config3):
    """Full-size launch (1920x1080, 4.5 M voxels, C = 64), compared on seeded whole tiles the tile-culled oracle renders."""
    import torch
    import paper_2606_23031_b200 as dvx
    sc = config3
    cam = sc.cameras[0]
    n_ch = 64
    mask = _tile_mask(cam, 64, 91)
    feats = _features(sc, n_ch, 5)
    rs = np.random.RandomState(6)
    img = rs.uniform(-1.0, 1.0, size=(cam.height, cam.width, n_ch)).astype(np.float32) * mask[:, :, None]
    dev = dvx.SceneOnDevice(ctx, sc)
    _, _, alpha, frame = dev.render()
    F = frame.render_features(_cat(feats), cam.height, cam.width)
    v_total = sum(t.n_voxels for t in sc.octrees)
    num = torch.zeros((v_total, n_ch), device="cuda")
    frame.fuse_features(torch.from_numpy(img).cuda(), num)       # the image is zero outside the sample
    torch.cuda.synchronize()
    ref = O.render_features(sc, feats=feats, img=img, mode=1, mask=mask)
    m = mask.astype(bool)
    err = np.abs(F.cpu().numpy().astype(np.float64)[m] - ref["features"][m]).max()
    assert err <= FEAT_TOL, err
    ref_num = np.concatenate(ref["num"], axis=0)
    scale = max(np.concatenate(ref["wsum"]).max(), 1.0)
    _check_fuse(num.cpu().numpy(), ref_num, scale, "num")
    frame.release()
    for t in dev.trees:
        t.close()


def test_feature_argument_errors_and_empty_scene(ctx, config1):
    import torch
    import paper_2606_23031_b200 as dvx
    from helpers import axis_camera, empty_tree, scene
    dev = dvx.SceneOnDevice(ctx, config1)
    cam = config1.cameras[0]
    rgb, depth, alpha, none = dev.render(save=False)
    assert none is None
    _, _, _, frame = dev.render()
    v_total = sum(t.n_voxels for t in config1.octrees)
    with pytest.raises(dvx.DvxError):
        frame.render_features(torch.zeros((v_total, 513), device="cuda"), cam.height, cam.width)
    with pytest.raises(dvx.DvxError):
        ctx.check(ctx.lib.dvx_render_features(ctx.h, frame.h, 0, torch.zeros(4, device="cuda").data_ptr(), torch.zeros(4, device="cuda").data_ptr()))
    with pytest.raises(dvx.DvxError):
        ctx.check(ctx.lib.dvx_render_features(ctx.h, frame.h, 4, None, None))
    frame.release()
    with pytest.raises(dvx.DvxError):   # the naive walker keeps no tile lists to replay
        _, _, _, fr = dev.render(flags=dvx.FLAG_NAIVE)
        try:
            fr.weights()
        finally:
            fr.release()
    # a scene without voxels: nnz = 0, the feature image is zero
    sc = scene(empty_tree(), cam=axis_camera(width=20, height=18))
    dev0 = dvx.SceneOnDevice(ctx, sc)
    _, _, _, fr = dev0.render()
    nnz, rows, vox, w = fr.weights()
    assert nnz == 0
    F = fr.render_features(torch.zeros((1, 4), device="cuda"), 18, 20)
    torch.cuda.synchronize()
    assert float(F.abs().max()) == 0.0
    fr.release()
