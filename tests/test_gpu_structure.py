"""Row N4 through the C ABI against oracle/structure.py: proximity subdivision rounds and pruning bit-exact,
the Eq. 1 density prior within fp32 rounding; small cases in full, the static octree of config 2 at full size."""
import numpy as np
import pytest

import dvx_scenes as S
from dvx_scenes import octree as so
from oracle import grid as G
from oracle import structure as T

pytestmark = pytest.mark.gpu

PRIOR_TOL = 2e-6   # fp32 output of an fp64 evaluation: half an ulp of |v| <= 10 is 4.8e-7; the search cut-off adds < 4e-8


@pytest.fixture(scope="module")
def ctx():
    import paper_2606_23031_b200 as dvx
    c = dvx.Context(0)
    yield c
    c.close()


def _dev_code(code):
    import torch
    return torch.from_numpy(np.ascontiguousarray(code).view(np.int64)).cuda()


def _dev_pts(pts):
    import torch
    return torch.from_numpy(np.ascontiguousarray(pts, dtype=np.float32).reshape(-1, 3)).cuda()


def _surface_points(tree, n, seed, jitter):
    """Seeded stand-in for LiDAR returns: points near the centres of randomly chosen leaves (float32, like a sensor's output)."""
    rs = np.random.RandomState(seed)
    lo, hi = T.voxel_boxes(tree.code, tree.center, tree.side)
    pick = rs.randint(0, tree.code.shape[0], size=n)
    c = 0.5 * (lo[pick] + hi[pick])
    return (c + rs.randn(n, 3) * jitter).astype(np.float32)


def _round_trip_subdivide(ctx, code, center, side, pts, thr, cell, max_level=16):
    import torch
    cloud = ctx.cloud(_dev_pts(pts), cell)
    new, split = ctx.subdivide_near(cloud, _dev_code(code), center, side, thr, max_level)
    torch.cuda.synchronize()
    ref_new, ref_split = T.subdivide_near(code, np.asarray(center, np.float64), float(side), pts.astype(np.float64), float(np.float32(thr)), max_level)
    assert np.array_equal(split.cpu().numpy().astype(bool), ref_split)
    assert np.array_equal(new.cpu().numpy().view(np.uint64), ref_new)
    cloud.close()
    return ref_new, ref_split


def test_subdivision_rounds_small(ctx):
    for seed in (1, 2, 3):
        sc = S.tiny_random_scene(seed, n_static=60)
        tree = sc.static
        side = float(tree.side)
        pts = _surface_points(tree, 80, seed, 0.02 * side)
        code = tree.code
        for rnd, cell in enumerate((0.05 * side, 0.2 * side, 0.011 * side)):   # cells smaller / larger than the threshold
            code, split = _round_trip_subdivide(ctx, code, tree.center, side, pts, 0.03 * side, cell)
            assert split.any()
    # threshold 0 (only leaves that contain a point), a threshold larger than the scene, an empty cloud, max_level
    tree = S.tiny_random_scene(4, n_static=40).static
    pts = _surface_points(tree, 30, 9, 0.0)
    _round_trip_subdivide(ctx, tree.code, tree.center, float(tree.side), pts, 0.0, 0.1 * float(tree.side))
    _, sp = _round_trip_subdivide(ctx, tree.code, tree.center, float(tree.side), pts, 10.0 * float(tree.side), 0.5 * float(tree.side))
    assert sp.all()
    _, sp = _round_trip_subdivide(ctx, tree.code, tree.center, float(tree.side), np.zeros((0, 3), np.float32), 1.0, 1.0)
    assert not sp.any()
    lvl = int(so.decode(tree.code)[3].max())
    _, sp = _round_trip_subdivide(ctx, tree.code, tree.center, float(tree.side), pts, 10.0 * float(tree.side), 1.0, max_level=lvl)
    assert sp.any() and not sp.all()


def test_inclusive_threshold_exact_case(ctx):
    # box [0,2]^3 of a 4 m cube; a point exactly 0.5 above the top face: distance == threshold must split (R26: <=)
    code = so.encode(np.array([1]), np.array([1]), np.array([1]), 1)
    pts = np.array([[1.0, 1.0, 2.5]], np.float32)
    _, sp = _round_trip_subdivide(ctx, code, (0.0, 0.0, 0.0), 4.0, pts, 0.5, 0.5)
    assert sp[0]
    _, sp = _round_trip_subdivide(ctx, code, (0.0, 0.0, 0.0), 4.0, pts, 0.49999, 0.5)
    assert not sp[0]


def test_density_prior_small(ctx):
    import torch
    for seed in (5, 6):
        sc = S.tiny_random_scene(seed, n_static=80)
        tree = sc.static
        side = float(tree.side)
        lvl = int(so.decode(tree.code)[3].max())
        s_min = side / (1 << lvl)
        pts = _surface_points(tree, 120, seed, 0.5 * s_min)
        grid = ctx.grid(_dev_code(tree.code))
        for cell in (3.1 * s_min, 0.7 * s_min, 20 * s_min):
            cloud = ctx.cloud(_dev_pts(pts), cell)
            dens = ctx.density_prior(cloud, _dev_code(tree.code), tree.center, side, grid, s_min)
            torch.cuda.synchronize()
            ref = T.density_prior(tree.code, np.asarray(tree.center, np.float64), side, pts.astype(np.float64), float(np.float32(s_min)))
            assert ref.max() > -9.0 and ref.min() < -9.99
            assert np.abs(dens.cpu().numpy().astype(np.float64) - ref).max() <= PRIOR_TOL
            cloud.close()
        # other constants, and an empty cloud
        cloud = ctx.cloud(_dev_pts(pts), s_min)
        dens = ctx.density_prior(cloud, _dev_code(tree.code), tree.center, side, grid, s_min, v_close=1.5, v_far=-4.0)
        ref = T.density_prior(tree.code, np.asarray(tree.center, np.float64), side, pts.astype(np.float64), float(np.float32(s_min)), 1.5, -4.0)
        assert np.abs(dens.cpu().numpy().astype(np.float64) - ref).max() <= PRIOR_TOL
        cloud.close()
        empty = ctx.cloud(_dev_pts(np.zeros((0, 3))), 1.0)
        dens = ctx.density_prior(empty, _dev_code(tree.code), tree.center, side, grid, s_min)
        assert bool((dens == -10.0).all())
        empty.close()
        grid.close()


def test_prune(ctx):
    import torch
    sc = S.make_config(1)
    tree = sc.static
    code, geo = _dev_code(tree.code), torch.from_numpy(tree.geo).cuda()
    for thr in (float(np.median(tree.geo.max(axis=1))), -1e9, 1e9):
        kept, idx = ctx.prune(code, geo, thr)
        ref_code, ref_idx = T.prune(tree.code, tree.geo, float(np.float32(thr)))
        assert np.array_equal(kept.cpu().numpy().view(np.uint64), ref_code)
        assert np.array_equal(idx.cpu().numpy().view(np.uint32), ref_idx)


def test_structure_pipeline_config2_static(ctx):
    """Full size: the static octree of config 2 (0.5 M leaves) against a 200 k-point cloud: one subdivision round (bit-exact),
    then grid tables and the Eq. 1 prior on the refined tree (2e-6), then pruning by the prior (bit-exact)."""
    import torch
    sc = S.make_config(2)
    tree = sc.static
    side = float(tree.side)
    level = so.decode(tree.code)[3]
    s_min = side / (1 << int(level.max()))
    pts = _surface_points(tree, 200_000, 17, 2.0 * s_min)
    thr = 1.5 * s_min
    new, split = _round_trip_subdivide(ctx, tree.code, tree.center, side, pts, thr, thr, max_level=int(level.max()) + 1)
    assert 0.02 < split.mean() < 0.98
    grid = ctx.grid(_dev_code(new))
    s2 = 0.5 * s_min
    cloud = ctx.cloud(_dev_pts(pts), 3.1 * s2)
    dens = ctx.density_prior(cloud, _dev_code(new), tree.center, side, grid, s2)
    torch.cuda.synchronize()
    ref = T.density_prior(new, np.asarray(tree.center, np.float64), side, pts.astype(np.float64), float(np.float32(s2)))
    assert grid.n_points == ref.shape[0]
    assert np.abs(dens.cpu().numpy().astype(np.float64) - ref).max() <= PRIOR_TOL
    geo = torch.empty((new.shape[0], 8), device="cuda")
    grid.gather(dens, geo)
    kept, idx = ctx.prune(_dev_code(new), geo, -9.5)
    ref_code, ref_idx = T.prune(new, G.grid_gather(dens.cpu().numpy(), G.grid_tables(new)[0]), float(np.float32(-9.5)))
    assert np.array_equal(kept.cpu().numpy().view(np.uint64), ref_code) and np.array_equal(idx.cpu().numpy().view(np.uint32), ref_idx)
    assert 0 < ref_code.shape[0] < new.shape[0]
    cloud.close()
    grid.close()


def test_structure_argument_errors(ctx):
    import torch
    import paper_2606_23031_b200 as dvx
    p = torch.zeros((4, 3), device="cuda")
    with pytest.raises(dvx.DvxError):
        ctx.cloud(p, 0.0)
    bad = p.clone()
    bad[1, 2] = float("inf")
    with pytest.raises(dvx.DvxError):
        ctx.cloud(bad, 1.0)
    wide = torch.tensor([[0.0, 0.0, 0.0], [1e7, 0.0, 0.0]], device="cuda")
    with pytest.raises(dvx.DvxError):
        ctx.cloud(wide, 1.0)      # more than 2^21 cells along x
    cloud = ctx.cloud(p, 1.0)
    code = _dev_code(so.encode(np.array([0]), np.array([0]), np.array([0]), 1))
    with pytest.raises(dvx.DvxError):
        ctx.subdivide_near(cloud, code, (0, 0, 0), 4.0, -1.0)
    grid = ctx.grid(code)
    with pytest.raises(dvx.DvxError):
        ctx.density_prior(cloud, code, (0, 0, 0), 4.0, grid, 0.0)
    grid.close()
    cloud.close()


def test_subdivide_near_beyond_2_27_leaves(ctx):
    """the flag kernels index warps as (block * threads + thread) >> 5; with one warp per leaf that product passes
    2^32 at 2^27 leaves, inside the documented range V < 2^28.  2^27 + 8192 level-10 leaves (a dense Morton prefix of the
    cube), a handful of points inside the LAST leaves: only leaves with an index above 2^27 may be flagged, and they must be
    flagged exactly as the oracle flags them on that tail (the head is checked to be all clear)."""
    import torch
    n = (1 << 27) + 8192
    idx = torch.arange(n, dtype=torch.int64, device="cuda")
    code = (idx << 18) | (10 << 48)               # 30-bit Morton path left-aligned in 48 bits, level 10
    side, center = 1024.0, (0.0, 0.0, 0.0)        # level-10 cells of 1 m
    tail = code[-64:].cpu().numpy().view(np.uint64)
    lo, hi = T.voxel_boxes(tail, center, side)
    rs = np.random.RandomState(5)
    pts = (0.5 * (lo[::7] + hi[::7]) + rs.uniform(-0.2, 0.2, size=lo[::7].shape)).astype(np.float32)
    thr = 0.45
    cloud = ctx.cloud(_dev_pts(pts), 1.0)
    desc_code = code.contiguous()
    split = torch.zeros(n, dtype=torch.uint8, device="cuda")
    import ctypes as C
    import paper_2606_23031_b200.binding as B
    desc = B.OctreeDesc(n, 0, (C.c_float * 3)(*center), side, desc_code.data_ptr(), None, None)
    n_out = C.c_uint64()
    ctx.check(ctx.lib.dvx_subdivide_near(ctx.h, cloud.h, C.byref(desc), thr, 11, None, 0, C.byref(n_out), split.data_ptr()))
    torch.cuda.synchronize()
    # reference on the last 4096 leaves (every point is inside one of the last 64), zero elsewhere
    m = 4096
    ref_new, ref_split = T.subdivide_near(code[-m:].cpu().numpy().view(np.uint64), np.asarray(center, np.float64), side,
                                          pts.astype(np.float64), float(np.float32(thr)), 11)
    got = split[-m:].cpu().numpy().astype(bool)
    assert ref_split.sum() >= 10 and np.array_equal(got, ref_split)
    assert int(split[:-m].sum().item()) == 0
    assert n_out.value == n + 7 * int(ref_split.sum())
    cloud.close()
    del code, split, idx
    ctx.trim()


def test_subdivide_fill_matches_the_oracle_and_keeps_the_image(ctx):
    """dvx_subdivide_fill (R29) against oracle/structure.py on config 1's static octree after a proximity round: corner
    densities bit for bit (sums of at most 8 fp32 values with power-of-two weights are exact in fp64 on both sides), SH
    copied; and the refined octree renders the image of the original one up to the quadrature (finer voxels, more samples)."""
    import torch
    import paper_2606_23031_b200 as dvx
    sc = S.make_config(1)
    tree = sc.static
    side = float(tree.side)
    pts = _surface_points(tree, 400, 23, 0.3)
    cloud = ctx.cloud(_dev_pts(pts), 1.0)
    code = _dev_code(tree.code)
    new, split = ctx.subdivide_near(cloud, code, tree.center, side, 0.5, 7)
    torch.cuda.synchronize()
    geo, sh = torch.from_numpy(tree.geo).cuda(), torch.from_numpy(tree.sh).cuda()
    g2, s2 = ctx.subdivide_fill(split, geo, sh, tree.sh_degree, int(new.shape[0]))
    torch.cuda.synchronize()
    rg, rs = T.subdivide_fill(split.cpu().numpy(), tree.geo, tree.sh)
    assert 0.05 < float(split.float().mean()) < 0.95
    assert np.array_equal(g2.cpu().numpy(), rg.astype(np.float32)) and np.array_equal(s2.cpu().numpy(), rs.astype(np.float32))
    # render both octrees (static only) with the library: same field, finer quadrature
    old = ctx.octree(code, geo, sh, tree.center, side, tree.sh_degree)
    ref = ctx.octree(new.contiguous(), g2, s2, tree.center, side, tree.sh_degree)
    cam = dvx.camera_from(sc.cameras[0])
    a = ctx.render(cam, old, save=False)
    b = ctx.render(cam, ref, save=False)
    torch.cuda.synchronize()
    assert float(a[2].max()) > 0.5
    assert float((a[2] - b[2]).abs().max()) < 3e-2 and float((a[0] - b[0]).abs().max()) < 3e-2
    assert float((a[2] - b[2]).abs().mean()) < 2e-3
    old.close(); ref.close(); cloud.close()
