"""Row N2 through the C ABI against oracle/grid.py: grid-point tables bit-exact, gather / reduce / Adam
within fp32 rounding, and one whole training step (render, backward, optimizer, render again) against the oracle."""
import copy

import numpy as np
import pytest

import dvx_scenes as S
from dvx_scenes import octree as so
from oracle import grid as G
from oracle import oracle as O

pytestmark = pytest.mark.gpu

HP = dict(lr=0.02, beta1=0.9, beta2=0.99, eps=1e-8)


@pytest.fixture(scope="module")
def ctx():
    import paper_2606_23031_b200 as dvx
    c = dvx.Context(0)
    yield c
    c.close()


def _dev_code(code):
    import torch
    return torch.from_numpy(np.ascontiguousarray(code).view(np.int64)).cuda()


def _tables(grid):
    import torch
    torch.cuda.synchronize()
    return (grid.point_of().cpu().numpy().view(np.uint32), grid.offsets().cpu().numpy().view(np.uint32),
            grid.slots().cpu().numpy().view(np.uint32))


def _check_tables(ctx, code):
    ref_po, ref_off, ref_sl, keys = G.grid_tables(code)
    grid = ctx.grid(_dev_code(code))
    po, off, sl = _tables(grid)
    assert grid.n_points == keys.shape[0]
    assert np.array_equal(po, ref_po)
    assert np.array_equal(off, ref_off)
    assert np.array_equal(sl, ref_sl)
    return grid, ref_po


def test_grid_tables_bit_exact_small(ctx, config1):
    for tree in config1.octrees:
        _check_tables(ctx, tree.code)[0].close()
    for seed in (1, 2, 3):
        sc = S.tiny_random_scene(seed, n_static=50, n_actor=12)
        for tree in sc.octrees:
            _check_tables(ctx, tree.code)[0].close()
    n = 8  # full 8^3 grid: (n+1)^3 points (pin P16)
    i, j, k = np.meshgrid(np.arange(n), np.arange(n), np.arange(n), indexing="ij")
    grid, _ = _check_tables(ctx, so.encode(i.reshape(-1), j.reshape(-1), k.reshape(-1), 3))
    assert grid.n_points == 9 ** 3
    grid.close()


def test_grid_degenerate_sizes(ctx):
    import torch
    g0 = ctx.grid(torch.zeros(0, dtype=torch.int64, device="cuda"))
    assert g0.n_points == 0 and g0.n_voxels == 0
    g0.gather(torch.zeros(1, device="cuda"), torch.zeros(1, device="cuda"))   # no-ops
    g0.close()
    # one voxel at the deepest level, in the far corner: lattice coordinate 65536 (bit 16) appears
    top = (1 << 16) - 1
    code = so.encode(np.array([top]), np.array([top]), np.array([top]), 16)
    grid, po = _check_tables(ctx, code)
    assert grid.n_points == 8
    grid.close()
    # the root split once, plus a deepest-level voxel far from the others
    code = np.concatenate([so.encode(np.array([0, 1]), np.array([0, 0]), np.array([0, 0]), 1), so.encode(np.array([5]), np.array([top]), np.array([9]), 16)])
    _check_tables(ctx, code)[0].close()


def test_grid_tables_config3_static(ctx, config3):
    """Full size (4.0 M voxels, 32 M corner keys, several thousand sort tiles): bit-exact against the oracle."""
    import torch
    code = config3.static.code
    grid, ref_po = _check_tables(ctx, code)
    # gather at full size is exact
    rs = np.random.RandomState(0)
    dens = rs.randn(grid.n_points).astype(np.float32)
    d = torch.from_numpy(dens).cuda()
    geo = torch.empty((code.shape[0], 8), dtype=torch.float32, device="cuda")
    grid.gather(d, geo)
    torch.cuda.synchronize()
    assert np.array_equal(geo.cpu().numpy(), G.grid_gather(dens, ref_po))
    grid.close()


def _close(got, ref, rtol, atol, what):
    got = np.asarray(got, dtype=np.float64)
    err = np.abs(got - ref)
    bound = rtol * np.abs(ref) + atol
    assert (err <= bound).all(), "%s: worst excess %g at |ref| max %g" % (what, (err - bound).max(), np.abs(ref).max())


def test_grid_reduce_and_adam_steps(ctx, config1):
    import torch
    code = config1.static.code
    V = code.shape[0]
    grid, po = _check_tables(ctx, code)
    Gn = grid.n_points
    rs = np.random.RandomState(4)
    dens = rs.randn(Gn).astype(np.float32)
    d = torch.from_numpy(dens).cuda()
    m = torch.zeros(Gn, device="cuda")
    v = torch.zeros(Gn, device="cuda")
    geo = torch.empty((V, 8), device="cuda")
    grid.gather(d, geo)
    rd, rm, rv = dens.astype(np.float64), np.zeros(Gn), np.zeros(Gn)
    for t in range(1, 6):
        dgeo_h = (rs.randn(V, 8) * 10.0 ** rs.randint(-5, 1, size=(V, 1))).astype(np.float32)
        if t == 2:
            dgeo_h[::2] = 0.0        # untouched voxels
        dgeo = torch.from_numpy(dgeo_h).cuda()
        dd = torch.empty(Gn, device="cuda")
        grid.reduce(dgeo, dd)
        ref_g = G.grid_reduce(dgeo_h, po, Gn)
        mag = G.grid_reduce(np.abs(dgeo_h), po, Gn)
        torch.cuda.synchronize()
        assert (np.abs(dd.cpu().numpy() - ref_g) <= 4e-7 * mag + 1e-30).all()   # 8-term fp32 sum
        grid.adam_step(d, m, v, dgeo, geo, step=t, **HP)
        rd, rm, rv, rgeo = G.grid_adam_step(rd, rm, rv, dgeo_h, po, HP["lr"], HP["beta1"], HP["beta2"], HP["eps"], t)
        torch.cuda.synchronize()
        assert float(dgeo.abs().max()) == 0.0, "gradients must be zeroed"
        assert np.array_equal(geo.cpu().numpy(), d.cpu().numpy()[po.astype(np.int64)]), "geo must be the gather of density"
        # m, v: a few fp32 roundings per step, plus the rounding of the 8-term gradient sum (4e-7 mag, which is a large
        # RELATIVE error where the terms cancel); density: each step moves at most ~lr, error a few ulp of that + of |p|
        _close(m.cpu().numpy(), rm, 2e-5, 4e-7 * mag, "m step %d" % t)
        _close(v.cpu().numpy(), rv, 4e-5, 1e-8 * mag * mag, "v step %d" % t)
        _close(d.cpu().numpy(), rd, 2e-6, HP["lr"] * 1e-4, "density step %d" % t)
    grid.close()


@pytest.mark.parametrize("n", [1, 3, 4, 1027, (1 << 20) + 2])
def test_adam_step_elementwise(ctx, n):
    import torch
    rs = np.random.RandomState(n % 97)
    p_h, g_h = rs.randn(n).astype(np.float32), (rs.randn(n) * 10.0 ** rs.randint(-5, 1, size=n)).astype(np.float32)
    m_h, v_h = (rs.randn(n) * 0.01).astype(np.float32), (rs.rand(n) * 1e-3).astype(np.float32)
    p, m, v, g = [torch.from_numpy(a.copy()).cuda() for a in (p_h, m_h, v_h, g_h)]
    ctx.adam_step(p, m, v, g, step=3, **HP)
    rp, rm, rv = G.adam_step(p_h, m_h, v_h, g_h, HP["lr"], HP["beta1"], HP["beta2"], HP["eps"], 3)
    torch.cuda.synchronize()
    assert float(g.abs().max()) == 0.0
    # m = b1 m + (1-b1) g can cancel: bound by the magnitude of the two terms
    _close(m.cpu().numpy(), rm, 2e-6, 3e-7 * (0.9 * np.abs(m_h) + 0.1 * np.abs(g_h)), "m")
    _close(v.cpu().numpy(), rv, 2e-6, 1e-20, "v")
    # the step is step_size m / denom: the rounding of m (above) and of the quotient (a few ulp) carried through it
    dm = 3e-7 * (0.9 * np.abs(m_h) + 0.1 * np.abs(g_h)) + 2e-6 * np.abs(rm)
    step_size = HP["lr"] / (1 - HP["beta1"] ** 3)
    denom = np.sqrt(rv / (1 - HP["beta2"] ** 3)) + HP["eps"]
    _close(p.cpu().numpy(), rp, 2e-7, step_size * dm / denom + 1e-6 * np.abs(rp - p_h), "p")


def test_batched_steps_equal_single_calls(ctx, config1):
    """dvx_grid_adam_step_n / dvx_adam_step_n over all octrees of config 1 (one launch) == one call per octree, bit for bit;
    empty arrays in the batch are skipped."""
    import torch
    rs = np.random.RandomState(9)
    hp = dict(HP, step=2)
    grids, single, batch = [], [], []
    for tree in config1.octrees:
        grid = ctx.grid(_dev_code(tree.code))
        V, Gn = tree.n_voxels, grid.n_points
        arrs = [rs.randn(Gn), rs.randn(Gn) * 0.1, rs.rand(Gn) * 0.01, rs.randn(V, 8), np.zeros((V, 8))]
        grids.append(grid)
        single.append([torch.from_numpy(a.astype(np.float32)).cuda() for a in arrs])
        batch.append([t.clone() for t in single[-1]])
    empty = ctx.grid(torch.zeros(0, dtype=torch.int64, device="cuda"))
    z = torch.zeros(4, device="cuda")
    for grid, ts in zip(grids, single):
        grid.adam_step(*ts, **hp)
    ctx.grid_adam_step_n([(grids[0], *batch[0]), (empty, z, z, z, z, z)] + [(g, *ts) for g, ts in zip(grids[1:], batch[1:])], **hp)
    torch.cuda.synchronize()
    for a, b in zip(single, batch):
        for x, y in zip(a, b):
            assert torch.equal(x, y)
    sizes = [5, 4096, 0, 4097, 12289, 3]
    one = [[torch.from_numpy(rs.randn(n).astype(np.float32)).cuda().abs() * s for s in (1, 0.1, 0.01, 1)] for n in sizes]
    many = [[t.clone() for t in ts] for ts in one]
    for ts in one:
        ctx.adam_step(*ts, **hp)
    ctx.adam_step_n([tuple(ts) for ts in many], **hp)
    torch.cuda.synchronize()
    for a, b in zip(one, many):
        for x, y in zip(a, b):
            assert torch.equal(x, y)
    for g in grids + [empty]:
        g.close()


def test_adam_argument_errors(ctx):
    import torch
    import paper_2606_23031_b200 as dvx
    a = torch.zeros(8, device="cuda")
    with pytest.raises(dvx.DvxError):
        ctx.adam_step(a, a, a, a, lr=0.0, beta1=0.9, beta2=0.99, eps=1e-8, step=1)
    with pytest.raises(dvx.DvxError):
        ctx.adam_step(a, a, a, a, lr=0.1, beta1=1.0, beta2=0.99, eps=1e-8, step=1)
    with pytest.raises(dvx.DvxError):
        ctx.adam_step(a, a, a, a, lr=0.1, beta1=0.9, beta2=0.99, eps=1e-8, step=0)
    with pytest.raises(dvx.DvxError):
        ctx.adam_step(a[1:], a[1:], a[1:], a[1:], lr=0.1, beta1=0.9, beta2=0.99, eps=1e-8, step=1)  # misaligned


def test_training_step_config1(ctx, config1):
    """render -> backward -> grid Adam on the densities + Adam on the SH coefficients -> render, against the oracle doing
    the same in double precision (images of the second render within the R16 tolerances)."""
    import torch
    import paper_2606_23031_b200 as dvx
    sc = copy.deepcopy(config1)
    gin = sc.image_grads(rgb_std=1e-2, depth_std=1e-3, alpha_std=1e-2)
    dev = dvx.SceneOnDevice(ctx, sc)
    rgb, depth, alpha, frame = dev.render()
    g = [torch.from_numpy(gin[k]).cuda() for k in ("rgb", "depth", "alpha")]
    grads = frame.backward(g[0], g[1], g[2])
    frame.release()
    ref = O.render(sc, mode=0, grads_in=gin)
    # eps well above the gradient tolerance (abs 1e-6): Adam's first step is lr g/(|g|+eps), and with a tiny eps a
    # parameter whose gradient is rounding noise would move by +-lr depending on the noise's sign
    hp = dict(HP, lr=0.05, eps=1e-4)
    state = []
    for n, tree in enumerate(sc.octrees):
        grid = ctx.grid(_dev_code(tree.code))
        po, off, sl = _tables(grid)
        ref_po = G.grid_tables(tree.code)[0]
        assert np.array_equal(po, ref_po)
        Gn = grid.n_points
        dens_h = np.zeros(Gn)
        dens_h[po.reshape(-1).astype(np.int64)] = tree.geo.reshape(-1)       # the scene's geo is consistent on shared corners
        d = torch.from_numpy(dens_h.astype(np.float32)).cuda()
        m, v = torch.zeros(Gn, device="cuda"), torch.zeros(Gn, device="cuda")
        dgeo, dsh = grads[n]
        t_dev = dev.trees[n]
        grid.adam_step(d, m, v, dgeo, t_dev.geo, step=1, **hp)
        ms, vs = torch.zeros_like(dsh), torch.zeros_like(dsh)
        ctx.adam_step(t_dev.sh, ms, vs, dsh, step=1, **hp)
        state.append((grid, d, m, v, ms, vs))
        # the oracle's step
        _, _, _, geo2 = G.grid_adam_step(dens_h, np.zeros(Gn), np.zeros(Gn), ref["dgeo"][n], ref_po, hp["lr"], hp["beta1"], hp["beta2"], hp["eps"], 1)
        sh2, _, _ = G.adam_step(tree.sh, np.zeros_like(ref["dsh"][n]), np.zeros_like(ref["dsh"][n]), ref["dsh"][n], hp["lr"], hp["beta1"], hp["beta2"], hp["eps"], 1)
        tree.geo = np.ascontiguousarray(geo2, dtype=tree.geo.dtype)
        tree.sh = np.ascontiguousarray(sh2, dtype=tree.sh.dtype)
    rgb2, depth2, alpha2, _ = dev.render(save=False)
    torch.cuda.synchronize()
    ref2 = O.render(sc, mode=0)
    assert np.abs(ref2["rgb"] - ref["rgb"]).max() > 1e-2, "the step must have changed the image"
    err = np.abs(rgb2.cpu().numpy() - ref2["rgb"]).max()
    # gradient tolerance (rel 1e-3 + abs 1e-6) through the step: |d param| <= lr (1e-3 |g| + 1e-6)/(|g| + eps) <= 5e-4
    assert err <= 1e-3, err
    assert np.abs(alpha2.cpu().numpy() - ref2["alpha"]).max() <= 1e-3
    for grid, *_ in state:
        grid.close()
