"""Pins of oracle/grid.py (widening row N2: shared grid-point densities + Adam) against things other than itself.

P16 closed form: a full uniform grid of n^3 voxels has (n+1)^3 grid points with 1/2/4/8 sharers by position
P17 hand count: 8 level-1 voxels, one of them split into 8 level-2 voxels -> 27 + 19 = 46 points (7 of them hanging)
P18 brute force: exact-fraction corner positions deduplicated with a dict, ordered by a bit-loop Morton key
P19 adjointness: <gather(d), w> = <d, reduce(w)>; torch autograd through an index gives the same reduction
P20 Adam against torch.optim.Adam in float64 and against the closed form of the first step
P21 grid_adam_step: isolated voxels reduce to elementwise Adam on the corner record
"""
from fractions import Fraction

import numpy as np
import pytest
import torch

import dvx_scenes
from dvx_scenes import octree as so
from oracle import grid as og


def _uniform_codes(level):
    n = 1 << level
    i, j, k = np.meshgrid(np.arange(n), np.arange(n), np.arange(n), indexing="ij")
    return so.encode(i.reshape(-1), j.reshape(-1), k.reshape(-1), level)


@pytest.mark.parametrize("level", [1, 2, 3])
def test_p16_uniform_grid_closed_form(level):
    code = _uniform_codes(level)
    n = 1 << level
    point_of, offsets, slots, keys = og.grid_tables(code)
    G = keys.shape[0]
    assert G == (n + 1) ** 3
    assert offsets[-1] == 8 * n ** 3 and offsets.shape[0] == G + 1
    share = np.diff(offsets.astype(np.int64))
    # a lattice point with a of its 3 coordinates on the boundary is shared by 2^(3-a) voxels
    expect = {8: (n - 1) ** 3, 4: 6 * (n - 1) ** 2, 2: 12 * (n - 1), 1: 8}
    for s, cnt in expect.items():
        assert int((share == s).sum()) == cnt, (s, cnt)
    assert np.all(np.diff(keys.astype(np.int64)) > 0)


def test_p17_two_level_hand_count():
    lvl1 = [(i, j, k) for i in range(2) for j in range(2) for k in range(2) if (i, j, k) != (0, 0, 0)]
    code = [so.encode(np.array([i]), np.array([j]), np.array([k]), 1)[0] for i, j, k in lvl1]
    code += [so.encode(np.array([i]), np.array([j]), np.array([k]), 2)[0] for i in range(2) for j in range(2) for k in range(2)]
    code = np.array(code, dtype=np.uint64)
    point_of, offsets, slots, keys = og.grid_tables(code)
    assert keys.shape[0] == 46
    # the centre of the root cube is a corner of all 7 coarse voxels and of one fine voxel
    share = np.diff(offsets.astype(np.int64))
    assert share.max() == 8 and int((share == 8).sum()) == 1 + 1  # root centre, centre of the split octant
    # every one of the 15 voxels contributes 8 corner slots, hanging nodes included
    assert int(share.sum()) == 8 * 15


def _py_morton(x, y, z):
    key = 0
    for b in range(17):
        key |= ((x >> b) & 1) << (3 * b + 2) | ((y >> b) & 1) << (3 * b + 1) | ((z >> b) & 1) << (3 * b)
    return key


@pytest.mark.parametrize("seed", [3, 11, 29])
def test_p18_brute_force_fractions(seed):
    scene = dvx_scenes.tiny_random_scene(seed, n_static=40, n_actor=10)
    for tree in [scene.static] + list(scene.actors):
        code = tree.code
        i, j, k, level = so.decode(code)
        pos = {}
        per_slot = []
        for v in range(code.shape[0]):
            n = 1 << int(level[v])
            for c in range(8):
                q = (Fraction(int(i[v]) + ((c >> 2) & 1), n), Fraction(int(j[v]) + ((c >> 1) & 1), n),
                     Fraction(int(k[v]) + (c & 1), n))
                pos.setdefault(q, []).append(8 * v + c)
                per_slot.append(q)
        order = sorted(pos, key=lambda q: _py_morton(int(q[0] * 65536), int(q[1] * 65536), int(q[2] * 65536)))
        index = {q: r for r, q in enumerate(order)}
        point_of, offsets, slots, keys = og.grid_tables(code)
        assert keys.shape[0] == len(order)
        assert [index[q] for q in per_slot] == point_of.reshape(-1).tolist()
        for r, q in enumerate(order):
            assert slots[offsets[r]:offsets[r + 1]].tolist() == sorted(pos[q])
            assert int(keys[r]) == _py_morton(int(q[0] * 65536), int(q[1] * 65536), int(q[2] * 65536))


def test_p19_adjoint_and_autograd():
    scene = dvx_scenes.tiny_random_scene(5, n_static=60, n_actor=10)
    code = scene.static.code
    point_of, offsets, slots, keys = og.grid_tables(code)
    G = keys.shape[0]
    rs = np.random.RandomState(0)
    d = rs.randn(G)
    w = rs.randn(code.shape[0], 8)
    lhs = float((og.grid_gather(d, point_of) * w).sum())
    red = og.grid_reduce(w, point_of, G)
    assert abs(lhs - float((d * red).sum())) < 1e-10 * max(1.0, abs(lhs))
    td = torch.tensor(d, dtype=torch.float64, requires_grad=True)
    geo = td[torch.from_numpy(point_of.astype(np.int64))]
    (geo * torch.from_numpy(w)).sum().backward()
    np.testing.assert_allclose(red, td.grad.numpy(), rtol=1e-12, atol=1e-12)
    # the scene generator draws corner densities per lattice point, so its geo must be a gather of something
    geo_s = scene.static.geo.astype(np.float64)
    first = np.zeros(G)
    first[point_of.reshape(-1)] = geo_s.reshape(-1)
    np.testing.assert_array_equal(og.grid_gather(first, point_of), geo_s)


def test_p20_adam_vs_torch_and_first_step():
    rs = np.random.RandomState(1)
    n = 257
    p0 = rs.randn(n)
    lr, b1, b2, eps = 0.025, 0.9, 0.99, 1e-15
    tp = torch.tensor(p0, dtype=torch.float64, requires_grad=True)
    opt = torch.optim.Adam([tp], lr=lr, betas=(b1, b2), eps=eps)
    p, m, v = p0.copy(), np.zeros(n), np.zeros(n)
    for t in range(1, 7):
        g = rs.randn(n) * 10.0 ** rs.randint(-6, 2, size=n)
        if t == 3:
            g[::3] = 0.0
        tp.grad = torch.tensor(g, dtype=torch.float64)
        opt.step()
        p, m, v = og.adam_step(p, m, v, g, lr, b1, b2, eps, t)
        np.testing.assert_allclose(p, tp.detach().numpy(), rtol=1e-12, atol=1e-14)
        if t == 1:  # mhat = g, vhat = g^2
            np.testing.assert_allclose(p, p0 - lr * g / (np.abs(g) + eps), rtol=1e-12, atol=1e-14)


def test_p21_isolated_voxels_reduce_to_elementwise():
    # voxels two cells apart share no corner
    i = np.arange(0, 16, 2)
    code = so.encode(i, i[::-1].copy(), (i * 3) % 16, 4)
    point_of, offsets, slots, keys = og.grid_tables(code)
    G = keys.shape[0]
    assert G == 8 * code.shape[0]
    rs = np.random.RandomState(2)
    d, m, v = rs.randn(G), rs.randn(G) * 0.1, rs.rand(G) * 0.01
    dgeo = rs.randn(code.shape[0], 8)
    hp = (0.01, 0.9, 0.999, 1e-8, 4)
    d2, m2, v2, geo2 = og.grid_adam_step(d, m, v, dgeo, point_of, *hp)
    ge, me, ve = og.adam_step(og.grid_gather(d, point_of), og.grid_gather(m, point_of), og.grid_gather(v, point_of), dgeo, *hp)
    np.testing.assert_allclose(geo2, ge, rtol=1e-13)
    np.testing.assert_allclose(og.grid_gather(m2, point_of), me, rtol=1e-13)
    np.testing.assert_allclose(og.grid_gather(v2, point_of), ve, rtol=1e-13)
