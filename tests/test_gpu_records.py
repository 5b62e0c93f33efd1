"""The forward's hit records and the backward that replays them (include/dvx.h "Hit records"; hot-path step 5,
PAPER.md:113).  The replay, the list-walking backward (DVX_FLAG_NO_RECORDS) and the device-side fall-back after a pool
overflow must all give the oracle's gradients; the forward image must not depend on whether records are written."""
import numpy as np
import pytest

import dvx_scenes as S
from oracle import oracle as O

pytestmark = pytest.mark.gpu

GRAD_REL, GRAD_ABS = 1e-3, 1e-6


@pytest.fixture(scope="module")
def ctx():
    import paper_2606_23031_b200 as dvx
    c = dvx.Context(0)
    yield c
    c.close()


def _check(got, ref, what):
    got = got.cpu().numpy().astype(np.float64)
    excess = np.abs(got - ref) - (GRAD_REL * np.abs(ref) + GRAD_ABS)
    assert excess.size == 0 or excess.max() <= 0, "%s: worst excess %g" % (what, excess.max())


def _backward_all(dev, sc, gin, **kw):
    import torch
    rgb, depth, alpha, frame = dev.render(**kw)
    st = frame.record_stats()
    g = [None if gin[k] is None else torch.from_numpy(gin[k]).cuda() for k in ("rgb", "depth", "alpha")]
    grads = frame.backward(g[0], g[1], g[2])
    torch.cuda.synchronize()
    frame.release()
    return (rgb, depth, alpha), grads, st


def test_replay_walk_and_overflow_fallback_agree_with_the_oracle(ctx, config1):
    import paper_2606_23031_b200 as dvx
    import torch
    sc = config1
    gin = sc.image_grads(rgb_std=1e-2, depth_std=1e-3, alpha_std=1e-2)
    ref = O.render(sc, mode=0, grads_in=gin)
    dev = dvx.SceneOnDevice(ctx, sc)
    img_r, g_r, st_r = _backward_all(dev, sc, gin)                                    # records + replay
    img_w, g_w, st_w = _backward_all(dev, sc, gin, flags=dvx.FLAG_NO_RECORDS)         # list walk
    ctx.set_record_budget(3 * 16384)                                                  # three chunks: certain overflow
    try:
        img_o, g_o, st_o = _backward_all(dev, sc, gin)                                # replay refuses, the walk runs
    finally:
        ctx.set_record_budget(0)
    assert st_r["bytes_used"] > 0 and st_r["bytes_used"] <= st_r["bytes_capacity"] and not st_r["overflowed"]
    assert st_w == {"bytes_used": 0, "bytes_capacity": 0, "overflowed": False}
    assert st_o["overflowed"] and st_o["bytes_capacity"] == 3 * 16384
    for a, b, c in zip(img_r, img_w, img_o):   # writing records must not change a bit of the image
        assert torch.equal(a, b) and torch.equal(a, c)
    for t in range(len(sc.octrees)):
        for k, name in ((0, "dgeo"), (1, "dsh")):
            want = ref[name][t]
            _check(g_r[t][k], want, "%s[%d] replay" % (name, t))
            _check(g_w[t][k], want, "%s[%d] walk" % (name, t))
            _check(g_o[t][k], want, "%s[%d] overflow fall-back" % (name, t))
            scale = g_w[t][k].abs().max().item()
            assert (g_r[t][k] - g_w[t][k]).abs().max().item() <= 2e-5 * scale + 1e-9   # same terms, other summation order
    # the hit count the records imply is the forward's own: used bytes cover at least n_used records of 40 bytes
    n_hits = int(ref["n_used"].sum())
    assert st_r["bytes_used"] >= 40 * n_hits * 0.98
    for t in dev.trees:
        t.close()


@pytest.mark.parametrize("seed,activation,t_stop", [(3, 0, 1e-4), (11, 1, 0.0), (5, 0, 0.3)])
def test_replay_on_small_scenes_with_actor_cuts_and_early_termination(ctx, seed, activation, t_stop):
    """Tiny random scenes (an actor box cutting static voxels in two, exp-linear activation, an aggressive t_stop so that
    most rays stop early): replay == walk == oracle, all gradient entries, with depth and alpha gradients."""
    import paper_2606_23031_b200 as dvx
    sc = S.tiny_random_scene(seed, sh_degree=1, width=40, height=24)
    sc.activation, sc.t_stop = activation, t_stop
    if t_stop >= 0.1:
        for t in sc.octrees:
            t.geo = (t.geo + np.float32(2.5)).astype(np.float32)
    gin = sc.image_grads(0, 1e-2, 1e-3, 1e-2)   # the config-1 recipe; R16's absolute floor is sized for it
    ref = O.render(sc, grads_in=gin)
    if t_stop >= 0.1:
        full = O.render(sc, t_stop=0.0)
        assert (ref["n_used"] < full["n_used"]).mean() > 0.2
    dev = dvx.SceneOnDevice(ctx, sc)
    _, g_r, st = _backward_all(dev, sc, gin)
    _, g_w, _ = _backward_all(dev, sc, gin, flags=dvx.FLAG_NO_RECORDS)
    assert not st["overflowed"]
    for t in range(len(sc.octrees)):
        for k, name in ((0, "dgeo"), (1, "dsh")):
            _check(g_r[t][k], ref[name][t], "%s[%d] replay" % (name, t))
            _check(g_w[t][k], ref[name][t], "%s[%d] walk" % (name, t))
    for t in dev.trees:
        t.close()


def test_pool_sizing_follows_the_previous_frames(ctx):
    """Automatic sizing: the first saved frame of a context gets 48 hits per pixel; later frames 1.25 x what the recent
    frames used, so a workload with more hits per pixel overflows at most on its first frame and still returns the
    right gradients on that frame (the fall-back)."""
    import paper_2606_23031_b200 as dvx
    import torch
    c2 = dvx.Context(0)
    try:
        sc = S.make_config(2)
        dev = dvx.SceneOnDevice(c2, sc)
        g = torch.from_numpy(sc.image_grads(rgb_std=1e-2)["rgb"]).cuda()
        stats, grads = [], []
        for it in range(3):
            _, _, _, fr = dev.render()
            stats.append(fr.record_stats())
            grads.append(fr.backward(g))
            torch.cuda.synchronize()
            fr.release()
        assert not stats[1]["overflowed"] and not stats[2]["overflowed"]
        assert stats[2]["bytes_capacity"] <= 1.6 * stats[2]["bytes_used"] + (1 << 22)
        ref = grads[2][0][0].abs().max().item()
        for it in (0, 1):
            assert (grads[it][0][0] - grads[2][0][0]).abs().max().item() <= 2e-5 * ref + 1e-9
        for t in dev.trees:
            t.close()
    finally:
        c2.close()


def test_a_pool_the_allocator_cannot_give_is_not_an_error(ctx, config1):
    """dvx.h 'Hit records': when the allocator returns NULL for the record pool the frame simply keeps no records and the
    backward walks the tile lists - same gradients."""
    import torch
    sc = config1
    gin = sc.image_grads(rgb_std=1e-2, depth_std=1e-3, alpha_std=1e-2)
    ref = O.render(sc, mode=0, grads_in=gin)
    import paper_2606_23031_b200 as dvx
    dev = dvx.SceneOnDevice(ctx, sc)
    ctx.set_record_budget(1 << 46)          # 64 TiB: torch's allocator refuses, the callback returns NULL
    try:
        img, grads, st = _backward_all(dev, sc, gin)
    finally:
        ctx.set_record_budget(0)
    assert st == {"bytes_used": 0, "bytes_capacity": 0, "overflowed": False}
    for t in range(len(sc.octrees)):
        _check(grads[t][0], ref["dgeo"][t], "dgeo[%d] without a pool" % t)
        _check(grads[t][1], ref["dsh"][t], "dsh[%d] without a pool" % t)
    for t in dev.trees:
        t.close()


def test_batch_entry_points_argument_errors(ctx, config1):
    """dvx_render_batch / dvx_backward_batch: an invalid camera anywhere in the batch fails the whole call with
    DVX_ERR_INVALID_ARG and hands out no frame; empty batches are no-ops; frames with a normal map are refused by the batched
    backward (their post-pass writes dgeo)."""
    import ctypes as C
    import torch
    import paper_2606_23031_b200 as dvx
    sc = config1
    dev = dvx.SceneOnDevice(ctx, sc)
    good = dev.cams[0]
    bad = dvx.camera_from(sc.cameras[0]); bad.fx = 0.0
    with pytest.raises(dvx.DvxError) as e:
        ctx.render_batch([good, bad], dev.trees[0], dev.trees[1:], dev.poses, dev.box_half)
    assert e.value.status == -1
    outs, frames = ctx.render_batch([], dev.trees[0], dev.trees[1:], dev.poses, dev.box_half)
    assert outs == [] and frames == []
    ctx.backward_batch([], [], dev.zero_grads())
    # a frame with a normal map goes through dvx_backward_n, not the batch
    rgb, depth, alpha, normal, fr = dev.render(normals=True)
    g = torch.zeros_like(rgb)
    with pytest.raises(dvx.DvxError) as e:
        ctx.backward_batch([fr], [g], dev.zero_grads())
    assert e.value.status == -5
    fr.release()
    # and the context still works
    outs, frames = ctx.render_batch([good, good], dev.trees[0], dev.trees[1:], dev.poses, dev.box_half)
    torch.cuda.synchronize()
    assert torch.equal(outs[0][0], outs[1][0]) and torch.equal(outs[0][0], rgb)
    for f in frames:
        f.release()
    for t in dev.trees:
        t.close()
