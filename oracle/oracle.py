"""ctypes front end of the CPU oracle (oracle/dvx_oracle.c).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module.  It never imports the CUDA package.
"""
import ctypes as C
import os
import subprocess
import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "dvx_oracle.c")
_LIB = os.path.join(_HERE, "libdvx_oracle.so")
_lib = None


def build(force=False):
    """gcc -O2 -fopenmp (never tuned; SURVEY.md §8(d) "CPU baseline beside it")."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-std=c99", "-shared", "-fPIC", "-o", _LIB, _SRC, "-lm"])
    return _LIB


class _Octree(C.Structure):
    _fields_ = [("n_voxels", C.c_uint32), ("sh_degree", C.c_uint32), ("center", C.c_double * 3), ("side", C.c_double),
                ("code", C.c_void_p), ("geo_f", C.c_void_p), ("geo_d", C.c_void_p), ("sh_f", C.c_void_p), ("sh_d", C.c_void_p)]


class _Camera(C.Structure):
    _fields_ = [("width", C.c_uint32), ("height", C.c_uint32), ("fx", C.c_double), ("fy", C.c_double), ("cx", C.c_double),
                ("cy", C.c_double), ("c2w", C.c_double * 12), ("near_", C.c_double), ("far_", C.c_double)]


class _Opts(C.Structure):
    _fields_ = [("k_samples", C.c_uint32), ("activation", C.c_uint32), ("t_stop", C.c_double), ("mode", C.c_uint32)]


class _Sky(C.Structure):
    _fields_ = [("width", C.c_uint32), ("height", C.c_uint32), ("tex", C.c_void_p), ("dtex", C.c_void_p)]


class _Grad(C.Structure):
    _fields_ = [("dgeo", C.c_void_p), ("dsh", C.c_void_p)]


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.orc_tile_hit_list.restype = C.c_int64
        _lib.orc_ray_segments.restype = C.c_int64
        _lib.orc_order_key.restype = C.c_uint64
        _lib.orc_order_key.argtypes = [C.c_uint64, C.c_int]
    return _lib


def num_threads():
    return int(lib().orc_num_threads())


def _ptr(a):
    return a.ctypes.data_as(C.c_void_p) if a is not None else None


class _Packed:
    """Keeps the numpy arrays alive next to the C structs built from a scene."""

    def __init__(self, scene, cam_index=0, mode=0, k_samples=None, activation=None, t_stop=None):
        trees = scene.octrees
        self.keep = []
        self.trees = (_Octree * len(trees))()
        for n, t in enumerate(trees):
            o = self.trees[n]
            o.n_voxels, o.sh_degree = t.n_voxels, t.sh_degree
            o.center = (C.c_double * 3)(*[float(x) for x in t.center])
            o.side = float(t.side)
            code = np.ascontiguousarray(t.code, dtype=np.uint64)
            geo, sh = np.ascontiguousarray(t.geo), np.ascontiguousarray(t.sh)
            self.keep += [code, geo, sh]
            o.code = _ptr(code)
            if geo.dtype == np.float64:
                o.geo_d = _ptr(geo)
            else:
                assert geo.dtype == np.float32
                o.geo_f = _ptr(geo)
            if sh.dtype == np.float64:
                o.sh_d = _ptr(sh)
            else:
                assert sh.dtype == np.float32
                o.sh_f = _ptr(sh)
        cam = scene.cameras[cam_index]
        self.cam = _Camera(cam.width, cam.height, cam.fx, cam.fy, cam.cx, cam.cy,
                           (C.c_double * 12)(*[float(x) for x in cam.c2w]), cam.near, cam.far)
        self.poses = np.ascontiguousarray(scene.poses, dtype=np.float64).reshape(-1)
        self.half = np.ascontiguousarray(scene.box_half, dtype=np.float64).reshape(-1)
        self.opts = _Opts(scene.k_samples if k_samples is None else k_samples,
                          scene.activation if activation is None else activation,
                          scene.t_stop if t_stop is None else t_stop, mode)
        self.n_trees = len(trees)
        self.hw = (cam.height, cam.width)


def render(scene, cam_index=0, mode=0, mask=None, grads_in=None, want_grads=None, sky=None, normals=False, **opt):
    """Forward (and backward when ``grads_in`` is given) in double precision.

    grads_in: dict with 'rgb' [H,W,3] and optional 'depth', 'alpha' [H,W].
    sky: optional equirectangular map [Hs,Ws,3] (O10 / Eq. 2, reading R21); with grads_in also returns 'dsky'.
    normals: also return the normal map 'normal' [H,W,3] (O11, reading R22); grads_in may then hold 'normal' [H,W,3].
    Returns dict(rgb, depth, alpha, n_used [, dgeo list, dsh list, dsky]).
    """
    p = _Packed(scene, cam_index, mode, **opt)
    H, W = p.hw
    rgb = np.zeros((H, W, 3)); depth = np.zeros((H, W)); alpha = np.zeros((H, W))
    n_used = np.zeros((H, W), dtype=np.uint32)
    m = None if mask is None else np.ascontiguousarray(mask, dtype=np.uint8)
    g_rgb = g_depth = g_alpha = None
    cgrads = None
    out = {}
    if grads_in is not None:
        g_rgb = np.ascontiguousarray(grads_in["rgb"], dtype=np.float64)
        g_depth = None if grads_in.get("depth") is None else np.ascontiguousarray(grads_in["depth"], dtype=np.float64)
        g_alpha = None if grads_in.get("alpha") is None else np.ascontiguousarray(grads_in["alpha"], dtype=np.float64)
        cgrads = (_Grad * p.n_trees)()
        out["dgeo"], out["dsh"] = [], []
        for n, t in enumerate(scene.octrees):
            dg = np.zeros((t.n_voxels, 8)); ds = np.zeros((t.n_voxels, t.n_sh, 3))
            out["dgeo"].append(dg); out["dsh"].append(ds)
            cgrads[n].dgeo, cgrads[n].dsh = _ptr(dg), _ptr(ds)
    csky = None
    if sky is not None:
        tex = np.ascontiguousarray(sky, dtype=np.float64)
        assert tex.ndim == 3 and tex.shape[2] == 3
        dtex = np.zeros_like(tex) if grads_in is not None else None
        csky = C.byref(_Sky(tex.shape[1], tex.shape[0], _ptr(tex), _ptr(dtex)))
        if dtex is not None:
            out["dsky"] = dtex
    normal = np.zeros((H, W, 3)) if (normals or (grads_in is not None and grads_in.get("normal") is not None)) else None
    g_normal = None
    if grads_in is not None and grads_in.get("normal") is not None:
        g_normal = np.ascontiguousarray(grads_in["normal"], dtype=np.float64)
    rc = lib().orc_render_full(C.byref(p.cam), p.n_trees, p.trees, _ptr(p.poses), _ptr(p.half), C.byref(p.opts), _ptr(m),
                               _ptr(rgb), _ptr(depth), _ptr(alpha), _ptr(g_rgb), _ptr(g_depth), _ptr(g_alpha), cgrads,
                               _ptr(n_used), csky, _ptr(normal), _ptr(g_normal))
    if normal is not None:
        out["normal"] = normal
    if rc != 0:
        raise ValueError("orc_render: invalid arguments")
    out.update(rgb=rgb, depth=depth, alpha=alpha, n_used=n_used)
    return out


class _Feat(C.Structure):
    _fields_ = [("n_channels", C.c_uint32), ("feat", C.POINTER(C.c_void_p)), ("out", C.c_void_p), ("img", C.c_void_p),
                ("num", C.POINTER(C.c_void_p)), ("wsum", C.POINTER(C.c_void_p))]


def render_features(scene, feats=None, img=None, cam_index=0, mode=0, mask=None, **opt):
    """O12 (row N3, reading R25).  feats: list of [V_t, C] arrays per octree -> 'features' [H,W,C] = sum_j T_j alpha_j f_j.
    img: [H,W,C] 2-D features -> 'num' (list of [V_t,C]) and 'wsum' (list of [V_t]): the fuse pass, the transpose of the
    feature render.  Also returns 'alpha'.  Double precision."""
    p = _Packed(scene, cam_index, mode, **opt)
    H, W = p.hw
    nt = p.n_trees
    fx = _Feat()
    out = {}
    keep = []
    if feats is not None:
        fs = [np.ascontiguousarray(f, dtype=np.float64) for f in feats]
        n_ch = fs[0].shape[1] if fs[0].ndim == 2 else int(np.asarray(feats[0]).shape[-1])
        assert all(f.shape == (t.n_voxels, n_ch) for f, t in zip(fs, scene.octrees))
        arr = (C.c_void_p * nt)(*[f.ctypes.data for f in fs])
        fx.feat = C.cast(arr, C.POINTER(C.c_void_p))
        F = np.zeros((H, W, n_ch))
        fx.out = _ptr(F)
        out["features"] = F
        keep += [fs, arr]
    if img is not None:
        im = np.ascontiguousarray(img, dtype=np.float64)
        n_ch = im.shape[2]
        assert im.shape == (H, W, n_ch)
        num = [np.zeros((t.n_voxels, n_ch)) for t in scene.octrees]
        ws = [np.zeros(t.n_voxels) for t in scene.octrees]
        a1 = (C.c_void_p * nt)(*[a.ctypes.data for a in num])
        a2 = (C.c_void_p * nt)(*[a.ctypes.data for a in ws])
        fx.img, fx.num, fx.wsum = _ptr(im), C.cast(a1, C.POINTER(C.c_void_p)), C.cast(a2, C.POINTER(C.c_void_p))
        out["num"], out["wsum"] = num, ws
        keep += [im, a1, a2]
    fx.n_channels = n_ch
    alpha = np.zeros((H, W))
    m = None if mask is None else np.ascontiguousarray(mask, dtype=np.uint8)
    rc = lib().orc_render_features(C.byref(p.cam), p.n_trees, p.trees, _ptr(p.poses), _ptr(p.half), C.byref(p.opts), _ptr(m),
                                   C.byref(fx), _ptr(alpha))
    if rc != 0:
        raise ValueError("orc_render_features: invalid arguments")
    out["alpha"] = alpha
    return out


def tile_hit_list(scene, tx, ty, tree, octant, cam_index=0):
    p = _Packed(scene, cam_index, 0)
    cap = scene.octrees[tree].n_voxels
    ids = np.zeros(max(cap, 1), dtype=np.uint32)
    n = lib().orc_tile_hit_list(C.byref(p.cam), p.n_trees, p.trees, _ptr(p.poses), _ptr(p.half), C.byref(p.opts),
                                int(tx), int(ty), int(tree), int(octant), _ptr(ids), C.c_int64(cap))
    return ids[:n].copy()


def ray_segments(scene, u, v, cam_index=0, cap=1 << 16):
    p = _Packed(scene, cam_index, 0)
    tree = np.zeros(cap, dtype=np.uint32); vox = np.zeros(cap, dtype=np.uint32)
    a = np.zeros(cap); b = np.zeros(cap)
    n = lib().orc_ray_segments(C.byref(p.cam), p.n_trees, p.trees, _ptr(p.poses), _ptr(p.half), C.byref(p.opts),
                               int(u), int(v), _ptr(tree), _ptr(vox), _ptr(a), _ptr(b), C.c_int64(cap))
    n = min(n, cap)
    return tree[:n], vox[:n], a[:n], b[:n]


def sky_footprint(width, height, direction):
    d = (C.c_double * 3)(*[float(x) for x in direction])
    idx = (C.c_int64 * 4)(); wt = (C.c_double * 4)()
    lib().orc_sky_footprint(C.c_uint32(width), C.c_uint32(height), d, idx, wt)
    return np.array(list(idx)), np.array(list(wt))


def order_key(code, q):
    return np.array([lib().orc_order_key(int(c), int(q)) for c in np.atleast_1d(code)], dtype=np.uint64)


def sh_basis(direction):
    d = (C.c_double * 3)(*[float(x) for x in direction])
    Y = (C.c_double * 16)()
    lib().orc_sh_basis(d, Y)
    return np.array(list(Y))


def ray(scene, u, v, cam_index=0):
    p = _Packed(scene, cam_index, 0)
    o = (C.c_double * 3)(); d = (C.c_double * 3)()
    lib().orc_ray(C.byref(p.cam), int(u), int(v), o, d)
    return np.array(list(o)), np.array(list(d))


def ray_box(pose, half, o, d, near=0.05, far=1e9):
    P = (C.c_double * 12)(*[float(x) for x in np.asarray(pose).reshape(12)])
    h = (C.c_double * 3)(*[float(x) for x in half])
    oo = (C.c_double * 3)(*[float(x) for x in o]); dd = (C.c_double * 3)(*[float(x) for x in d])
    tin = C.c_double(); tout = C.c_double()
    hit = lib().orc_ray_box(P, h, oo, dd, C.c_double(near), C.c_double(far), C.byref(tin), C.byref(tout))
    return (tin.value, tout.value) if hit else None
