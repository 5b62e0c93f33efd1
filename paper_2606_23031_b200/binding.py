"""Thin ctypes binding of libdvx.so (include/dvx.h): argument marshalling only.

Every step of the hot path runs in the CUDA kernels behind the C ABI; PyTorch is used for device memory
(``torch.empty`` through the allocator callbacks) and the stream.  There is no CPU fallback: importing works
anywhere (so the symbol table can be checked), but creating a ``Context`` without a CUDA device raises.
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libdvx.so")

DVX_OK = 0
ERRORS = {-1: "DVX_ERR_INVALID_ARG", -2: "DVX_ERR_BAD_OCTREE", -3: "DVX_ERR_OOM", -4: "DVX_ERR_CUDA",
          -5: "DVX_ERR_NOT_IMPLEMENTED"}
STAGES = ("preprocess", "sort", "composite", "backward", "backward_composite", "backward_sh", "gap_host_sync", "gap_fwd_bwd")
FLAG_COUNTERS = 1
FLAG_NAIVE = 2
FLAG_NO_RECORDS = 4

EXPORTS = ["dvx_create", "dvx_destroy", "dvx_octree_create", "dvx_octree_refresh_structure", "dvx_octree_destroy",
           "dvx_render", "dvx_backward", "dvx_backward_n", "dvx_frame_release", "dvx_debug_tile_list", "dvx_frame_counters",
           "dvx_frame_stage_ms", "dvx_last_error", "dvx_sort_pairs", "dvx_launch_count", "dvx_stage_ms_collect", "dvx_render_host",
           "dvx_backward_host", "dvx_grid_create", "dvx_grid_destroy", "dvx_grid_gather", "dvx_grid_reduce",
           "dvx_grid_adam_step", "dvx_adam_step", "dvx_grid_adam_step_n", "dvx_adam_step_n",
           "dvx_frame_weights", "dvx_render_features", "dvx_fuse_features",
           "dvx_cloud_create", "dvx_cloud_destroy", "dvx_density_prior", "dvx_subdivide_near", "dvx_prune",
           "dvx_set_record_budget", "dvx_frame_record_stats", "dvx_trim", "dvx_microbench_fma", "dvx_render_batch", "dvx_backward_batch", "dvx_subdivide_fill", "dvx_sort_pairs_no_alloc", "dvx_host_io_wait"]


class DvxError(RuntimeError):
    def __init__(self, status, text):
        super().__init__("%s (%d): %s" % (ERRORS.get(status, "?"), status, text))
        self.status = status


class OctreeDesc(C.Structure):
    _fields_ = [("n_voxels", C.c_uint32), ("sh_degree", C.c_uint32), ("center", C.c_float * 3), ("side", C.c_float),
                ("code", C.c_void_p), ("geo", C.c_void_p), ("sh", C.c_void_p)]


class Camera(C.Structure):
    _fields_ = [("width", C.c_uint32), ("height", C.c_uint32), ("fx", C.c_float), ("fy", C.c_float), ("cx", C.c_float),
                ("cy", C.c_float), ("c2w", C.c_float * 12), ("near_", C.c_float), ("far_", C.c_float)]


class Sky(C.Structure):
    _fields_ = [("width", C.c_uint32), ("height", C.c_uint32), ("tex", C.c_void_p), ("dtex", C.c_void_p)]


class RenderOpts(C.Structure):
    _fields_ = [("k_samples", C.c_uint32), ("activation", C.c_uint32), ("t_stop", C.c_float), ("flags", C.c_uint32),
                ("sky", C.POINTER(Sky))]


class Image(C.Structure):
    _fields_ = [("rgb", C.c_void_p), ("depth", C.c_void_p), ("alpha", C.c_void_p), ("normal", C.c_void_p)]


class Grad(C.Structure):
    _fields_ = [("dgeo", C.c_void_p), ("dsh", C.c_void_p)]


class GridTables(C.Structure):
    _fields_ = [("n_points", C.c_uint32), ("point_of", C.c_void_p), ("offsets", C.c_void_p), ("slots", C.c_void_p)]


class Adam(C.Structure):
    _fields_ = [("lr", C.c_float), ("beta1", C.c_float), ("beta2", C.c_float), ("eps", C.c_float), ("step", C.c_uint32)]


class Weights(C.Structure):
    _fields_ = [("nnz", C.c_uint64), ("row_start", C.c_void_p), ("voxel", C.c_void_p), ("weight", C.c_void_p)]


class GridAdamItem(C.Structure):
    _fields_ = [("grid", C.c_void_p), ("density", C.c_void_p), ("m", C.c_void_p), ("v", C.c_void_p), ("dgeo", C.c_void_p),
                ("geo", C.c_void_p)]


class AdamItem(C.Structure):
    _fields_ = [("n", C.c_uint64), ("p", C.c_void_p), ("m", C.c_void_p), ("v", C.c_void_p), ("g", C.c_void_p)]


ALLOC_FN = C.CFUNCTYPE(C.c_void_p, C.c_size_t, C.c_void_p)
FREE_FN = C.CFUNCTYPE(None, C.c_void_p, C.c_void_p)

_lib = None


def load():
    """dlopen libdvx.so (built in-tree by paper_2606_23031_b200.build) and declare the signatures."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError("libdvx.so is missing: run `python -m paper_2606_23031_b200.build` (there is no CPU fallback)")
    lib = C.CDLL(LIB_PATH)
    P = C.c_void_p
    lib.dvx_create.argtypes = [C.c_int, P, ALLOC_FN, FREE_FN, P, C.POINTER(P)]
    lib.dvx_destroy.argtypes = [P]
    lib.dvx_destroy.restype = None
    lib.dvx_octree_create.argtypes = [P, C.POINTER(OctreeDesc), C.POINTER(P)]
    lib.dvx_octree_refresh_structure.argtypes = [P, P, C.POINTER(OctreeDesc)]
    lib.dvx_octree_destroy.argtypes = [P, P]
    lib.dvx_octree_destroy.restype = None
    lib.dvx_render.argtypes = [P, C.POINTER(Camera), P, C.c_uint32, C.POINTER(P), P, P, C.POINTER(RenderOpts), Image,
                               C.POINTER(P)]
    lib.dvx_backward.argtypes = [P, P, P, P, P, Grad, C.POINTER(Grad)]
    lib.dvx_backward_n.argtypes = [P, P, P, P, P, P, Grad, C.POINTER(Grad)]
    lib.dvx_frame_release.argtypes = [P, P]
    lib.dvx_frame_release.restype = None
    lib.dvx_debug_tile_list.argtypes = [P, P, C.c_uint32, C.c_uint32, C.c_uint32, P, C.c_uint32, C.POINTER(C.c_uint32)]
    lib.dvx_frame_counters.argtypes = [P, P] + [C.POINTER(C.c_uint64)] * 5
    lib.dvx_frame_stage_ms.argtypes = [P, P, C.POINTER(C.c_float)]
    lib.dvx_last_error.argtypes = [P]
    lib.dvx_last_error.restype = C.c_char_p
    lib.dvx_sort_pairs.argtypes = [P, P, P, C.c_uint64, C.c_uint32]
    lib.dvx_launch_count.argtypes = []
    lib.dvx_stage_ms_collect.argtypes = [P, C.POINTER(C.c_float), C.POINTER(C.c_uint32)]
    lib.dvx_render_host.argtypes = lib.dvx_render.argtypes
    lib.dvx_backward_host.argtypes = lib.dvx_backward.argtypes
    lib.dvx_grid_create.argtypes = [P, P, C.c_uint32, C.POINTER(P), C.POINTER(GridTables)]
    lib.dvx_grid_destroy.argtypes = [P, P]
    lib.dvx_grid_destroy.restype = None
    lib.dvx_grid_gather.argtypes = [P, P, P, P]
    lib.dvx_grid_reduce.argtypes = [P, P, P, P]
    lib.dvx_grid_adam_step.argtypes = [P, P, C.POINTER(Adam), P, P, P, P, P]
    lib.dvx_adam_step.argtypes = [P, C.POINTER(Adam), C.c_uint64, P, P, P, P]
    lib.dvx_frame_weights.argtypes = [P, P, C.POINTER(Weights)]
    lib.dvx_render_features.argtypes = [P, P, C.c_uint32, P, P]
    lib.dvx_fuse_features.argtypes = [P, P, C.c_uint32, P, P, P]
    lib.dvx_cloud_create.argtypes = [P, P, C.c_uint64, C.c_float, C.POINTER(P)]
    lib.dvx_cloud_destroy.argtypes = [P, P]
    lib.dvx_cloud_destroy.restype = None
    lib.dvx_density_prior.argtypes = [P, P, C.POINTER(OctreeDesc), P, C.c_float, C.c_float, C.c_float, P]
    lib.dvx_subdivide_near.argtypes = [P, P, C.POINTER(OctreeDesc), C.c_float, C.c_uint32, P, C.c_uint64, C.POINTER(C.c_uint64), P]
    lib.dvx_prune.argtypes = [P, C.c_uint32, P, P, C.c_float, P, P, C.POINTER(C.c_uint32)]
    lib.dvx_grid_adam_step_n.argtypes = [P, C.POINTER(Adam), C.c_uint32, C.POINTER(GridAdamItem)]
    lib.dvx_adam_step_n.argtypes = [P, C.POINTER(Adam), C.c_uint32, C.POINTER(AdamItem)]
    lib.dvx_render_batch.argtypes = [P, C.c_uint32, C.POINTER(Camera), P, C.c_uint32, C.POINTER(P), P, P, C.POINTER(RenderOpts),
                                     C.POINTER(Image), C.POINTER(P)]
    lib.dvx_backward_batch.argtypes = [P, C.c_uint32, C.POINTER(P), C.POINTER(P), C.POINTER(P), C.POINTER(P), Grad, C.POINTER(Grad)]
    lib.dvx_subdivide_fill.argtypes = [P, C.c_uint32, P, P, P, C.c_uint32, P, P, C.c_uint64, C.POINTER(C.c_uint64)]
    lib.dvx_sort_pairs_no_alloc.argtypes = [C.c_int, P, P, P, C.c_uint64, C.c_uint32, C.c_char_p, C.c_size_t]
    lib.dvx_host_io_wait.argtypes = [P]
    lib.dvx_trim.argtypes = [P, C.POINTER(C.c_uint64)]
    lib.dvx_microbench_fma.argtypes = [P, C.c_uint32, C.POINTER(C.c_double), C.POINTER(C.c_double), C.POINTER(C.c_float)]
    lib.dvx_set_record_budget.argtypes = [P, C.c_uint64]
    lib.dvx_frame_record_stats.argtypes = [P, P, C.POINTER(C.c_uint64), C.POINTER(C.c_uint64), C.POINTER(C.c_uint32)]
    for name in EXPORTS:
        if name not in ("dvx_destroy", "dvx_octree_destroy", "dvx_frame_release", "dvx_last_error", "dvx_launch_count",
                        "dvx_grid_destroy", "dvx_cloud_destroy"):
            getattr(lib, name).restype = C.c_int32
    lib.dvx_launch_count.restype = C.c_uint64
    _lib = lib
    return lib


SORT_NO_ALLOC_MAX_PAIRS = 1 << 20


def sort_pairs_no_alloc(keys, vals, key_bits, device=0, stream_ptr=None):
    """dvx_sort_pairs_no_alloc: sorts CUDA int64 keys / int32 vals in place using the library's static scratch (no context,
    no allocation; at most SORT_NO_ALLOC_MAX_PAIRS pairs).  Raises DvxError with the library's message."""
    lib = load()
    buf = C.create_string_buffer(256)
    n = int(keys.shape[0])
    rc = lib.dvx_sort_pairs_no_alloc(device, C.c_void_p(stream_ptr), keys.data_ptr() if n else None, vals.data_ptr() if n else None,
                                     n, key_bits, buf, 256)
    if rc != DVX_OK:
        raise DvxError(rc, buf.value.decode())


class Context:
    """dvx_create on a CUDA device; device scratch comes from the PyTorch caching allocator."""

    def __init__(self, device=0, stream=None, torch_alloc=True):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("libdvx needs a CUDA device (sm_100a); there is no CPU fallback")
        self.lib = load()
        self.torch = torch
        self.device = torch.device("cuda", device)
        self._blocks = {}
        self._alloc_cb = ALLOC_FN(self._alloc)
        self._free_cb = FREE_FN(self._free)
        self.stream = stream
        handle = C.c_void_p()
        with torch.cuda.device(self.device):
            st = stream.cuda_stream if stream is not None else torch.cuda.current_stream().cuda_stream
        self._stream_ptr = st
        if torch_alloc:
            rc = self.lib.dvx_create(device, C.c_void_p(st), self._alloc_cb, self._free_cb, None, C.byref(handle))
        else:
            rc = self.lib.dvx_create(device, C.c_void_p(st), ALLOC_FN(0), FREE_FN(0), None, C.byref(handle))
        if rc != DVX_OK:
            raise DvxError(rc, "dvx_create failed")
        self.h = handle

    def _alloc(self, nbytes, _user):
        try:
            t = self.torch.empty(int(nbytes), dtype=self.torch.uint8, device=self.device)
        except Exception:  # out of memory -> NULL -> DVX_ERR_OOM
            return None
        self._blocks[t.data_ptr()] = t
        return t.data_ptr()

    def _free(self, ptr, _user):
        self._blocks.pop(ptr, None)

    def stage_ms_collect(self):
        """Sum of the stage times of all frames released since the last call -> (dict of ms sums, n_frames)."""
        ms = (C.c_float * 8)()
        n = C.c_uint32()
        self.check(self.lib.dvx_stage_ms_collect(self.h, ms, C.byref(n)))
        return dict(zip(STAGES, list(ms)[:8])), n.value

    def microbench_fma(self, iters=1 << 14):
        """dvx_microbench_fma -> dict(lane_fma_per_s, warp_instr_per_s, ms)."""
        a, b, ms = C.c_double(), C.c_double(), C.c_float()
        self.check(self.lib.dvx_microbench_fma(self.h, iters, C.byref(a), C.byref(b), C.byref(ms)))
        return {"lane_fma_per_s": a.value, "warp_instr_per_s": b.value, "ms": ms.value}

    def host_io_wait(self):
        """dvx_host_io_wait: the context's stream waits for every host copy-out still in flight."""
        self.check(self.lib.dvx_host_io_wait(self.h))

    def trim(self):
        """dvx_trim: hand every cached scratch block back to the allocator -> bytes freed."""
        n = C.c_uint64()
        self.check(self.lib.dvx_trim(self.h, C.byref(n)))
        return n.value

    def set_record_budget(self, nbytes):
        """dvx_set_record_budget: bytes of hit records per saved frame (0 = automatic sizing)."""
        self.check(self.lib.dvx_set_record_budget(self.h, int(nbytes)))

    def check(self, rc):
        if rc != DVX_OK:
            raise DvxError(rc, self.lib.dvx_last_error(self.h).decode())

    def close(self):
        if self.h:
            self.lib.dvx_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ------------------------------------------------------------------ octrees
    def octree(self, code, geo, sh, center, side, sh_degree):
        return Octree(self, code, geo, sh, center, side, sh_degree)

    # ------------------------------------------------------------------ row N2: grid points + optimizer
    def grid(self, code):
        """dvx_grid_create for a CUDA uint64 (stored as int64) code tensor [V]."""
        return Grid(self, code)

    def adam_step(self, p, m, v, g, lr, beta1, beta2, eps, step):
        """dvx_adam_step over contiguous CUDA float32 tensors of equal size; g is zeroed."""
        hp = Adam(lr, beta1, beta2, eps, step)
        self.check(self.lib.dvx_adam_step(self.h, C.byref(hp), p.numel(), p.data_ptr(), m.data_ptr(), v.data_ptr(),
                                          g.data_ptr()))

    # ------------------------------------------------------------------ row N4: LiDAR-guided structure operations
    def cloud(self, points, cell):
        """dvx_cloud_create for a CUDA float32 [n, 3] tensor of points in the octree's frame."""
        return Cloud(self, points, cell)

    @staticmethod
    def _structure_desc(code, center, side):
        n = int(code.shape[0])
        return OctreeDesc(n, 0, (C.c_float * 3)(*[float(x) for x in center]), float(side), code.data_ptr() if n else None, None, None)

    def density_prior(self, cloud, code, center, side, grid, s_min, v_close=-2.0, v_far=-10.0):
        """dvx_density_prior (Eq. 1) -> CUDA float32 [G]."""
        out = self.torch.empty(grid.n_points, dtype=self.torch.float32, device=self.device)
        desc = self._structure_desc(code, center, side)
        self.check(self.lib.dvx_density_prior(self.h, cloud.h, C.byref(desc), grid.h, s_min, v_close, v_far, out.data_ptr()))
        return out

    def subdivide_near(self, cloud, code, center, side, threshold, max_level=16):
        """dvx_subdivide_near -> (new codes int64 [V'], split uint8 [V])."""
        torch = self.torch
        n = int(code.shape[0])
        desc = self._structure_desc(code, center, side)
        out = torch.empty(8 * n, dtype=torch.int64, device=self.device)
        split = torch.zeros(n, dtype=torch.uint8, device=self.device)
        n_out = C.c_uint64()
        self.check(self.lib.dvx_subdivide_near(self.h, cloud.h, C.byref(desc), threshold, max_level, out.data_ptr(), 8 * n,
                                               C.byref(n_out), split.data_ptr()))
        return out[:n_out.value], split

    def subdivide_fill(self, split, geo, sh, sh_degree, n_out):
        """dvx_subdivide_fill -> (geo [n_out, 8], sh [n_out, C_sh, 3]) of the leaves after the round (n_out from subdivide_near)."""
        torch = self.torch
        n = int(split.shape[0])
        geo_out = torch.empty((n_out, 8), dtype=torch.float32, device=self.device)
        sh_out = torch.empty((n_out,) + tuple(sh.shape[1:]), dtype=torch.float32, device=self.device)
        got = C.c_uint64()
        self.check(self.lib.dvx_subdivide_fill(self.h, n, split.data_ptr(), geo.data_ptr(), sh.data_ptr(), sh_degree,
                                               geo_out.data_ptr(), sh_out.data_ptr(), n_out, C.byref(got)))
        assert got.value == n_out
        return geo_out, sh_out

    def prune(self, code, geo, threshold):
        """dvx_prune -> (kept codes int64 [V'], kept indices int32 [V'])."""
        torch = self.torch
        n = int(code.shape[0])
        out = torch.empty(n, dtype=torch.int64, device=self.device)
        idx = torch.empty(n, dtype=torch.int32, device=self.device)
        n_out = C.c_uint32()
        self.check(self.lib.dvx_prune(self.h, n, code.data_ptr(), geo.data_ptr(), threshold, out.data_ptr(), idx.data_ptr(),
                                      C.byref(n_out)))
        return out[:n_out.value], idx[:n_out.value]

    def grid_adam_step_n(self, items, lr, beta1, beta2, eps, step):
        """dvx_grid_adam_step_n: items = [(Grid, density, m, v, dgeo, geo), ...], all octrees in one launch."""
        hp = Adam(lr, beta1, beta2, eps, step)
        arr = (GridAdamItem * max(len(items), 1))(*[GridAdamItem(g.h, *[t.data_ptr() for t in ts]) for g, *ts in items])
        self.check(self.lib.dvx_grid_adam_step_n(self.h, C.byref(hp), len(items), arr))

    def adam_step_n(self, items, lr, beta1, beta2, eps, step):
        """dvx_adam_step_n: items = [(p, m, v, g), ...] contiguous CUDA float32 tensors."""
        hp = Adam(lr, beta1, beta2, eps, step)
        arr = (AdamItem * max(len(items), 1))(*[AdamItem(p.numel(), p.data_ptr(), m.data_ptr(), v.data_ptr(), g.data_ptr())
                                                for p, m, v, g in items])
        self.check(self.lib.dvx_adam_step_n(self.h, C.byref(hp), len(items), arr))

    # ------------------------------------------------------------------ batched render / backward (config 5)
    def render_batch(self, cams, static, actors=(), poses=None, box_half=None, k_samples=8, activation=0, t_stop=1e-4, flags=0,
                     save=True, outs=None):
        """dvx_render_batch: cams = list of binding.Camera; outs = list of (rgb, depth, alpha) device tensors or None.
        Returns (list of (rgb, depth, alpha), list of Frame or None)."""
        torch = self.torch
        n_c = len(cams)
        if outs is None:
            outs = [(torch.empty((c.height, c.width, 3), dtype=torch.float32, device=self.device),
                     torch.empty((c.height, c.width), dtype=torch.float32, device=self.device),
                     torch.empty((c.height, c.width), dtype=torch.float32, device=self.device)) for c in cams]
        n = len(actors)
        handles = (C.c_void_p * max(n, 1))(*[a.h for a in actors])
        poses = np.ascontiguousarray(np.zeros((0, 12)) if poses is None else poses, dtype=np.float32).reshape(-1)
        half = np.ascontiguousarray(np.zeros((0, 3)) if box_half is None else box_half, dtype=np.float32).reshape(-1)
        assert poses.size == 12 * n and half.size == 3 * n
        opts = RenderOpts(k_samples, activation, t_stop, flags, None)
        cam_arr = (Camera * n_c)(*cams)
        img_arr = (Image * n_c)(*[Image(o[0].data_ptr(), o[1].data_ptr(), o[2].data_ptr(), None) for o in outs])
        fh = (C.c_void_p * n_c)()
        self.check(self.lib.dvx_render_batch(self.h, n_c, cam_arr, static.h, n, handles, poses.ctypes.data_as(C.c_void_p),
                                             half.ctypes.data_as(C.c_void_p), C.byref(opts), img_arr, fh if save else None))
        frames = [Frame(self, C.c_void_p(fh[i]), [static] + list(actors)) for i in range(n_c)] if save else None
        return outs, frames

    def backward_batch(self, frames, dL_drgb, grads, dL_ddepth=None, dL_dalpha=None):
        """dvx_backward_batch: frames / dL_drgb lists of equal length; grads = list of (dgeo, dsh) per octree (accumulated)."""
        n_f = len(frames)
        ptrs = lambda ts: None if ts is None else (C.c_void_p * n_f)(*[None if t is None else t.data_ptr() for t in ts])
        g = [Grad(a.data_ptr() if a is not None else None, b.data_ptr() if b is not None else None) for a, b in grads]
        arr = (Grad * max(len(g) - 1, 1))(*g[1:])
        fr = (C.c_void_p * n_f)(*[f.h for f in frames])
        self.check(self.lib.dvx_backward_batch(self.h, n_f, fr, ptrs(dL_drgb), ptrs(dL_ddepth), ptrs(dL_dalpha), g[0], arr))
        return grads

    # ------------------------------------------------------------------ render / backward
    def render(self, cam, static, actors=(), poses=None, box_half=None, k_samples=8, activation=0, t_stop=1e-4, flags=0,
               save=True, out=None, host=False, sky=None, dsky=None, normals=False):
        """dvx_render (host=False: device image tensors) or dvx_render_host (host=True: ``out`` must be three pinned
        CPU tensors).  cam: binding.Camera; poses [N,12] / box_half [N,3] host float32 arrays.
        sky: optional CUDA float32 tensor [Hs,Ws,3] (Eq. 2); dsky: tensor of the same shape that dvx_backward accumulates
        the texture gradient into.  normals=True also renders the normal map (O11) and returns
        (rgb, depth, alpha, normal [H,W,3], Frame or None) instead of (rgb [H,W,3], depth [H,W], alpha [H,W], Frame or None)."""
        torch = self.torch
        H, W = cam.height, cam.width
        if host and out is None:
            out = (torch.empty((H, W, 3), dtype=torch.float32).pin_memory(), torch.empty((H, W), dtype=torch.float32).pin_memory(),
                   torch.empty((H, W), dtype=torch.float32).pin_memory())
        if out is None:
            rgb = torch.empty((H, W, 3), dtype=torch.float32, device=self.device)
            depth = torch.empty((H, W), dtype=torch.float32, device=self.device)
            alpha = torch.empty((H, W), dtype=torch.float32, device=self.device)
        else:
            rgb, depth, alpha = out
        n = len(actors)
        handles = (C.c_void_p * max(n, 1))(*[a.h for a in actors])
        poses = np.ascontiguousarray(np.zeros((0, 12)) if poses is None else poses, dtype=np.float32).reshape(-1)
        half = np.ascontiguousarray(np.zeros((0, 3)) if box_half is None else box_half, dtype=np.float32).reshape(-1)
        assert poses.size == 12 * n and half.size == 3 * n
        opts = RenderOpts(k_samples, activation, t_stop, flags, None)
        if sky is not None:
            assert sky.is_cuda and sky.dtype == torch.float32 and sky.dim() == 3 and sky.shape[2] == 3 and sky.is_contiguous()
            csky = Sky(sky.shape[1], sky.shape[0], sky.data_ptr(), dsky.data_ptr() if dsky is not None else None)
            opts.sky = C.pointer(csky)
        normal = None
        if normals:
            normal = torch.empty((H, W, 3), dtype=torch.float32).pin_memory() if host else \
                torch.empty((H, W, 3), dtype=torch.float32, device=self.device)
        img = Image(rgb.data_ptr(), depth.data_ptr(), alpha.data_ptr(), normal.data_ptr() if normals else None)
        fh = C.c_void_p()
        fn = self.lib.dvx_render_host if host else self.lib.dvx_render
        rc = fn(self.h, C.byref(cam), static.h, n, handles, poses.ctypes.data_as(C.c_void_p),
                half.ctypes.data_as(C.c_void_p), C.byref(opts), img, C.byref(fh) if save else None)
        self.check(rc)
        frame = Frame(self, fh, [static] + list(actors)) if save else None
        if frame is not None:
            frame.keep = (sky, dsky)   # the library borrows these until the frame is released
        if normals:
            return rgb, depth, alpha, normal, frame
        return rgb, depth, alpha, frame


class Octree:
    """dvx_octree_create over caller-owned CUDA tensors (kept alive here)."""

    def __init__(self, ctx, code, geo, sh, center, side, sh_degree):
        torch = ctx.torch
        self.ctx = ctx
        self.code = code.contiguous()
        self.geo = geo.contiguous()
        self.sh = sh.contiguous()
        assert self.code.dtype in (torch.int64, torch.uint64) and self.geo.dtype == torch.float32 and self.sh.dtype == torch.float32
        self.n_voxels = int(self.code.shape[0])
        self.sh_degree = int(sh_degree)
        self.n_sh = (self.sh_degree + 1) ** 2
        self.desc = OctreeDesc(self.n_voxels, self.sh_degree, (C.c_float * 3)(*[float(x) for x in center]), float(side),
                               self.code.data_ptr() if self.n_voxels else None,
                               self.geo.data_ptr() if self.n_voxels else None,
                               self.sh.data_ptr() if self.n_voxels else None)
        h = C.c_void_p()
        ctx.check(ctx.lib.dvx_octree_create(ctx.h, C.byref(self.desc), C.byref(h)))
        self.h = h

    def close(self):
        if self.h and self.ctx.h:
            self.ctx.lib.dvx_octree_destroy(self.ctx.h, self.h)
        self.h = None


class Cloud:
    """LiDAR points binned into a uniform cell grid (dvx_cloud_create)."""

    def __init__(self, ctx, points, cell):
        self.ctx = ctx
        points = points.contiguous()
        h = C.c_void_p()
        n = int(points.shape[0])
        ctx.check(ctx.lib.dvx_cloud_create(ctx.h, points.data_ptr() if n else None, n, cell, C.byref(h)))
        self.h = h

    def close(self):
        if self.h and self.ctx.h:
            self.ctx.lib.dvx_cloud_destroy(self.ctx.h, self.h)
        self.h = None


class Grid:
    """Grid-point tables of one octree (dvx_grid_create): argument marshalling only."""

    def __init__(self, ctx, code):
        self.ctx = ctx
        self.n_voxels = int(code.shape[0])
        h = C.c_void_p()
        self.tables = GridTables()
        ctx.check(ctx.lib.dvx_grid_create(ctx.h, code.data_ptr() if self.n_voxels else None, self.n_voxels, C.byref(h),
                                          C.byref(self.tables)))
        self.h = h
        self.n_points = int(self.tables.n_points)

    def _view(self, ptr, n):
        """The library allocated the table through this context's torch allocator: view that block, no copy."""
        torch = self.ctx.torch
        if n == 0:
            return torch.empty(0, dtype=torch.int32, device=self.ctx.device)
        block = self.ctx._blocks.get(ptr)
        if block is None:
            raise RuntimeError("grid tables are only viewable with torch_alloc=True")
        return block.view(torch.int32)[:n]

    def point_of(self):
        return self._view(self.tables.point_of, self.n_voxels * 8).view(self.n_voxels, 8)

    def offsets(self):
        return self._view(self.tables.offsets, self.n_points + 1)

    def slots(self):
        return self._view(self.tables.slots, self.n_voxels * 8)

    def gather(self, density, geo):
        self.ctx.check(self.ctx.lib.dvx_grid_gather(self.ctx.h, self.h, density.data_ptr(), geo.data_ptr()))

    def reduce(self, dgeo, ddensity):
        self.ctx.check(self.ctx.lib.dvx_grid_reduce(self.ctx.h, self.h, dgeo.data_ptr(), ddensity.data_ptr()))

    def adam_step(self, density, m, v, dgeo, geo, lr, beta1, beta2, eps, step):
        hp = Adam(lr, beta1, beta2, eps, step)
        self.ctx.check(self.ctx.lib.dvx_grid_adam_step(self.ctx.h, self.h, C.byref(hp), density.data_ptr(), m.data_ptr(),
                                                       v.data_ptr(), dgeo.data_ptr(), geo.data_ptr()))

    def close(self):
        if self.h and self.ctx.h:
            self.ctx.lib.dvx_grid_destroy(self.ctx.h, self.h)
        self.h = None


class Frame:
    def __init__(self, ctx, h, trees):
        self.ctx, self.h, self.trees = ctx, h, trees

    def backward(self, dL_drgb, dL_ddepth=None, dL_dalpha=None, grads=None, host=False, dL_dnormal=None):
        """dvx_backward (device image gradients) or dvx_backward_host (host=True: pinned CPU tensors).
        grads: list of (dgeo, dsh) tensors per octree (accumulated into); None = fresh zeros.
        Returns the list of (dgeo, dsh)."""
        ctx, torch = self.ctx, self.ctx.torch
        if grads is None:
            grads = [(torch.zeros((t.n_voxels, 8), dtype=torch.float32, device=ctx.device),
                      torch.zeros((t.n_voxels, t.n_sh, 3), dtype=torch.float32, device=ctx.device)) for t in self.trees]
        g = [Grad(a.data_ptr() if a is not None else None, b.data_ptr() if b is not None else None) for a, b in grads]
        n = len(self.trees) - 1
        arr = (Grad * max(n, 1))(*g[1:])
        ptr = lambda t: None if t is None else t.data_ptr()
        if dL_dnormal is not None:
            assert not host
            ctx.check(ctx.lib.dvx_backward_n(ctx.h, self.h, ptr(dL_drgb), ptr(dL_ddepth), ptr(dL_dalpha), ptr(dL_dnormal), g[0], arr))
            return grads
        fn = ctx.lib.dvx_backward_host if host else ctx.lib.dvx_backward
        ctx.check(fn(ctx.h, self.h, ptr(dL_drgb), ptr(dL_ddepth), ptr(dL_dalpha), g[0], arr))
        return grads

    # ------------------------------------------------------------------ row N3: feature compositing
    def weights(self):
        """dvx_frame_weights -> (nnz, row_start [H*W+1], voxel [nnz], weight [nnz]) as zero-copy views of the frame's CSR."""
        ctx, torch = self.ctx, self.ctx.torch
        w = Weights()
        ctx.check(ctx.lib.dvx_frame_weights(ctx.h, self.h, C.byref(w)))

        def view(ptr, n, dtype):
            if n == 0:
                return torch.empty(0, dtype=dtype, device=ctx.device)
            return ctx._blocks[ptr].view(dtype)[:n]
        nnz = int(w.nnz)
        return nnz, ctx._blocks[w.row_start].view(torch.int32), view(w.voxel, nnz, torch.int32), view(w.weight, nnz, torch.float32)

    def render_features(self, feat, height, width):
        """dvx_render_features: feat CUDA float32 [V_total, C] (octrees end to end) -> [H, W, C]."""
        ctx, torch = self.ctx, self.ctx.torch
        n_ch = int(feat.shape[1])
        out = torch.empty((height, width, n_ch), dtype=torch.float32, device=ctx.device)
        ctx.check(ctx.lib.dvx_render_features(ctx.h, self.h, n_ch, feat.data_ptr(), out.data_ptr()))
        return out

    def fuse_features(self, img, num, wsum=None):
        """dvx_fuse_features: img [H, W, C]; num [V_total, C] and wsum [V_total] are accumulated into."""
        ctx = self.ctx
        ctx.check(ctx.lib.dvx_fuse_features(ctx.h, self.h, int(img.shape[2]), img.data_ptr(), num.data_ptr(),
                                            wsum.data_ptr() if wsum is not None else None))

    def tile_list(self, tile, octree, octant):
        ctx = self.ctx
        n = C.c_uint32()
        ctx.check(ctx.lib.dvx_debug_tile_list(ctx.h, self.h, tile, octree, octant, None, 0, C.byref(n)))
        ids = np.zeros(max(n.value, 1), dtype=np.uint32)
        ctx.check(ctx.lib.dvx_debug_tile_list(ctx.h, self.h, tile, octree, octant, ids.ctypes.data_as(C.c_void_p), n.value,
                                              C.byref(n)))
        return ids[:n.value]

    def counters(self):
        ctx = self.ctx
        v = [C.c_uint64() for _ in range(5)]
        ctx.check(ctx.lib.dvx_frame_counters(ctx.h, self.h, *[C.byref(x) for x in v]))
        return dict(zip(("v_vis", "pairs", "pairs_eff", "q_test", "q_hit"), [x.value for x in v]))

    def record_stats(self):
        """dvx_frame_record_stats -> dict(bytes_used, bytes_capacity, overflowed)."""
        ctx = self.ctx
        used, cap, over = C.c_uint64(), C.c_uint64(), C.c_uint32()
        ctx.check(ctx.lib.dvx_frame_record_stats(ctx.h, self.h, C.byref(used), C.byref(cap), C.byref(over)))
        return {"bytes_used": used.value, "bytes_capacity": cap.value, "overflowed": bool(over.value)}

    def stage_ms(self):
        ctx = self.ctx
        ms = (C.c_float * 8)()
        ctx.check(ctx.lib.dvx_frame_stage_ms(ctx.h, self.h, ms))
        return dict(zip(STAGES, list(ms)[:8]))

    def release(self):
        if self.h and self.ctx.h:
            self.ctx.lib.dvx_frame_release(self.ctx.h, self.h)
        self.h = None


def camera_from(cam):
    """dvx_scenes.Camera (or anything with the same attributes) -> binding.Camera."""
    return Camera(cam.width, cam.height, cam.fx, cam.fy, cam.cx, cam.cy,
                  (C.c_float * 12)(*[float(x) for x in np.asarray(cam.c2w).reshape(12)]), cam.near, cam.far)


class SceneOnDevice:
    """Uploads a dvx_scenes.Scene (host numpy) to the GPU and creates the octree handles."""

    def __init__(self, ctx, scene):
        torch = ctx.torch
        self.ctx, self.scene = ctx, scene
        self.trees = []
        for t in scene.octrees:
            code = torch.from_numpy(np.ascontiguousarray(t.code).view(np.int64)).to(ctx.device)
            geo = torch.from_numpy(np.ascontiguousarray(t.geo, dtype=np.float32)).to(ctx.device)
            sh = torch.from_numpy(np.ascontiguousarray(t.sh, dtype=np.float32)).to(ctx.device)
            self.trees.append(ctx.octree(code, geo, sh, t.center, t.side, t.sh_degree))
        self.poses = np.ascontiguousarray(scene.poses, dtype=np.float32)
        self.box_half = np.ascontiguousarray(scene.box_half, dtype=np.float32)
        self.cams = [camera_from(c) for c in scene.cameras]

    def render(self, cam_index=0, save=True, flags=0, out=None, host=False, sky=None, dsky=None, normals=False, **opt):
        s = self.scene
        kw = dict(k_samples=s.k_samples, activation=s.activation, t_stop=s.t_stop)
        kw.update(opt)
        return self.ctx.render(self.cams[cam_index], self.trees[0], self.trees[1:], self.poses, self.box_half, flags=flags,
                               save=save, out=out, host=host, sky=sky, dsky=dsky, normals=normals, **kw)

    def render_batch(self, cam_indices=None, save=True, flags=0, outs=None, **opt):
        s = self.scene
        kw = dict(k_samples=s.k_samples, activation=s.activation, t_stop=s.t_stop)
        kw.update(opt)
        cams = [self.cams[c] for c in (range(len(self.cams)) if cam_indices is None else cam_indices)]
        return self.ctx.render_batch(cams, self.trees[0], self.trees[1:], self.poses, self.box_half, flags=flags, save=save,
                                     outs=outs, **kw)

    def zero_grads(self):
        torch = self.ctx.torch
        return [(torch.zeros((t.n_voxels, 8), dtype=torch.float32, device=self.ctx.device),
                 torch.zeros((t.n_voxels, t.n_sh, 3), dtype=torch.float32, device=self.ctx.device)) for t in self.trees]
