"""paper_2606_23031_b200 - B200-native (sm_100a) hot path of "Driving Voxels" (arxiv/paper_2606_23031):
the single-pass compositional sparse-voxel tile rasterizer, forward and backward, behind the C ABI of
include/dvx.h (libdvx.so, hand-written CUDA).  This package is the thin Python binding; see DESIGN.md.
"""
from .binding import (Context, Octree, Frame, Camera, SceneOnDevice, DvxError, camera_from, load, LIB_PATH, EXPORTS,  # noqa: F401
                      FLAG_COUNTERS, FLAG_NAIVE, FLAG_NO_RECORDS, sort_pairs_no_alloc, SORT_NO_ALLOC_MAX_PAIRS)
