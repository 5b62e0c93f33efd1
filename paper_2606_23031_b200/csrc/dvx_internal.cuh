// dvx_internal.cuh - structures and launch prototypes shared by the translation units of libdvx.
// Nothing here is visible through include/dvx.h.  Notation follows the paper and DESIGN.md.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <atomic>
#include "../../include/dvx.h"

#define DVX_MAX_TREES (DVX_MAX_ACTORS + 1)

// One octree as the kernels of one frame see it (device array of n_trees entries; [0] = static O_bg).
struct TreeFrame {
  const uint64_t *code;  // [V]        R14a
  const float *geo;      // [V][8]     raw corner densities v_geo
  const float *sh;       // [V][n_sh][3]
  const uint32_t *rank;  // [8][V]     step-0 tables: rank of voxel v under octant q at rank[q*V + v]
  float *dgeo;           // backward only
  float *dsh;            // backward only
  uint32_t n_voxels, n_sh, base, is_actor;  // base = first global voxel id of this tree
  double lo[3];          // cube min corner w_c - w_s/2 (tree frame)
  double cell;           // w_s / 2^16 : edge of a level-16 cell
  double o_l[3];         // camera origin in the tree frame: R_o^T (o_c - t_o)
  double rel0[3];        // lo - o_l: cube min corner relative to the camera origin (tree frame)
  double Nd[9];          // R_o^T R_c in fp64 (N below is its fp32 rounding)
  float ol_f[3];         // o_l rounded to fp32 (debug walker's ray-OBB test only)
  float inv_cell_f;      // 1 / cell rounded to fp32
  float N[9];            // R_o^T R_c: d_l[a] = N[3a] x' + N[3a+1] y' + N[3a+2];  p_cam[c] = sum_a N[3a+c] rel[a]
  float R[9];            // local -> world rotation R_o (row-major; identity for the static tree): world normals (R22)
  float half[3];         // OBB half extents (actors)
  int box_rect[4];       // pixel rectangle of the OBB (x0,y0,x1,y1 inclusive; x1<x0 = not visible); set on device
};

struct FrameParams {
  uint32_t width, height, tiles_x, tiles_y, n_tiles, n_trees;
  float fx, fy, cx, cy, near_, far_, zclip;
  double inv_fx, inv_fy, cx_d, cy_d;  // fp64 copies for the per-pixel ray set-up of the tile kernel
  float cull_t[4];   // tan of the frustum's side planes, one pixel outside the image: x/z in [t[0], t[1]], y/z in [t[2], t[3]]
  float cull_l[4];   // sqrt(1 + t^2): length of the planes' normals (step 1's bounding-sphere pre-cull)
  double Rc[9];                       // camera rotation (row-major, camera -> world): world direction of a pixel (sky)
  uint32_t k_samples, activation, flags;
  float t_stop, inv_k;  // inv_k = 1 / k_samples
  uint32_t rank_bits;   // sort key = ((tile*8 + octant) << rank_bits) | (tree base + rank); rank_bits = bits_for(v_total)
  uint32_t v_total;     // sum of n_voxels
  uint32_t n_buckets;   // n_tiles * n_trees * 8
};

// Per visible voxel, per frame (32 bytes, indexed by global voxel id).
struct __align__(16) FrameVox {
  float rel[3];   // voxel min corner minus camera origin, tree frame (computed in fp64, rounded once)
  float s;        // voxel edge length
  float rgb[3];   // max(0, 1/2 + sum_i Y_i(dir_v) k_i)  (R8)
  uint32_t meta;  // bits 0-2: colour channel clamped at 0 (gradient blocked)
};

enum { CNT_PAIRS = 0, CNT_VVIS = 1, CNT_QTEST = 2, CNT_QHIT = 3, CNT_PAIRS_EFF = 4, CNT_OVERFLOW = 5, CNT_EMIT = 6,
       CNT_REC_CHUNKS = 7,    // hit-record chunks handed out by the forward (may exceed the capacity: then CNT_REC_OVERFLOW is set)
       CNT_REC_OVERFLOW = 8,  // != 0: the record pool was too small, the backward re-walks the lists instead of replaying
       CNT_PREV_REC = 9,      // chunks the context's latest frame with a backward (or released without one) needed ...
       CNT_PREV_NPIX = 10,    // ... and its pixel count: copied in by step 1, read by the host with the pair count (pool sizing)
       CNT_N = 12 };

// ---- hit records (forward -> backward): what the forward composited, in the order it composited it ------------------
// The forward kernel processes its (pixel, voxel) hits in batches of up to 32 per warp (phase B/C of dvx_composite_tile.cu).
// When a frame is saved for a backward pass, every batch is also written to a per-warp stream in HBM, so that the
// backward replays the batches instead of walking the tile lists and testing every candidate voxel again.
// One batch = DVX_REC_BATCH_BYTES, structure-of-arrays so that each of the three record stores / loads of a warp is one
// contiguous run:
//   [   0,  512)  32 x {id, meta, delta, mid}      voxel, owning pixel's lane | tree << 8 | level << 16, (b - a) / K, (a + b) / 2
//   [ 512, 1024)  32 x {p_x, p_y, p_z, q_x}        local coordinates u(lambda) = p + q lambda on the clipped segment
//   [1024, 1280)  32 x {q_y, q_z}
//   [1280, 1408)  32 x ownership mask              bit i of word l: item i of the batch belongs to the warp's pixel l
// Batches are grouped in chunks of DVX_REC_CHUNK, handed out from one pool by an atomic counter; chunk c starts at
// rec_pool + c * DVX_REC_CHUNK_STRIDE (a power of two, pool base aligned to it, so that "the chunk is full" is a test on the
// low bits of the write pointer); rec_next links a warp's chunks, rec_tab[2 * warp] = first chunk, rec_tab[2 * warp + 1] =
// number of batches (warp = tile * 8 + 4x8 block).
#define DVX_REC_BATCH_BYTES 1408u
#define DVX_REC_CHUNK 11u
#define DVX_REC_CHUNK_STRIDE 16384u   // 11 * 1408 = 15488 bytes used

struct CompositeArgs {
  FrameParams p;
  const TreeFrame *trees;
  const FrameVox *fvox;
  const ushort4 *pxrect;       // [v_total] pixel rectangle of each voxel (x0,y0,x1,y1 inclusive)
  const uint32_t *ids;         // [P] sorted global voxel ids
  const uint32_t *range_beg;   // [n_buckets]
  const uint32_t *range_end;   // [n_buckets]
  const unsigned long long *actor_mask;  // [n_tiles]
  const uint32_t *tile_order;  // [n_tiles] CTA -> tile, heaviest tiles first, or NULL (CTA i serves tile i)
  float *rgb, *depth, *alpha;  // caller's images
  float *sv_rgbd;              // [H*W][4] saved C_final, D_final (frame-owned; may be NULL when nothing is saved)
  float *sv_T;                 // [H*W]
  uint32_t *sv_nused;          // [H*W]
  unsigned long long *counters;
  uint32_t *eff_end;           // [n_buckets] furthest list position any warp streamed (DVX_FLAG_COUNTERS only, else NULL)
  const float4 *vnrm;          // [v_total] per-voxel world normal (R22), or NULL when no normal map was requested
  float *normal;               // caller's normal image [H][W][3] or NULL
  float *sv_nrm;               // [H*W][4] saved N_final (frame-owned) or NULL
  const float *g_normal;       // backward: dL/dN [H][W][3] or NULL
  float *dnrm;                 // backward scratch [v_total][4]: dL/dn_v (world frame)
  const float *sky_tex;        // [sky_h][sky_w][3] or NULL (Eq. 2)
  float *sky_dtex;             // backward: texture gradient, or NULL
  uint32_t sky_w, sky_h;
  // backward
  const float *g_rgb, *g_depth, *g_alpha;
  float *drgb;                 // [v_total][4] scratch: dL/drgb_v
  // hit records (see above); rec_pool == NULL: nothing is recorded / the backward walks the lists
  unsigned char *rec_pool;     // [rec_cap chunks][DVX_REC_CHUNK][DVX_REC_BATCH_BYTES]
  uint32_t *rec_next;          // [rec_cap]
  uint32_t *rec_tab;           // [n_tiles * 8][2]
  uint32_t rec_cap;            // chunks in the pool
  // weight export (row N3)
  const uint32_t *exp_row;     // [H*W + 1] CSR row starts
  uint32_t *exp_vox;           // [nnz] global voxel id
  float *exp_w;                // [nnz] T_j alpha_j
};

// Number of kernels launched by this library since it was loaded (bench.py's gpu_launches claim).
extern std::atomic<unsigned long long> g_dvx_launches;
#define DVX_COUNT_LAUNCH(n) (g_dvx_launches.fetch_add((unsigned long long)(n), std::memory_order_relaxed))

// ---- dvx_sort.cu
size_t dvx_sort_scratch_bytes(uint64_t n);
// Sorts by bits [0,key_bits) ascending, stable.  Result lands in keys_a/vals_a or keys_b/vals_b; returns 0 or 1 (which).
int dvx_sort_launch(uint64_t *keys_a, uint32_t *vals_a, uint64_t *keys_b, uint32_t *vals_b, uint64_t n, uint32_t key_bits,
                    void *scratch, cudaStream_t st);
void dvx_scan_u32_launch(uint32_t *data, uint64_t n, uint32_t *scratch, cudaStream_t st);  // exclusive, in place

// ---- dvx_preprocess.cu
void dvx_rank_keys_launch(const uint64_t *code, uint32_t n, int q, uint64_t *keys, uint32_t *vals, cudaStream_t st);
void dvx_rank_scatter_launch(const uint32_t *perm, uint32_t n, uint32_t *rank, cudaStream_t st);
void dvx_validate_launch(const uint64_t *code_sorted_keys, const uint32_t *perm, const uint64_t *code, uint32_t n,
                         uint32_t *bad_flag, cudaStream_t st);
void dvx_tree_setup_launch(const FrameParams &p, TreeFrame *trees, unsigned long long *counters, const unsigned long long *rec_last,
                           cudaStream_t st);
void dvx_tile_masks_launch(const FrameParams &p, const TreeFrame *trees, uint8_t *octmask, unsigned long long *actor_mask,
                           cudaStream_t st);
void dvx_preprocess_launch(const FrameParams &p, const TreeFrame *trees, const uint8_t *octmask, FrameVox *fvox,
                           ushort4 *pxrect, float4 *vnrm, unsigned long long *counters, cudaStream_t st);
void dvx_normal_backward_launch(const FrameParams &p, const TreeFrame *trees, const float *dnrm, cudaStream_t st);
void dvx_emit_pairs_launch(const FrameParams &p, const TreeFrame *trees, const uint8_t *octmask, const ushort4 *pxrect,
                           const FrameVox *fvox, uint64_t *keys, uint32_t *vals, unsigned long long capacity,
                           unsigned long long *counters, cudaStream_t st);
void dvx_ranges_launch(const uint64_t *keys, uint64_t n, uint32_t rank_bits, const TreeFrame *trees, uint32_t n_trees,
                       uint32_t *range_beg, uint32_t *range_end, uint32_t *tile_cost, cudaStream_t st);
void dvx_tile_order_launch(const uint32_t *tile_cost, uint32_t n_tiles, uint32_t *tile_order /* [2 n_tiles] */, cudaStream_t st);
struct DvxGradTable { float *dgeo[DVX_MAX_TREES]; float *dsh[DVX_MAX_TREES]; };
// also publishes the frame's record-chunk count to the context's rec_last[2] = {chunks, pixels} (either may be NULL)
void dvx_patch_grads_launch(TreeFrame *trees, uint32_t n_trees, const DvxGradTable &tbl, const unsigned long long *counters,
                            unsigned long long *rec_last, unsigned long long npix, cudaStream_t st);
void dvx_publish_rec_launch(const unsigned long long *counters, unsigned long long *rec_last, unsigned long long npix, cudaStream_t st);
void dvx_sh_backward_launch(const FrameParams &p, const TreeFrame *trees, const FrameVox *fvox, const float *drgb,
                            cudaStream_t st);

// ---- dvx_grid.cu (row N2: shared grid-point densities, optimizer step)
void dvx_corner_keys_launch(const uint64_t *code, uint64_t n_slots, uint64_t *keys, uint32_t *vals, cudaStream_t st);
void dvx_grid_heads_launch(const uint64_t *skeys, uint64_t n, uint32_t *flag, cudaStream_t st);
void dvx_grid_count_launch(const uint64_t *skeys, const uint32_t *excl, uint64_t n, uint32_t *n_points, cudaStream_t st);
void dvx_grid_tables_launch(const uint64_t *skeys, const uint32_t *svals, const uint32_t *excl, uint64_t n,
                            uint32_t *point_of, uint32_t *offsets, uint32_t *slots, cudaStream_t st);
void dvx_grid_gather_launch(const float *density, const uint32_t *point_of, uint64_t n_slots, float *geo, cudaStream_t st);
void dvx_grid_reduce_launch(const float *dgeo, const uint32_t *offsets, const uint32_t *slots, uint32_t n_points,
                            float *ddensity, cudaStream_t st);
struct DvxGridAdamItem {
  const uint32_t *offsets, *slots, *point_of;
  uint32_t n_points, n_voxels;
  float *density, *m, *v, *dgeo, *geo;
};
struct DvxAdamItem {
  uint64_t n;
  float *p, *m, *v, *g;
};
// all items in as few launches as possible (32 arrays per launch)
void dvx_grid_adam_launch(float lr, float beta1, float beta2, float eps, uint32_t step, uint32_t n,
                          const DvxGridAdamItem *items, cudaStream_t st);
void dvx_adam_launch(float lr, float beta1, float beta2, float eps, uint32_t step, uint32_t n, const DvxAdamItem *items,
                     cudaStream_t st);

// ---- dvx_structure.cu (row N4: LiDAR-guided structure operations)
struct DvxCloudData {
  double origin[3];            // lower corner of cell (0,0,0)
  double cell;                 // cell edge
  uint32_t dims[3];            // cells per axis
  uint32_t n_cells;            // occupied cells
  uint64_t n;                  // points
  const uint64_t *cell_key;    // [n_cells] ascending linear index (z * ny + y) * nx + x
  const uint32_t *cell_start;  // [n_cells + 1]
  const float4 *pts;           // [n] in cell order
};
void dvx_cloud_bounds_launch(const float *pts, uint64_t n, uint32_t *minmax6, cudaStream_t st);
void dvx_cloud_keys_launch(const float *pts, uint64_t n, const DvxCloudData &d, uint64_t *keys, uint32_t *vals, cudaStream_t st);
void dvx_cloud_gather_launch(const float *pts, const uint32_t *perm, uint64_t n, float4 *out, cudaStream_t st);
void dvx_cloud_cells_launch(const uint64_t *skeys, const uint32_t *excl, uint64_t n, uint64_t *cell_key, uint32_t *cell_start,
                            cudaStream_t st);
void dvx_density_prior_launch(const DvxCloudData &d, const uint64_t *code, const uint32_t *offsets, const uint32_t *slots,
                              uint32_t n_points, const double center[3], double side, double s_min, double reach,
                              double v_close, double v_far, float *density, cudaStream_t st);
void dvx_near_flags_launch(const DvxCloudData &d, const uint64_t *code, uint32_t n_voxels, const double center[3], double side,
                           double threshold, uint32_t max_level, uint32_t *count, uint8_t *split, cudaStream_t st);
void dvx_expand_launch(const uint64_t *code, uint32_t n_voxels, const uint32_t *offsets, uint64_t *out, cudaStream_t st);
void dvx_split_counts_launch(const uint8_t *split, uint32_t n_voxels, uint32_t *count, cudaStream_t st);
void dvx_subdivide_fill_launch(const uint32_t *offsets, uint32_t n_voxels, const float *geo_in, const float *sh_in, uint32_t sh_floats,
                               float *geo_out, float *sh_out, cudaStream_t st);
void dvx_prune_flags_launch(const float *geo, uint32_t n_voxels, float threshold, uint32_t *keep, cudaStream_t st);
void dvx_prune_scatter_launch(const uint64_t *code, uint32_t n_voxels, const uint32_t *offsets, uint64_t *code_out,
                              uint32_t *index_out, cudaStream_t st);

// ---- dvx_microbench.cu
uint64_t dvx_microbench_fma_launch(float *out, uint32_t blocks, uint32_t iters, cudaStream_t st);
uint32_t dvx_microbench_threads(void);

// ---- dvx_features.cu (row N3).  img == NULL: render (feat, out);  img != NULL: fuse (img, num, wsum)
void dvx_features_launch(uint32_t width, uint32_t height, uint32_t n_channels, const uint32_t *row_start, const uint32_t *voxel,
                         const float *weight, const float *feat, float *out, const float *img, float *num, float *wsum,
                         cudaStream_t st);

// ---- dvx_composite_tile.cu (production) / dvx_composite_naive.cu (DVX_FLAG_NAIVE: one thread walks one ray, debug)
void dvx_composite_tile_launch(const CompositeArgs &a, bool backward, cudaStream_t st);
void dvx_composite_naive_launch(const CompositeArgs &a, bool backward, cudaStream_t st);
void dvx_composite_export_launch(const CompositeArgs &a, cudaStream_t st);
// Backward from the hit records (returns at once when the frame's record pool overflowed); a list-walking backward launched
// with a.rec_pool != NULL is its complement (it returns at once unless the pool overflowed).
void dvx_composite_replay_launch(const CompositeArgs &a, cudaStream_t st);
inline void dvx_composite_launch(const CompositeArgs &a, bool backward, cudaStream_t st) {
  if (a.p.flags & DVX_FLAG_NAIVE) dvx_composite_naive_launch(a, backward, st);
  else dvx_composite_tile_launch(a, backward, st);
}
