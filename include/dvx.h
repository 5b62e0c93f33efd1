/*
 * dvx.h - C ABI of libdvx: the single-pass compositional sparse-voxel tile rasterizer of
 * "Driving Voxels" (arxiv/paper_2606_23031), forward and backward, for one NVIDIA B200 (sm_100a).
 *
 * What the calls compute (PAPER.md = the paper text; R# = readings listed in DESIGN.md section 3):
 *   render   : Algorithm 1 "Scene Rendering with Segmented Volume Rendering" over
 *              one static world-frame octree O_bg and N rigid actor octrees O_i under poses T_t^i
 *              (PAPER.md:63, :73-75), per-ray ray-OBB intervals sorted front to back (PAPER.md:101-105,
 *              :295), accumulation function F over Morton-ordered per-tile voxel lists with the state
 *              S = (C, D, T, tau_curr), T_final returned as alpha (Eq. 2, :111).
 *   backward : "Gradients flow through each voxel segment independently": gradients of the
 *              8 corner raw densities v_geo and of the per-voxel SH colour coefficients.
 *
 * Conventions
 *   - Plain C.  No exception, abort, exit or print ever crosses this boundary; every call returns a
 *     dvx_status (0 = DVX_OK, negative = error) and dvx_last_error() gives the text of the last failure.
 *   - "DEVICE" pointers are CUDA device pointers on the context's device, owned by the caller and only
 *     borrowed by the library; "HOST" pointers are ordinary host memory, read before the call returns.
 *   - All GPU work is enqueued on the context's stream.  dvx_render synchronises that stream once
 *     internally (it has to learn the number of (tile, voxel) pairs to size the sort); dvx_backward does
 *     not synchronise.  The caller synchronises before reading outputs.
 *   - There is no CPU fallback: without a CUDA device dvx_create fails with DVX_ERR_CUDA.
 */
#ifndef DVX_H_
#define DVX_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef int32_t dvx_status;
#define DVX_OK 0
#define DVX_ERR_INVALID_ARG (-1)     /* null pointer, n_actors > 64, sh_degree > 3, k_samples not in [1,8], bad camera, pose not rigid */
#define DVX_ERR_BAD_OCTREE (-2)      /* level not in [1,16], code bits below the level not zero, duplicate or nested leaves */
#define DVX_ERR_OOM (-3)             /* the allocator returned NULL */
#define DVX_ERR_CUDA (-4)            /* CUDA runtime error (sticky); text via dvx_last_error */
#define DVX_ERR_NOT_IMPLEMENTED (-5)

#define DVX_MAX_ACTORS 64
#define DVX_MAX_LEVEL 16
#define DVX_TILE 16 /* 16x16 pixel tiles (BASELINE.json north_star (1)) */

typedef struct dvx_ctx dvx_ctx;       /* opaque: device, stream, scratch cache */
typedef struct dvx_octree dvx_octree; /* opaque: borrowed array pointers + cached per-octant rank tables (step 0) */
typedef struct dvx_frame dvx_frame;   /* opaque: what dvx_backward needs from one dvx_render call */

/* Device memory comes from the caller (the PyTorch caching allocator in practice).  Both NULL = cudaMalloc/cudaFree. */
typedef void *(*dvx_alloc_fn)(size_t bytes, void *user);
typedef void (*dvx_free_fn)(void *ptr, void *user);

/* device: CUDA ordinal.  cuda_stream: a cudaStream_t (NULL = the legacy default stream). */
dvx_status dvx_create(int device, void *cuda_stream, dvx_alloc_fn alloc, dvx_free_fn free_, void *user, dvx_ctx **out);
void dvx_destroy(dvx_ctx *ctx);
/* The context keeps released scratch blocks (sort buffers, per-frame tables, record pools) for reuse, matched by size, so a
 * steady-state loop allocates nothing.  A workload whose sizes keep growing (subdivision rounds) leaves the smaller blocks
 * behind: dvx_trim synchronises the stream and returns every cached block to the allocator.  bytes_freed may be NULL. */
dvx_status dvx_trim(dvx_ctx *ctx, uint64_t *bytes_freed);

/* One leaf-only octree.  All three arrays are DEVICE pointers, borrowed until dvx_octree_destroy;
 * geo and sh may change in place between renders (they are re-read every frame), code may not (see refresh). */
typedef struct {
  uint32_t n_voxels;    /* V >= 0 */
  uint32_t sh_degree;   /* 0..3; C_sh = (deg+1)^2 basis functions */
  float center[3];      /* w_c: cube centre in the octree's own frame */
  float side;           /* w_s: root cube edge length (> 0) */
  const uint64_t *code; /* [V] bits 48-52 = level l in [1,16]; bits 0-47 = Morton path left-aligned: 3-bit group
                           m in [0,l) at bits [45-3m,47-3m] = 4 x_m + 2 y_m + z_m, x_m = bit (l-1-m) of the cell
                           coordinate i; groups m >= l are zero (R14a) */
  const float *geo;     /* [V][8] raw corner densities, corner c = 4 b_x + 2 b_y + b_z (R7); 32-byte aligned */
  const float *sh;      /* [V][C_sh][3] SH colour coefficients (R8); 16-byte aligned */
} dvx_octree_desc;

/* Validates the leaf set and builds the per-octant rank tables (hot-path step 0: rank of every voxel under the key
 * morton48 XOR q*0x249249249249, q = 4 s_x + 2 s_y + s_z, s_a = (d_a < 0); R14b).  Synchronises the stream. */
dvx_status dvx_octree_create(dvx_ctx *ctx, const dvx_octree_desc *desc, dvx_octree **out);
/* The leaf set (code / n_voxels) changed: revalidate and rebuild the rank tables. */
dvx_status dvx_octree_refresh_structure(dvx_ctx *ctx, dvx_octree *tree, const dvx_octree_desc *desc);
void dvx_octree_destroy(dvx_ctx *ctx, dvx_octree *tree);

/* Pinhole camera (R10): pixel centres at half-integers; camera axes x right, y down, z forward. */
typedef struct {
  uint32_t width, height;
  float fx, fy, cx, cy;
  float c2w[12]; /* row-major 3x4 [R_c | o_c] */
  float near_;   /* tau starts here (R11), > 0 */
  float far_;    /* tau_max */
} dvx_camera;

/* Sky ("Sky Modeling", Eq. 2 :111): C = C_voxels + T_final * C_sky, C_sky = bilinear sample of a 2-D spherical
 * map at the ray's WORLD direction d (z up).  Reading R21: equirectangular, phi = atan2(d_y, d_x), theta = acos(d_z), texel
 * coordinates s = (phi/2pi + 1/2) W - 1/2 (wraps), t = (theta/pi) H - 1/2 (clamped to [0, H-1]).  Depth and alpha are not
 * affected.  dvx_backward accumulates (+=) the texture gradient into dtex when it is not NULL. */
typedef struct {
  uint32_t width, height; /* W, H >= 1 */
  const float *tex;       /* DEVICE [H][W][3], borrowed until the frame is released */
  float *dtex;            /* DEVICE [H][W][3] or NULL */
} dvx_sky;

typedef struct {
  uint32_t k_samples;  /* K midpoint samples per clipped ray-voxel segment, 1..8 (R6) */
  uint32_t activation; /* 0 = exp (default), 1 = exp-linear with theta = 1.1 (R5) */
  float t_stop;        /* early termination T < t_stop, tested after every voxel (R3); 0 disables */
  uint32_t flags;      /* DVX_FLAG_* */
  const dvx_sky *sky;  /* HOST pointer, read before the call returns; NULL = no sky (C_sky = 0) */
} dvx_render_opts;
#define DVX_FLAG_COUNTERS 1u /* maintain q_test / q_hit / pairs_eff (slower; off in timed runs) */
#define DVX_FLAG_NAIVE 2u    /* debug: per-thread in-order walker instead of the cooperative tile kernel */
#define DVX_FLAG_NO_RECORDS 4u /* saved frames only: keep no hit records; dvx_backward then walks the tile lists again
                                  (same gradients up to the order of the float reductions; slower, no record pool) */

typedef struct {
  float *rgb;   /* DEVICE [H][W][3] */
  float *depth; /* DEVICE [H][W]  D = sum T_j alpha_j (a_j+b_j)/2, Euclidean ray distance (R9) */
  float *alpha; /* DEVICE [H][W]  1 - T_final */
  float *normal; /* DEVICE [H][W][3] or NULL (not computed).  N = sum T_j alpha_j n_j, the N of the state tuple S
                    (PAPER.md:107, :297); n_j = the voxel's normal in the WORLD frame, reading R22: minus the gradient of
                    its trilinear raw density at the voxel centre, divided by max(|g|, 1e-6) */
} dvx_image;

/* Steps 1-4 of the hot path.  All work is enqueued on the context's stream; the call blocks the host ONCE, between step 1
 * and step 2, to read the number of (tile, octant, voxel) pairs that sizes the sort buffers and the sort's grid (dvx_render_batch
 * amortises that round trip over its cameras).  The GPU does not idle meanwhile: key generation only needs a capacity, which
 * the context takes from its recent frames (x 1.25), and is enqueued before the wait; a frame with more pairs than that
 * repeats it.  poses_l2w: HOST [N][12] row-major [R_i | t_i] local->world;
 * box_half: HOST [N][3] half extents of the oriented box in the actor frame.  opts NULL = defaults
 * (K=8, exp, t_stop=1e-4, flags 0).  saved: if non-NULL receives a frame handle for dvx_backward / introspection
 * (release with dvx_frame_release); NULL = inference, nothing kept. */
dvx_status dvx_render(dvx_ctx *ctx, const dvx_camera *cam, const dvx_octree *static_tree, uint32_t n_actors,
                      const dvx_octree *const *actors, const float *poses_l2w, const float *box_half,
                      const dvx_render_opts *opts, dvx_image out, dvx_frame **saved);

typedef struct {
  float *dgeo; /* DEVICE [V][8]       same shape as geo; ACCUMULATED (+=); may be NULL (skipped) */
  float *dsh;  /* DEVICE [V][C_sh][3] same shape as sh;  ACCUMULATED (+=); may be NULL (skipped) */
} dvx_grad;

/* Step 5.  dL_drgb DEVICE [H][W][3]; dL_ddepth / dL_dalpha DEVICE [H][W] or NULL (= zero).
 * static_grad for the static octree, actor_grads HOST array [N] of DEVICE pointers, same order as in dvx_render.
 * No gradient flows to geometry (camera, poses, voxel positions) nor through the per-voxel view direction. */
dvx_status dvx_backward(dvx_ctx *ctx, dvx_frame *saved, const float *dL_drgb, const float *dL_ddepth,
                        const float *dL_dalpha, dvx_grad static_grad, const dvx_grad *actor_grads);
/* dvx_backward with a gradient of the normal map as well (the frame must have been rendered with out.normal != NULL):
 * dL_dnormal DEVICE [H][W][3] or NULL.  The corner densities receive it through the compositing weights and through
 * the voxel normals themselves (R22). */
dvx_status dvx_backward_n(dvx_ctx *ctx, dvx_frame *saved, const float *dL_drgb, const float *dL_ddepth,
                          const float *dL_dalpha, const float *dL_dnormal, dvx_grad static_grad,
                          const dvx_grad *actor_grads);
void dvx_frame_release(dvx_ctx *ctx, dvx_frame *frame);

/* Several cameras at once (BASELINE.json configs[4]: six surround cameras sharing the octrees, the poses of one timestamp
 * and ONE gradient set, one forward + backward per training iteration).  Results are those of n_cams
 * dvx_render / n_frames dvx_backward calls in the same order (gradients up to float summation order).  What differs is the
 * schedule: step 1 of every camera is enqueued first and the pair counts of all of them come back in ONE host round trip
 * instead of one per camera; camera c's key generation and sort (step 2) run on a second, library-owned high-priority
 * stream under camera c-1's compositing kernel; in the backward, frame c's per-voxel SH post-pass runs there under frame
 * c+1's replay.  Events order the two streams against the context's stream on entry and on exit, so the caller sees one
 * stream as before.  cams: HOST [n_cams]; outs: HOST [n_cams] of DEVICE image pointers; saved: HOST [n_cams] frame handles
 * out, or NULL (inference); dL_drgb: HOST [n_frames] of DEVICE pointers, dL_ddepth / dL_dalpha likewise or NULL (arrays
 * or their entries).  Frames rendered with a normal map take dvx_backward_n, one by one (its post-pass writes dgeo). */
dvx_status dvx_render_batch(dvx_ctx *ctx, uint32_t n_cams, const dvx_camera *cams, const dvx_octree *static_tree,
                            uint32_t n_actors, const dvx_octree *const *actors, const float *poses_l2w,
                            const float *box_half, const dvx_render_opts *opts, const dvx_image *outs, dvx_frame **saved);
dvx_status dvx_backward_batch(dvx_ctx *ctx, uint32_t n_frames, dvx_frame *const *frames, const float *const *dL_drgb,
                              const float *const *dL_ddepth, const float *const *dL_dalpha, dvx_grad static_grad,
                              const dvx_grad *actor_grads);

/* Hit records.  When dvx_render is given a `saved` handle, the compositing kernel also writes what it composited -
 * per (pixel, voxel) hit 44 bytes: voxel, octree, owning pixel, the clipped segment in the voxel's local coordinates, its length / K
 * and midpoint, in the order the pixel blended them (Alg. 1's sequence) - into a pool obtained from
 * the caller's allocator, and dvx_backward streams those records instead of walking the sorted tile
 * lists and testing every candidate voxel a second time.  The pool is sized from the hit counts of the context's recent
 * frames (first frame: 48 hits per pixel); a frame that needs more falls back to the list walk on the device, without
 * a host round trip, with identical results up to float summation order.  dvx_set_record_budget fixes the pool size
 * instead (bytes per frame; 0 = back to automatic sizing).  dvx_frame_record_stats (synchronises the stream) reports
 * what one frame used. */
dvx_status dvx_set_record_budget(dvx_ctx *ctx, uint64_t bytes_per_frame);
dvx_status dvx_frame_record_stats(dvx_ctx *ctx, const dvx_frame *frame, uint64_t *bytes_used, uint64_t *bytes_capacity,
                                  uint32_t *overflowed);

/* The same two calls with HOST image buffers (pinned memory recommended), for end-to-end use from a host
 * data pipeline: dvx_render_host renders into device staging owned by the context and enqueues the device->host
 * copies of RGB, depth and alpha (out_host.* are HOST pointers; valid after the stream is synchronised);
 * dvx_backward_host enqueues the host->device copies of the incoming image gradients (HOST pointers; depth / alpha
 * may be NULL) and then runs step 5.  The copies run on a second, library-owned stream so that they overlap the compute
 * on the context's stream (copy-out of frame i with the backward of frame i and the start of frame i+1 - the staging is
 * double-buffered -, copy-in with the forward); events order them.  The host images of dvx_render_host are valid once the
 * context's stream has been synchronised after dvx_host_io_wait(ctx), which makes that stream wait for every copy-out still
 * in flight (a device-wide synchronisation covers them too; with saved == NULL the render call itself orders the stream
 * behind its copies).  Octree arrays and gradient buffers stay DEVICE pointers (they are model
 * state that lives in HBM across steps).  Bytes moved per call: 20 W H out, 12 W H (+4 W H each for depth/alpha) in. */
dvx_status dvx_render_host(dvx_ctx *ctx, const dvx_camera *cam, const dvx_octree *static_tree, uint32_t n_actors,
                           const dvx_octree *const *actors, const float *poses_l2w, const float *box_half,
                           const dvx_render_opts *opts, dvx_image out_host, dvx_frame **saved);
dvx_status dvx_backward_host(dvx_ctx *ctx, dvx_frame *saved, const float *dL_drgb_host, const float *dL_ddepth_host,
                             const float *dL_dalpha_host, dvx_grad static_grad, const dvx_grad *actor_grads);
dvx_status dvx_host_io_wait(dvx_ctx *ctx);

/* Introspection for the parity tests and the benchmark (each synchronises the stream).
 * dvx_debug_tile_list: the sorted voxel list (voxel indices within octree `octree`, 0 = static, i = actor i-1) of
 * tile `tile` (row-major tile index) for ray-direction octant `octant`; ids_host HOST [capacity]; *n_out = full length. */
dvx_status dvx_debug_tile_list(dvx_ctx *ctx, const dvx_frame *frame, uint32_t tile, uint32_t octree, uint32_t octant,
                               uint32_t *ids_host, uint32_t capacity, uint32_t *n_out);
/* v_vis: voxels surviving culling; pairs: (tile, octant, voxel) pairs sorted; the last three need DVX_FLAG_COUNTERS. */
dvx_status dvx_frame_counters(dvx_ctx *ctx, const dvx_frame *frame, uint64_t *v_vis, uint64_t *pairs,
                              uint64_t *pairs_eff, uint64_t *q_test, uint64_t *q_hit);
/* Device milliseconds (CUDA events on the context's stream) of the stages of the frame's dvx_render call:
 * [0] preprocess (step 1), [1] key generation + sort + ranges (step 2), [2] compositing kernel (steps 3+4);
 * after dvx_backward also [3] all of step 5, [4] its compositing-replay kernel alone, [5] its per-voxel SH
 * post-pass alone; [6] the gap between the end of step 1 and the start of step 2 (near zero when key generation could be
 * enqueued before the pair count was known, see dvx_render; else the host round trip, during which the GPU idles), [7] the gap between the end of compositing and the start of step 5 (whatever the caller or a copy
 * put in between).  HOST out[8].  Synchronises the stream. */
dvx_status dvx_frame_stage_ms(dvx_ctx *ctx, const dvx_frame *frame, float *ms_out8);
/* The same eight times SUMMED over every frame released (or rendered with saved = NULL) since the last call;
 * *n_frames = how many.  Lets a benchmark time the stages of the very steps it measures without keeping frames alive.
 * HOST ms_out8[8], HOST n_frames.  Synchronises the stream. */
dvx_status dvx_stage_ms_collect(dvx_ctx *ctx, float *ms_out8, uint32_t *n_frames);
/* The device's fp32 FMA rate, measured now: a kernel of independent FFMA chains on every warp slot of every SM, timed
 * with CUDA events on the context's stream (synchronises).  One FFMA per lane per clock per SM sub-partition is both the
 * fp32 peak and the instruction-issue peak, so this is the denominator of the issue-rate roofline that bounds the
 * compositing kernels (SURVEY.md 8(d) asks for a measured FMA peak from the same run).  iters: loop trips of 64 FFMA per
 * thread (1 << 14 runs for about a millisecond).  Any output pointer may be NULL. */
dvx_status dvx_microbench_fma(dvx_ctx *ctx, uint32_t iters, double *lane_fma_per_s, double *warp_instr_per_s, float *ms);
/* Kernels launched by the library in this process so far (all contexts). */
uint64_t dvx_launch_count(void);
const char *dvx_last_error(const dvx_ctx *ctx);

/* Stand-alone entry to hot-path step 2's sort (tests and sort-throughput measurement): sorts n (key, value) pairs by
 * the low key_bits bits of the key, ascending, stable.  keys / vals DEVICE arrays, sorted in place. */
dvx_status dvx_sort_pairs(dvx_ctx *ctx, uint64_t *keys, uint32_t *vals, uint64_t n, uint32_t key_bits);

/* The same sort for callers that may not allocate device memory (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc): needs no context and calls no cudaMalloc, cudaFree or allocator callback.  Its
 * ping-pong buffers and one-sweep scratch live in a file-scope device array of fixed size inside the library
 * (DVX_SORT_NO_ALLOC_MAX_PAIRS pairs: about 15 MB, held by every GPU that loads the library until the process exits).
 * n > DVX_SORT_NO_ALLOC_MAX_PAIRS is rejected with DVX_ERR_INVALID_ARG and a message; use dvx_sort_pairs then.
 * device: CUDA device index (made current); cuda_stream: the stream to enqueue on (NULL = default stream); keys / vals
 * DEVICE arrays, sorted in place, ascending by the low key_bits bits, stable; err: HOST buffer [err_cap] that receives the
 * error text (may be NULL).  Does not synchronise.  ALL calls share the one static array: calls that overlap on the GPU
 * (different streams or threads without ordering between them) race - order them, e.g. on one stream.  The array keeps
 * the last call's contents; whatever must start at zero is cleared by every call. */
#define DVX_SORT_NO_ALLOC_MAX_PAIRS (1u << 20)
dvx_status dvx_sort_pairs_no_alloc(int device, void *cuda_stream, uint64_t *keys, uint32_t *vals, uint64_t n,
                                   uint32_t key_bits, char *err, size_t err_cap);

/* ---- Widening row N2: shared grid-point corner densities and the optimizer step -----------------------
 * The corner densities "are optimized during training".  Reading R23: coincident corners of
 * neighbouring voxels are ONE parameter (a grid point), identified by the corner's integer coordinate on the level-16
 * lattice of the octree (hanging nodes are grid points of their own); grid points are numbered in ascending order of
 * the 51-bit Morton key of that coordinate (bit b of x at 3b+2, of y at 3b+1, of z at 3b).  Reading R24: the optimizer
 * is Adam (Kingma & Ba 2015, Algorithm 1, with bias correction).  The [V][8] corner record stays what the rasterizer
 * reads and what dvx_backward accumulates into; these calls tie it to the per-grid-point parameter array. */
typedef struct dvx_grid dvx_grid; /* opaque: owns the three tables below */
typedef struct {
  uint32_t n_points;         /* G */
  const uint32_t *point_of;  /* DEVICE [V][8]: grid point of corner c of voxel v */
  const uint32_t *offsets;   /* DEVICE [G+1]: CSR row starts into slots */
  const uint32_t *slots;     /* DEVICE [8V]: slots[offsets[p] .. offsets[p+1]) = the corner slots 8v+c that are point p, ascending */
} dvx_grid_tables;

/* Builds the tables from the leaf set (code DEVICE [V], the dvx_octree_desc format, already validated by
 * dvx_octree_create; V < 2^27).  One radix sort of 8V keys.  tables (HOST, may be NULL) receives borrowed pointers valid
 * until dvx_grid_destroy.  Synchronises the stream.  V = 0 gives G = 0. */
dvx_status dvx_grid_create(dvx_ctx *ctx, const uint64_t *code, uint32_t n_voxels, dvx_grid **out, dvx_grid_tables *tables);
void dvx_grid_destroy(dvx_ctx *ctx, dvx_grid *grid);
/* geo[v][c] = density[point_of[v][c]].  density DEVICE [G], geo DEVICE [V][8] (overwritten). */
dvx_status dvx_grid_gather(dvx_ctx *ctx, const dvx_grid *grid, const float *density, float *geo);
/* ddensity[p] = sum over the slots of p of dgeo (ascending slot order, no atomics: deterministic).  dgeo DEVICE [V][8],
 * ddensity DEVICE [G] (overwritten, not accumulated). */
dvx_status dvx_grid_reduce(dvx_ctx *ctx, const dvx_grid *grid, const float *dgeo, float *ddensity);

typedef struct {
  float lr, beta1, beta2, eps; /* lr > 0, 0 <= beta < 1, eps >= 0 */
  uint32_t step;               /* t >= 1: the bias corrections 1 - beta^t are taken on the host in double */
} dvx_adam;
/* One fused optimizer step of the corner densities of one octree: g = dvx_grid_reduce(dgeo); Adam on (density, m, v)
 * DEVICE [G]; the new densities are written back into every corner slot of geo DEVICE [V][8]; dgeo DEVICE [V][8] is
 * ZEROED (ready for the next dvx_backward).  Does not synchronise. */
dvx_status dvx_grid_adam_step(dvx_ctx *ctx, const dvx_grid *grid, const dvx_adam *hp, float *density, float *m, float *v,
                              float *dgeo, float *geo);
/* Elementwise Adam over n floats (the SH coefficients, the sky texture): p, m, v updated in place, g ZEROED.
 * All four DEVICE, 16-byte aligned.  n < 2^43.  Does not synchronise. */
dvx_status dvx_adam_step(dvx_ctx *ctx, const dvx_adam *hp, uint64_t n, float *p, float *m, float *v, float *g);

/* The same two steps for SEVERAL parameter arrays in one kernel launch per 32 arrays (the static octree and the actor
 * octrees of a scene: an actor's few thousand parameters would otherwise cost a launch of their own).  items HOST [n],
 * read before the call returns; the fields mean what the arguments of the single-array calls mean.  Entries with an
 * empty grid / n = 0 are skipped.  Results are identical to n single-array calls. */
typedef struct {
  const dvx_grid *grid;
  float *density, *m, *v; /* DEVICE [G] */
  float *dgeo, *geo;      /* DEVICE [V][8] */
} dvx_grid_adam_item;
typedef struct {
  uint64_t n;
  float *p, *m, *v, *g; /* DEVICE [n], 16-byte aligned */
} dvx_adam_item;
dvx_status dvx_grid_adam_step_n(dvx_ctx *ctx, const dvx_adam *hp, uint32_t n, const dvx_grid_adam_item *items);
dvx_status dvx_adam_step_n(dvx_ctx *ctx, const dvx_adam *hp, uint32_t n, const dvx_adam_item *items);

/* ---- Widening row N3: feature compositing and the feature fuser -----------------------------------------
 * "substituting the standard RGB color rendering step with a high-dimensional feature accumulation pass" and
 * the "feature volume fuser".  Reading R25: with w_j = T_j alpha_j the compositing weight of the j-th
 * composited sub-segment of a pixel's ray (the weights that blend the colour; early termination as rendered),
 *   render:  F[p][c]    = sum_j w_j feat[v_j][c]                     (no view dependence, no sky term)
 *   fuse:    num[v][c] += sum over (p, j) with v_j = v of w_j img[p][c],   wsum[v] += the same sum of w_j
 * so num / wsum is the weight-averaged 2-D feature a voxel saw, and fuse is the transpose of render.
 * Voxels are addressed by their FRAME-GLOBAL index: the octrees of the dvx_render call laid end to end (static octree
 * first, then actor 0 .. N-1), i.e. row = (sum of n_voxels of the octrees before it) + voxel index.  V_total = that sum
 * over all octrees.  All three calls need a frame rendered with saved != NULL and still alive. */
typedef struct {
  uint64_t nnz;              /* = sum over pixels of the number of composited sub-segments */
  const uint32_t *row_start; /* DEVICE [H*W + 1], row-major pixels */
  const uint32_t *voxel;     /* DEVICE [nnz] frame-global voxel index, front to back within a row */
  const float *weight;       /* DEVICE [nnz] w_j */
} dvx_weights;
/* The compositing weights of the frame as a CSR matrix [H*W x V_total].  Built on the first call by one replay of the
 * compositing pass (the per-pixel counts were saved by dvx_render), then cached in the frame until dvx_frame_release;
 * the pointers are borrowed.  out may be NULL (build only).  Synchronises the stream (it has to learn nnz). */
dvx_status dvx_frame_weights(dvx_ctx *ctx, dvx_frame *frame, dvx_weights *out);
/* F = W feat.  n_channels C in [1, 512]; feat DEVICE [V_total][C], out DEVICE [H][W][C] (overwritten), both 16-byte
 * aligned.  Builds the weights if dvx_frame_weights has not been called.  Does not synchronise otherwise. */
dvx_status dvx_render_features(dvx_ctx *ctx, dvx_frame *frame, uint32_t n_channels, const float *feat, float *out);
/* num += W^T img, wsum += W^T 1.  img DEVICE [H][W][C]; num DEVICE [V_total][C] ACCUMULATED; wsum DEVICE [V_total]
 * ACCUMULATED, or NULL.  Float atomics: the sums are order-dependent in the last bits. */
dvx_status dvx_fuse_features(dvx_ctx *ctx, dvx_frame *frame, uint32_t n_channels, const float *img, float *num, float *wsum);

/* ---- Widening row N4: LiDAR-guided structure operations of the static octree ------------
 * "Proximity-Based Voxel Subdivision: ... In each round, voxels closer than a distance threshold to a LiDAR point are
 * subdivided" (:87) and "Soft Density Initialization Prior: ... For each grid corner, the euclidean distance d to the
 * nearest LiDAR point is computed and mapped to an initial density" v = v_far + (v_close - v_far) exp(-2 d^2 / s^2) (Eq. 1,
 * :91; the paper sets v_close = -2, v_far = -10, s = the minimum voxel size).  Readings R26-R28: the distance
 * of a point to a voxel is the Euclidean distance to its closed box (0 inside), "closer than" is <=; Eq. 1 is evaluated per
 * grid point of R23; a leaf is pruned when the largest of its 8 raw corner densities is below a threshold.  Geometry is
 * evaluated in fp64 from the fp32 inputs, so split / keep decisions are exact.  After a structure change the caller rebuilds
 * the step-0 tables (dvx_octree_refresh_structure) and the grid tables (dvx_grid_create). */
typedef struct dvx_cloud dvx_cloud; /* opaque: the LiDAR points binned into a uniform cell grid */
/* points DEVICE [n][3] fp32 in the octree's frame (copied, not borrowed), n < 2^31.  cell > 0: the edge of the binning
 * cells; queries cost least when it is about the query radius (the subdivision threshold, 3.1 s for Eq. 1).
 * Synchronises the stream.  n = 0 is valid (nothing is ever near). */
dvx_status dvx_cloud_create(dvx_ctx *ctx, const float *points, uint64_t n, float cell, dvx_cloud **out);
void dvx_cloud_destroy(dvx_ctx *ctx, dvx_cloud *cloud);
/* Eq. 1 for every grid point of `grid` (built from desc->code): density DEVICE [G] overwritten.  desc supplies center,
 * side and code; geo / sh are not read.  Points further than 3.1 s_min from a grid point cannot change its fp32 result and
 * are not searched.  Does not synchronise. */
dvx_status dvx_density_prior(dvx_ctx *ctx, const dvx_cloud *cloud, const dvx_octree_desc *desc, const dvx_grid *grid,
                             float s_min, float v_close, float v_far, float *density);
/* One subdivision round: every leaf with level < max_level that has a point within `threshold` of its box is replaced by its
 * 8 children (octant order 4x+2y+z), the others are kept; input order is preserved.  *n_out (HOST) = number of leaves of
 * the result; code_out DEVICE [capacity] is written only if capacity >= *n_out (8 V always suffices).  split DEVICE [V]
 * bytes (1 = was subdivided) or NULL.  Synchronises the stream. */
dvx_status dvx_subdivide_near(dvx_ctx *ctx, const dvx_cloud *cloud, const dvx_octree_desc *desc, float threshold,
                              uint32_t max_level, uint64_t *code_out, uint64_t capacity, uint64_t *n_out, uint8_t *split);
/* Parameters of the leaves a subdivision round produced (reading R29; the paper only says the structure "is only modified
 * during an adaptive pruning and progressive subdivision", following SVRaster): in dvx_subdivide_near's output
 * order, a kept leaf keeps its 8 corner densities and its SH coefficients; child o = 4 ox + 2 oy + oz of a split leaf gets,
 * at its corner c = 4 bx + 2 by + bz, the parent's trilinear raw density at u = (o + b) / 2 - the continuous density field
 * is unchanged by the split - and a copy of the parent's SH coefficients.  split DEVICE [V] as written by
 * dvx_subdivide_near; geo_in DEVICE [V][8], sh_in DEVICE [V][C_sh][3] or NULL; geo_out DEVICE [capacity][8], sh_out DEVICE
 * [capacity][C_sh][3] or NULL (sh_in and sh_out go together); *n_out HOST = leaves after the round (capacity must be at
 * least that; 8 V always suffices).  geo arrays 32-byte aligned.  Synchronises the stream. */
dvx_status dvx_subdivide_fill(dvx_ctx *ctx, uint32_t n_voxels, const uint8_t *split, const float *geo_in, const float *sh_in,
                              uint32_t sh_degree, float *geo_out, float *sh_out, uint64_t capacity, uint64_t *n_out);
/* Pruning: keeps the leaves whose largest raw corner density is >= threshold, in order.  code DEVICE [V], geo DEVICE
 * [V][8] (32-byte aligned); code_out DEVICE [V]; index_out DEVICE [V] (the kept leaves' old indices, for gathering geo and
 * sh) or NULL; *n_out HOST.  Synchronises the stream. */
dvx_status dvx_prune(dvx_ctx *ctx, uint32_t n_voxels, const uint64_t *code, const float *geo, float threshold,
                     uint64_t *code_out, uint32_t *index_out, uint32_t *n_out);

#ifdef __cplusplus
}
#endif
#endif /* DVX_H_ */
