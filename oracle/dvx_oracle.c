/*
 * dvx_oracle.c - TEST INFRASTRUCTURE ONLY.  Plain, slow, double-precision CPU restatement of the
 * DrivingVoxels compositional sparse-voxel renderer (forward + backward) written from the paper.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * build, load or call this file.  It shares no code with paper_2606_23031_b200/csrc (the CUDA
 * path) and never includes include/dvx.h.
 *
 * What it follows (PAPER.md = /root/reference/PAPER.md; O#/R# = DESIGN.md oracle steps/readings):
 *   O1 ray                r(tau) = o + tau d                      PAPER.md:101 (Sec. 3.4)
 *   O2 ray-OBB intervals  [tau_in^i, tau_out^i], local frame by (T_t^i)^-1
 *   O3 segment schedule   Algorithm 1
 *   O4 candidate filter   "only the primitives that reside within the active bounded interval"
 *                                                                  PAPER.md:297 (App. A)
 *   O5 ordering           sort by true ray distance               BASELINE.json north_star
 *   O6 voxel integral     8 corner raw densities, trilinear, numerical integration, activation
 *                                                                  PAPER.md:63 (Sec. 3.1), :107
 *   O7 colour             SH per leaf voxel
 *   O8 compositing        state S=(C,D,T), weighted by accumulated transmittance, T<eps stop
 *                                                                  PAPER.md:107, :297, Alg.1 l.8-9, Eq.2 :111
 *   O9 backward           reverse-mode tape per ray
 *   O10 sky composite     C = C_voxels + T_final C_sky, C_sky = bilinear sample of a 2-D spherical map at the
 *                         ray's world direction, texture updated by backpropagation
 *                                                                  PAPER.md:65 (Sky Modeling), Eq. 2 :111; R21
 *   O11 normal map        N = sum_j T_j alpha_j n_j, n_j = the voxel's normal (state tuple S = (C, D, N, T, tau_curr))
 *                                                                  PAPER.md:107, :297; R22
 *
 * Pinned by tests/test_oracle_pins.py (closed forms P1/P2/P10/P11, Morton-vs-depth order P3,
 * world-frame rewrite P4, empty box P5, finite differences P6, partition of unity P7,
 * subdivision P8, dense-sampling ray-box P9, SH orthonormality P12, culled==brute P13; early termination
 * P32 (threshold crossed / not crossed closed forms, crossing voxel included, strict '<'), the exp-linear
 * derivative and the truncated tape P33 (finite differences), orc_tile_hit_list P34 (hand-written lists and a
 * dense-sampling cross-check)).  tests/test_oracle_sanitizers.py runs this file under ASan + UBSan.
 * Parity-unpinned against the AUTHORS' implementation: readings R1, R2, R5, R8, R9 (the paper
 * prints no worked numeric example); see DESIGN.md.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_MAX_LEVEL 16
#define ORC_TILE 16

typedef struct {
  uint32_t n_voxels;
  uint32_t sh_degree;
  double center[3];
  double side;
  const uint64_t *code;  /* [V] key format R14a */
  const float *geo_f;    /* [V][8] raw corner densities (fp32 inputs) ... */
  const double *geo_d;   /* ... or doubles (finite-difference tests); exactly one is non-NULL */
  const float *sh_f;     /* [V][(deg+1)^2][3] */
  const double *sh_d;
} orc_octree;

typedef struct {
  uint32_t width, height;
  double fx, fy, cx, cy;
  double c2w[12]; /* row-major 3x4 [R_c | o_c], camera x right / y down / z forward (R10) */
  double near_, far_;
} orc_camera;

typedef struct {
  uint32_t k_samples;  /* K midpoint samples per clipped segment (R6) */
  uint32_t activation; /* 0 exp, 1 exp-linear (R5) */
  double t_stop;       /* early termination threshold (R3); 0 disables */
  uint32_t mode;       /* 0 brute force over all voxels; 1 tile-culled candidates (P13) */
} orc_opts;

typedef struct {
  double *dgeo; /* [V][8]   accumulated (+=) */
  double *dsh;  /* [V][C][3] accumulated (+=) */
} orc_grad;

/* R21: the sky is an equirectangular map tex[H][W][3] over the WORLD direction d (z up): azimuth phi = atan2(d_y, d_x),
 * polar angle theta = acos(d_z); continuous texel coordinates s = (phi/2pi + 1/2) W - 1/2 (wraps), t = (theta/pi) H - 1/2
 * (clamped to [0, H-1]); bilinear between the four surrounding texel centres. */
typedef struct orc_sky_s {
  uint32_t width, height;
  const double *tex; /* [H][W][3] */
  double *dtex;      /* [H][W][3] accumulated (+=), or NULL */
} orc_sky;

/* O12 (widening row N3, "substituting the standard RGB color rendering step with a high-dimensional feature
 * accumulation pass", and the "feature volume fuser" of :241).  Reading R25: with w_j = T_j alpha_j the compositing
 * weight of the j-th composited sub-segment of a ray (the same weights that blend the colour, :107),
 *   render:  F[p][c]        = sum_j w_j feat[tree_j][v_j][c]                  (no view dependence, no sky term)
 *   fuse:    num[t][v][c]  += sum over rays p, sub-segments j of (t, v):  w_j img[p][c],   wsum[t][v] += the same sum of w_j
 * so that num/wsum is the weight-averaged 2-D feature seen by the voxel, and fuse is the transpose of render. */
typedef struct {
  uint32_t n_channels;
  const double *const *feat; /* [n_trees] -> [V_t][C], or NULL (no feature image) */
  double *out;               /* [H][W][C] (untouched where masked out), or NULL */
  const double *img;         /* [H][W][C] 2-D features to fuse, or NULL */
  double *const *num;        /* [n_trees] -> [V_t][C], accumulated (+=) */
  double *const *wsum;       /* [n_trees] -> [V_t],    accumulated (+=) */
} orc_feat;

static const double ORC_PI = 3.14159265358979323846;

/* texel indices (into [H][W]) and weights of the bilinear footprint of world direction d */
static void sky_footprint(const orc_sky *sky, const double d[3], size_t idx[4], double wt[4]) {
  double W = (double)sky->width, H = (double)sky->height;
  double dz = d[2] > 1 ? 1 : (d[2] < -1 ? -1 : d[2]);
  double s = (atan2(d[1], d[0]) / (2 * ORC_PI) + 0.5) * W - 0.5;
  double t = acos(dz) / ORC_PI * H - 0.5;
  if (t < 0) t = 0;
  if (t > H - 1) t = H - 1;
  double fs = floor(s), ft = floor(t);
  double as = s - fs, at = t - ft;
  long i0 = (long)fs, j0 = (long)ft, w = (long)sky->width, h = (long)sky->height;
  long i1 = i0 + 1, j1 = j0 + 1 < h ? j0 + 1 : h - 1;
  i0 = ((i0 % w) + w) % w; i1 = ((i1 % w) + w) % w;
  idx[0] = (size_t)(j0 * w + i0); wt[0] = (1 - as) * (1 - at);
  idx[1] = (size_t)(j0 * w + i1); wt[1] = as * (1 - at);
  idx[2] = (size_t)(j1 * w + i0); wt[2] = (1 - as) * at;
  idx[3] = (size_t)(j1 * w + i1); wt[3] = as * at;
}

/* ------------------------------------------------------------------ small helpers ---------- */

static double geo_at(const orc_octree *t, uint32_t v, int c) {
  return t->geo_d ? t->geo_d[(size_t)v * 8 + c] : (double)t->geo_f[(size_t)v * 8 + c];
}
static double sh_at(const orc_octree *t, uint32_t v, int i, int ch) {
  size_t n = (size_t)(t->sh_degree + 1) * (t->sh_degree + 1);
  size_t idx = ((size_t)v * n + i) * 3 + ch;
  return t->sh_d ? t->sh_d[idx] : (double)t->sh_f[idx];
}

/* R14a: bits 48-52 level; bits 0-47 Morton path left-aligned, group m at bits [45-3m,47-3m]
 * = 4 x_m + 2 y_m + z_m with x_m = bit (l-1-m) of i. */
void orc_decode(uint64_t code, int *i, int *j, int *k, int *level) {
  int l = (int)((code >> 48) & 31);
  int x = 0, y = 0, z = 0;
  for (int m = 0; m < l; ++m) {
    int g = (int)((code >> (45 - 3 * m)) & 7);
    x = (x << 1) | ((g >> 2) & 1);
    y = (y << 1) | ((g >> 1) & 1);
    z = (z << 1) | (g & 1);
  }
  *i = x; *j = y; *k = z; *level = l;
}

/* R14b: order key for direction octant q = 4 s_x + 2 s_y + s_z, s_a = (d_a < 0). */
uint64_t orc_order_key(uint64_t code, int q) {
  return (code & 0xFFFFFFFFFFFFull) ^ ((uint64_t)q * 0x249249249249ull);
}

static void voxel_box(const orc_octree *t, uint32_t v, double mn[3], double *size) {
  int i, j, k, l;
  orc_decode(t->code[v], &i, &j, &k, &l);
  double s = t->side / (double)(1u << l);
  mn[0] = t->center[0] - 0.5 * t->side + i * s;
  mn[1] = t->center[1] - 0.5 * t->side + j * s;
  mn[2] = t->center[2] - 0.5 * t->side + k * s;
  *size = s;
}

/* O1: pixel (u,v) -> world ray.  d_cam = ((u+1/2-cx)/fx, (v+1/2-cy)/fy, 1), d = R_c d_cam/|d_cam|. */
void orc_ray(const orc_camera *cam, int u, int v, double o[3], double d[3]) {
  double dc[3] = {(u + 0.5 - cam->cx) / cam->fx, (v + 0.5 - cam->cy) / cam->fy, 1.0};
  double n = sqrt(dc[0] * dc[0] + dc[1] * dc[1] + dc[2] * dc[2]);
  for (int r = 0; r < 3; ++r) {
    d[r] = (cam->c2w[4 * r + 0] * dc[0] + cam->c2w[4 * r + 1] * dc[1] + cam->c2w[4 * r + 2] * dc[2]) / n;
    o[r] = cam->c2w[4 * r + 3];
  }
}

/* Slab test of the ray o + tau d against the axis-aligned box [mn, mx] (O2 / O4).
 * Axis with d_a == 0: miss when the origin is outside the HALF-OPEN slab [mn_a, mx_a), else no constraint
 * (reading R20: a ray lying exactly in a face shared by two voxels belongs to one of them only,
 * so subdivision invariance P8 holds for such rays too).
 * Returns 0 on a certain miss; otherwise *t0 = max_a min(t1,t2), *t1 = min_a max(t1,t2). */
static int slab(const double o[3], const double d[3], const double mn[3], const double mx[3], double *t0,
                double *t1) {
  double lo = -INFINITY, hi = INFINITY;
  for (int a = 0; a < 3; ++a) {
    if (d[a] != 0.0) {
      double ta = (mn[a] - o[a]) / d[a], tb = (mx[a] - o[a]) / d[a];
      double tn = ta < tb ? ta : tb, tf = ta < tb ? tb : ta;
      if (tn > lo) lo = tn;
      if (tf < hi) hi = tf;
    } else if (o[a] < mn[a] || o[a] >= mx[a]) {
      return 0;
    }
  }
  *t0 = lo; *t1 = hi;
  return 1;
}

/* local ray of actor pose [R|t]: o_l = R^T (o - t), d_l = R^T d   (Alg.1 l.5) */
static void to_local(const double *pose, const double o[3], const double d[3], double ol[3], double dl[3]) {
  for (int c = 0; c < 3; ++c) {
    ol[c] = 0; dl[c] = 0;
    for (int r = 0; r < 3; ++r) {
      ol[c] += pose[4 * r + c] * (o[r] - pose[4 * r + 3]);
      dl[c] += pose[4 * r + c] * d[r];
    }
  }
}

/* O2: ray-OBB.  Hit iff tau_out > max(tau_in, near); then tau_in<-max(tau_in,near), tau_out<-min(tau_out,far). */
int orc_ray_box(const double *pose, const double half[3], const double o[3], const double d[3], double near_,
                double far_, double *tin, double *tout) {
  double ol[3], dl[3], mn[3] = {-half[0], -half[1], -half[2]}, mx[3] = {half[0], half[1], half[2]};
  double a, b;
  to_local(pose, o, d, ol, dl);
  if (!slab(ol, dl, mn, mx, &a, &b)) return 0;
  if (!(b > (a > near_ ? a : near_))) return 0;
  *tin = a > near_ ? a : near_;
  *tout = b < far_ ? b : far_;
  return 1;
}

/* R8: real spherical harmonics up to degree 3 of the unit vector (x,y,z). */
void orc_sh_basis(const double dir[3], double Y[16]) {
  const double c0 = 0.28209479177387814, c1 = 0.4886025119029199;
  const double c2a = 1.0925484305920792, c2b = 0.31539156525252005, c2c = 0.5462742152960396;
  const double c3a = 0.5900435899266435, c3b = 2.890611442640554, c3c = 0.4570457994644658;
  const double c3d = 0.3731763325901154, c3e = 1.445305721320277;
  double x = dir[0], y = dir[1], z = dir[2];
  Y[0] = c0;
  Y[1] = -c1 * y; Y[2] = c1 * z; Y[3] = -c1 * x;
  Y[4] = c2a * x * y; Y[5] = -c2a * y * z; Y[6] = c2b * (2 * z * z - x * x - y * y);
  Y[7] = -c2a * x * z; Y[8] = c2c * (x * x - y * y);
  Y[9] = -c3a * y * (3 * x * x - y * y); Y[10] = c3b * x * y * z;
  Y[11] = -c3c * y * (4 * z * z - x * x - y * y); Y[12] = c3d * z * (2 * z * z - 3 * x * x - 3 * y * y);
  Y[13] = -c3c * x * (4 * z * z - x * x - y * y); Y[14] = c3e * z * (x * x - y * y);
  Y[15] = -c3a * x * (x * x - 3 * y * y);
}

/* R5 activation and its derivative */
static double act(double x, int kind) {
  if (kind == 0) return exp(x);
  const double th = 1.1;
  return x > th ? x : exp(x / th - 1.0 + log(th));
}
static double dact(double x, int kind) {
  if (kind == 0) return exp(x);
  const double th = 1.1;
  return x > th ? 1.0 : exp(x / th - 1.0 + log(th)) / th;
}

/* ------------------------------------------------------------------ per-ray tape ----------- */

typedef struct {
  double a, b;     /* clipped sub-segment */
  uint32_t tree, v;
} seg_t;

static int seg_cmp(const void *pa, const void *pb) {
  const seg_t *x = (const seg_t *)pa, *y = (const seg_t *)pb;
  if (x->a != y->a) return x->a < y->a ? -1 : 1;
  if (x->b != y->b) return x->b < y->b ? -1 : 1; /* deterministic whatever the candidate order */
  if (x->tree != y->tree) return x->tree < y->tree ? -1 : 1;
  return x->v < y->v ? -1 : (x->v > y->v);
}

typedef struct { seg_t *s; size_t n, cap; } segvec;
static void seg_push(segvec *sv, seg_t s) {
  if (sv->n == sv->cap) {
    sv->cap = sv->cap ? 2 * sv->cap : 256;
    sv->s = (seg_t *)realloc(sv->s, sv->cap * sizeof(seg_t));
  }
  sv->s[sv->n++] = s;
}

typedef struct { double lo, hi; } ival;

typedef struct {
  int n_trees;               /* 1 + N */
  const orc_octree *trees;   /* [0] static */
  const double *poses;       /* [N][12] */
  const double *half;        /* [N][3] */
  const orc_camera *cam;
  const orc_opts *opt;
  const struct orc_sky_s *sky; /* NULL = no sky (Eq. 2 with C_sky = 0) */
  const orc_feat *fx;          /* NULL = no feature pass (O12) */
} scene_t;

/* O3: the allowed intervals.  Sort hit actors by (tau_in, index); tau_curr never moves backwards (R2). */
typedef struct { double tin, tout; int idx; } hit_t;
static int hit_cmp(const void *pa, const void *pb) {
  const hit_t *x = (const hit_t *)pa, *y = (const hit_t *)pb;
  if (x->tin != y->tin) return x->tin < y->tin ? -1 : 1;
  return x->idx - y->idx;
}

/* builds bg[] (static intervals, returns count) and act[i] (one interval per actor, lo>=hi if none) */
static int schedule(const scene_t *sc, const double o[3], const double d[3], ival *bg, ival *actv, hit_t *hits) {
  int N = sc->n_trees - 1, m = 0, nbg = 0;
  double near_ = sc->cam->near_, far_ = sc->cam->far_;
  for (int i = 0; i < N; ++i) {
    actv[i].lo = 1; actv[i].hi = 0;
    double tin, tout;
    if (orc_ray_box(sc->poses + 12 * i, sc->half + 3 * i, o, d, near_, far_, &tin, &tout)) {
      hits[m].tin = tin; hits[m].tout = tout; hits[m].idx = i; ++m;
    }
  }
  qsort(hits, m, sizeof(hit_t), hit_cmp);
  double cur = near_;
  for (int h = 0; h < m; ++h) {
    double lo = hits[h].tin > cur ? hits[h].tin : cur;
    if (hits[h].tin > cur) { bg[nbg].lo = cur; bg[nbg].hi = hits[h].tin; ++nbg; }
    if (hits[h].tout > lo) { actv[hits[h].idx].lo = lo; actv[hits[h].idx].hi = hits[h].tout; }
    if (hits[h].tout > cur) cur = hits[h].tout;
  }
  if (far_ > cur) { bg[nbg].lo = cur; bg[nbg].hi = far_; ++nbg; }
  return nbg;
}

/* O4 for one voxel of one tree: ray-AABB in the tree's frame, intersected with the allowed intervals. */
static void candidate(const orc_octree *t, uint32_t tree, uint32_t v, const double o[3], const double d[3],
                      const ival *iv, int niv, segvec *out) {
  double mn[3], mx[3], s, a, b;
  voxel_box(t, v, mn, &s);
  mx[0] = mn[0] + s; mx[1] = mn[1] + s; mx[2] = mn[2] + s;
  if (!slab(o, d, mn, mx, &a, &b)) return;
  for (int n = 0; n < niv; ++n) {
    double lo = a > iv[n].lo ? a : iv[n].lo, hi = b < iv[n].hi ? b : iv[n].hi;
    if (hi > lo) { seg_t sg = {lo, hi, tree, v}; seg_push(out, sg); }
  }
}

/* O6: K-point midpoint rule on the clipped segment; returns tau_v, optionally fills per-sample raw & weights */
static double integrate(const orc_octree *t, uint32_t v, const double o[3], const double d[3], double a, double b,
                        const orc_opts *opt, double *raw_k /*[K]*/, double *w_k /*[K][8]*/) {
  double mn[3], s;
  voxel_box(t, v, mn, &s);
  int K = (int)opt->k_samples;
  double delta = (b - a) / K, sum = 0;
  for (int k = 0; k < K; ++k) {
    double tk = a + (k + 0.5) * delta, u[3];
    for (int ax = 0; ax < 3; ++ax) {
      u[ax] = (o[ax] + tk * d[ax] - mn[ax]) / s;
      if (u[ax] < 0) u[ax] = 0;
      if (u[ax] > 1) u[ax] = 1;
    }
    double raw = 0;
    for (int c = 0; c < 8; ++c) { /* corner c = 4 bx + 2 by + bz (R7) */
      double w = ((c & 4) ? u[0] : 1 - u[0]) * ((c & 2) ? u[1] : 1 - u[1]) * ((c & 1) ? u[2] : 1 - u[2]);
      raw += geo_at(t, v, c) * w;
      if (w_k) w_k[8 * k + c] = w;
    }
    if (raw_k) raw_k[k] = raw;
    sum += act(raw, (int)opt->activation);
  }
  return delta * sum;
}

/* O7: rgb_v = max(0, 1/2 + sum_i Y_i(dir_v) k_i), dir_v from the camera origin IN THE TREE'S FRAME to the centre */
static void voxel_colour(const orc_octree *t, uint32_t v, const double o_frame[3], double rgb[3], double pre[3],
                         double Y[16]) {
  double mn[3], s, dir[3], n = 0;
  voxel_box(t, v, mn, &s);
  for (int a = 0; a < 3; ++a) { dir[a] = mn[a] + 0.5 * s - o_frame[a]; n += dir[a] * dir[a]; }
  n = sqrt(n);
  for (int a = 0; a < 3; ++a) dir[a] /= n;
  orc_sh_basis(dir, Y);
  int nsh = (int)((t->sh_degree + 1) * (t->sh_degree + 1));
  for (int ch = 0; ch < 3; ++ch) {
    double acc = 0.5;
    for (int i = 0; i < nsh; ++i) acc += Y[i] * sh_at(t, v, i, ch);
    pre[ch] = acc;
    rgb[ch] = acc > 0 ? acc : 0;
  }
}

/* R22: the voxel's normal = minus the gradient of its trilinear raw density at the voxel centre, normalised:
 * g_a = 1/4 sum over the four corner pairs along axis a of (geo[b_a = 1] - geo[b_a = 0]) (so a constant voxel has g = 0
 * exactly), n_local = -g / max(|g|, ORC_NRM_EPS) (a flat voxel fades to no normal instead of a random unit vector),
 * rotated into the WORLD frame by the actor's R_i (identity for the static octree).
 * Outputs: nw[3] world normal; g[3] local gradient, gn = |g| (for the backward). */
#define ORC_NRM_EPS 1e-6
static void voxel_normal(const scene_t *sc, uint32_t tree, uint32_t v, double nw[3], double g[3], double *gn) {
  const orc_octree *t = &sc->trees[tree];
  for (int a = 0; a < 3; ++a) {
    int bit = 4 >> a;
    double acc = 0;
    for (int c = 0; c < 8; ++c)
      if (!(c & bit)) acc += geo_at(t, v, c | bit) - geo_at(t, v, c);
    g[a] = 0.25 * acc;
  }
  *gn = sqrt(g[0] * g[0] + g[1] * g[1] + g[2] * g[2]);
  double den = *gn > ORC_NRM_EPS ? *gn : ORC_NRM_EPS;
  double nl[3] = {-g[0] / den, -g[1] / den, -g[2] / den};
  if (tree == 0) { memcpy(nw, nl, sizeof nl); return; }
  const double *P = sc->poses + 12 * (tree - 1);
  for (int r = 0; r < 3; ++r) nw[r] = P[4 * r] * nl[0] + P[4 * r + 1] * nl[1] + P[4 * r + 2] * nl[2];
}
/* adjoint of voxel_normal: gnw = dL/dn_world -> accumulates dL/dgeo[v][0..8) */
static void voxel_normal_backward(const scene_t *sc, uint32_t tree, uint32_t v, const double gnw[3], double *dgeo_v) {
  double nw[3], g[3], gn;
  voxel_normal(sc, tree, v, nw, g, &gn);
  double gl[3];
  if (tree == 0) memcpy(gl, gnw, sizeof gl);
  else {
    const double *P = sc->poses + 12 * (tree - 1);
    for (int c = 0; c < 3; ++c) gl[c] = P[c] * gnw[0] + P[4 + c] * gnw[1] + P[8 + c] * gnw[2]; /* R^T */
  }
  double dg[3];
  if (gn > ORC_NRM_EPS) { /* d(-g/|g|)/dg = -(I - n n^T)/|g| */
    double nl[3] = {-g[0] / gn, -g[1] / gn, -g[2] / gn};
    double dot = nl[0] * gl[0] + nl[1] * gl[1] + nl[2] * gl[2];
    for (int a = 0; a < 3; ++a) dg[a] = -(gl[a] - nl[a] * dot) / gn;
  } else {
    for (int a = 0; a < 3; ++a) dg[a] = -gl[a] / ORC_NRM_EPS;
  }
  for (int a = 0; a < 3; ++a) {
    int bit = 4 >> a;
    for (int c = 0; c < 8; ++c) {
      double val = 0.25 * ((c & bit) ? dg[a] : -dg[a]);
#pragma omp atomic
      dgeo_v[c] += val;
    }
  }
}

typedef struct {
  segvec segs;
  ival *bg, *actv;
  hit_t *hits;
  double *tau, *Tb; /* tape: tau_v and T before the voxel */
  size_t tape_cap;
} ray_ws;

static void ws_init(ray_ws *w, int n_trees) {
  memset(w, 0, sizeof(*w));
  w->bg = (ival *)malloc(sizeof(ival) * (size_t)(n_trees + 1));
  w->actv = (ival *)malloc(sizeof(ival) * (size_t)(n_trees + 1));
  w->hits = (hit_t *)malloc(sizeof(hit_t) * (size_t)(n_trees + 1));
}
static void ws_free(ray_ws *w) { free(w->segs.s); free(w->bg); free(w->actv); free(w->hits); free(w->tau); free(w->Tb); }

/* One ray: O1-O8 (+O9 when g_* given).  cand[t]/ncand[t] = candidate voxel ids of tree t (NULL = all voxels).
 * out5 = {R,G,B,depth,alpha}; *n_used = number of sub-segments composited. */
static void render_ray(const scene_t *sc, int u, int v, const uint32_t *const *cand, const uint32_t *ncand,
                       ray_ws *w, double out5[5], const double *g5 /* or NULL */, orc_grad *grads, uint32_t *n_used,
                       double *nout /* [3] or NULL */, const double *gN /* [3] or NULL */) {
  double o[3], d[3];
  orc_ray(sc->cam, u, v, o, d);
  int nbg = schedule(sc, o, d, w->bg, w->actv, w->hits);
  w->segs.n = 0;
  for (int t = 0; t < sc->n_trees; ++t) {
    const orc_octree *tr = &sc->trees[t];
    double ol[3], dl[3];
    const ival *iv; int niv;
    if (t == 0) { memcpy(ol, o, sizeof ol); memcpy(dl, d, sizeof dl); iv = w->bg; niv = nbg; }
    else {
      if (!(w->actv[t - 1].hi > w->actv[t - 1].lo)) continue;
      to_local(sc->poses + 12 * (t - 1), o, d, ol, dl); iv = &w->actv[t - 1]; niv = 1;
    }
    if (cand && cand[t]) for (uint32_t n = 0; n < ncand[t]; ++n) candidate(tr, (uint32_t)t, cand[t][n], ol, dl, iv, niv, &w->segs);
    else if (!cand) for (uint32_t vx = 0; vx < tr->n_voxels; ++vx) candidate(tr, (uint32_t)t, vx, ol, dl, iv, niv, &w->segs);
  }
  if (w->segs.n > 1) qsort(w->segs.s, w->segs.n, sizeof(seg_t), seg_cmp); /* O5 (guard: no NULL base for an empty list) */
  if (w->segs.n > w->tape_cap) {
    w->tape_cap = w->segs.n * 2;
    w->tau = (double *)realloc(w->tau, sizeof(double) * w->tape_cap);
    w->Tb = (double *)realloc(w->Tb, sizeof(double) * w->tape_cap);
  }
  double C[3] = {0, 0, 0}, D = 0, T = 1, Nacc[3] = {0, 0, 0};
  size_t used = 0;
  for (size_t n = 0; n < w->segs.n; ++n) { /* O8 */
    const seg_t *sg = &w->segs.s[n];
    const orc_octree *tr = &sc->trees[sg->tree];
    double ol[3], dl[3], rgb[3], pre[3], Y[16];
    if (sg->tree == 0) { memcpy(ol, o, sizeof ol); memcpy(dl, d, sizeof dl); }
    else to_local(sc->poses + 12 * (sg->tree - 1), o, d, ol, dl);
    double tau = integrate(tr, sg->v, ol, dl, sg->a, sg->b, sc->opt, NULL, NULL);
    double alpha = 1.0 - exp(-tau);
    voxel_colour(tr, sg->v, ol, rgb, pre, Y);
    double wgt = T * alpha;
    w->tau[n] = tau; w->Tb[n] = T;
    for (int ch = 0; ch < 3; ++ch) C[ch] += wgt * rgb[ch];
    D += wgt * 0.5 * (sg->a + sg->b);
    if (nout) { /* O11 */
      double nw[3], gg[3], gn;
      voxel_normal(sc, sg->tree, sg->v, nw, gg, &gn);
      for (int a = 0; a < 3; ++a) Nacc[a] += wgt * nw[a];
    }
    T *= exp(-tau);
    used = n + 1;
    if (T < sc->opt->t_stop) break;
  }
  size_t sk_idx[4] = {0, 0, 0, 0};
  double sk_wt[4] = {0, 0, 0, 0}, sky_rgb[3] = {0, 0, 0};
  if (sc->sky) { /* O10, Eq. 2: C = C_voxels + T_final C_sky */
    sky_footprint(sc->sky, d, sk_idx, sk_wt);
    for (int ch = 0; ch < 3; ++ch) {
      for (int n = 0; n < 4; ++n) sky_rgb[ch] += sk_wt[n] * sc->sky->tex[3 * sk_idx[n] + ch];
      C[ch] += T * sky_rgb[ch];
    }
  }
  out5[0] = C[0]; out5[1] = C[1]; out5[2] = C[2]; out5[3] = D; out5[4] = 1.0 - T;
  if (nout) memcpy(nout, Nacc, sizeof Nacc);
  if (n_used) *n_used = (uint32_t)used;
  if (sc->fx) { /* O12: the tape holds T before each composited sub-segment and its tau */
    const orc_feat *fx = sc->fx;
    const size_t C = fx->n_channels, p = (size_t)v * sc->cam->width + (size_t)u;
    if (fx->feat && fx->out)
      for (size_t c = 0; c < C; ++c) fx->out[p * C + c] = 0.0;
    for (size_t n = 0; n < used; ++n) {
      const seg_t *sg = &w->segs.s[n];
      const double wgt = w->Tb[n] * (1.0 - exp(-w->tau[n]));
      if (fx->feat && fx->out)
        for (size_t c = 0; c < C; ++c) fx->out[p * C + c] += wgt * fx->feat[sg->tree][(size_t)sg->v * C + c];
      if (fx->img) {
        for (size_t c = 0; c < C; ++c) {
          const double val = wgt * fx->img[p * C + c];
#pragma omp atomic
          fx->num[sg->tree][(size_t)sg->v * C + c] += val;
        }
#pragma omp atomic
        fx->wsum[sg->tree][sg->v] += wgt;
      }
    }
  }
  if (!g5 || !grads) return;
  /* O9: reverse sweep over the tape.  Adjoint of T after the last voxel comes from alpha = 1 - T and from Eq. 2. */
  double gT = -g5[4];
  if (sc->sky) {
    for (int ch = 0; ch < 3; ++ch) {
      gT += g5[ch] * sky_rgb[ch];
      if (sc->sky->dtex)
        for (int n = 0; n < 4; ++n) {
          double val = g5[ch] * T * sk_wt[n];
#pragma omp atomic
          sc->sky->dtex[3 * sk_idx[n] + ch] += val;
        }
    }
  }
  int K = (int)sc->opt->k_samples;
  double raw_k[64], w_k[64 * 8];
  for (size_t n = used; n-- > 0;) {
    const seg_t *sg = &w->segs.s[n];
    const orc_octree *tr = &sc->trees[sg->tree];
    double ol[3], dl[3], rgb[3], pre[3], Y[16];
    if (sg->tree == 0) { memcpy(ol, o, sizeof ol); memcpy(dl, d, sizeof dl); }
    else to_local(sc->poses + 12 * (sg->tree - 1), o, d, ol, dl);
    double tau = w->tau[n], Tb = w->Tb[n], e = exp(-tau), alpha = 1.0 - e, wgt = Tb * alpha;
    voxel_colour(tr, sg->v, ol, rgb, pre, Y);
    double mid = 0.5 * (sg->a + sg->b);
    double g_w = g5[0] * rgb[0] + g5[1] * rgb[1] + g5[2] * rgb[2] + g5[3] * mid;
    if (gN) {
      double nw[3], gg[3], gn;
      voxel_normal(sc, sg->tree, sg->v, nw, gg, &gn);
      g_w += gN[0] * nw[0] + gN[1] * nw[1] + gN[2] * nw[2];
      if (grads[sg->tree].dgeo) {
        double gnw[3] = {wgt * gN[0], wgt * gN[1], wgt * gN[2]};
        voxel_normal_backward(sc, sg->tree, sg->v, gnw, grads[sg->tree].dgeo + (size_t)sg->v * 8);
      }
    }
    double g_alpha = g_w * Tb;
    double g_Tb = g_w * alpha + gT * e;
    double g_tau = g_alpha * e - gT * Tb * e;
    gT = g_Tb;
    int nsh = (int)((tr->sh_degree + 1) * (tr->sh_degree + 1));
    if (grads[sg->tree].dsh)
      for (int ch = 0; ch < 3; ++ch)
        if (pre[ch] > 0)
          for (int i = 0; i < nsh; ++i) {
            double val = Y[i] * wgt * g5[ch];
#pragma omp atomic
            grads[sg->tree].dsh[((size_t)sg->v * nsh + i) * 3 + ch] += val;
          }
    if (grads[sg->tree].dgeo) {
      integrate(tr, sg->v, ol, dl, sg->a, sg->b, sc->opt, raw_k, w_k);
      double delta = (sg->b - sg->a) / K;
      for (int c = 0; c < 8; ++c) {
        double acc = 0;
        for (int k = 0; k < K; ++k) acc += dact(raw_k[k], (int)sc->opt->activation) * w_k[8 * k + c];
        double val = g_tau * delta * acc;
#pragma omp atomic
        grads[sg->tree].dgeo[(size_t)sg->v * 8 + c] += val;
      }
    }
  }
}

/* ------------------------------------------------------------------ tile-culled candidates -- */
/* P13: per-tile candidate sets from exact double-precision corner projection.  A voxel (clipped to the
 * actor box for actors) is kept for a tile when the bounding rectangle of its projection, after clipping
 * the 12 edges against z_cam = z_clip, overlaps the tile (1 px margin).  Points on any ray at tau >= near
 * have z_cam >= near * min_pixels(1/|d_cam|) > z_clip, so nothing a ray can hit is lost. */
typedef struct { int x0, y0, x1, y1; } rect_t; /* inclusive tile rect; x1<x0 = culled */

static rect_t voxel_tiles(const scene_t *sc, int t, uint32_t v, double zclip) {
  const orc_camera *cam = sc->cam;
  const orc_octree *tr = &sc->trees[t];
  double mn[3], mx[3], s;
  rect_t r = {0, 0, -1, -1};
  voxel_box(tr, v, mn, &s);
  for (int a = 0; a < 3; ++a) mx[a] = mn[a] + s;
  if (t > 0) { /* actor voxels only matter inside the box (R18) */
    const double *h = sc->half + 3 * (t - 1);
    for (int a = 0; a < 3; ++a) {
      if (mn[a] < -h[a]) mn[a] = -h[a];
      if (mx[a] > h[a]) mx[a] = h[a];
      if (!(mx[a] >= mn[a])) return r;
    }
  }
  double pc[8][3];
  for (int c = 0; c < 8; ++c) {
    double p[3] = {(c & 4) ? mx[0] : mn[0], (c & 2) ? mx[1] : mn[1], (c & 1) ? mx[2] : mn[2]}, pw[3];
    if (t > 0) {
      const double *P = sc->poses + 12 * (t - 1);
      for (int rr = 0; rr < 3; ++rr) pw[rr] = P[4 * rr] * p[0] + P[4 * rr + 1] * p[1] + P[4 * rr + 2] * p[2] + P[4 * rr + 3];
    } else memcpy(pw, p, sizeof pw);
    for (int cc = 0; cc < 3; ++cc) {
      pc[c][cc] = 0;
      for (int rr = 0; rr < 3; ++rr) pc[c][cc] += cam->c2w[4 * rr + cc] * (pw[rr] - cam->c2w[4 * rr + 3]);
    }
  }
  double xmin = INFINITY, xmax = -INFINITY, ymin = INFINITY, ymax = -INFINITY;
  int any = 0;
#define ACC(P) do { double px = cam->fx * (P)[0] / (P)[2] + cam->cx, py = cam->fy * (P)[1] / (P)[2] + cam->cy; \
    xmin = fmin(xmin, px); xmax = fmax(xmax, px); ymin = fmin(ymin, py); ymax = fmax(ymax, py); any = 1; } while (0)
  for (int c = 0; c < 8; ++c) if (pc[c][2] >= zclip) ACC(pc[c]);
  for (int c = 0; c < 8; ++c)
    for (int ax = 1; ax <= 4; ax <<= 1) {
      int c2 = c | ax;
      if (c2 == c) continue;
      double za = pc[c][2], zb = pc[c2][2];
      if ((za < zclip) != (zb < zclip)) {
        double f = (zclip - za) / (zb - za), q[3];
        for (int a = 0; a < 3; ++a) q[a] = pc[c][a] + f * (pc[c2][a] - pc[c][a]);
        q[2] = zclip;
        ACC(q);
      }
    }
#undef ACC
  if (!any) return r;
  xmin -= 1; ymin -= 1; xmax += 1; ymax += 1;
  if (xmax < 0 || ymax < 0 || xmin >= cam->width || ymin >= cam->height) return r;
  int tw = ((int)cam->width + ORC_TILE - 1) / ORC_TILE, th = ((int)cam->height + ORC_TILE - 1) / ORC_TILE;
  r.x0 = xmin <= 0 ? 0 : (int)(xmin / ORC_TILE);
  r.y0 = ymin <= 0 ? 0 : (int)(ymin / ORC_TILE);
  r.x1 = xmax >= cam->width ? tw - 1 : (int)(xmax / ORC_TILE);
  r.y1 = ymax >= cam->height ? th - 1 : (int)(ymax / ORC_TILE);
  if (r.x1 > tw - 1) r.x1 = tw - 1;
  if (r.y1 > th - 1) r.y1 = th - 1;
  return r;
}

typedef struct {
  size_t *start; /* [n_tiles * n_trees + 1] */
  uint32_t *ids;
} tilelists;

static double z_clip_of(const orc_camera *cam) {
  double m = 1.0;
  int us[2] = {0, (int)cam->width - 1}, vs[2] = {0, (int)cam->height - 1};
  for (int a = 0; a < 2; ++a)
    for (int b = 0; b < 2; ++b) {
      double x = (us[a] + 0.5 - cam->cx) / cam->fx, y = (vs[b] + 0.5 - cam->cy) / cam->fy;
      double c = 1.0 / sqrt(x * x + y * y + 1.0);
      if (c < m) m = c;
    }
  return 0.5 * cam->near_ * m;
}

static void build_tilelists(const scene_t *sc, tilelists *tl) {
  const orc_camera *cam = sc->cam;
  int tw = ((int)cam->width + ORC_TILE - 1) / ORC_TILE, th = ((int)cam->height + ORC_TILE - 1) / ORC_TILE;
  size_t nb = (size_t)tw * th * sc->n_trees;
  double zclip = z_clip_of(cam);
  tl->start = (size_t *)calloc(nb + 1, sizeof(size_t));
  rect_t **rects = (rect_t **)malloc(sizeof(rect_t *) * sc->n_trees);
  for (int t = 0; t < sc->n_trees; ++t) {
    uint32_t V = sc->trees[t].n_voxels;
    rects[t] = (rect_t *)malloc(sizeof(rect_t) * (V ? V : 1));
#pragma omp parallel for schedule(static)
    for (int64_t v = 0; v < (int64_t)V; ++v) rects[t][v] = voxel_tiles(sc, t, (uint32_t)v, zclip);
    for (uint32_t v = 0; v < V; ++v) {
      rect_t r = rects[t][v];
      for (int y = r.y0; y <= r.y1; ++y)
        for (int x = r.x0; x <= r.x1; ++x) tl->start[((size_t)y * tw + x) * sc->n_trees + t + 1]++;
    }
  }
  for (size_t b = 0; b < nb; ++b) tl->start[b + 1] += tl->start[b];
  tl->ids = (uint32_t *)malloc(sizeof(uint32_t) * (tl->start[nb] ? tl->start[nb] : 1));
  size_t *fill = (size_t *)malloc(sizeof(size_t) * nb);
  memcpy(fill, tl->start, sizeof(size_t) * nb);
  for (int t = 0; t < sc->n_trees; ++t) {
    for (uint32_t v = 0; v < sc->trees[t].n_voxels; ++v) {
      rect_t r = rects[t][v];
      for (int y = r.y0; y <= r.y1; ++y)
        for (int x = r.x0; x <= r.x1; ++x) tl->ids[fill[((size_t)y * tw + x) * sc->n_trees + t]++] = v;
    }
    free(rects[t]);
  }
  free(rects); free(fill);
}

/* ------------------------------------------------------------------ exported entry points --- */

/* Renders every pixel whose mask byte is non-zero (mask NULL = all).  Outputs are [H][W][3], [H][W], [H][W]
 * doubles (untouched where masked out).  When g_rgb != NULL also runs O9 and accumulates into grads[n_trees]
 * (g_depth / g_alpha may be NULL = zero).  n_used (optional, [H][W]) = sub-segments composited per ray.
 * Returns 0, or -1 on invalid arguments. */
static int render_impl(const orc_camera *cam, int n_trees, const orc_octree *trees, const double *poses, const double *half,
                       const orc_opts *opt, const uint8_t *mask, double *rgb, double *depth, double *alpha,
                       const double *g_rgb, const double *g_depth, const double *g_alpha, orc_grad *grads,
                       uint32_t *n_used, const orc_sky *sky, double *normal /* [H][W][3] or NULL */,
                       const double *g_normal /* [H][W][3] or NULL */, const orc_feat *fx) {
  if (!cam || !trees || !opt || n_trees < 1 || opt->k_samples < 1 || opt->k_samples > 64) return -1;
  if (sky && (!sky->tex || sky->width < 1 || sky->height < 1)) return -1;
  scene_t sc = {n_trees, trees, poses, half, cam, opt, sky, fx};
  int W = (int)cam->width, H = (int)cam->height;
  int tw = (W + ORC_TILE - 1) / ORC_TILE, th = (H + ORC_TILE - 1) / ORC_TILE;
  tilelists tl = {0, 0};
  if (opt->mode == 1) build_tilelists(&sc, &tl);
#pragma omp parallel
  {
    ray_ws w;
    ws_init(&w, n_trees);
    const uint32_t **cand = (const uint32_t **)malloc(sizeof(uint32_t *) * n_trees);
    uint32_t *ncand = (uint32_t *)malloc(sizeof(uint32_t) * n_trees);
#pragma omp for schedule(dynamic, 1)
    for (int tile = 0; tile < tw * th; ++tile) {
      int tx = tile % tw, ty = tile / tw;
      if (opt->mode == 1)
        for (int t = 0; t < n_trees; ++t) {
          size_t b = (size_t)tile * n_trees + t;
          cand[t] = tl.ids + tl.start[b];
          ncand[t] = (uint32_t)(tl.start[b + 1] - tl.start[b]);
        }
      for (int v = ty * ORC_TILE; v < (ty + 1) * ORC_TILE && v < H; ++v)
        for (int u = tx * ORC_TILE; u < (tx + 1) * ORC_TILE && u < W; ++u) {
          size_t p = (size_t)v * W + u;
          if (mask && !mask[p]) continue;
          double out5[5], g5[5];
          if (g_rgb) {
            g5[0] = g_rgb[3 * p]; g5[1] = g_rgb[3 * p + 1]; g5[2] = g_rgb[3 * p + 2];
            g5[3] = g_depth ? g_depth[p] : 0; g5[4] = g_alpha ? g_alpha[p] : 0;
          }
          uint32_t used;
          render_ray(&sc, u, v, opt->mode == 1 ? cand : NULL, ncand, &w, out5, g_rgb ? g5 : NULL, grads, &used,
                     normal ? normal + 3 * p : NULL, (g_rgb && g_normal) ? g_normal + 3 * p : NULL);
          if (rgb) { rgb[3 * p] = out5[0]; rgb[3 * p + 1] = out5[1]; rgb[3 * p + 2] = out5[2]; }
          if (depth) depth[p] = out5[3];
          if (alpha) alpha[p] = out5[4];
          if (n_used) n_used[p] = used;
        }
    }
    ws_free(&w); free(cand); free(ncand);
  }
  free(tl.start); free(tl.ids);
  return 0;
}

int orc_render_full(const orc_camera *cam, int n_trees, const orc_octree *trees, const double *poses, const double *half,
                    const orc_opts *opt, const uint8_t *mask, double *rgb, double *depth, double *alpha,
                    const double *g_rgb, const double *g_depth, const double *g_alpha, orc_grad *grads,
                    uint32_t *n_used, const orc_sky *sky, double *normal, const double *g_normal) {
  if (!rgb || !depth || !alpha) return -1;
  return render_impl(cam, n_trees, trees, poses, half, opt, mask, rgb, depth, alpha, g_rgb, g_depth, g_alpha, grads, n_used,
                     sky, normal, g_normal, NULL);
}

/* O12: feature image and / or fusion over every pixel whose mask byte is non-zero; alpha (optional) = 1 - T_final. */
int orc_render_features(const orc_camera *cam, int n_trees, const orc_octree *trees, const double *poses,
                        const double *half, const orc_opts *opt, const uint8_t *mask, const orc_feat *fx, double *alpha) {
  if (!fx || fx->n_channels < 1) return -1;
  if (fx->feat && !fx->out) return -1;
  if (fx->img && (!fx->num || !fx->wsum)) return -1;
  return render_impl(cam, n_trees, trees, poses, half, opt, mask, NULL, NULL, alpha, NULL, NULL, NULL, NULL, NULL, NULL, NULL,
                     NULL, fx);
}

int orc_render_sky(const orc_camera *cam, int n_trees, const orc_octree *trees, const double *poses, const double *half,
                   const orc_opts *opt, const uint8_t *mask, double *rgb, double *depth, double *alpha,
                   const double *g_rgb, const double *g_depth, const double *g_alpha, orc_grad *grads,
                   uint32_t *n_used, const orc_sky *sky) {
  return orc_render_full(cam, n_trees, trees, poses, half, opt, mask, rgb, depth, alpha, g_rgb, g_depth, g_alpha, grads,
                         n_used, sky, NULL, NULL);
}

int orc_render(const orc_camera *cam, int n_trees, const orc_octree *trees, const double *poses, const double *half,
               const orc_opts *opt, const uint8_t *mask, double *rgb, double *depth, double *alpha,
               const double *g_rgb, const double *g_depth, const double *g_alpha, orc_grad *grads,
               uint32_t *n_used) {
  return orc_render_sky(cam, n_trees, trees, poses, half, opt, mask, rgb, depth, alpha, g_rgb, g_depth, g_alpha, grads,
                        n_used, NULL);
}

/* the bilinear footprint alone (pin P14) */
void orc_sky_footprint(uint32_t width, uint32_t height, const double d[3], int64_t idx[4], double wt[4]) {
  orc_sky sky = {width, height, NULL, NULL};
  size_t i4[4];
  sky_footprint(&sky, d, i4, wt);
  for (int n = 0; n < 4; ++n) idx[n] = (int64_t)i4[n];
}

static int key_cmp(const void *a, const void *b) {
  uint64_t x = *(const uint64_t *)a, y = *(const uint64_t *)b;
  return x < y ? -1 : (x > y);
}

/* T1 reference: voxels of tree `tree` that contribute a sub-segment longer than 1e-5 * s_l to at least one
 * pixel of tile (tx,ty) whose ray has direction octant `octant` in that tree's frame, sorted by the R14b key.
 * Early termination is ignored (every potentially needed voxel counts).  Returns the count (ids filled up to cap). */
int64_t orc_tile_hit_list(const orc_camera *cam, int n_trees, const orc_octree *trees, const double *poses,
                          const double *half, const orc_opts *opt, int tx, int ty, int tree, int octant,
                          uint32_t *ids, int64_t cap) {
  scene_t sc = {n_trees, trees, poses, half, cam, opt};
  int W = (int)cam->width, H = (int)cam->height;
  const orc_octree *tr = &trees[tree];
  uint8_t *hitflag = (uint8_t *)calloc(tr->n_voxels ? tr->n_voxels : 1, 1);
  ray_ws w;
  ws_init(&w, n_trees);
  for (int v = ty * ORC_TILE; v < (ty + 1) * ORC_TILE && v < H; ++v)
    for (int u = tx * ORC_TILE; u < (tx + 1) * ORC_TILE && u < W; ++u) {
      double o[3], d[3], ol[3], dl[3];
      orc_ray(cam, u, v, o, d);
      int nbg = schedule(&sc, o, d, w.bg, w.actv, w.hits);
      const ival *iv; int niv;
      if (tree == 0) { memcpy(ol, o, sizeof ol); memcpy(dl, d, sizeof dl); iv = w.bg; niv = nbg; }
      else {
        if (!(w.actv[tree - 1].hi > w.actv[tree - 1].lo)) continue;
        to_local(poses + 12 * (tree - 1), o, d, ol, dl); iv = &w.actv[tree - 1]; niv = 1;
      }
      int q = 4 * (dl[0] < 0) + 2 * (dl[1] < 0) + (dl[2] < 0); /* R12 */
      if (q != octant) continue;
      w.segs.n = 0;
      for (uint32_t vx = 0; vx < tr->n_voxels; ++vx) candidate(tr, (uint32_t)tree, vx, ol, dl, iv, niv, &w.segs);
      for (size_t n = 0; n < w.segs.n; ++n) {
        double mn[3], s;
        voxel_box(tr, w.segs.s[n].v, mn, &s);
        if (w.segs.s[n].b - w.segs.s[n].a > 1e-5 * s) hitflag[w.segs.s[n].v] = 1;
      }
    }
  ws_free(&w);
  /* sort the flagged voxels by the R14b key (insertion into an index array + qsort on keys) */
  int64_t n = 0;
  for (uint32_t vx = 0; vx < tr->n_voxels; ++vx) n += hitflag[vx];
  uint64_t *keys = (uint64_t *)malloc(sizeof(uint64_t) * 2 * (size_t)(n ? n : 1));
  int64_t m = 0;
  for (uint32_t vx = 0; vx < tr->n_voxels; ++vx)
    if (hitflag[vx]) { keys[2 * m] = orc_order_key(tr->code[vx], octant); keys[2 * m + 1] = vx; ++m; }
  qsort(keys, (size_t)n, 2 * sizeof(uint64_t), key_cmp);
  for (int64_t i = 0; i < n && i < cap; ++i) ids[i] = (uint32_t)keys[2 * i + 1];
  free(keys); free(hitflag);
  return n;
}

/* Per-ray list of composited sub-segments (for P3 and debugging): fills tree/voxel/a/b in compositing order. */
int64_t orc_ray_segments(const orc_camera *cam, int n_trees, const orc_octree *trees, const double *poses,
                         const double *half, const orc_opts *opt, int u, int v, uint32_t *tree_out,
                         uint32_t *vox_out, double *a_out, double *b_out, int64_t cap) {
  scene_t sc = {n_trees, trees, poses, half, cam, opt};
  ray_ws w;
  double out5[5];
  uint32_t used;
  ws_init(&w, n_trees);
  orc_opts o2 = *opt;
  o2.t_stop = 0; /* list everything */
  sc.opt = &o2;
  render_ray(&sc, u, v, NULL, NULL, &w, out5, NULL, NULL, &used, NULL, NULL);
  int64_t n = (int64_t)w.segs.n;
  for (int64_t i = 0; i < n && i < cap; ++i) {
    tree_out[i] = w.segs.s[i].tree; vox_out[i] = w.segs.s[i].v; a_out[i] = w.segs.s[i].a; b_out[i] = w.segs.s[i].b;
  }
  ws_free(&w);
  return n;
}

int orc_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}
