// dvx_composite_tile.cu - hot-path steps 3, 4 and 5, the production kernels.
//   step 3  per-ray ray-OBB intervals [tau_in^i, tau_out^i] sorted front to back
//   step 4  Algorithm 1: F over Morton-ordered per-tile voxel lists, segment by segment, carrying
//           S = (C, D, T, tau_curr); trilinear raw density, K midpoint samples, activation,
//           alpha = 1 - exp(-sum sigma dt), blend weighted by T
//   step 5  the matching backward, segment-reduced over the warp before the vector atomics
//
// One CTA per 16x16 tile, one warp per 8x4 pixel block, one lane per pixel.  The work of a warp is split into three
// kinds of phases so that the expensive arithmetic always runs on full warps:
//   A  geometry   the warp walks the tile's sorted list 32 entries at a time (lane = entry: coalesced id load, gather of
//                 the per-frame voxel record, pixel-rectangle pre-filter by ballot); for every surviving entry all lanes
//                 (= pixels) run the ray-AABB slab test, clip to their current interval of Algorithm 1 and apply the
//                 gating rule; hits are appended to a per-warp queue in shared memory as (voxel, pixel, a, b) items,
//                 ordered by list position - which is each pixel's own front-to-back order.
//   B  integrate  as soon as 32 items are queued: lane = item.  The trilinear raw density restricted to a ray segment
//                 is a cubic in the segment parameter, so the 8 corner values are folded into 4 coefficients once and
//                 each of the K samples costs a Horner evaluation and one ex2.  tau_v goes back to the queue.
//   C  blend      lane = pixel again: every pixel consumes its own items of the batch in order (T, C, D update and the
//                 T < t_stop test after every voxel, R3).  In the backward this phase produces dL/dtau_v and T alpha g_C
//                 per item, and a second lane = item phase (B2) turns them into corner gradients, reduces runs of items
//                 of the same voxel with shuffles and issues one 16-byte vector atomic per 4 floats.
// Gating (which list entry ends a pixel's current background / actor interval) is purely geometric, so phase A never
// needs T; early termination only removes pixels from later batches.
#include "dvx_ray.cuh"

namespace {

constexpr int TILE_THREADS = 256;
constexpr int TILE_WARPS = TILE_THREADS / 32;
constexpr int QCAP = 64;              // queue capacity per warp: at most 31 left-over items + 32 of one entry
constexpr uint32_t NONE = 0xFFFFFFFFu;
constexpr float LOG2E = 1.4426950408889634f;

template <bool BWD>
struct WarpQueue {
  uint32_t id[QCAP];     // item: global voxel id
  uint32_t meta[QCAP];   // item: pixel lane | tree << 8
  float a[QCAP], b[QCAP];  // item: clipped sub-segment [a,b] (O4)
  float tau[QCAP];       // phase B: tau_v;  backward phase C overwrites it with dL/dtau_v
  uint32_t e_id[QCAP];   // entry (one list element hit by >= 1 pixel): voxel id, hit-lane mask, index of its first item
  uint32_t e_mask[QCAP];
  uint32_t e_base[QCAP];
  float wg[BWD ? QCAP * 3 : 1];  // backward phase C: T alpha g_C per item, zero where the colour clamp is active
};

struct Pix {
  float C0, C1, C2, D, T;
  uint32_t n_used;
  bool done;
  float gC0, gC1, gC2, gD, gA, Xtot, Xpre, T_final;  // backward only
  uint32_t n_stop;
};

struct WarpCtx {
  int lane, u0, v0;     // u0,v0: pixel of lane 0 of this warp
  uint32_t lt;          // lanes below this one
};

__device__ __forceinline__ uint32_t warp_min_u32(uint32_t v) { return __reduce_min_sync(0xffffffffu, v); }

// ---- phase B arithmetic -------------------------------------------------------------------------------------------
// Coefficients of raw(lambda) = trilinear(g, p + q lambda), lambda in [0,1]; corner c = 4 b_x + 2 b_y + b_z (R7).
__device__ __forceinline__ void cubic_coeffs(const float g[8], const float p[3], const float q[3], float c[4]) {
  float A[4], B[4];
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const float dz = g[2 * i + 1] - g[2 * i];
    A[i] = fmaf(dz, p[2], g[2 * i]);
    B[i] = dz * q[2];
  }
  float Q[2][3];
#pragma unroll
  for (int bx = 0; bx < 2; ++bx) {
    const float dA = A[2 * bx + 1] - A[2 * bx], dB = B[2 * bx + 1] - B[2 * bx];
    Q[bx][0] = fmaf(dA, p[1], A[2 * bx]);
    Q[bx][1] = fmaf(dA, q[1], fmaf(dB, p[1], B[2 * bx]));
    Q[bx][2] = dB * q[1];
  }
  const float d0 = Q[1][0] - Q[0][0], d1 = Q[1][1] - Q[0][1], d2 = Q[1][2] - Q[0][2];
  c[0] = fmaf(d0, p[0], Q[0][0]);
  c[1] = fmaf(d0, q[0], fmaf(d1, p[0], Q[0][1]));
  c[2] = fmaf(d1, q[0], fmaf(d2, p[0], Q[0][2]));
  c[3] = d2 * q[0];
}

struct ItemGeom {
  float p[3], q[3];  // local coordinates u(lambda) = p + q lambda on the clipped segment
  float delta;       // (b - a) / K
};

// O6 for one queued item: K-point midpoint rule on [a,b].  Returns tau_v; with GRAD also the moments
// M_j = sum_k act'(raw_k) lambda_k^j (j = 0..3) from which phase B2 rebuilds sum_k act'(raw_k) w_c(u_k) for all corners.
template <bool GRAD>
__device__ __forceinline__ float integrate_item(const CompositeArgs &A, const WarpCtx &W, uint32_t id, uint32_t meta, float a,
                                                float b, ItemGeom &G, float M[4]) {
  const TreeFrame &T = A.trees[meta >> 8];
  const int pl = (int)(meta & 31u);
  const float xp = dvx_cam_x(A.p, W.u0 + (pl & 7)), yp = dvx_cam_y(A.p, W.v0 + (pl >> 3));
  const float rn = rsqrtf(xp * xp + yp * yp + 1.0f);
  const float4 f0 = __ldg(reinterpret_cast<const float4 *>(A.fvox + id));
  const float4 *gp = reinterpret_cast<const float4 *>(T.geo + (size_t)(id - T.base) * 8);
  const float4 g0 = __ldg(gp), g1 = __ldg(gp + 1);
  const float g[8] = {g0.x, g0.y, g0.z, g0.w, g1.x, g1.y, g1.z, g1.w};
  const float rel[3] = {f0.x, f0.y, f0.z};
  const float inv_s = 1.0f / f0.w;
  const float len = b - a;
#pragma unroll
  for (int ax = 0; ax < 3; ++ax) {
    const float d = dvx_dir_comp(T.N, ax, xp, yp) * rn;
    const float pa = __saturatef((a * d - rel[ax]) * inv_s);   // u clamped to [0,1]^3 (O6)
    const float pb = __saturatef((b * d - rel[ax]) * inv_s);
    G.p[ax] = pa;
    G.q[ax] = pb - pa;
  }
  float c[4];
  cubic_coeffs(g, G.p, G.q, c);
  const uint32_t K = A.p.k_samples, kind = A.p.activation;
  const float invK = 1.0f / (float)K;
  G.delta = len * invK;
  float S = 0.f;
  if (GRAD) M[0] = M[1] = M[2] = M[3] = 0.f;
  if (kind == 0) {  // exp: sigma = ex2(raw * log2 e), act' = act
    const float c0 = c[0] * LOG2E, c1 = c[1] * LOG2E, c2 = c[2] * LOG2E, c3 = c[3] * LOG2E;
    float lam = 0.5f * invK;
#pragma unroll 8
    for (uint32_t k = 0; k < K; ++k) {
      const float sig = exp2f(fmaf(fmaf(fmaf(c3, lam, c2), lam, c1), lam, c0));
      S += sig;
      if (GRAD) {
        M[0] += sig;
        float t = sig * lam; M[1] += t;
        t *= lam; M[2] += t;
        t *= lam; M[3] += t;
      }
      lam += invK;
    }
  } else {
    float lam = 0.5f * invK;
    for (uint32_t k = 0; k < K; ++k) {
      const float raw = fmaf(fmaf(fmaf(c[3], lam, c[2]), lam, c[1]), lam, c[0]);
      S += act_fn(raw, kind);
      if (GRAD) {
        const float ds = dact_fn(raw, kind);
        M[0] += ds;
        float t = ds * lam; M[1] += t;
        t *= lam; M[2] += t;
        t *= lam; M[3] += t;
      }
      lam += invK;
    }
  }
  return G.delta * S;
}

// sum_k act'(raw_k) w_c(u_k) for the 8 corners from the moments: w_c(lambda) = X_bx Y_by Z_bz with
// X_1 = p_x + q_x lambda, X_0 = (1 - p_x) - q_x lambda, ...  Contract the moments with Z, then Y, then X.
__device__ __forceinline__ void corner_sums(const ItemGeom &G, const float M[4], float out[8]) {
  float Nz[2][3];
#pragma unroll
  for (int bz = 0; bz < 2; ++bz) {
    const float z0 = bz ? G.p[2] : 1.0f - G.p[2], z1 = bz ? G.q[2] : -G.q[2];
#pragma unroll
    for (int j = 0; j < 3; ++j) Nz[bz][j] = fmaf(z1, M[j + 1], z0 * M[j]);
  }
  float Oy[2][2][2];
#pragma unroll
  for (int by = 0; by < 2; ++by) {
    const float y0 = by ? G.p[1] : 1.0f - G.p[1], y1 = by ? G.q[1] : -G.q[1];
#pragma unroll
    for (int bz = 0; bz < 2; ++bz)
#pragma unroll
      for (int j = 0; j < 2; ++j) Oy[by][bz][j] = fmaf(y1, Nz[bz][j + 1], y0 * Nz[bz][j]);
  }
#pragma unroll
  for (int bx = 0; bx < 2; ++bx) {
    const float x0 = bx ? G.p[0] : 1.0f - G.p[0], x1 = bx ? G.q[0] : -G.q[0];
#pragma unroll
    for (int by = 0; by < 2; ++by)
#pragma unroll
      for (int bz = 0; bz < 2; ++bz) out[4 * bx + 2 * by + bz] = fmaf(x1, Oy[by][bz][1], x0 * Oy[by][bz][0]);
  }
}

__device__ __forceinline__ void red_add_v4(float *addr, float x, float y, float z, float w) {
  asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(addr), "f"(x), "f"(y), "f"(z), "f"(w) : "memory");
}

// ---- phases B, C (and B2) over the first min(n_items, 32) queued items; the rest is shifted to the queue front ----
template <bool BWD>
__device__ __forceinline__ void flush_batch(const CompositeArgs &A, const WarpCtx &W, WarpQueue<BWD> &Q, int &n_items,
                                            int &n_ent, Pix &S) {
  const int lane = W.lane;
  const int count = n_items < 32 ? n_items : 32;
  __syncwarp();
  // -- B: lane = item
  ItemGeom G;
  float M[4];
  uint32_t my_id = NONE, my_meta = 0;
  if (lane < count) {
    my_id = Q.id[lane];
    my_meta = Q.meta[lane];
    Q.tau[lane] = integrate_item<BWD>(A, W, my_id, my_meta, Q.a[lane], Q.b[lane], G, M);
  }
  __syncwarp();
  // -- C: lane = pixel; entries in list order, i.e. in this pixel's front-to-back order
  int j = 0;
  uint32_t strad_mask = 0;  // hit lanes of an entry cut by the batch boundary that were NOT consumed
  bool strad = false;
  for (; j < n_ent; ++j) {
    const int base = (int)Q.e_base[j];
    if (base >= count) break;
    const uint32_t mask = Q.e_mask[j];
    const bool mine = (mask >> lane) & 1u;
    const int pos = base + __popc(mask & W.lt);
    const bool in_batch = mine && pos < count;
    if (base + __popc(mask) > count) {  // the entry straddles the boundary: keep the lanes beyond it for the next batch
      strad = true;
      strad_mask = mask & ~__ballot_sync(0xffffffffu, in_batch);
    }
    if (in_batch) {
      if (!S.done) {
        const float4 f1 = __ldg(reinterpret_cast<const float4 *>(A.fvox + Q.e_id[j]) + 1);
        const float tau = Q.tau[pos];
        const float ca = Q.a[pos], cb = Q.b[pos];
        const float e = exp2f(-tau * LOG2E);
        const float alpha = tau < 1e-3f ? tau * fmaf(-0.5f, tau, 1.0f) : 1.0f - e;  // 1 - exp(-tau) without cancellation
        const float w = S.T * alpha;
        const float mid = 0.5f * (ca + cb);
        if (!BWD) {
          S.C0 = fmaf(w, f1.x, S.C0); S.C1 = fmaf(w, f1.y, S.C1); S.C2 = fmaf(w, f1.z, S.C2);
          S.D = fmaf(w, mid, S.D);
        } else {
          const float X = S.gC0 * f1.x + S.gC1 * f1.y + S.gC2 * f1.z + S.gD * mid;
          S.Xpre = fmaf(w, X, S.Xpre);
          Q.tau[pos] = S.T * e * X - (S.Xtot - S.Xpre) + S.gA * S.T_final;  // dL/dtau_v
          const uint32_t cm = __float_as_uint(f1.w);
          Q.wg[3 * pos + 0] = (cm & 1u) ? 0.f : w * S.gC0;
          Q.wg[3 * pos + 1] = (cm & 2u) ? 0.f : w * S.gC1;
          Q.wg[3 * pos + 2] = (cm & 4u) ? 0.f : w * S.gC2;
        }
        S.T *= e;
        S.n_used++;
        if (!BWD) {
          if (S.T < A.p.t_stop) S.done = true;  // R3: tested after every voxel
        } else {
          if (S.n_used >= S.n_stop) S.done = true;
        }
      } else if (BWD) {  // queued before this pixel finished its replay: contributes nothing
        Q.tau[pos] = 0.f;
        Q.wg[3 * pos + 0] = 0.f; Q.wg[3 * pos + 1] = 0.f; Q.wg[3 * pos + 2] = 0.f;
      }
    }
  }
  const int j_keep = strad ? j - 1 : j;  // first entry that stays in the queue
  __syncwarp();
  // -- B2 (backward): lane = item again; corner gradients, run-reduced by voxel, vector atomics
  if (BWD) {
    float val[11];
#pragma unroll
    for (int c = 0; c < 11; ++c) val[c] = 0.f;
    if (lane < count) {
      const float dtau = Q.tau[lane] * G.delta;
      float cs[8];
      corner_sums(G, M, cs);
#pragma unroll
      for (int c = 0; c < 8; ++c) val[c] = dtau * cs[c];
      val[8] = Q.wg[3 * lane]; val[9] = Q.wg[3 * lane + 1]; val[10] = Q.wg[3 * lane + 2];
    }
    // items of one voxel are contiguous: segmented suffix sums, the first lane of each run ends up with the run total
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const uint32_t oid = __shfl_down_sync(0xffffffffu, my_id, o);
      const bool take = (lane + o < 32) && oid == my_id;
#pragma unroll
      for (int c = 0; c < 11; ++c) {
        const float x = __shfl_down_sync(0xffffffffu, val[c], o);
        if (take) val[c] += x;
      }
    }
    const uint32_t prev = __shfl_up_sync(0xffffffffu, my_id, 1);
    if (my_id != NONE && (lane == 0 || prev != my_id)) {
      const TreeFrame &T = A.trees[my_meta >> 8];
      if (T.dgeo) {
        float *dg = T.dgeo + (size_t)(my_id - T.base) * 8;
        red_add_v4(dg, val[0], val[1], val[2], val[3]);
        red_add_v4(dg + 4, val[4], val[5], val[6], val[7]);
      }
      red_add_v4(A.drgb + (size_t)my_id * 4, val[8], val[9], val[10], 0.f);
    }
  }
  // -- shift what is left to the queue front
  const int rem = n_items - count;
  const int ent_left = n_ent - j_keep;
  uint32_t t_id = 0, t_meta = 0, t_eid = 0, t_emask = 0, t_ebase = 0;
  float t_a = 0.f, t_b = 0.f;
  if (lane < rem) {
    t_id = Q.id[count + lane]; t_meta = Q.meta[count + lane]; t_a = Q.a[count + lane]; t_b = Q.b[count + lane];
  }
  if (lane < ent_left) {
    t_eid = Q.e_id[j_keep + lane];
    t_emask = Q.e_mask[j_keep + lane];
    t_ebase = Q.e_base[j_keep + lane];
    if (lane == 0 && strad) { t_emask = strad_mask; t_ebase = 0; }
    else t_ebase -= (uint32_t)count;
  }
  __syncwarp();
  if (lane < rem) { Q.id[lane] = t_id; Q.meta[lane] = t_meta; Q.a[lane] = t_a; Q.b[lane] = t_b; }
  if (lane < ent_left) { Q.e_id[lane] = t_eid; Q.e_mask[lane] = t_emask; Q.e_base[lane] = t_ebase; }
  __syncwarp();
  n_items = rem;
  n_ent = ent_left;
}

// ---- the kernel ------------------------------------------------------------------------------------------------------
template <bool BWD>
__global__ void __launch_bounds__(TILE_THREADS, 2) composite_tile_kernel(const CompositeArgs A) {
  __shared__ WarpQueue<BWD> s_queue[TILE_WARPS];
  const FrameParams &p = A.p;
  const int tile = blockIdx.x;
  const int warp = threadIdx.x >> 5;
  WarpCtx W;
  W.lane = threadIdx.x & 31;
  W.lt = (1u << W.lane) - 1u;
  W.u0 = (tile % p.tiles_x) * DVX_TILE + (warp & 1) * 8;
  W.v0 = (tile / p.tiles_x) * DVX_TILE + (warp >> 1) * 4;
  WarpQueue<BWD> &Q = s_queue[warp];
  const int lane = W.lane;
  const int u = W.u0 + (lane & 7), v = W.v0 + (lane >> 3);
  const bool inside = u < (int)p.width && v < (int)p.height;
  const size_t pix = (size_t)v * p.width + u;
  const bool counters = (p.flags & DVX_FLAG_COUNTERS) != 0;

  Pix S;
  S.C0 = S.C1 = S.C2 = 0.f; S.D = 0.f; S.T = 1.f; S.n_used = 0; S.done = !inside;
  S.Xpre = 0.f; S.n_stop = 0;
  if (BWD && inside) {
    S.gC0 = A.g_rgb[3 * pix]; S.gC1 = A.g_rgb[3 * pix + 1]; S.gC2 = A.g_rgb[3 * pix + 2];
    S.gD = A.g_depth ? A.g_depth[pix] : 0.f;
    S.gA = A.g_alpha ? A.g_alpha[pix] : 0.f;
    const float4 cd = reinterpret_cast<const float4 *>(A.sv_rgbd)[pix];
    S.Xtot = S.gC0 * cd.x + S.gC1 * cd.y + S.gC2 * cd.z + S.gD * cd.w;
    S.T_final = A.sv_T[pix];
    S.n_stop = A.sv_nused[pix];
    if (S.n_stop == 0) S.done = true;
  }
  const float xp = dvx_cam_x(p, u), yp = dvx_cam_y(p, v);
  const float rn = rsqrtf(xp * xp + yp * yp + 1.0f);

  // ---- step 3: intervals of the actors in this tile's mask, insertion-sorted by (tau_in, actor index) (O2, O3)
  float h_in[DVX_MAX_ACTORS], h_out[DVX_MAX_ACTORS];
  unsigned char h_idx[DVX_MAX_ACTORS];
  int m = 0;
  {
    unsigned long long am = A.actor_mask[tile];
    while (am) {
      const int i = __ffsll((long long)am) - 1;
      am &= am - 1;
      if (S.done) continue;
      const TreeFrame &T = A.trees[1 + i];
      Ray r; int q;
      make_ray(T.N, xp, yp, rn, r, q);
      float tin, tout;
      if (ray_box(T, r, p.near_, p.far_, tin, tout)) {
        int j = m++;
        while (j > 0 && h_in[j - 1] > tin) {  // ties keep the lower actor index first
          h_in[j] = h_in[j - 1]; h_out[j] = h_out[j - 1]; h_idx[j] = h_idx[j - 1];
          --j;
        }
        h_in[j] = tin; h_out[j] = tout; h_idx[j] = (unsigned char)i;
      }
    }
  }

  // ---- step 4: Algorithm 1 as a per-lane state machine; the warp serves one (tree, octant) list at a time
  float cur = p.near_;   // tau_curr
  int h = 0;             // next entry of the hit list
  int stage = 0;         // 0: background before hit h (or the final background), 1: actor of hit h, 2: finished
  uint32_t cur0 = NONE;  // this pixel's cursor in the static list of its octant (persists across background intervals)
  int n_items = 0, n_ent = 0;
  unsigned long long q_test = 0;
  const uint32_t wu0 = (uint32_t)W.u0, wv0 = (uint32_t)W.v0, wu1 = wu0 + 7u, wv1 = wv0 + 3u;

  uint32_t seg_tree = NONE;  // pending segment of this lane: tree and interval [lo, hi]
  float lo = 0.f, hi = 0.f;
  for (;;) {
    // -- this lane's next non-empty segment of Algorithm 1 (kept until the warp serves its tree)
    if (S.done) seg_tree = NONE;
    while (seg_tree == NONE && !S.done && stage != 2) {
      if (stage == 0) {
        if (h < m) {
          const float tin = h_in[h];
          stage = 1;
          if (tin > cur) { seg_tree = 0; lo = cur; hi = tin; break; }           // background before object entry
        } else {
          stage = 2;
          if (p.far_ > cur) { seg_tree = 0; lo = cur; hi = p.far_; break; }     // remaining background
        }
      } else {
        const float tin = h_in[h], tout = h_out[h];
        const float l = fmaxf(tin, cur);
        const uint32_t t = 1u + h_idx[h];
        cur = fmaxf(cur, tout);
        ++h;
        stage = 0;
        if (tout > l) { seg_tree = t; lo = l; hi = tout; break; }                // object in its canonical local space
      }
    }
    const uint32_t t = warp_min_u32(seg_tree);
    if (t == NONE) break;
    const bool part = seg_tree == t;
    const TreeFrame &T = A.trees[t];
    Ray r; int q = 0;
    make_ray(T.N, xp, yp, rn, r, q);
    uint32_t omask = __reduce_or_sync(0xffffffffu, part ? (1u << q) : 0u);
    while (omask) {
      const int qq = __ffs(omask) - 1;
      omask &= omask - 1;
      const size_t bucket = ((size_t)tile * p.n_trees + t) * 8 + qq;
      const uint32_t beg = __ldg(A.range_beg + bucket), end = __ldg(A.range_end + bucket);
      bool active = part && q == qq;
      uint32_t c_l = beg;
      if (t == 0 && cur0 != NONE) c_l = cur0;
      uint32_t pos = warp_min_u32(active ? c_l : NONE);
      while (pos < end && __any_sync(0xffffffffu, active)) {
        const uint32_t n = min(32u, end - pos);
        uint32_t id = 0;
        float4 f0 = make_float4(0.f, 0.f, 0.f, 0.f);
        bool c = false;
        if ((uint32_t)lane < n) {
          id = __ldg(A.ids + pos + lane);
          const ushort4 rc = __ldg(A.pxrect + id);
          f0 = __ldg(reinterpret_cast<const float4 *>(A.fvox + id));
          c = rc.x <= wu1 && rc.z >= wu0 && rc.y <= wv1 && rc.w >= wv0;
        }
        uint32_t cand = __ballot_sync(0xffffffffu, c);
        while (cand) {
          const int j = __ffs(cand) - 1;
          cand &= cand - 1;
          const uint32_t e = pos + j;
          const uint32_t id_e = __shfl_sync(0xffffffffu, id, j);
          const float rel[3] = {__shfl_sync(0xffffffffu, f0.x, j), __shfl_sync(0xffffffffu, f0.y, j),
                                __shfl_sync(0xffffffffu, f0.z, j)};
          const float s = __shfl_sync(0xffffffffu, f0.w, j);
          bool emit = false;
          float ca = 0.f, cb = 0.f;
          if (active && c_l <= e) {
            float a, b;
            if (counters) ++q_test;
            if (slab_rel(r, rel, s, a, b) && b > a) {
              if (a >= hi) {            // the voxel starts at or beyond the interval end: gate here
                active = false; c_l = e;
              } else {
                ca = fmaxf(a, lo); cb = fminf(b, hi);   // R1: clip to the interval
                emit = cb > ca;
                if (b > hi) { active = false; c_l = e; }  // sticks out: it may own a second piece after the box
              }
            }
          }
          const uint32_t mk = __ballot_sync(0xffffffffu, emit);
          if (mk) {
            if (lane == 0) { Q.e_id[n_ent] = id_e; Q.e_mask[n_ent] = mk; Q.e_base[n_ent] = (uint32_t)n_items; }
            if (emit) {
              const int at = n_items + __popc(mk & W.lt);
              Q.id[at] = id_e; Q.meta[at] = (uint32_t)lane | (t << 8); Q.a[at] = ca; Q.b[at] = cb;
            }
            ++n_ent;
            n_items += __popc(mk);
            if (n_items >= 32) {
              flush_batch<BWD>(A, W, Q, n_items, n_ent, S);
              active = active && !S.done;
            }
          }
          if (!__any_sync(0xffffffffu, active)) break;
        }
        pos += 32;
      }
      if (part && q == qq) {
        if (active) c_l = end;          // walked off the list: nothing left for later intervals either
        if (t == 0) cur0 = c_l;
      }
    }
    if (part) seg_tree = NONE;          // served
  }
  while (n_items > 0) flush_batch<BWD>(A, W, Q, n_items, n_ent, S);

  if (!BWD && inside) {
    A.rgb[3 * pix] = S.C0; A.rgb[3 * pix + 1] = S.C1; A.rgb[3 * pix + 2] = S.C2;
    A.depth[pix] = S.D;
    A.alpha[pix] = 1.0f - S.T;
    if (A.sv_rgbd) {
      reinterpret_cast<float4 *>(A.sv_rgbd)[pix] = make_float4(S.C0, S.C1, S.C2, S.D);
      A.sv_T[pix] = S.T;
      A.sv_nused[pix] = S.n_used;
    }
  }
  if (counters && !BWD) {
    unsigned long long qt = q_test, qh = S.n_used;
    for (int o = 16; o > 0; o >>= 1) {
      qt += __shfl_xor_sync(0xffffffffu, qt, o);
      qh += __shfl_xor_sync(0xffffffffu, qh, o);
    }
    if (lane == 0) {
      atomicAdd(&A.counters[CNT_QTEST], qt);
      atomicAdd(&A.counters[CNT_QHIT], qh);
    }
  }
}

}  // namespace

void dvx_composite_tile_launch(const CompositeArgs &a, bool backward, cudaStream_t st) {
  if (a.p.n_tiles == 0) return;
  DVX_COUNT_LAUNCH(1);
  if (backward)
    composite_tile_kernel<true><<<a.p.n_tiles, TILE_THREADS, 0, st>>>(a);
  else
    composite_tile_kernel<false><<<a.p.n_tiles, TILE_THREADS, 0, st>>>(a);
}
