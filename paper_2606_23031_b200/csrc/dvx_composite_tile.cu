// dvx_composite_tile.cu - hot-path steps 3, 4 and 5, the production kernels.
//   step 3  per-ray ray-OBB intervals [tau_in^i, tau_out^i] sorted front to back
//   step 4  Algorithm 1: F over Morton-ordered per-tile voxel lists, segment by segment, carrying
//           S = (C, D, T, tau_curr); trilinear raw density, K midpoint samples, activation,
//           alpha = 1 - exp(-sum sigma dt), blend weighted by T
//   step 5  the matching backward, run-reduced over the warp before the vector atomics
//
// One CTA per 16x16 tile, one warp per 4x8 pixel block (DVX_WARP_W x 32/DVX_WARP_W; 4x8 measured best on config 3), one lane per pixel.  The work of a warp is split into phases so
// that the expensive arithmetic always runs on full warps:
//   A  geometry   the warp walks the tile's sorted list 32 entries at a time.  First lane = entry: coalesced id load,
//                 pixel-rectangle pre-filter, Morton decode and - in fp64, once per (warp, entry) - the voxel centre
//                 split into its distance t0 along the warp's reference direction d0 and the small remainder m0.
//                 Then lane = pixel: for every surviving entry the slab test runs on small, well-conditioned numbers
//                 (x(tau) - c = s' d + (t0 e - m0), s' = tau - t0, e = d - d0), is clipped to the pixel's current interval
//                 of Algorithm 1 (R1) and gated; hits go to a per-warp ring in shared memory as items, ordered by list
//                 position = each pixel's own front-to-back order.
//   B  integrate  as soon as 32 items are queued: lane = item.  The trilinear raw density restricted to a ray segment
//                 is a cubic in the segment parameter: the 8 corner values fold into 4 coefficients once, each of the
//                 K samples is a Horner evaluation and one ex2.
//   C  blend      lane = pixel again: every pixel consumes its own items of the batch in order (a per-lane bit mask of
//                 ring positions): T, C, D update and the T < t_stop test after every voxel (R3).  In the backward this
//                 phase produces dL/dtau_v and T alpha g_C per item, and a second lane = item phase (B2) turns them
//                 into corner gradients, reduces runs of items of the same voxel with shuffles and issues 16-byte
//                 vector reductions (red.global.add.v4.f32).
// Gating (which list entry ends a pixel's current background / actor interval) is purely geometric, so phase A never
// needs T; early termination only removes pixels from later batches.
#include "dvx_ray.cuh"

namespace {

constexpr int DVX_TILE_SPLIT = 2;  // CTAs per 16x16 tile (1, 2, 4 or 8): a CTA holds 8 / DVX_TILE_SPLIT of the tile's warps.  Measured on
                          // B200, step ms for 1 / 2 / 4: config 3 4.00 / 3.92 / 3.98, config 4 5.32 / 5.25 / 5.32 (finer tail)
constexpr int TILE_SPLIT = DVX_TILE_SPLIT;
constexpr int TILE_THREADS = 256 / TILE_SPLIT;
constexpr int TILE_WARPS = TILE_THREADS / 32;
constexpr int DVX_TILE_MIN_CTAS = (3 * DVX_TILE_SPLIT);
// Backward run reduction: runs of one voxel are reduced in pieces of at most 4 lanes (1, 2, 8, 16, 32 measured slower) unless the
// whole batch is ONE voxel: then the run is reduced whole (phase_B2).
constexpr int DVX_CAND_GROUPS = 8;  // phase A: bands of rows of the warp's pixel block that walk their candidates independently.  Forward
                           // compositing of a saved frame, config 3 / config 4, ms, for 1, 2, 4, 8 bands: 1.378 1.377 1.354 1.312 / 1.934 1.943 1.935 1.888
constexpr int DVX_WARP_W = 4;  // a warp covers DVX_WARP_W x (32 / DVX_WARP_W) pixels
constexpr int WARP_W = DVX_WARP_W, WARP_H = 32 / DVX_WARP_W, WARPS_X = DVX_TILE / WARP_W;
constexpr int QCAP = 64;              // ring capacity per warp: at most 31 left-over items + 32 of one entry
constexpr uint32_t NONE = 0xFFFFFFFFu;
constexpr float LOG2E = 1.4426950408889634f;

// One list entry as phase A (lane = pixel) sees it, staged by the lane that owns the entry.
struct __align__(16) EntryRec {
  float t0;       // distance of the voxel centre along the warp's reference direction d0
  float m0[3];    // centre - t0 d0 (tree frame)
  uint32_t id;    // global voxel id                 } same order as the head of Item: phase A's item store takes the
  uint32_t meta;  // tree << 8 | level << 16         } pair as it was loaded
  float hs;       // half edge length
  uint32_t pad;
};

// One queued (pixel, voxel) hit: 48 bytes, written with three 16-byte stores in phase A.
struct __align__(16) Item {
  uint32_t id;        // global voxel id
  uint32_t meta;      // tree << 8 | level << 16 (the low byte is free here; see pad)
  float ca, cb;       // clipped sub-segment, relative to t0 (O4, R1)
  float w[3];         // x(tau) - centre = s' d + w
  float mid;          // (a + b) / 2, absolute ray distance (depth, R9)
  float d[3];         // ray direction in the tree frame
  float pad;          // as bits: the lane (0..31) of the pixel that owns the item; item_geom ORs it into the low byte of meta
};

// phase B -> C (-> B2), per batch item (written by the item's lane, read by the pixel's lane):
template <bool NRM>
struct BatchShared {
  float4 eam[32];               // forward: exp(-tau_v), alpha_v, (a+b)/2, voxel id (the weight export reads it);
                                // backward: exp(-tau_v), alpha_v, X_v = g_C . rgb_v + g_D mid_v (+ g_N . n_v); phase C then
                                // overwrites .z with dL/dtau_v and .w with the blend weight T alpha for phase B2
  float4 rgbm[32];              // forward: the voxel's RGB and clamp bits
  float4 nrm[NRM ? 32 : 1];     // the voxel's world normal (O11)
  // backward: the incoming gradients of the warp's 32 pixels (g_C, g_D) and (g_N), filled once per kernel.  An item's lane
  // reads its pixel's entry in phase B (the pixel's lane index travels in the low byte of the item's meta word), so that
  // everything of dL/dtau_v that does not depend on the blend order is computed with all lanes busy
  float4 pg[32];
  float4 pn[NRM ? 32 : 1];
};

// Everything only the batch phases touch lives in shared memory, not in registers: the candidate loop of phase A runs
// under an 80-register cap, and what it does not need must not be live across it (the compiler otherwise re-derives lane,
// warp and queue addresses from tid.x inside the loop: 6 % of the forward's instructions in profiles/r02a).
template <bool NRM>
struct WarpQueue {
  EntryRec ent[32];
  Item item[QCAP];              // ring
  double d0[3];                 // the warp's reference direction for the list being served
  BatchShared<NRM> b;
  float4 dir[32];               // per pixel: its ray direction in the frame of the list being served, .w = the pixel's lane
                                // index as bits (copied into every item)
  float4 acc[32];               // forward, per pixel between batches: C (rgb) and D
  float2 tn[32];                //          T and n_used (as bits)
  float4 nacc[NRM ? 32 : 1];    //          N (O11)
  uint32_t rec_n;               // chunks this warp has taken for its hit-record stream (dvx_internal.cuh); lane 0 only
};

struct Pix {
  float C0, C1, C2, D, T;
  uint32_t n_used;
  uint32_t done;  // 0 / 1 (a full register: as a bool it was packed into a byte lane with PRMT)
  float gC0, gC1, gC2, gD, gA, Xtot, Xpre, T_final;  // backward only
  uint32_t n_stop;
  float N0, N1, N2;     // normal map (O11), forward
  float gN0, gN1, gN2;  // dL/dN, backward
  uint32_t exp_pos;     // weight export (row N3): start of this pixel's row in the CSR arrays
};

__device__ __forceinline__ uint32_t warp_min_u32(uint32_t v) { return __reduce_min_sync(0xffffffffu, v); }
__device__ __forceinline__ float ex2_approx(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ uint32_t lanemask_lt() {  // one S2R where it is used; kept in a register it was rebuilt from tid.x
  uint32_t m;
  asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m));
  return m;
}
__device__ __forceinline__ double shfl_double(double v, int src) {
  int lo = __double2loint(v), hi = __double2hiint(v);
  lo = __shfl_sync(0xffffffffu, lo, src);
  hi = __shfl_sync(0xffffffffu, hi, src);
  return __hiloint2double(hi, lo);
}
__device__ __forceinline__ double rcp_double(double x) {  // 1/x to ~1e-14 relative: fp32 seed + one Newton step
  double r = (double)__frcp_rn((float)x);
  return r * (2.0 - x * r);
}

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

// One queued item (ring slot `at`) as phase B needs it: voxel, tree / level, and the clipped segment in the voxel's local
// coordinates, u(lambda) = p + q lambda with u clamped to [0,1]^3 (O6).
template <bool NRM>
__device__ __forceinline__ void item_geom(const CompositeArgs &A, const WarpQueue<NRM> &Q, const uint4 *s_tree, int at,
                                          uint32_t &id, uint32_t &meta, ItemGeom &G, float &mid) {
  const float4 i0 = *reinterpret_cast<const float4 *>(&Q.item[at]);        // id, meta, ca, cb
  const float4 i1 = *(reinterpret_cast<const float4 *>(&Q.item[at]) + 1);  // w, mid
  const float4 i2 = *(reinterpret_cast<const float4 *>(&Q.item[at]) + 2);  // d
  id = __float_as_uint(i0.x);
  meta = __float_as_uint(i0.y) | __float_as_uint(i2.w);  // low byte: lane of the pixel that owns the item
  mid = i1.w;
  const uint32_t level = __float_as_uint(i0.y) >> 16;
  // 1 / edge length = (1 / level-16 cell) * 2^(level - 16): exact power-of-two scaling
  const float inv_s = __uint_as_float(s_tree[(meta >> 8) & 0xFFu].w) * __uint_as_float((111u + level) << 23);
  const float ca = i0.z, cb = i0.w;
  const float dd[3] = {i2.x, i2.y, i2.z}, ww[3] = {i1.x, i1.y, i1.z};
#pragma unroll
  for (int ax = 0; ax < 3; ++ax) {
    const float d = dd[ax], w = ww[ax];
    const float pa = __saturatef(fmaf(fmaf(ca, d, w), inv_s, 0.5f));
    const float pb = __saturatef(fmaf(fmaf(cb, d, w), inv_s, 0.5f));
    G.p[ax] = pa;
    G.q[ax] = pb - pa;
  }
  G.delta = (cb - ca) * A.p.inv_k;
}

// O6 for one item: K-point midpoint rule on the clipped segment.  Returns tau_v; with BWD also the moments
// M_j = sum_k act'(raw_k) lambda_k^j (j = 0..3), from which phase B2 rebuilds sum_k act'(raw_k) w_c(u_k).
template <bool BWD>
__device__ __forceinline__ float integrate_geom(const CompositeArgs &A, const uint4 *s_tree, uint32_t id, uint32_t meta,
                                                const ItemGeom &G, float M[4]) {
  const uint4 tf = s_tree[(meta >> 8) & 0xFFu];  // geo pointer, base, 1 / cell of the item's octree (per-CTA table)
  const float *geo = reinterpret_cast<const float *>(((unsigned long long)tf.y << 32) | tf.x);
  const float4 *gp = reinterpret_cast<const float4 *>(geo + (size_t)(id - tf.z) * 8);
  const float4 g0 = __ldg(gp), g1 = __ldg(gp + 1);
  const float g[8] = {g0.x, g0.y, g0.z, g0.w, g1.x, g1.y, g1.z, g1.w};
  float c[4];
  cubic_coeffs(g, G.p, G.q, c);
  const uint32_t K = A.p.k_samples, kind = A.p.activation;
  const float invK = A.p.inv_k;
  float S = 0.f;
  if (BWD) M[0] = M[1] = M[2] = M[3] = 0.f;
  float lam = 0.5f * invK;
  if (kind == 0 && K == 8) {  // the configured case: exp, 8 samples at lambda = (k + 1/2) / 8 as immediates
    const float c0 = c[0] * LOG2E, c1 = c[1] * LOG2E, c2 = c[2] * LOG2E, c3 = c[3] * LOG2E;
#pragma unroll
    for (int k = 0; k < 8; ++k) {
      const float l8 = (float)(2 * k + 1) * 0.0625f;   // lambda_k and its powers are exact in fp32 (odd / 16, / 256, / 4096)
      const float sig = ex2_approx(fmaf(fmaf(fmaf(c3, l8, c2), l8, c1), l8, c0));
      S += sig;
      if (BWD) {  // one FFMA per moment with an immediate power of lambda_k
        M[1] = fmaf(sig, l8, M[1]);
        M[2] = fmaf(sig, l8 * l8, M[2]);
        M[3] = fmaf(sig, l8 * l8 * l8, M[3]);
      }
    }
    if (BWD) M[0] = S;  // act' = act for exp
  } else if (kind == 1 && K == 8) {  // exp-linear (R5, theta = 1.1) at the configured K: unrolled like the exp case
    constexpr float TH = 1.1f, A1 = LOG2E / TH, A0 = (0.09531017980432493f - 1.0f) * LOG2E;  // ex2(A1 raw + A0) = exp(raw/theta - 1 + ln theta)
#pragma unroll
    for (int k = 0; k < 8; ++k) {
      const float l8 = (float)(2 * k + 1) * 0.0625f;
      const float raw = fmaf(fmaf(fmaf(c[3], l8, c[2]), l8, c[1]), l8, c[0]);
      const float ex = ex2_approx(fmaf(raw, A1, A0));
      const bool lin = raw > TH;
      S += lin ? raw : ex;
      if (BWD) {
        const float ds = lin ? 1.0f : ex * (1.0f / TH);
        M[0] += ds;
        M[1] = fmaf(ds, l8, M[1]);
        M[2] = fmaf(ds, l8 * l8, M[2]);
        M[3] = fmaf(ds, l8 * l8 * l8, M[3]);
      }
    }
  } else if (kind == 0) {  // exp: sigma = ex2(raw * log2 e), act' = act
    const float c0 = c[0] * LOG2E, c1 = c[1] * LOG2E, c2 = c[2] * LOG2E, c3 = c[3] * LOG2E;
#pragma unroll 4
    for (uint32_t k = 0; k < K; ++k) {
      const float sig = ex2_approx(fmaf(fmaf(fmaf(c3, lam, c2), lam, c1), lam, c0));
      S += sig;
      if (BWD) {
        M[0] += sig;
        float t = sig * lam; M[1] += t;
        t *= lam; M[2] += t;
        t *= lam; M[3] += t;
      }
      lam += invK;
    }
  } else {
    for (uint32_t k = 0; k < K; ++k) {
      const float raw = fmaf(fmaf(fmaf(c[3], lam, c[2]), lam, c[1]), lam, c[0]);
      S += act_fn(raw, kind);
      if (BWD) {
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
  // the b = 1 factor of an axis is u = p + q lambda, the b = 0 factor is 1 - u: contract with u, get the other half by
  // subtracting from the uncontracted sums: 33 instructions instead of 44.  Every term is a sum of non-negative products
  // (act' >= 0, u in [0,1]), so a difference loses accuracy only relative to a corner weight that is itself ~0: the error
  // stays ~1e-7 of the voxel's largest corner gradient (parity tolerance 1e-3 relative, 1e-6 absolute).
  // Replay 1.062 -> 1.044 ms on config 3, 1.742 -> 1.705 on config 4.
  float Nz[2][3];
#pragma unroll
  for (int j = 0; j < 3; ++j) {
    Nz[1][j] = fmaf(G.q[2], M[j + 1], G.p[2] * M[j]);
    Nz[0][j] = M[j] - Nz[1][j];
  }
  float Oy[2][2][2];
#pragma unroll
  for (int bz = 0; bz < 2; ++bz)
#pragma unroll
    for (int j = 0; j < 2; ++j) {
      Oy[1][bz][j] = fmaf(G.q[1], Nz[bz][j + 1], G.p[1] * Nz[bz][j]);
      Oy[0][bz][j] = Nz[bz][j] - Oy[1][bz][j];
    }
#pragma unroll
  for (int by = 0; by < 2; ++by)
#pragma unroll
    for (int bz = 0; bz < 2; ++bz) {
      const float hi = fmaf(G.q[0], Oy[by][bz][1], G.p[0] * Oy[by][bz][0]);
      out[4 + 2 * by + bz] = hi;
      out[2 * by + bz] = Oy[by][bz][0] - hi;
    }
}

__device__ __forceinline__ void red_add_v4(float *addr, float x, float y, float z, float w) {
  asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(addr), "f"(x), "f"(y), "f"(z), "f"(w) : "memory");
}

// ---- phases B, C and B2 of one batch of up to 32 items ---------------------------------------------------------------
// The list-walking kernels take the batch from the head of the warp's ring (flush_batch), the replay kernel from the hit
// records the forward wrote (composite_replay_kernel); from there on both run the same three phases.

// -- B: lane = item (lanes < count).  tau_v, exp(-tau_v), alpha_v, the voxel's colour (and normal) -> shared memory, so that
// C's serial per-pixel loop contains no transcendental and no global load.
// The colour (and normal) loads go out before the integration so their latency hides under it - in the backward too since
// the pixels' gradients left the registers for the shared-memory table (before that the four extra live registers spilled
// there; end of round 2: replay 1.114 -> 1.083 ms with the early load).
template <bool BWD, bool NRM>
__device__ __forceinline__ void phase_B(const CompositeArgs &A, const uint4 *s_tree, int lane, BatchShared<NRM> &bs, uint32_t id,
                                        uint32_t meta, const ItemGeom &G, float mid, float M[4], float gv[NRM ? 6 : 3]) {
  float4 f1, nv = make_float4(0.f, 0.f, 0.f, 0.f);
  f1 = __ldg(reinterpret_cast<const float4 *>(A.fvox + id) + 1);
  if (NRM) nv = __ldg(A.vnrm + id);
  const float tau = integrate_geom<BWD>(A, s_tree, id, meta, G, M);
  const float e = ex2_approx(-tau * LOG2E);
  const float alpha = tau < 1e-3f ? tau * fmaf(-0.5f, tau, 1.0f) : 1.0f - e;  // 1 - exp(-tau) without cancellation
  if (!BWD) {
    bs.eam[lane] = make_float4(e, alpha, mid, __uint_as_float(id));
    bs.rgbm[lane] = f1;
    if (NRM) bs.nrm[lane] = nv;
  } else {
    // what phase C needs of this item besides the blend order: X_v = g_C . rgb_v + g_D mid_v (+ g_N . n_v) with the gradients
    // of the item's pixel; what phase B2 needs: the pixel's g_C with the clamped channels zeroed (O7) (and g_N)
    const uint32_t pl = meta & 31u;
    const float4 g = bs.pg[pl];
    float X = g.x * f1.x + g.y * f1.y + g.z * f1.z + g.w * mid;
    const uint32_t cm = __float_as_uint(f1.w);  // colour clamp active: no gradient through that channel (O7)
    gv[0] = (cm & 1u) ? 0.f : g.x; gv[1] = (cm & 2u) ? 0.f : g.y; gv[2] = (cm & 4u) ? 0.f : g.z;
    if (NRM) {
      const float4 gn = bs.pn[pl];
      X += gn.x * nv.x + gn.y * nv.y + gn.z * nv.z;
      gv[3] = gn.x; gv[4] = gn.y; gv[5] = gn.z;
    }
    bs.eam[lane] = make_float4(e, alpha, X, 0.f);
  }
}

// -- C: lane = pixel; its own items of the batch (bit i of `mine` = item i) in batch order = front-to-back order along its
// ray: T, C, D update and the T < t_stop test after every voxel (R3).  The backward leaves dL/dtau_v and T alpha g_C (g_N)
// per item in shared memory for B2.
template <bool BWD, bool NRM, bool EXP>
__device__ __forceinline__ void phase_C(const CompositeArgs &A, BatchShared<NRM> &bs, uint32_t mine, Pix &S) {
  while (mine) {
    const int i = __ffs(mine) - 1;
    mine &= mine - 1;
    if (!S.done) {
      const float4 ea = bs.eam[i];
      const float e = ea.x;
      const float w = S.T * ea.y;
      if (EXP) {  // row N3: the compositing weight of this (pixel, voxel), in the pixel's front-to-back order
        if (S.n_used < S.n_stop) {
          const uint32_t at = S.exp_pos + S.n_used;
          A.exp_vox[at] = __float_as_uint(ea.w);
          A.exp_w[at] = w;
        }
      }
      if (!BWD) {
        const float4 f1 = bs.rgbm[i];
        const float mid = ea.z;
        S.C0 = fmaf(w, f1.x, S.C0); S.C1 = fmaf(w, f1.y, S.C1); S.C2 = fmaf(w, f1.z, S.C2);
        S.D = fmaf(w, mid, S.D);
        if (NRM) {
          const float4 nv = bs.nrm[i];
          S.N0 = fmaf(w, nv.x, S.N0); S.N1 = fmaf(w, nv.y, S.N1); S.N2 = fmaf(w, nv.z, S.N2);
        }
      } else {
        const float X = ea.z;  // phase B: g_C . rgb_v + g_D mid_v (+ g_N . n_v)
        S.Xpre = fmaf(w, X, S.Xpre);
        const float dtau = S.T * e * X - (S.Xtot - S.Xpre) + S.gA * S.T_final;  // dL/dtau_v
        *reinterpret_cast<float2 *>(&bs.eam[i].z) = make_float2(dtau, w);
      }
      S.T *= e;
      S.n_used++;
      if (!BWD) {
        if (S.T < A.p.t_stop) S.done = true;  // R3: tested after every voxel
      } else {
        if (S.n_used >= S.n_stop) S.done = true;
      }
    } else if (BWD) {  // queued before this pixel finished its replay: contributes nothing
      *reinterpret_cast<float2 *>(&bs.eam[i].z) = make_float2(0.f, 0.f);
    }
  }
}

// -- B2 (backward): lane = item again; corner gradients, run-reduced by voxel, vector reductions
template <bool NRM>
__device__ __forceinline__ void phase_B2(const CompositeArgs &A, int lane, int count, const BatchShared<NRM> &bs, const uint4 *s_tree,
                                         float *const *s_dgeo, uint32_t my_id, uint32_t my_meta, const ItemGeom &G, const float M[4],
                                         const float gv[NRM ? 6 : 3]) {
  constexpr int NV = NRM ? 14 : 11;  // 8 corner gradients, 3 colour, (3 normal)
  // Every lane computes: lanes past the batch's items (my_id == NONE, only in a warp's last batch) hold defined but
  // meaningless G / M / gv (the caller initialises them), form pieces of their own and issue no reduction.  (With the
  // values zeroed first and the arithmetic under `lane < count`: replay 1.114 -> 1.095 ms without.)
  float val[NV];
  {
    const float2 dw = *reinterpret_cast<const float2 *>(&bs.eam[lane].z);  // phase C: dL/dtau_v, T alpha
    const float dtau = dw.x * G.delta;
    float cs[8];
    corner_sums(G, M, cs);
#pragma unroll
    for (int c = 0; c < 8; ++c) val[c] = dtau * cs[c];
    val[8] = dw.y * gv[0]; val[9] = dw.y * gv[1]; val[10] = dw.y * gv[2];
    if (NRM) { val[NV - 3] = dw.y * gv[3]; val[NV - 2] = dw.y * gv[4]; val[NV - 1] = dw.y * gv[5]; }
  }
  // Items of one voxel sit next to each other in the batch (the pixels one list entry hit in one trip of phase A).  They are
  // summed in pieces: ADJACENT lanes with the same voxel id inside one aligned group of 4 lanes - two segmented shuffle steps,
  // no ballots and no run numbering, the piece a lane belongs to follows from its neighbours' ids alone (adjacency matters: a
  // voxel cut in two by a box is queued twice, with other voxels in between, and those stay separate pieces).  The first
  // lane of a piece issues its reductions; a run that straddles a group boundary, or is longer than 4, issues several: the L2
  // absorbs ~3x more reductions cheaper than three more shuffle rounds (pieces of 1, 2, 8, 16, 32 lanes measured slower).
  // Not so where many warps hammer the same voxel: a batch that is ONE voxel (it covers the warp's 4x8 pixels, so its
  // neighbours' too) is summed whole, see below.  Warp-uniform choice.
  // Round 2: pieces were first defined relative to the run's start (a ballot of run heads, clz, a second ballot, popc):
  // ten more instructions per batch, fewer reductions; the aligned form is faster on config 3 (replay 1.152 -> 1.133 ms)
  // and on config 4 (1.932 -> 1.890 ms).
  if (__all_sync(0xffffffffu, my_id == __shfl_sync(0xffffffffu, my_id, 0))) {
    // The whole batch is ONE voxel (coarse voxels near the camera cover whole 4x8 blocks, trip after trip; common on config 4's
    // coarse static octree).  All 32 lanes are summed, by a transposing butterfly: at the step over lane bit b a lane keeps the half of its
    // values whose index has the matching bit, gets the partner's copy of that half and hands over the other half, so the
    // number of values per lane halves as the number of lanes per sum doubles - 8 + 4 + 2 + 1 + 1 shuffles instead of 5 x NV.
    // Lane 2 i then holds the total of value i and issues one scalar reduction (the 11 or 14 of them are one instruction).
    // Against five plain shuffle steps into lane 0: replay 1.781 -> 1.742 ms on config 4, unchanged on config 3 (1.06 ms).
    float v[16];
#pragma unroll
    for (int c = 0; c < 16; ++c) v[c] = c < NV ? val[c] : 0.f;
#pragma unroll
    for (int h = 8; h >= 1; h >>= 1) {      // h values survive the step over lane bit 2 h
      const bool up = (lane & (2 * h)) != 0;
#pragma unroll
      for (int c = 0; c < h; ++c) {
        const float keep = up ? v[c + h] : v[c], send = up ? v[c] : v[c + h];
        v[c] = keep + __shfl_xor_sync(0xffffffffu, send, 2 * h);
      }
    }
    v[0] += __shfl_xor_sync(0xffffffffu, v[0], 1);
    const int idx = lane >> 1;             // bits 4..1 of the lane = bits 3..0 of the value's index
    if (!(lane & 1) && idx < NV && my_id != NONE) {
      if (idx < 8) {
        const uint32_t ti = (my_meta >> 8) & 0xFFu;
        if (s_dgeo[ti]) atomicAdd(s_dgeo[ti] + (size_t)(my_id - s_tree[ti].z) * 8 + idx, v[0]);
      } else if (idx < 11) {
        atomicAdd(A.drgb + (size_t)my_id * 4 + (idx - 8), v[0]);
      } else if (NRM) {
        atomicAdd(A.dnrm + (size_t)my_id * 4 + (idx - 11), v[0]);
      }
    }
    return;
  }
  const uint32_t prev = __shfl_up_sync(0xffffffffu, my_id, 1);
  const uint32_t id1 = __shfl_down_sync(0xffffffffu, my_id, 1), id2 = __shfl_down_sync(0xffffffffu, my_id, 2);
  const int sub = lane & 3;
  const bool take1 = sub < 3 && id1 == my_id;
  const bool take2 = sub < 2 && take1 && id2 == my_id;
  const bool is_head2 = sub == 0 || prev != my_id;
#pragma unroll
  for (int c = 0; c < NV; ++c) {
    const float x = __shfl_down_sync(0xffffffffu, val[c], 1);
    if (take1) val[c] += x;
  }
#pragma unroll
  for (int c = 0; c < NV; ++c) {
    const float x = __shfl_down_sync(0xffffffffu, val[c], 2);
    if (take2) val[c] += x;
  }
  if (my_id != NONE && is_head2) {
    const uint32_t ti = (my_meta >> 8) & 0xFFu;
    if (s_dgeo[ti]) {
      float *dg = s_dgeo[ti] + (size_t)(my_id - s_tree[ti].z) * 8;
      red_add_v4(dg, val[0], val[1], val[2], val[3]);
      red_add_v4(dg + 4, val[4], val[5], val[6], val[7]);
    }
    red_add_v4(A.drgb + (size_t)my_id * 4, val[8], val[9], val[10], 0.f);
    if (NRM) red_add_v4(A.dnrm + (size_t)my_id * 4, val[NV - 3], val[NV - 2], val[NV - 1], 0.f);
  }
}

// The next batch slot of this warp's hit-record stream, or NULL once the pool is exhausted (warp-uniform).
// `ptr` is the warp's write pointer: REC_PTR_START before the first batch, else the address of the next slot - or, after
// the pool ran out, the same byte offsets with a zero high word (which no device address has): the warp then writes
// nothing but keeps COUNTING the chunks it would have taken, so that CNT_REC_CHUNKS ends up as what the frame needed and
// the next frame's pool is sized right.  Chunks start at multiples of DVX_REC_CHUNK_STRIDE and hold DVX_REC_CHUNK batches,
// so the low bits of the pointer say when a new chunk is due; it is taken from the pool with one atomic and linked behind
// the previous one.  The fast path is two 32-bit tests and an add.
constexpr uint32_t REC_CHUNK_USED = DVX_REC_CHUNK * DVX_REC_BATCH_BYTES;
constexpr unsigned long long REC_PTR_START = REC_CHUNK_USED;
template <bool NRM>
__device__ __forceinline__ unsigned char *rec_next_block(const CompositeArgs &A, int lane, int tile, int warp, WarpQueue<NRM> &Q,
                                                         unsigned long long &ptr) {
  if (((uint32_t)ptr & (DVX_REC_CHUNK_STRIDE - 1u)) == REC_CHUNK_USED) {  // rare path: first batch or chunk boundary
    uint32_t c = 0;
    if (lane == 0) c = (uint32_t)atomicAdd(&A.counters[CNT_REC_CHUNKS], 1ull);
    c = __shfl_sync(0xffffffffu, c, 0);
    if (c >= A.rec_cap) {  // the counter only grows: from here on this warp always lands here
      if (lane == 0) atomicOr(reinterpret_cast<unsigned int *>(&A.counters[CNT_REC_OVERFLOW]), 1u);
      ptr = 0;             // counting mode: a virtual chunk
    } else {
      if (lane == 0) {
        if (ptr == REC_PTR_START) A.rec_tab[2 * ((uint32_t)tile * 8u + (uint32_t)warp)] = c;
        else A.rec_next[(ptr - reinterpret_cast<unsigned long long>(A.rec_pool)) / DVX_REC_CHUNK_STRIDE] = c;
        Q.rec_n += 1;  // chunks taken so far
      }
      ptr = reinterpret_cast<unsigned long long>(A.rec_pool) + (unsigned long long)c * DVX_REC_CHUNK_STRIDE;
    }
  }
  unsigned char *blk = (uint32_t)(ptr >> 32) ? reinterpret_cast<unsigned char *>(ptr) : nullptr;
  ptr += DVX_REC_BATCH_BYTES;
  return blk;
}

// Phases B, C (and B2) over the first min(n_items, 32) queued items of the ring.
// Ring slot of the i-th queued item: (head + i) & (QCAP-1).  my_bits: bit i set <=> queued item i belongs to this pixel.
template <bool BWD, bool NRM, bool EXP, bool REC>
__device__ __forceinline__ void flush_batch(const CompositeArgs &A, int lane, WarpQueue<NRM> &Q, const uint4 *s_tree,
                                            float *const *s_dgeo, int &n_items, int &head, unsigned long long &my_bits, Pix &S,
                                            int tile, int warp, unsigned long long &rec_ptr) {
  const int count = n_items < 32 ? n_items : 32;
  unsigned char *blk = nullptr;
  if (REC) blk = rec_next_block<NRM>(A, lane, tile, warp, Q, rec_ptr);
  __syncwarp();
  ItemGeom G = {};
  float M[4] = {}, gv[NRM ? 6 : 3] = {};
  uint32_t my_id = NONE, my_meta = 0;
  if (lane < count) {
    float mid;
    item_geom<NRM>(A, Q, s_tree, (head + lane) & (QCAP - 1), my_id, my_meta, G, mid);
    if (REC && blk) {
      unsigned char *mine_rec = blk + 16 * lane;
      __stcs(reinterpret_cast<float4 *>(mine_rec), make_float4(__uint_as_float(my_id), __uint_as_float(my_meta), G.delta, mid));
      __stcs(reinterpret_cast<float4 *>(mine_rec + 512), make_float4(G.p[0], G.p[1], G.p[2], G.q[0]));
      __stcs(reinterpret_cast<float2 *>(blk + 1024 + 8 * lane), make_float2(G.q[1], G.q[2]));
    }
    phase_B<BWD, NRM>(A, s_tree, lane, Q.b, my_id, my_meta, G, mid, M, gv);
  }
  uint32_t mine = (uint32_t)my_bits;
  if (count < 32) mine &= (1u << count) - 1u;
  if (REC && blk) __stcs(reinterpret_cast<uint32_t *>(blk + 1280) + lane, mine);
  __syncwarp();
  if (!BWD) {  // the pixel's running sums live in shared memory between batches
    const float4 a4 = Q.acc[lane];
    const float2 t2 = Q.tn[lane];
    S.C0 = a4.x; S.C1 = a4.y; S.C2 = a4.z; S.D = a4.w; S.T = t2.x; S.n_used = __float_as_uint(t2.y);
    if (NRM) { const float4 n4 = Q.nacc[lane]; S.N0 = n4.x; S.N1 = n4.y; S.N2 = n4.z; }
  }
  phase_C<BWD, NRM, EXP>(A, Q.b, mine, S);
  if (!BWD) {
    Q.acc[lane] = make_float4(S.C0, S.C1, S.C2, S.D);
    Q.tn[lane] = make_float2(S.T, __uint_as_float(S.n_used));
    if (NRM) Q.nacc[lane] = make_float4(S.N0, S.N1, S.N2, 0.f);
  }
  my_bits >>= count;
  __syncwarp();
  if (BWD) {
    phase_B2<NRM>(A, lane, count, Q.b, s_tree, s_dgeo, my_id, my_meta, G, M, gv);
    __syncwarp();
  }
  head = (head + count) & (QCAP - 1);
  n_items -= count;
}

// ---- the kernel ------------------------------------------------------------------------------------------------------
// Per-pixel ray in fp64 (O1): d_cam = ((u+1/2-cx)/fx, (v+1/2-cy)/fy, 1) / |.|.  Recomputed where needed (once per served
// list) instead of being held in six registers.
__device__ __forceinline__ void pixel_ray_d(const FrameParams &p, int u, int v, double &xd, double &yd, double &rnd) {
  xd = ((double)u + 0.5 - p.cx_d) * p.inv_fx;
  yd = ((double)v + 0.5 - p.cy_d) * p.inv_fy;
  rnd = rsqrt(xd * xd + yd * yd + 1.0);
}

// R20, the measure-zero case of a ray component that is exactly 0: that axis puts no constraint on tau, and the ray meets
// the voxel only if the camera coordinate lies in [min, max) of the slab.  Decided exactly, from the voxel's integer
// coordinates in fp64 (the staged fp32 centre is not exact enough to settle a ray lying IN a voxel face).
__device__ __noinline__ float2 axis_parallel_fix(const TreeFrame *T, uint32_t id, uint32_t level, uint32_t zmask, float hs,
                                                 float k0, float k1, float k2, float c0, float c1, float c2) {
  uint32_t XYZ[3], lv;
  dvx_decode16(__ldg(T->code + (id - T->base)), XYZ[0], XYZ[1], XYZ[2], lv);
  const uint32_t size = 1u << (DVX_MAX_LEVEL - level);
  const float c[3] = {c0, c1, c2}, k[3] = {k0, k1, k2};  // k = |1/d|
  float sa = -INFINITY, sb = INFINITY;
  bool inside = true;
  for (int a = 0; a < 3; ++a) {
    if ((zmask >> a) & 1u) {
      const double mn = fma(T->cell, (double)XYZ[a], T->rel0[a]);  // slab minimum relative to the camera
      inside = inside && mn <= 0.0 && mn + T->cell * (double)size > 0.0;
    } else {
      sa = fmaxf(sa, fmaf(-hs, k[a], -c[a]));
      sb = fminf(sb, fmaf(hs, k[a], -c[a]));
    }
  }
  return inside ? make_float2(sa, sb) : make_float2(INFINITY, -INFINITY);
}

// Per-pixel state of a backward pass: incoming gradients, the forward's saved totals, where the replay stops (R3).
template <bool NRM>
__device__ __forceinline__ void backward_pixel_init(const CompositeArgs &A, int u, int v, size_t pix, Pix &S) {
  S.gC0 = A.g_rgb[3 * pix]; S.gC1 = A.g_rgb[3 * pix + 1]; S.gC2 = A.g_rgb[3 * pix + 2];
  S.gD = A.g_depth ? A.g_depth[pix] : 0.f;
  S.gA = A.g_alpha ? A.g_alpha[pix] : 0.f;
  const float4 cd = reinterpret_cast<const float4 *>(A.sv_rgbd)[pix];
  S.Xtot = S.gC0 * cd.x + S.gC1 * cd.y + S.gC2 * cd.z + S.gD * cd.w;
  if (NRM) {
    S.gN0 = A.g_normal[3 * pix]; S.gN1 = A.g_normal[3 * pix + 1]; S.gN2 = A.g_normal[3 * pix + 2];
    const float4 nf = reinterpret_cast<const float4 *>(A.sv_nrm)[pix];
    S.Xtot += S.gN0 * nf.x + S.gN1 * nf.y + S.gN2 * nf.z;
  }
  S.T_final = A.sv_T[pix];
  S.n_stop = A.sv_nused[pix];
  // Eq. 2: dL/dT_final also has g_C . C_sky; with alpha = 1 - T_final that is an alpha gradient of -(g_C . C_sky)
  if (A.sky_tex) S.gA -= dvx_sky_backward(&A, u, v, S.gC0, S.gC1, S.gC2, S.T_final);
  if (S.n_stop == 0) S.done = true;
}

__device__ __forceinline__ void pixel_state_zero(Pix &S, bool inside) {
  S.C0 = S.C1 = S.C2 = 0.f; S.D = 0.f; S.T = 1.f; S.n_used = 0; S.done = !inside;
  S.gC0 = S.gC1 = S.gC2 = S.gD = S.gA = S.Xtot = S.T_final = 0.f;
  S.Xpre = 0.f; S.n_stop = 0;
  S.N0 = S.N1 = S.N2 = 0.f; S.gN0 = S.gN1 = S.gN2 = 0.f;
  S.exp_pos = 0;
}

// REC (forward, frame saved for a backward): every batch is also appended to the warp's hit-record stream.
// A BWD launch with a record pool attached is the fall-back of the replay kernel: it only runs when the pool overflowed.
template <bool BWD, bool CNT, bool NRM, bool EXP = false, bool REC = false>
__global__ void __launch_bounds__(TILE_THREADS, DVX_TILE_MIN_CTAS) composite_tile_kernel(const __grid_constant__ CompositeArgs A) {
  if (BWD && A.rec_pool && A.counters[CNT_REC_OVERFLOW] == 0ull) return;  // the replay kernel did this frame's backward
  __shared__ WarpQueue<NRM> s_queue[TILE_WARPS];
  // what phase B needs of an item's octree, 16 bytes each: one shared-memory load instead of three dependent global ones
  __shared__ uint4 s_tree[DVX_MAX_ACTORS + 1];
  __shared__ float *s_dgeo[BWD ? DVX_MAX_ACTORS + 1 : 1];
  const FrameParams &p = A.p;
  for (uint32_t i = threadIdx.x; i < p.n_trees; i += TILE_THREADS) {
    const TreeFrame &Ti = A.trees[i];
    const unsigned long long ga = reinterpret_cast<unsigned long long>(Ti.geo);
    s_tree[i] = make_uint4((uint32_t)ga, (uint32_t)(ga >> 32), Ti.base, __float_as_uint(Ti.inv_cell_f));
    if (BWD) s_dgeo[i] = Ti.dgeo;
  }
  const int tile = A.tile_order ? (int)__ldg(A.tile_order + blockIdx.x / TILE_SPLIT) : (int)(blockIdx.x / TILE_SPLIT);
  const int warp_l = threadIdx.x >> 5;                                  // warp of this CTA
  const int warp = (int)(blockIdx.x % TILE_SPLIT) * TILE_WARPS + warp_l;  // warp of the tile: which 4x8 pixel block
  const int lane = threadIdx.x & 31;
  const int wu0 = (tile % p.tiles_x) * DVX_TILE + (warp % WARPS_X) * WARP_W;   // pixel of lane 0 of this warp
  const int wv0 = (tile / p.tiles_x) * DVX_TILE + (warp / WARPS_X) * WARP_H;
  WarpQueue<NRM> &Q = s_queue[warp_l];
  const int u = wu0 + lane % WARP_W, v = wv0 + lane / WARP_W;
  const bool inside = u < (int)p.width && v < (int)p.height;
  const size_t pix = (size_t)v * p.width + u;

  Pix S;
  pixel_state_zero(S, inside);
  if (EXP && inside) {  // the row lengths are the n_used the rendering pass saved
    S.exp_pos = A.exp_row[pix];
    S.n_stop = A.exp_row[pix + 1] - S.exp_pos;
  }
  if (BWD && inside) backward_pixel_init<NRM>(A, u, v, pix, S);
  if (BWD) {  // pixels outside the image own no items; their entries are zero
    Q.b.pg[lane] = make_float4(S.gC0, S.gC1, S.gC2, S.gD);
    if (NRM) Q.b.pn[lane] = make_float4(S.gN0, S.gN1, S.gN2, 0.f);
  }
  unsigned long long rec_ptr = REC_PTR_START;
  if (!BWD) {
    Q.acc[lane] = make_float4(0.f, 0.f, 0.f, 0.f);
    Q.tn[lane] = make_float2(1.f, __uint_as_float(0u));
    if (NRM) Q.nacc[lane] = make_float4(0.f, 0.f, 0.f, 0.f);
  }
  if (REC && lane == 0) Q.rec_n = 0;

  // ---- step 3: intervals of the actors in this tile's mask, insertion-sorted by (tau_in, actor index) (O2, O3)
  float h_in[DVX_MAX_ACTORS], h_out[DVX_MAX_ACTORS];
  unsigned char h_idx[DVX_MAX_ACTORS];
  int m = 0;
  {
    unsigned long long am = A.actor_mask[tile];
    if (am) {
      double xd, yd, rnd;
      pixel_ray_d(p, u, v, xd, yd, rnd);
      while (am) {
        const int i = __ffsll((long long)am) - 1;
        am &= am - 1;
        if (S.done) continue;
        const TreeFrame &T = A.trees[1 + i];
        double lo = -1.0e300, hi = 1.0e300;
        bool miss = false;
#pragma unroll
        for (int a = 0; a < 3; ++a) {
          const double da = (T.Nd[3 * a] * xd + T.Nd[3 * a + 1] * yd + T.Nd[3 * a + 2]) * rnd;
          const double o = T.o_l[a], hh = (double)T.half[a];
          if (da == 0.0) {
            miss = miss || !(o >= -hh && o < hh);
          } else {
            const double inv = rcp_double(da);
            const double t1 = (-hh - o) * inv, t2 = (hh - o) * inv;
            lo = fmax(lo, fmin(t1, t2));
            hi = fmin(hi, fmax(t1, t2));
          }
        }
        if (miss || !(hi > fmax(lo, (double)p.near_))) continue;
        const float tin = (float)fmax(lo, (double)p.near_), tout = (float)fmin(hi, (double)p.far_);
        int j = m++;
        while (j > 0 && h_in[j - 1] > tin) {  // ties keep the lower actor index first
          h_in[j] = h_in[j - 1]; h_out[j] = h_out[j - 1]; h_idx[j] = h_idx[j - 1];
          --j;
        }
        h_in[j] = tin; h_out[j] = tout; h_idx[j] = (unsigned char)i;
      }
    }
  }

  __syncthreads();  // s_tree / s_dgeo
  // ---- step 4: Algorithm 1 as a per-lane state machine; the warp serves one (tree, octant) list at a time
  float cur = p.near_;   // tau_curr
  int h = 0;             // next entry of the hit list
  int stage = 0;         // 0: background before hit h (or the final background), 1: actor of hit h, 2: finished
  uint32_t cur0 = NONE;  // this pixel's cursor in the static list of its octant (persists across background intervals)
  int n_items = 0, head = 0;
  unsigned long long my_bits = 0;
  unsigned long long q_test = 0;
  const uint32_t ru0 = (uint32_t)wu0, rv0 = (uint32_t)wv0, ru1 = ru0 + WARP_W - 1, rv1 = rv0 + WARP_H - 1;
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
          if (tin > cur) { seg_tree = 0; lo = cur; hi = tin; }              // background before object entry
        } else {
          stage = 2;
          if (p.far_ > cur) { seg_tree = 0; lo = cur; hi = p.far_; }        // remaining background
        }
      } else {
        const float tin = h_in[h], tout = h_out[h];
        const float l = fmaxf(tin, cur);
        const uint32_t ta = 1u + h_idx[h];
        cur = fmaxf(cur, tout);
        ++h;
        stage = 0;
        if (tout > l) { seg_tree = ta; lo = l; hi = tout; }                  // object in its canonical local space
      }
    }
    const uint32_t t = warp_min_u32(seg_tree);
    if (t == NONE) break;
    const bool part = seg_tree == t;
    const TreeFrame &T = A.trees[t];
    // ray of this pixel in the frame of tree t: fp64 direction, its fp32 rounding, reciprocal, octant, and the small
    // difference e to the warp's reference direction d0 (= the direction of lane 0's pixel, kept in shared memory)
    float inv[3], e[3];
    int q = 0;
    uint32_t zmask = 0;  // axes on which this ray is exactly axis-parallel (R20), almost always 0
    {
      double xd, yd, rnd;
      pixel_ray_d(p, u, v, xd, yd, rnd);
      const float xp = dvx_cam_x(p, u), yp = dvx_cam_y(p, v);  // fp32 copy: only the octant decision uses it (R12)
      __syncwarp();
      float d[3];
#pragma unroll
      for (int a = 0; a < 3; ++a) {
        const double da = (T.Nd[3 * a] * xd + T.Nd[3 * a + 1] * yd + T.Nd[3 * a + 2]) * rnd;
        const double d0a = shfl_double(da, 0);
        if (lane == 0) Q.d0[a] = d0a;
        e[a] = (float)(da - d0a);
        d[a] = (float)da;
        q |= (dvx_dir_comp(T.N, a, xp, yp) < 0.f) ? (4 >> a) : 0;  // R12: s_a = (d_a < 0), same fp32 formula as step 1
        inv[a] = d[a] != 0.f ? 1.0f / d[a] : 0.f;
        if (d[a] == 0.f) zmask |= 1u << a;
      }
      Q.dir[lane] = make_float4(d[0], d[1], d[2], __uint_as_float((uint32_t)lane));  // read back by this lane only, at every emit
      __syncwarp();
    }
    // warp-uniform "some lane is axis-parallel": keeps the R20 test out of the per-candidate loop (the forward otherwise
    // rebuilt zmask from d[] there, 9 instructions per candidate: forward 1.254 -> 1.218 ms on config 3)
    const bool z_any = __any_sync(0xffffffffu, zmask != 0u);
    uint32_t omask = __reduce_or_sync(0xffffffffu, part ? (1u << q) : 0u);
    while (omask) {
      const int qq = __ffs(omask) - 1;
      omask &= omask - 1;
      const size_t bucket = ((size_t)tile * p.n_trees + t) * 8 + qq;
      const uint32_t beg = __ldg(A.range_beg + bucket), end = __ldg(A.range_end + bucket);
      uint32_t c_l = beg;
      if (t == 0 && cur0 != NONE) c_l = cur0;
      uint32_t c_t = (part && q == qq) ? c_l : NONE;  // first entry this pixel still tests; NONE = not (or no longer) walking
      uint32_t pos = warp_min_u32(c_t);
      // the id of this lane's entry of the NEXT round is loaded one round ahead, and an entry's pixel rectangle and code are
      // loaded together (the code of an entry that fails the rectangle test is wasted, 8 bytes from L2): one exposed load
      // latency per round of 32 entries instead of three dependent ones
      uint32_t id_next = pos + lane < end ? __ldg(A.ids + pos + lane) : 0u;
      while (pos < end && __any_sync(0xffffffffu, c_t != NONE)) {
        const uint32_t n = min(32u, end - pos);
        // -- lane = entry: pre-filter and fp64 centre decomposition
        bool c = false;
        uint32_t ry0 = 1u, ry1 = 0u;  // rows of the entry's pixel rectangle
        const uint32_t id_cur = id_next;
        if (pos + 32u + lane < end) id_next = __ldg(A.ids + pos + 32u + lane);
        if ((uint32_t)lane < n) {
          const uint32_t id = id_cur;
          const uint64_t code_v = __ldg(T.code + (id - T.base));
          const ushort4 rc = __ldg(A.pxrect + id);
          c = rc.x <= ru1 && rc.z >= ru0 && rc.y <= rv1 && rc.w >= rv0;
          ry0 = rc.y; ry1 = rc.w;
          if (c) {
            uint32_t X, Y, Z, lv;
            dvx_decode16(code_v, X, Y, Z, lv);
            const uint32_t size = 1u << (DVX_MAX_LEVEL - lv);
            const double hc = 0.5 * T.cell;
            const double d0x = Q.d0[0], d0y = Q.d0[1], d0z = Q.d0[2];
            const double cx = fma(hc, (double)(2u * X + size), T.rel0[0]);
            const double cy = fma(hc, (double)(2u * Y + size), T.rel0[1]);
            const double cz = fma(hc, (double)(2u * Z + size), T.rel0[2]);
            const float t0 = (float)(cx * d0x + cy * d0y + cz * d0z);
            const double t0d = (double)t0;
            EntryRec rec;
            rec.t0 = t0;
            rec.m0[0] = (float)(cx - t0d * d0x); rec.m0[1] = (float)(cy - t0d * d0y); rec.m0[2] = (float)(cz - t0d * d0z);
            rec.hs = (float)(hc * (double)size);
            rec.id = id; rec.meta = (t << 8) | (lv << 16); rec.pad = 0;
            Q.ent[lane] = rec;
          }
        }
        // The warp's 4x8 pixel block is cut into DVX_CAND_GROUPS bands of rows; every band walks its own candidates (the
        // entries whose pixel rectangle reaches into the band), so one trip of the loop below tests up to DVX_CAND_GROUPS
        // different entries.  A pixel still meets its entries in list order, and items are queued in (trip, lane) order,
        // so every pixel's items stay in its own front-to-back order.
        uint32_t cand = 0;
        {
          constexpr int BAND_H = WARP_H / DVX_CAND_GROUPS, BAND_LANES = 32 / DVX_CAND_GROUPS;
#pragma unroll
          for (int g = 0; g < DVX_CAND_GROUPS; ++g) {
            const uint32_t b = __ballot_sync(0xffffffffu, c && ry0 <= rv0 + (g + 1) * BAND_H - 1 && ry1 >= rv0 + g * BAND_H);
            if (lane / BAND_LANES == g) cand = b;
          }
        }
        __syncwarp();
        // -- lane = pixel
        while (__any_sync(0xffffffffu, cand != 0u)) {
          const bool act = cand != 0u;
          const int j = act ? __ffs(cand) - 1 : 0;
          cand &= cand - 1;
          const uint32_t ei = pos + j;
          const float4 r0 = *reinterpret_cast<const float4 *>(&Q.ent[j]);          // t0, m0
          const uint4 r1 = *(reinterpret_cast<const uint4 *>(&Q.ent[j]) + 1);      // id, meta, hs
          const float hs = __uint_as_float(r1.z);
          const float w0 = fmaf(r0.x, e[0], -r0.y), w1 = fmaf(r0.x, e[1], -r0.z), w2 = fmaf(r0.x, e[2], -r0.w);
          const float c0 = w0 * inv[0], c1 = w1 * inv[1], c2 = w2 * inv[2];
          float sa = fmaxf(fmaxf(fmaf(-hs, fabsf(inv[0]), -c0), fmaf(-hs, fabsf(inv[1]), -c1)), fmaf(-hs, fabsf(inv[2]), -c2));
          float sb = fminf(fminf(fmaf(hs, fabsf(inv[0]), -c0), fmaf(hs, fabsf(inv[1]), -c1)), fmaf(hs, fabsf(inv[2]), -c2));
          if (z_any && zmask) {
            const float2 f = axis_parallel_fix(&T, r1.x, r1.y >> 16, zmask, hs, fabsf(inv[0]), fabsf(inv[1]), fabsf(inv[2]), c0, c1, c2);
            sa = f.x; sb = f.y;
          }
          const float lo_r = lo - r0.x, hi_r = hi - r0.x;
          const float ca = fmaxf(sa, lo_r), cb = fminf(sb, hi_r);       // R1: clip to the interval
          const bool live = act && c_t <= ei && sb > sa;                // this pixel's ray meets the voxel
          const bool emit = live && cb > ca;
          if (CNT) q_test += (act && c_t <= ei) ? 1u : 0u;
          // gate: the voxel reaches beyond the interval end (it may own a second piece after the box), or starts beyond it
          if (live && sb > hi_r) { c_t = NONE; c_l = ei; }
          const uint32_t mk = __ballot_sync(0xffffffffu, emit);
          if (mk) {
            if (emit) {
              const int rel_at = n_items + __popc(mk & lanemask_lt());
              float4 *it = reinterpret_cast<float4 *>(&Q.item[(head + rel_at) & (QCAP - 1)]);
              it[0] = make_float4(__uint_as_float(r1.x), __uint_as_float(r1.y), ca, cb);
              it[1] = make_float4(w0, w1, w2, r0.x + 0.5f * (ca + cb));
              it[2] = Q.dir[lane];
              my_bits |= 1ull << rel_at;
            }
            n_items += __popc(mk);
            if (n_items >= 32) {
              flush_batch<BWD, NRM, EXP, REC>(A, lane, Q, s_tree, s_dgeo, n_items, head, my_bits, S, tile, warp, rec_ptr);
              if (S.done) c_t = NONE;
            }
          }
        }
        __syncwarp();
        pos += 32;
      }
      if (CNT && A.eff_end && lane == 0) atomicMax(A.eff_end + bucket, min(pos, end));
      if (part && q == qq) {
        if (c_t != NONE) c_l = end;     // walked off the list: nothing left for later intervals either
        if (t == 0) cur0 = c_l;
      }
    }
    if (part) seg_tree = NONE;          // served
  }
  while (n_items > 0) flush_batch<BWD, NRM, EXP, REC>(A, lane, Q, s_tree, s_dgeo, n_items, head, my_bits, S, tile, warp, rec_ptr);

  if (REC && lane == 0) {  // batches written = full chunks + the slots used of the last one
    const uint32_t used = ((uint32_t)rec_ptr & (DVX_REC_CHUNK_STRIDE - 1u)) / DVX_REC_BATCH_BYTES;
    A.rec_tab[2 * ((uint32_t)tile * 8u + (uint32_t)warp) + 1] = Q.rec_n ? (Q.rec_n - 1u) * DVX_REC_CHUNK + used : 0u;
  }
  if (!BWD) {
    const float4 a4 = Q.acc[lane];
    const float2 t2 = Q.tn[lane];
    S.C0 = a4.x; S.C1 = a4.y; S.C2 = a4.z; S.D = a4.w; S.T = t2.x; S.n_used = __float_as_uint(t2.y);
    if (NRM) { const float4 n4 = Q.nacc[lane]; S.N0 = n4.x; S.N1 = n4.y; S.N2 = n4.z; }
  }
  if (!BWD && !EXP && inside) {
    float3 sky = make_float3(0.f, 0.f, 0.f);
    if (A.sky_tex) sky = dvx_sky_forward(&A, u, v, S.T);  // Eq. 2: C = C_voxels + T_final C_sky
    A.rgb[3 * pix] = S.C0 + sky.x; A.rgb[3 * pix + 1] = S.C1 + sky.y; A.rgb[3 * pix + 2] = S.C2 + sky.z;
    A.depth[pix] = S.D;
    A.alpha[pix] = 1.0f - S.T;
    if (NRM) {
      A.normal[3 * pix] = S.N0; A.normal[3 * pix + 1] = S.N1; A.normal[3 * pix + 2] = S.N2;
      if (A.sv_nrm) reinterpret_cast<float4 *>(A.sv_nrm)[pix] = make_float4(S.N0, S.N1, S.N2, 0.f);
    }
    if (A.sv_rgbd) {
      reinterpret_cast<float4 *>(A.sv_rgbd)[pix] = make_float4(S.C0, S.C1, S.C2, S.D);
      A.sv_T[pix] = S.T;
      A.sv_nused[pix] = S.n_used;
    }
  }
  if (CNT && !BWD) {
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


// ---- backward from the hit records -------------------------------------------------------------------------------------
// Step 5 without steps 3-4's geometry: the forward left every batch it composited (voxel, local segment, owner masks) in the
// warp's record stream, so the backward needs no list walk, no slab test, no interval schedule and no queue: per batch it
// loads the records (three coalesced loads, the next batch prefetched under the current one), integrates with moments
// (phase B), replays the pixels' blend order (phase C) and reduces the gradients (phase B2).
// Same grid and warp -> pixel-block mapping as the forward.
constexpr int DVX_REPLAY_MIN_CTAS = 7;  // 72 registers, no spills; config 3 replay ms at 6 / 7 / 8 CTAs per SM: 1.272 / 1.189 / 1.207 (config 4: 2.114 / 1.996 / 2.045)
struct RecBatch {
  uint4 a;      // id, meta, delta, mid
  float4 b;     // p, q_x
  float2 c;     // q_y, q_z
  uint32_t mask;
};
__device__ __forceinline__ RecBatch rec_load(const unsigned char *blk, int lane) {
  RecBatch r;
  r.a = __ldcs(reinterpret_cast<const uint4 *>(blk) + lane);
  r.b = __ldcs(reinterpret_cast<const float4 *>(blk + 512) + lane);
  r.c = __ldcs(reinterpret_cast<const float2 *>(blk + 1024) + lane);
  r.mask = __ldcs(reinterpret_cast<const uint32_t *>(blk + 1280) + lane);
  return r;
}

template <bool NRM>
__global__ void __launch_bounds__(TILE_THREADS, DVX_REPLAY_MIN_CTAS) composite_replay_kernel(const __grid_constant__ CompositeArgs A) {
  if (A.counters[CNT_REC_OVERFLOW] != 0ull) return;  // incomplete records: the list-walking backward runs instead
  __shared__ BatchShared<NRM> s_b[TILE_WARPS];
  __shared__ uint4 s_tree[DVX_MAX_ACTORS + 1];
  __shared__ float *s_dgeo[DVX_MAX_ACTORS + 1];
  const FrameParams &p = A.p;
  for (uint32_t i = threadIdx.x; i < p.n_trees; i += TILE_THREADS) {
    const TreeFrame &Ti = A.trees[i];
    const unsigned long long ga = reinterpret_cast<unsigned long long>(Ti.geo);
    s_tree[i] = make_uint4((uint32_t)ga, (uint32_t)(ga >> 32), Ti.base, __float_as_uint(Ti.inv_cell_f));
    s_dgeo[i] = Ti.dgeo;
  }
  const int tile = A.tile_order ? (int)__ldg(A.tile_order + blockIdx.x / TILE_SPLIT) : (int)(blockIdx.x / TILE_SPLIT);
  const int warp_l = threadIdx.x >> 5;
  const int warp = (int)(blockIdx.x % TILE_SPLIT) * TILE_WARPS + warp_l;
  const int lane = threadIdx.x & 31;
  const int u = (tile % p.tiles_x) * DVX_TILE + (warp % WARPS_X) * WARP_W + lane % WARP_W;
  const int v = (tile / p.tiles_x) * DVX_TILE + (warp / WARPS_X) * WARP_H + lane / WARP_W;
  const bool inside = u < (int)p.width && v < (int)p.height;
  const size_t pix = (size_t)v * p.width + u;
  BatchShared<NRM> &bs = s_b[warp_l];
  // The per-pixel state stays in registers here (unlike in the forward): parked in shared memory between batches, with
  // two batch buffers in flight, the same loop ran 1.43-1.63 ms instead of 1.21 ms (config 3, 6-8 CTAs per SM).
  Pix S;
  pixel_state_zero(S, inside);
  if (inside) backward_pixel_init<NRM>(A, u, v, pix, S);
  bs.pg[lane] = make_float4(S.gC0, S.gC1, S.gC2, S.gD);
  if (NRM) bs.pn[lane] = make_float4(S.gN0, S.gN1, S.gN2, 0.f);
  const uint32_t warp_global = (uint32_t)tile * 8u + (uint32_t)warp;
  const uint32_t nb = A.rec_tab[2 * warp_global + 1];
  uint32_t chunk = nb ? A.rec_tab[2 * warp_global] : 0u;
  __syncthreads();  // s_tree / s_dgeo
  if (nb == 0) return;
  const unsigned char *blk = A.rec_pool + (size_t)chunk * DVX_REC_CHUNK_STRIDE;
  uint32_t slot = 0;
  RecBatch cur = rec_load(blk, lane);
  ItemGeom G = {};                        // lanes past a short batch's items keep these (phase B2 computes on every lane)
  float M[4] = {}, gv[NRM ? 6 : 3] = {};
  // No early exit once every pixel of the block has replayed its n_used voxels: the forward stops walking as soon as all of
  // a warp's pixels are done, so at most the batches still queued at that moment follow, and phase C gives their items zero
  // weight; the vote that tested for it cost more (replay 1.133 -> 1.114 ms on config 3, 1.890 -> 1.853 on config 4).
  for (uint32_t b = 0; b < nb; ++b) {
    // -- prefetch the next batch (a chunk's successor is read when its last slot has been used)
    RecBatch nxt = cur;
    if (b + 1 < nb) {
      blk += DVX_REC_BATCH_BYTES;
      if (++slot == DVX_REC_CHUNK) {
        slot = 0;
        chunk = __ldg(A.rec_next + chunk);
        blk = A.rec_pool + (size_t)chunk * DVX_REC_CHUNK_STRIDE;
      }
      nxt = rec_load(blk, lane);
    }
    const int count = __popc(__reduce_or_sync(0xffffffffu, cur.mask));  // every item of the batch has one owner
    uint32_t my_id = NONE, my_meta = 0;
    if (lane < count) {
      my_id = cur.a.x; my_meta = cur.a.y;
      G.delta = __uint_as_float(cur.a.z);
      G.p[0] = cur.b.x; G.p[1] = cur.b.y; G.p[2] = cur.b.z;
      G.q[0] = cur.b.w; G.q[1] = cur.c.x; G.q[2] = cur.c.y;
      phase_B<true, NRM>(A, s_tree, lane, bs, my_id, my_meta, G, __uint_as_float(cur.a.w), M, gv);
    }
    __syncwarp();
    phase_C<true, NRM, false>(A, bs, cur.mask, S);
    __syncwarp();
    phase_B2<NRM>(A, lane, count, bs, s_tree, s_dgeo, my_id, my_meta, G, M, gv);
    __syncwarp();
    cur = nxt;
  }
}

}  // namespace

// Row N3: the forward walk once more, writing the compositing weights (voxel, T alpha) of every pixel into the CSR rows
// whose lengths the rendering pass saved; no image is written.
void dvx_composite_export_launch(const CompositeArgs &a, cudaStream_t st) {
  if (a.p.n_tiles == 0) return;
  DVX_COUNT_LAUNCH(1);
  composite_tile_kernel<false, false, false, true><<<a.p.n_tiles * TILE_SPLIT, TILE_THREADS, 0, st>>>(a);
}

void dvx_composite_tile_launch(const CompositeArgs &a, bool backward, cudaStream_t st) {
  if (a.p.n_tiles == 0) return;
  DVX_COUNT_LAUNCH(1);
  const bool cnt = (a.p.flags & DVX_FLAG_COUNTERS) != 0;
  const bool nrm = backward ? (a.g_normal != nullptr) : (a.normal != nullptr);  // normal map requested (O11)
  const bool rec = !backward && a.rec_pool != nullptr;                           // forward of a saved frame: write hit records
  const unsigned grid = a.p.n_tiles * TILE_SPLIT;
  if (backward) {
    if (nrm) composite_tile_kernel<true, false, true><<<grid, TILE_THREADS, 0, st>>>(a);
    else composite_tile_kernel<true, false, false><<<grid, TILE_THREADS, 0, st>>>(a);
  } else if (nrm) {
    if (rec) composite_tile_kernel<false, false, true, false, true><<<grid, TILE_THREADS, 0, st>>>(a);
    else composite_tile_kernel<false, false, true><<<grid, TILE_THREADS, 0, st>>>(a);
  } else if (cnt) {
    if (rec) composite_tile_kernel<false, true, false, false, true><<<grid, TILE_THREADS, 0, st>>>(a);
    else composite_tile_kernel<false, true, false><<<grid, TILE_THREADS, 0, st>>>(a);
  } else {
    if (rec) composite_tile_kernel<false, false, false, false, true><<<grid, TILE_THREADS, 0, st>>>(a);
    else composite_tile_kernel<false, false, false><<<grid, TILE_THREADS, 0, st>>>(a);
  }
}

void dvx_composite_replay_launch(const CompositeArgs &a, cudaStream_t st) {
  if (a.p.n_tiles == 0) return;
  DVX_COUNT_LAUNCH(1);
  const unsigned grid = a.p.n_tiles * TILE_SPLIT;
  if (a.g_normal) composite_replay_kernel<true><<<grid, TILE_THREADS, 0, st>>>(a);
  else composite_replay_kernel<false><<<grid, TILE_THREADS, 0, st>>>(a);
}
