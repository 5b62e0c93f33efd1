// dvx_composite.cu - hot-path steps 3, 4 and 5:
//   step 3  per-ray ray-OBB intervals [tau_in^i, tau_out^i], sorted front to back
//   step 4  Algorithm 1: F(O_bg,[tau_curr,tau_in]) -> F(O_i,[tau_in,tau_out]) -> ... -> F(O_bg,[tau_curr,
//           tau_max]) carrying S = (C, D, T, tau_curr); inside F the ray-voxel segment, K midpoint samples of
//           the trilinear raw density, activation, alpha = 1 - exp(-sum sigma dt), blend weighted by T
//   step 5  the matching backward
// One CTA per 16x16 tile, one thread per pixel.
#include "dvx_ray.cuh"

namespace {

constexpr int TILE_THREADS = DVX_TILE * DVX_TILE;

// O6: K-point midpoint rule on the clipped segment [a,b]; returns tau_v.  With GRAD also G[c] = delta * sum_k act'(raw_k) w_c(u_k).
template <bool GRAD>
__device__ __forceinline__ float integrate(const Ray &r, const float rel[3], float s, const float g[8], float a, float b,
                                           uint32_t K, uint32_t kind, float *G) {
  const float inv_s = 1.0f / s;
  const float delta = (b - a) / (float)K;
  float sum = 0.f;
  if (GRAD) {
#pragma unroll
    for (int c = 0; c < 8; ++c) G[c] = 0.f;
  }
  for (uint32_t k = 0; k < K; ++k) {
    float t = a + ((float)k + 0.5f) * delta;
    float u[3];
#pragma unroll
    for (int ax = 0; ax < 3; ++ax) u[ax] = __saturatef((t * r.d[ax] - rel[ax]) * inv_s);
    float wx0 = 1.f - u[0], wy0 = 1.f - u[1], wz0 = 1.f - u[2];
    float w[8];
    w[0] = wx0 * wy0 * wz0; w[1] = wx0 * wy0 * u[2]; w[2] = wx0 * u[1] * wz0; w[3] = wx0 * u[1] * u[2];
    w[4] = u[0] * wy0 * wz0; w[5] = u[0] * wy0 * u[2]; w[6] = u[0] * u[1] * wz0; w[7] = u[0] * u[1] * u[2];
    float raw = 0.f;
#pragma unroll
    for (int c = 0; c < 8; ++c) raw += g[c] * w[c];
    sum += act_fn(raw, kind);
    if (GRAD) {
      float da = dact_fn(raw, kind);
#pragma unroll
      for (int c = 0; c < 8; ++c) G[c] += da * w[c];
    }
  }
  if (GRAD) {
#pragma unroll
    for (int c = 0; c < 8; ++c) G[c] *= delta;
  }
  return delta * sum;
}

struct PixelState {
  float C[3], D, T;
  uint32_t n_used;
  bool done;
  // backward
  float gC[3], gD, gA, Xtot, Xpre, T_final;
  uint32_t n_stop;
  unsigned long long q_test, q_hit;
};

// F over one octree's sorted tile list for the interval [lo, hi], starting at `cursor`.
// The cursor stops at the first voxel that starts at or beyond hi, or that sticks out of the interval (it may own a
// second piece after an actor box, R1).
template <bool BWD>
__device__ __forceinline__ void walk_list(const CompositeArgs &A, const TreeFrame &T, const Ray &r, uint32_t &cursor,
                                          uint32_t end, float lo, float hi, PixelState &S) {
  const uint32_t K = A.p.k_samples, kind = A.p.activation;
  while (cursor < end && !S.done) {
    const uint32_t id = __ldg(A.ids + cursor);
    const float4 f0 = __ldg(reinterpret_cast<const float4 *>(A.fvox + id));
    const float rel[3] = {f0.x, f0.y, f0.z};
    const float s = f0.w;
    float a, b;
    if (A.p.flags & DVX_FLAG_COUNTERS) S.q_test++;
    if (!slab_rel(r, rel, s, a, b)) { ++cursor; continue; }
    if (!(b > a)) { ++cursor; continue; }
    if (a >= hi) break;
    const float ca = fmaxf(a, lo), cb = fminf(b, hi);
    if (cb > ca) {
      if (A.p.flags & DVX_FLAG_COUNTERS) S.q_hit++;
      const float4 f1 = __ldg(reinterpret_cast<const float4 *>(A.fvox + id) + 1);
      const float4 *gp = reinterpret_cast<const float4 *>(T.geo + (size_t)(id - T.base) * 8);
      const float4 g0 = __ldg(gp), g1 = __ldg(gp + 1);
      const float g[8] = {g0.x, g0.y, g0.z, g0.w, g1.x, g1.y, g1.z, g1.w};
      float G[8];
      const float tau = integrate<BWD>(r, rel, s, g, ca, cb, K, kind, G);
      const float e = __expf(-tau);
      const float alpha = -expm1f(-tau);
      const float w = S.T * alpha;
      const float mid = 0.5f * (ca + cb);
      if (!BWD) {
        S.C[0] += w * f1.x; S.C[1] += w * f1.y; S.C[2] += w * f1.z;
        S.D += w * mid;
      } else {
        const float X = S.gC[0] * f1.x + S.gC[1] * f1.y + S.gC[2] * f1.z + S.gD * mid;
        S.Xpre += w * X;
        const float dtau = S.T * e * X - (S.Xtot - S.Xpre) + S.gA * S.T_final;
        const uint32_t meta = __float_as_uint(f1.w);
        float *dr = A.drgb + (size_t)id * 4;
        if (!(meta & 1u)) atomicAdd(dr + 0, w * S.gC[0]);
        if (!(meta & 2u)) atomicAdd(dr + 1, w * S.gC[1]);
        if (!(meta & 4u)) atomicAdd(dr + 2, w * S.gC[2]);
        if (T.dgeo) {
          float *dg = T.dgeo + (size_t)(id - T.base) * 8;
#pragma unroll
          for (int c = 0; c < 8; ++c) atomicAdd(dg + c, dtau * G[c]);
        }
      }
      S.T *= e;
      S.n_used++;
      if (!BWD) {
        if (S.T < A.p.t_stop) S.done = true;
      } else {
        if (S.n_used >= S.n_stop) S.done = true;
      }
    }
    if (b > hi) break;
    ++cursor;
  }
}

template <bool BWD>
__global__ void __launch_bounds__(TILE_THREADS) composite_naive_kernel(const __grid_constant__ CompositeArgs A) {
  const FrameParams &p = A.p;
  const int tile = blockIdx.x;
  const int tx = tile % p.tiles_x, ty = tile / p.tiles_x;
  const int u = tx * DVX_TILE + (threadIdx.x & 15), v = ty * DVX_TILE + (threadIdx.x >> 4);
  const bool inside = u < (int)p.width && v < (int)p.height;
  const size_t pix = (size_t)v * p.width + u;

  PixelState S;
  S.C[0] = S.C[1] = S.C[2] = 0.f; S.D = 0.f; S.T = 1.f; S.n_used = 0; S.done = !inside;
  S.q_test = S.q_hit = 0;
  S.Xpre = 0.f;
  if (BWD && inside) {
    S.gC[0] = A.g_rgb[3 * pix]; S.gC[1] = A.g_rgb[3 * pix + 1]; S.gC[2] = A.g_rgb[3 * pix + 2];
    S.gD = A.g_depth ? A.g_depth[pix] : 0.f;
    S.gA = A.g_alpha ? A.g_alpha[pix] : 0.f;
    const float4 cd = reinterpret_cast<const float4 *>(A.sv_rgbd)[pix];
    S.Xtot = S.gC[0] * cd.x + S.gC[1] * cd.y + S.gC[2] * cd.z + S.gD * cd.w;
    S.T_final = A.sv_T[pix];
    S.n_stop = A.sv_nused[pix];
    // Eq. 2: dL/dT_final also has g_C . C_sky; with alpha = 1 - T_final that is an alpha gradient of -(g_C . C_sky)
    if (A.sky_tex) S.gA -= dvx_sky_backward(&A, u, v, S.gC[0], S.gC[1], S.gC[2], S.T_final);
    if (S.n_stop == 0) S.done = true;
  }

  if (!S.done) {
    const float xp = dvx_cam_x(p, u), yp = dvx_cam_y(p, v);
    const float rn = rsqrtf(xp * xp + yp * yp + 1.0f);
    // step 3: intervals of the actors in this tile's mask, insertion-sorted by (tau_in, actor index)
    float h_in[DVX_MAX_ACTORS], h_out[DVX_MAX_ACTORS];
    unsigned char h_idx[DVX_MAX_ACTORS];
    int m = 0;
    unsigned long long am = A.actor_mask[tile];
    while (am) {
      const int i = __ffsll((long long)am) - 1;
      am &= am - 1;
      const TreeFrame &T = A.trees[1 + i];
      Ray r; int q;
      make_ray(T.N, xp, yp, rn, r, q);
      float tin, tout;
      if (ray_box(T, r, p.near_, p.far_, tin, tout)) {
        int j = m++;
        while (j > 0 && h_in[j - 1] > tin) {  // ties keep the lower actor index first (actors arrive in index order)
          h_in[j] = h_in[j - 1]; h_out[j] = h_out[j - 1]; h_idx[j] = h_idx[j - 1];
          --j;
        }
        h_in[j] = tin; h_out[j] = tout; h_idx[j] = (unsigned char)i;
      }
    }
    // step 4: Algorithm 1
    const TreeFrame &T0 = A.trees[0];
    Ray r0; int q0;
    make_ray(T0.N, xp, yp, rn, r0, q0);
    const size_t b0 = ((size_t)tile * p.n_trees + 0) * 8 + q0;
    uint32_t cur0 = A.range_beg[b0];
    const uint32_t end0 = A.range_end[b0];
    float cur = p.near_;
    for (int h = 0; h < m && !S.done; ++h) {
      const float tin = h_in[h], tout = h_out[h];
      const float lo = fmaxf(tin, cur);
      if (tin > cur) walk_list<BWD>(A, T0, r0, cur0, end0, cur, tin, S);  // background before object entry
      if (tout > lo && !S.done) {                                            // object in its canonical local space
        const TreeFrame &Ti = A.trees[1 + h_idx[h]];
        Ray ri; int qi;
        make_ray(Ti.N, xp, yp, rn, ri, qi);
        const size_t bi = ((size_t)tile * p.n_trees + 1 + h_idx[h]) * 8 + qi;
        uint32_t ci = A.range_beg[bi];
        walk_list<BWD>(A, Ti, ri, ci, A.range_end[bi], lo, tout, S);
      }
      cur = fmaxf(cur, tout);
    }
    if (!S.done && p.far_ > cur) walk_list<BWD>(A, T0, r0, cur0, end0, cur, p.far_, S);  // remaining background
  }

  if (!BWD && inside) {
    float3 sky = make_float3(0.f, 0.f, 0.f);
    if (A.sky_tex) sky = dvx_sky_forward(&A, u, v, S.T);  // Eq. 2: C = C_voxels + T_final C_sky
    A.rgb[3 * pix] = S.C[0] + sky.x; A.rgb[3 * pix + 1] = S.C[1] + sky.y; A.rgb[3 * pix + 2] = S.C[2] + sky.z;
    A.depth[pix] = S.D;
    A.alpha[pix] = 1.0f - S.T;
    if (A.sv_rgbd) {
      reinterpret_cast<float4 *>(A.sv_rgbd)[pix] = make_float4(S.C[0], S.C[1], S.C[2], S.D);
      A.sv_T[pix] = S.T;
      A.sv_nused[pix] = S.n_used;
    }
  }
  if (A.p.flags & DVX_FLAG_COUNTERS) {
    unsigned long long qt = S.q_test, qh = S.q_hit;
    for (int o = 16; o > 0; o >>= 1) {
      qt += __shfl_xor_sync(0xffffffffu, qt, o);
      qh += __shfl_xor_sync(0xffffffffu, qh, o);
    }
    if ((threadIdx.x & 31) == 0 && !BWD) {
      atomicAdd(&A.counters[CNT_QTEST], qt);
      atomicAdd(&A.counters[CNT_QHIT], qh);
    }
  }
}

}  // namespace

void dvx_composite_naive_launch(const CompositeArgs &a, bool backward, cudaStream_t st) {
  if (a.p.n_tiles == 0) return;
    if (backward) { DVX_COUNT_LAUNCH(1); composite_naive_kernel<true><<<a.p.n_tiles, TILE_THREADS, 0, st>>>(a); }
    else { DVX_COUNT_LAUNCH(1); composite_naive_kernel<false><<<a.p.n_tiles, TILE_THREADS, 0, st>>>(a); }
}
