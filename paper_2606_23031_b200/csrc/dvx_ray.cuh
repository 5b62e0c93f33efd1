// dvx_ray.cuh - per-ray geometry shared by the compositing kernels (hot-path steps 3 and 4): ray set-up in a tree frame,
// ray-AABB slab test in camera-relative coordinates, ray-OBB test, density activation (R5).
#pragma once
#include "dvx_device.cuh"

struct Ray {
  float d[3], inv[3];   // direction in the current tree frame and its reciprocal
  bool zero[3];         // d_a == 0 (slab rule of O2/O4 for axis-parallel rays)
  bool any_zero;
};

__device__ __forceinline__ void make_ray(const float *N, float xp, float yp, float rn, Ray &r, int &octant) {
  octant = 0;
  r.any_zero = false;
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    float f = dvx_dir_comp(N, a, xp, yp);
    octant |= (f < 0.f) ? (4 >> a) : 0;  // R12: s_a = (d_a < 0)
    r.d[a] = f * rn;
    r.zero[a] = (r.d[a] == 0.f);
    r.any_zero |= r.zero[a];
    r.inv[a] = r.zero[a] ? 0.f : 1.0f / r.d[a];
  }
}

// Slab test of the ray (origin at 0, tree frame, camera-relative coordinates) against [mn, mn+s]^3 given as `rel`.
// Returns false on a certain miss.  Axis-parallel rays: miss when the origin is outside the half-open slab (R20).
__device__ __forceinline__ bool slab_rel(const Ray &r, const float rel[3], float s, float &t0, float &t1) {
  float lo = -INFINITY, hi = INFINITY;
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    float ta = rel[a] * r.inv[a], tb = (rel[a] + s) * r.inv[a];
    float tn = fminf(ta, tb), tf = fmaxf(ta, tb);
    if (r.any_zero && r.zero[a]) {
      bool inside = (rel[a] <= 0.f) && (rel[a] + s > 0.f);  // mn <= o < mx
      if (!inside) return false;
      tn = -INFINITY; tf = INFINITY;
    }
    lo = fmaxf(lo, tn);
    hi = fminf(hi, tf);
  }
  t0 = lo; t1 = hi;
  return true;
}

__device__ __forceinline__ float act_fn(float x, uint32_t kind) {
  if (kind == 0) return __expf(x);
  const float th = 1.1f;
  return x > th ? x : __expf(x * (1.0f / th) - 1.0f + 0.09531017980432493f);  // ln 1.1
}
__device__ __forceinline__ float dact_fn(float x, uint32_t kind) {
  if (kind == 0) return __expf(x);
  const float th = 1.1f;
  return x > th ? 1.0f : __expf(x * (1.0f / th) - 1.0f + 0.09531017980432493f) * (1.0f / th);
}

// O2: ray-OBB in the actor frame.  Hit iff tau_out > max(tau_in, near).
__device__ __forceinline__ bool ray_box(const TreeFrame &T, const Ray &r, float near_, float far_, float &tin, float &tout) {
  float rel[3] = {-T.half[0] - T.ol_f[0], -T.half[1] - T.ol_f[1], -T.half[2] - T.ol_f[2]};
  float lo = -INFINITY, hi = INFINITY;
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    float mn = rel[a], mx = T.half[a] - T.ol_f[a];
    if (r.zero[a]) {
      if (!(mn <= 0.f && mx > 0.f)) return false;
    } else {
      float ta = mn * r.inv[a], tb = mx * r.inv[a];
      lo = fmaxf(lo, fminf(ta, tb));
      hi = fminf(hi, fmaxf(ta, tb));
    }
  }
  if (!(hi > fmaxf(lo, near_))) return false;
  tin = fmaxf(lo, near_);
  tout = fminf(hi, far_);
  return true;
}



// O10 / Eq. 2 (reading R21): bilinear footprint of pixel (u, v)'s WORLD direction in the equirectangular
// sky map.  Once per pixel, in fp64 up to the texel coordinates.  idx = texel indices into [H][W], wt = weights.
__device__ __forceinline__ void dvx_sky_footprint(const FrameParams &p, uint32_t W, uint32_t H, int u, int v, uint32_t idx[4],
                                                  float wt[4]) {
  const double xd = ((double)u + 0.5 - p.cx_d) * p.inv_fx, yd = ((double)v + 0.5 - p.cy_d) * p.inv_fy;
  const double rn = rsqrt(xd * xd + yd * yd + 1.0);
  const double dx = (p.Rc[0] * xd + p.Rc[1] * yd + p.Rc[2]) * rn, dy = (p.Rc[3] * xd + p.Rc[4] * yd + p.Rc[5]) * rn;
  const double dz = fmin(1.0, fmax(-1.0, (p.Rc[6] * xd + p.Rc[7] * yd + p.Rc[8]) * rn));
  const double PI = 3.14159265358979323846;
  const double s = (atan2(dy, dx) / (2.0 * PI) + 0.5) * (double)W - 0.5;
  const double t = fmin((double)H - 1.0, fmax(0.0, acos(dz) / PI * (double)H - 0.5));
  const double fs = floor(s), ft = floor(t);
  const float as = (float)(s - fs), at = (float)(t - ft);
  long long i0 = (long long)fs, j0 = (long long)ft;
  const long long w = (long long)W, h = (long long)H;
  long long i1 = i0 + 1;
  const long long j1 = j0 + 1 < h ? j0 + 1 : h - 1;
  i0 = ((i0 % w) + w) % w;
  i1 = ((i1 % w) + w) % w;
  idx[0] = (uint32_t)(j0 * w + i0); wt[0] = (1.f - as) * (1.f - at);
  idx[1] = (uint32_t)(j0 * w + i1); wt[1] = as * (1.f - at);
  idx[2] = (uint32_t)(j1 * w + i0); wt[2] = (1.f - as) * at;
  idx[3] = (uint32_t)(j1 * w + i1); wt[3] = as * at;
}
__device__ __forceinline__ void dvx_sky_colour(const float *tex, const uint32_t idx[4], const float wt[4], float rgb[3]) {
  rgb[0] = rgb[1] = rgb[2] = 0.f;
#pragma unroll
  for (int n = 0; n < 4; ++n) {
    const float *t = tex + 3 * (size_t)idx[n];
    rgb[0] = fmaf(wt[n], __ldg(t), rgb[0]); rgb[1] = fmaf(wt[n], __ldg(t + 1), rgb[1]); rgb[2] = fmaf(wt[n], __ldg(t + 2), rgb[2]);
  }
}

// Forward: T_final * C_sky for pixel (u, v) (added to C_voxels by the caller, Eq. 2).
static __device__ __noinline__ float3 dvx_sky_forward(const CompositeArgs *A, int u, int v, float T_final) {
  uint32_t idx[4];
  float wt[4], c[3];
  dvx_sky_footprint(A->p, A->sky_w, A->sky_h, u, v, idx, wt);
  dvx_sky_colour(A->sky_tex, idx, wt, c);
  return make_float3(T_final * c[0], T_final * c[1], T_final * c[2]);
}
// Backward of Eq. 2 for one pixel: dL/dtex += g_C T_final w (4 texels), and returns g_C . C_sky, the part of dL/dT_final
// that comes through the sky term (the caller folds it into the alpha gradient: alpha = 1 - T_final).
static __device__ __noinline__ float dvx_sky_backward(const CompositeArgs *A, int u, int v, float g0, float g1, float g2, float T_final) {
  uint32_t idx[4];
  float wt[4], c[3];
  dvx_sky_footprint(A->p, A->sky_w, A->sky_h, u, v, idx, wt);
  dvx_sky_colour(A->sky_tex, idx, wt, c);
  if (A->sky_dtex) {
#pragma unroll
    for (int n = 0; n < 4; ++n) {
      if (wt[n] == 0.f) continue;
      float *t = A->sky_dtex + 3 * (size_t)idx[n];
      const float k = T_final * wt[n];
      atomicAdd(t, g0 * k); atomicAdd(t + 1, g1 * k); atomicAdd(t + 2, g2 * k);
    }
  }
  return g0 * c[0] + g1 * c[1] + g2 * c[2];
}
