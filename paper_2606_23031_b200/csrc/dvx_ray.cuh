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

