// dvx_device.cuh - small __device__ helpers shared by the kernels (ray set-up, SH basis, Morton decode).
// The intrinsics with explicit rounding (__fmaf_rn, __fdiv_rn, ...) are used where two kernels must agree bit for bit
// on a sign decision (the ray-direction octant, reading R12): they are never contracted or re-associated by nvcc.
#pragma once
#include "dvx_internal.cuh"

// O1: d_cam = ((u+1/2-cx)/fx, (v+1/2-cy)/fy, 1).  Monotone in u and v.
__device__ __forceinline__ float dvx_cam_x(const FrameParams &p, int u) {
  return __fdiv_rn(__fadd_rn(__fadd_rn((float)u, 0.5f), -p.cx), p.fx);
}
__device__ __forceinline__ float dvx_cam_y(const FrameParams &p, int v) {
  return __fdiv_rn(__fadd_rn(__fadd_rn((float)v, 0.5f), -p.cy), p.fy);
}
// Un-normalised ray direction component a in a tree frame: f_a = N[3a] x' + N[3a+1] y' + N[3a+2].
// fmaf is monotone in each argument, so over a pixel rectangle the extremes of f_a sit at its corners: that is what
// lets the per-tile octant mask be computed from the four corner pixels only.
__device__ __forceinline__ float dvx_dir_comp(const float *N, int a, float xp, float yp) {
  return __fmaf_rn(N[3 * a], xp, __fmaf_rn(N[3 * a + 1], yp, N[3 * a + 2]));
}

// R14a: 48-bit left-aligned Morton path -> 16-bit cell coordinates at level-16 resolution (low 16-l bits zero).
__device__ __forceinline__ uint32_t dvx_compact3(uint64_t x) {
  x &= 0x1249249249249249ull;
  x = (x | (x >> 2)) & 0x10C30C30C30C30C3ull;
  x = (x | (x >> 4)) & 0x100F00F00F00F00Full;
  x = (x | (x >> 8)) & 0x001F0000FF0000FFull;
  x = (x | (x >> 16)) & 0x001F00000000FFFFull;
  x = (x | (x >> 32)) & 0xFFFFull;
  return (uint32_t)x;
}
__device__ __forceinline__ void dvx_decode16(uint64_t code, uint32_t &X, uint32_t &Y, uint32_t &Z, uint32_t &level) {
  uint64_t path = code & 0xFFFFFFFFFFFFull;
  level = (uint32_t)(code >> 48) & 31u;
  X = dvx_compact3(path >> 2);
  Y = dvx_compact3(path >> 1);
  Z = dvx_compact3(path);
}

// R8: real spherical harmonics up to degree 3 of the unit vector (x,y,z); constants as listed in DESIGN.md.
__device__ __forceinline__ void dvx_sh_basis(float x, float y, float z, float *Y, int n_sh) {
  Y[0] = 0.28209479177387814f;
  if (n_sh <= 1) return;
  const float c1 = 0.4886025119029199f;
  Y[1] = -c1 * y; Y[2] = c1 * z; Y[3] = -c1 * x;
  if (n_sh <= 4) return;
  const float c2a = 1.0925484305920792f, c2b = 0.31539156525252005f, c2c = 0.5462742152960396f;
  float xx = x * x, yy = y * y, zz = z * z;
  Y[4] = c2a * x * y; Y[5] = -c2a * y * z; Y[6] = c2b * (2.f * zz - xx - yy); Y[7] = -c2a * x * z; Y[8] = c2c * (xx - yy);
  if (n_sh <= 9) return;
  const float c3a = 0.5900435899266435f, c3b = 2.890611442640554f, c3c = 0.4570457994644658f;
  const float c3d = 0.3731763325901154f, c3e = 1.445305721320277f;
  Y[9] = -c3a * y * (3.f * xx - yy); Y[10] = c3b * x * y * z; Y[11] = -c3c * y * (4.f * zz - xx - yy);
  Y[12] = c3d * z * (2.f * zz - 3.f * xx - 3.f * yy); Y[13] = -c3c * x * (4.f * zz - xx - yy);
  Y[14] = c3e * z * (xx - yy); Y[15] = -c3a * x * (xx - 3.f * yy);
}

// Pixel rectangle (pixel-centre rule) of a convex body given its 8 camera-space corners, after clipping its 12 edges
// against z = zclip.  A ray through a pixel centre can only meet the body (at tau >= near) if the centre lies inside
// the bounding rectangle of the projection, so x0 = ceil(xmin - 1/2 - eps), x1 = floor(xmax - 1/2 + eps).
// Returns false when nothing is in front of the clip plane or the rectangle misses the image.
__device__ __forceinline__ bool dvx_pixel_rect(const float (*pc)[3], const FrameParams &p, int &x0, int &y0, int &x1, int &y1) {
  float xmin = 3.0e38f, xmax = -3.0e38f, ymin = 3.0e38f, ymax = -3.0e38f;
  bool any = false;
  const float zc = p.zclip;
#pragma unroll
  for (int c = 0; c < 8; ++c) {
    if (pc[c][2] >= zc) {
      float iz = 1.0f / pc[c][2];
      float px = p.fx * pc[c][0] * iz + p.cx, py = p.fy * pc[c][1] * iz + p.cy;
      xmin = fminf(xmin, px); xmax = fmaxf(xmax, px); ymin = fminf(ymin, py); ymax = fmaxf(ymax, py);
      any = true;
    }
  }
  bool behind = false;  // some corner lies behind the clip plane: only then can an edge cross it (almost never)
#pragma unroll
  for (int c = 0; c < 8; ++c) behind = behind || pc[c][2] < zc;
  if (behind) {
#pragma unroll
    for (int c = 0; c < 8; ++c) {
#pragma unroll
      for (int ax = 1; ax <= 4; ax <<= 1) {
        if (c & ax) continue;
        const int c2 = c | ax;
        float za = pc[c][2], zb = pc[c2][2];
        if ((za < zc) != (zb < zc)) {
          float f = (zc - za) / (zb - za);
          float qx = pc[c][0] + f * (pc[c2][0] - pc[c][0]), qy = pc[c][1] + f * (pc[c2][1] - pc[c][1]);
          float px = p.fx * qx / zc + p.cx, py = p.fy * qy / zc + p.cy;
          xmin = fminf(xmin, px); xmax = fmaxf(xmax, px); ymin = fminf(ymin, py); ymax = fmaxf(ymax, py);
          any = true;
        }
      }
    }
  }
  if (!any) return false;
  // relative slack for fp32 projection error plus 1/64 px absolute
  const float W = (float)p.width, H = (float)p.height;
  float ex = 0.015625f + 4e-6f * fmaxf(fabsf(xmin - p.cx), fabsf(xmax - p.cx));
  float ey = 0.015625f + 4e-6f * fmaxf(fabsf(ymin - p.cy), fabsf(ymax - p.cy));
  xmin -= 0.5f + ex; xmax += ex - 0.5f; ymin -= 0.5f + ey; ymax += ey - 0.5f;
  if (!(xmax >= 0.f) || !(ymax >= 0.f) || !(xmin <= W - 1.f) || !(ymin <= H - 1.f)) return false;
  x0 = xmin <= 0.f ? 0 : (int)ceilf(xmin);
  y0 = ymin <= 0.f ? 0 : (int)ceilf(ymin);
  x1 = xmax >= W - 1.f ? (int)p.width - 1 : (int)floorf(xmax);
  y1 = ymax >= H - 1.f ? (int)p.height - 1 : (int)floorf(ymax);
  return x1 >= x0 && y1 >= y0;
}


// R22: a voxel's normal = minus the gradient of its trilinear raw density at the voxel centre, normalised with
// max(|g|, 1e-6); g_a = 1/4 sum over the four corner pairs along axis a of (geo[b_a = 1] - geo[b_a = 0]).
#define DVX_NRM_EPS 1e-6f
__device__ __forceinline__ void dvx_centre_gradient(const float g[8], float grad[3]) {
  grad[0] = 0.25f * ((g[4] - g[0]) + (g[5] - g[1]) + (g[6] - g[2]) + (g[7] - g[3]));
  grad[1] = 0.25f * ((g[2] - g[0]) + (g[3] - g[1]) + (g[6] - g[4]) + (g[7] - g[5]));
  grad[2] = 0.25f * ((g[1] - g[0]) + (g[3] - g[2]) + (g[5] - g[4]) + (g[7] - g[6]));
}
