// dvx_features.cu - widening row N3: feature compositing and the feature fuser.
//
// "substituting the standard RGB color rendering step with a high-dimensional feature accumulation pass";
// the "feature volume fuser".  Reading R25: with w_j = T_j alpha_j the compositing weights of a ray,
//   render:  F[p][c]   = sum_j w_j feat[v_j][c]
//   fuse:    num[v][c] += sum_(p,j: v_j = v) w_j img[p][c],   wsum[v] += sum w_j        (the transpose of render)
//
// B200 design: the weights do not depend on the payload, so the traversal (the issue-bound part of the rasterizer) runs ONCE
// per frame and leaves the weights as a CSR matrix W [H*W x V_total] (dvx_composite_export_launch: row lengths = the n_used
// the rendering pass saved, 8 bytes per non-zero).  Feature rendering is then the SpMM  F = W feat  and fusing is
// num += W^T img, for any number of channels and any number of feature sets, and both are plain streaming kernels - the one
// part of the method that is bound by memory traffic rather than instruction issue:
//   CTA = one 16x16 tile, warp = its 4x8 pixel block, one pixel after the other; lanes = channels (float4 per lane when
//   C % 4 == 0).  A pixel's (voxel, weight) pairs are loaded 32 at a time, coalesced, and broadcast by shuffle; each
//   non-zero then costs one coalesced row read (render) or one vector reduction per lane (fuse).  The ~360 distinct voxel
//   rows a tile touches (C = 64: 92 KB) stay in L1 across its 256 pixels, so DRAM sees each row about once per tile.
#include "dvx_internal.cuh"

namespace {

constexpr int FEAT_THREADS = 256;
constexpr int FEAT_MAX_K = 4;  // float4 path: C <= 4 * 32 * FEAT_MAX_K = 512;  scalar path: C <= 32 * 4 * FEAT_MAX_K = 512

struct FeatArgs {
  uint32_t width, height, tiles_x, n_channels;
  const uint32_t *row_start;
  const uint32_t *voxel;
  const float *weight;
  const float *feat;  // render: [V_total][C]
  float *out;         // render: [H][W][C]
  const float *img;   // fuse:   [H][W][C]
  float *num;         // fuse:   [V_total][C]
  float *wsum;        // fuse:   [V_total] or NULL
};

__device__ __forceinline__ void red_add_v4f(float *addr, float4 v) {
  asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(addr), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w) : "memory");
}

// VEC = 4: lane holds channels 128 k + 4 lane .. +3;  VEC = 1: lane holds channels 32 k + lane (k < 4 FEAT_MAX_K)
template <int VEC, bool FUSE>
__global__ void __launch_bounds__(FEAT_THREADS) feature_kernel(const __grid_constant__ FeatArgs A) {
  constexpr int NK = VEC == 4 ? FEAT_MAX_K : 4 * FEAT_MAX_K;
  const int tile = blockIdx.x, warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int u0 = (tile % A.tiles_x) * DVX_TILE + (warp & 3) * 4;  // the compositor's 4x8 pixel block of this warp
  const int v0 = (tile / A.tiles_x) * DVX_TILE + (warp >> 2) * 8;
  const uint32_t C = A.n_channels;
  for (int px = 0; px < 32; ++px) {
    const int u = u0 + (px & 3), v = v0 + (px >> 2);
    if (u >= (int)A.width || v >= (int)A.height) continue;  // warp-uniform
    const size_t pix = (size_t)v * A.width + u;
    const uint32_t b = A.row_start[pix], e = A.row_start[pix + 1];
    float acc[NK * VEC];
#pragma unroll
    for (int k = 0; k < NK * VEC; ++k) acc[k] = 0.f;
    if (FUSE) {  // this pixel's 2-D feature, held in the accumulator registers
#pragma unroll
      for (int k = 0; k < NK; ++k) {
        const uint32_t ch = (uint32_t)(k * 32 + lane) * VEC;
        if (ch < C) {
          if (VEC == 4) {
            const float4 g = *reinterpret_cast<const float4 *>(A.img + pix * C + ch);
            acc[4 * k] = g.x; acc[4 * k + 1] = g.y; acc[4 * k + 2] = g.z; acc[4 * k + 3] = g.w;
          } else {
            acc[k] = A.img[pix * C + ch];
          }
        }
      }
    }
    for (uint32_t j0 = b; j0 < e; j0 += 32) {
      const uint32_t n = min(32u, e - j0);
      uint32_t my_vox = 0;
      float my_w = 0.f;
      if ((uint32_t)lane < n) {
        my_vox = __ldg(A.voxel + j0 + lane);
        my_w = __ldg(A.weight + j0 + lane);
      }
      if (FUSE && A.wsum && (uint32_t)lane < n) atomicAdd(A.wsum + my_vox, my_w);
#pragma unroll 4
      for (uint32_t i = 0; i < n; ++i) {
        const uint32_t id = __shfl_sync(0xffffffffu, my_vox, (int)i);
        const float w = __shfl_sync(0xffffffffu, my_w, (int)i);
#pragma unroll
        for (int k = 0; k < NK; ++k) {
          const uint32_t ch = (uint32_t)(k * 32 + lane) * VEC;
          if (ch < C) {
            if (!FUSE) {
              if (VEC == 4) {
                const float4 f = __ldg(reinterpret_cast<const float4 *>(A.feat + (size_t)id * C + ch));
                acc[4 * k] = fmaf(w, f.x, acc[4 * k]); acc[4 * k + 1] = fmaf(w, f.y, acc[4 * k + 1]);
                acc[4 * k + 2] = fmaf(w, f.z, acc[4 * k + 2]); acc[4 * k + 3] = fmaf(w, f.w, acc[4 * k + 3]);
              } else {
                acc[k] = fmaf(w, __ldg(A.feat + (size_t)id * C + ch), acc[k]);
              }
            } else {
              if (VEC == 4)
                red_add_v4f(A.num + (size_t)id * C + ch,
                            make_float4(w * acc[4 * k], w * acc[4 * k + 1], w * acc[4 * k + 2], w * acc[4 * k + 3]));
              else
                atomicAdd(A.num + (size_t)id * C + ch, w * acc[k]);
            }
          }
        }
      }
    }
    if (!FUSE) {
#pragma unroll
      for (int k = 0; k < NK; ++k) {
        const uint32_t ch = (uint32_t)(k * 32 + lane) * VEC;
        if (ch < C) {
          if (VEC == 4)
            *reinterpret_cast<float4 *>(A.out + pix * C + ch) = make_float4(acc[4 * k], acc[4 * k + 1], acc[4 * k + 2], acc[4 * k + 3]);
          else
            A.out[pix * C + ch] = acc[k];
        }
      }
    }
  }
}

// C = 4 LPR with LPR | 32 (C = 4 .. 128): a row is LPR float4 lanes, so the warp serves 32 / LPR non-zeros at once - every
// lane busy - each lane group with its own accumulator, summed across the groups by shuffles when the pixel is done.
template <int LPR, bool FUSE>
__global__ void __launch_bounds__(FEAT_THREADS) feature_grouped_kernel(const __grid_constant__ FeatArgs A) {
  constexpr int NG = 32 / LPR;
  const int tile = blockIdx.x, warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int grp = lane / LPR, sub = lane % LPR;
  const int u0 = (tile % A.tiles_x) * DVX_TILE + (warp & 3) * 4;
  const int v0 = (tile / A.tiles_x) * DVX_TILE + (warp >> 2) * 8;
  constexpr uint32_t C = 4 * LPR;
  for (int px = 0; px < 32; ++px) {
    const int u = u0 + (px & 3), v = v0 + (px >> 2);
    if (u >= (int)A.width || v >= (int)A.height) continue;  // warp-uniform
    const size_t pix = (size_t)v * A.width + u;
    const uint32_t b = A.row_start[pix], e = A.row_start[pix + 1];
    float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
    if (FUSE) acc = *reinterpret_cast<const float4 *>(A.img + pix * C + 4 * sub);
    for (uint32_t j0 = b; j0 < e; j0 += 32) {
      const uint32_t n = min(32u, e - j0);
      uint32_t my_vox = 0;
      float my_w = 0.f;
      if ((uint32_t)lane < n) {
        my_vox = __ldg(A.voxel + j0 + lane);
        my_w = __ldg(A.weight + j0 + lane);
      }
      if (FUSE && A.wsum && (uint32_t)lane < n) atomicAdd(A.wsum + my_vox, my_w);
#pragma unroll 4
      for (uint32_t i0 = 0; i0 < n; i0 += NG) {
        const uint32_t i = i0 + grp;
        const uint32_t id = __shfl_sync(0xffffffffu, my_vox, (int)(i & 31u));
        const float w = __shfl_sync(0xffffffffu, my_w, (int)(i & 31u));
        if (i < n) {
          if (!FUSE) {
            const float4 f = __ldg(reinterpret_cast<const float4 *>(A.feat + (size_t)id * C) + sub);
            acc.x = fmaf(w, f.x, acc.x); acc.y = fmaf(w, f.y, acc.y); acc.z = fmaf(w, f.z, acc.z); acc.w = fmaf(w, f.w, acc.w);
          } else {
            red_add_v4f(A.num + (size_t)id * C + 4 * sub, make_float4(w * acc.x, w * acc.y, w * acc.z, w * acc.w));
          }
        }
      }
    }
    if (!FUSE) {
#pragma unroll
      for (int o = LPR; o < 32; o <<= 1) {
        acc.x += __shfl_xor_sync(0xffffffffu, acc.x, o); acc.y += __shfl_xor_sync(0xffffffffu, acc.y, o);
        acc.z += __shfl_xor_sync(0xffffffffu, acc.z, o); acc.w += __shfl_xor_sync(0xffffffffu, acc.w, o);
      }
      if (grp == 0) *(reinterpret_cast<float4 *>(A.out + pix * C) + sub) = acc;
    }
  }
}

template <bool FUSE>
bool launch_grouped(const FeatArgs &A, unsigned tiles, cudaStream_t st) {
  switch (A.n_channels) {
    case 4: feature_grouped_kernel<1, FUSE><<<tiles, FEAT_THREADS, 0, st>>>(A); return true;
    case 8: feature_grouped_kernel<2, FUSE><<<tiles, FEAT_THREADS, 0, st>>>(A); return true;
    case 16: feature_grouped_kernel<4, FUSE><<<tiles, FEAT_THREADS, 0, st>>>(A); return true;
    case 32: feature_grouped_kernel<8, FUSE><<<tiles, FEAT_THREADS, 0, st>>>(A); return true;
    case 64: feature_grouped_kernel<16, FUSE><<<tiles, FEAT_THREADS, 0, st>>>(A); return true;
    case 128: feature_grouped_kernel<32, FUSE><<<tiles, FEAT_THREADS, 0, st>>>(A); return true;
    default: return false;
  }
}

}  // namespace

void dvx_features_launch(uint32_t width, uint32_t height, uint32_t n_channels, const uint32_t *row_start, const uint32_t *voxel,
                         const float *weight, const float *feat, float *out, const float *img, float *num, float *wsum,
                         cudaStream_t st) {
  FeatArgs A;
  A.width = width; A.height = height; A.tiles_x = (width + DVX_TILE - 1) / DVX_TILE; A.n_channels = n_channels;
  A.row_start = row_start; A.voxel = voxel; A.weight = weight;
  A.feat = feat; A.out = out; A.img = img; A.num = num; A.wsum = wsum;
  const unsigned tiles = A.tiles_x * ((height + DVX_TILE - 1) / DVX_TILE);
  if (tiles == 0) return;
  const bool fuse = img != nullptr;
  const bool v4 = (n_channels % 4) == 0;
  DVX_COUNT_LAUNCH(1);
  if (fuse ? launch_grouped<true>(A, tiles, st) : launch_grouped<false>(A, tiles, st)) return;
  if (fuse) {
    if (v4) feature_kernel<4, true><<<tiles, FEAT_THREADS, 0, st>>>(A);
    else feature_kernel<1, true><<<tiles, FEAT_THREADS, 0, st>>>(A);
  } else {
    if (v4) feature_kernel<4, false><<<tiles, FEAT_THREADS, 0, st>>>(A);
    else feature_kernel<1, false><<<tiles, FEAT_THREADS, 0, st>>>(A);
  }
}
