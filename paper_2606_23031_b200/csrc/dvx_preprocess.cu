// dvx_preprocess.cu - hot-path steps 0, 1 and the non-sort parts of step 2:
//   step 0  per-octree, per-octant rank tables under the key morton48 XOR q*0x249249249249 (R14b)
//   step 1  per-voxel projection under the octree's rigid transform, pixel/tile rectangle, frustum + OBB cull,
//           per-voxel view-dependent colour (R8)
//   step 2  (tile, octant, voxel) key generation and per-bucket ranges (the radix sort itself is dvx_sort.cu)
//   step 5b per-voxel SH post-pass of the backward
#include "dvx_device.cuh"

namespace {

constexpr int PRE_THREADS = 256;

__device__ __forceinline__ int find_tree(const uint32_t *s_base, int n_trees, uint32_t g) {
  int t = 0;
  while (t + 1 < n_trees && g >= s_base[t + 1]) ++t;
  return t;
}

// ------------------------------------------------------------------ step 0
__global__ void rank_keys_kernel(const uint64_t *code, uint32_t n, uint64_t flip, uint64_t *keys, uint32_t *vals) {
  uint32_t v = blockIdx.x * blockDim.x + threadIdx.x;
  if (v >= n) return;
  keys[v] = (code[v] & 0xFFFFFFFFFFFFull) ^ flip;
  vals[v] = v;
}
__global__ void rank_scatter_kernel(const uint32_t *perm, uint32_t n, uint32_t *rank) {
  uint32_t r = blockIdx.x * blockDim.x + threadIdx.x;
  if (r < n) rank[perm[r]] = r;
}
// Leaf-set validation on the q = 0 order: level in [1,16], bits below the level zero, no leaf equal to or nested in
// its successor (ancestors sort immediately before their descendants because of the zero padding).
__global__ void validate_kernel(const uint64_t *skeys, const uint32_t *perm, const uint64_t *code, uint32_t n,
                                uint32_t *bad) {
  uint32_t r = blockIdx.x * blockDim.x + threadIdx.x;
  if (r >= n) return;
  uint64_t c = code[perm[r]];
  uint32_t l = (uint32_t)(c >> 48) & 31u;
  bool ok = (c >> 53) == 0 && l >= 1 && l <= DVX_MAX_LEVEL;
  if (ok) {
    uint32_t sh = 3u * (DVX_MAX_LEVEL - l);
    uint64_t path = c & 0xFFFFFFFFFFFFull;
    if (sh && (path & ((1ull << sh) - 1ull))) ok = false;
    if (ok && r + 1 < n && ((skeys[r + 1] >> sh) == (path >> sh))) ok = false;  // duplicate or descendant follows
  }
  if (!ok) atomicOr(bad, 1u);
}

// ------------------------------------------------------------------ per-frame set-up
// One thread per tree: pixel rectangle of the actor's oriented box.
__global__ void tree_setup_kernel(FrameParams p, TreeFrame *trees, unsigned long long *counters, const unsigned long long *rec_last) {
  int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t == 0 && rec_last) {  // what the latest frame's hit records needed: travels to the host with this frame's pair count
    counters[CNT_PREV_REC] = rec_last[0];
    counters[CNT_PREV_NPIX] = rec_last[1];
  }
  if (t >= (int)p.n_trees) return;
  TreeFrame &T = trees[t];
  if (!T.is_actor) {
    T.box_rect[0] = 0; T.box_rect[1] = 0; T.box_rect[2] = (int)p.width - 1; T.box_rect[3] = (int)p.height - 1;
    return;
  }
  float pc[8][3];
  for (int c = 0; c < 8; ++c) {
    float rel[3];
    for (int a = 0; a < 3; ++a) {
      double x = ((c >> (2 - a)) & 1) ? (double)T.half[a] : -(double)T.half[a];
      rel[a] = (float)(x - T.o_l[a]);
    }
    for (int cc = 0; cc < 3; ++cc) pc[c][cc] = T.N[cc] * rel[0] + T.N[3 + cc] * rel[1] + T.N[6 + cc] * rel[2];
  }
  int x0, y0, x1, y1;
  if (dvx_pixel_rect(pc, p, x0, y0, x1, y1)) {
    T.box_rect[0] = x0; T.box_rect[1] = y0; T.box_rect[2] = x1; T.box_rect[3] = y1;
  } else {
    T.box_rect[0] = 1; T.box_rect[1] = 1; T.box_rect[2] = 0; T.box_rect[3] = 0;
  }
}

// One thread per tile: for every tree the set of ray-direction octants present among the tile's pixels (R12), and the
// 64-bit mask of actors whose box footprint touches the tile.
__global__ void tile_masks_kernel(FrameParams p, const TreeFrame *trees, uint8_t *octmask, unsigned long long *actor_mask) {
  int tile = blockIdx.x * blockDim.x + threadIdx.x;
  if (tile >= (int)p.n_tiles) return;
  int tx = tile % p.tiles_x, ty = tile / p.tiles_x;
  int u0 = tx * DVX_TILE, v0 = ty * DVX_TILE;
  int u1 = min(u0 + DVX_TILE, (int)p.width) - 1, v1 = min(v0 + DVX_TILE, (int)p.height) - 1;
  float xs[2] = {dvx_cam_x(p, u0), dvx_cam_x(p, u1)}, ys[2] = {dvx_cam_y(p, v0), dvx_cam_y(p, v1)};
  unsigned long long am = 0;
  for (int t = 0; t < (int)p.n_trees; ++t) {
    const TreeFrame &T = trees[t];
    uint8_t m = 0;
    bool overlap = T.box_rect[2] >= u0 && T.box_rect[0] <= u1 && T.box_rect[3] >= v0 && T.box_rect[1] <= v1;
    if (overlap) {
      int sset[3];  // bit 0: some pixel has s_a = 0 (d_a >= 0); bit 1: some pixel has s_a = 1
      for (int a = 0; a < 3; ++a) {
        int s = 0;
        for (int i = 0; i < 2; ++i)
          for (int j = 0; j < 2; ++j) s |= (dvx_dir_comp(T.N, a, xs[i], ys[j]) < 0.f) ? 2 : 1;
        sset[a] = s;
      }
      for (int q = 0; q < 8; ++q) {
        int sx = (q >> 2) & 1, sy = (q >> 1) & 1, sz = q & 1;
        if (((sset[0] >> sx) & 1) && ((sset[1] >> sy) & 1) && ((sset[2] >> sz) & 1)) m |= (uint8_t)(1u << q);
      }
      if (T.is_actor) am |= 1ull << (t - 1);
    }
    octmask[(size_t)tile * p.n_trees + t] = m;
  }
  actor_mask[tile] = am;
}

// ------------------------------------------------------------------ step 1
__device__ __forceinline__ bool voxel_rect(const FrameParams &p, const TreeFrame &T, uint64_t code, float rel_out[3],
                                           float &s_out, int &x0, int &y0, int &x1, int &y1) {
  uint32_t X, Y, Z, l;
  dvx_decode16(code, X, Y, Z, l);
  const double s = T.cell * (double)(1u << (DVX_MAX_LEVEL - l));
  double mn[3] = {T.lo[0] + T.cell * (double)X, T.lo[1] + T.cell * (double)Y, T.lo[2] + T.cell * (double)Z};
  double bmn[3], bmx[3];
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    rel_out[a] = (float)(mn[a] - T.o_l[a]);
    bmn[a] = mn[a];
    bmx[a] = mn[a] + s;
    if (T.is_actor) {  // actor voxels only matter inside the box (R18)
      bmn[a] = fmax(bmn[a], -(double)T.half[a]);
      bmx[a] = fmin(bmx[a], (double)T.half[a]);
    }
  }
  s_out = (float)s;
  if (!(bmx[0] >= bmn[0]) || !(bmx[1] >= bmn[1]) || !(bmx[2] >= bmn[2])) return false;
  {  // Cheap conservative pre-cull (59 % of config 3's voxels end here instead of in the 8-corner projection below): the voxel's
     // bounding sphere lies wholly outside one side plane of the frustum (taken one pixel outside the image) or wholly behind
     // the clip plane.  Everything the exact test keeps is inside the sphere (clipping to the box or to z = zclip only
     // removes points), and the margin covers the fp32 rounding of this test (1e-3 of |centre| + radius).  The visible set, the
     // pair count and every image are unchanged (checked on configs 3 and 4); step 1 0.199 -> 0.184 ms on config 3.
     // Tried on top of it in round 2, all slower or equal: the SH record staged through shared memory by cp.async (0.208 ms,
     // one CTA per SM less), four lanes per voxel reading 48 contiguous bytes each (0.187), an L2 prefetch of the record
     // before the pair counting (0.192), 4 or 6 CTAs per SM (0.193 / 0.196): the kernel is bound by the dependent chain
     // code -> octant masks -> record at 2.7 TB/s, not by how the record is read.
    const float hs = 0.5f * s_out, cxl = rel_out[0] + hs, cyl = rel_out[1] + hs, czl = rel_out[2] + hs;
    const float X = T.N[0] * cxl + T.N[3] * cyl + T.N[6] * czl, Y = T.N[1] * cxl + T.N[4] * cyl + T.N[7] * czl,
                Z = T.N[2] * cxl + T.N[5] * cyl + T.N[8] * czl;
    const float r = 1.7320508f * hs;
    const float m = r + 1e-3f * (fabsf(X) + fabsf(Y) + fabsf(Z) + r);
    if (Z + m < p.zclip) return false;
    if (p.cull_t[0] * Z - X > m * p.cull_l[0] || X - p.cull_t[1] * Z > m * p.cull_l[1] ||
        p.cull_t[2] * Z - Y > m * p.cull_l[2] || Y - p.cull_t[3] * Z > m * p.cull_l[3]) return false;
  }
  float pc[8][3];
#pragma unroll
  for (int c = 0; c < 8; ++c) {
    float r0 = (float)(((c & 4) ? bmx[0] : bmn[0]) - T.o_l[0]);
    float r1 = (float)(((c & 2) ? bmx[1] : bmn[1]) - T.o_l[1]);
    float r2 = (float)(((c & 1) ? bmx[2] : bmn[2]) - T.o_l[2]);
#pragma unroll
    for (int cc = 0; cc < 3; ++cc) pc[c][cc] = T.N[cc] * r0 + T.N[3 + cc] * r1 + T.N[6 + cc] * r2;
  }
  return dvx_pixel_rect(pc, p, x0, y0, x1, y1);
}

__device__ __forceinline__ uint32_t count_pairs(const FrameParams &p, const uint8_t *octmask, int t, int x0, int y0,
                                                int x1, int y1) {
  uint32_t n = 0;
  for (int ty = y0 >> 4; ty <= (y1 >> 4); ++ty)
    for (int tx = x0 >> 4; tx <= (x1 >> 4); ++tx)
      n += __popc((uint32_t)octmask[(size_t)(ty * p.tiles_x + tx) * p.n_trees + t]);
  return n;
}

// A voxel whose rectangle spans more than BIG_TILES tiles (ground next to the camera, a voxel around the camera) is
// handled by its whole warp, 32 tiles per step, instead of by one thread walking up to thousands of tiles.
constexpr int BIG_TILES = 24;

__device__ __forceinline__ int rect_tiles(int x0, int y0, int x1, int y1) {
  return ((x1 >> 4) - (x0 >> 4) + 1) * ((y1 >> 4) - (y0 >> 4) + 1);
}

// Warp-cooperative count_pairs for the voxel held by lane `src` (all lanes call; every lane gets the total).
__device__ __forceinline__ uint32_t count_pairs_warp(const FrameParams &p, const uint8_t *octmask, int src, int t, int x0,
                                                     int y0, int x1, int y1) {
  t = __shfl_sync(0xffffffffu, t, src);
  const int tx0 = __shfl_sync(0xffffffffu, x0, src) >> 4, ty0 = __shfl_sync(0xffffffffu, y0, src) >> 4;
  const int tx1 = __shfl_sync(0xffffffffu, x1, src) >> 4, ty1 = __shfl_sync(0xffffffffu, y1, src) >> 4;
  const int w = tx1 - tx0 + 1, n = w * (ty1 - ty0 + 1);
  uint32_t c = 0;
  for (int i = threadIdx.x & 31; i < n; i += 32) {
    const int tile = (ty0 + i / w) * (int)p.tiles_x + tx0 + i % w;
    c += __popc((uint32_t)octmask[(size_t)tile * p.n_trees + t]);
  }
  for (int o = 16; o > 0; o >>= 1) c += __shfl_xor_sync(0xffffffffu, c, o);
  return c;
}

constexpr int DVX_PRE_MIN_CTAS = 5;  // 48 registers, no spills; config 3 step-1 ms for 4 / 5 / 6 CTAs per SM: 0.203 / 0.199 / 0.203
template <bool NRM>
__global__ void __launch_bounds__(PRE_THREADS, DVX_PRE_MIN_CTAS) preprocess_kernel(FrameParams p, const TreeFrame *trees,
                                                                 const uint8_t *octmask, FrameVox *fvox,
                                                                 ushort4 *pxrect, float4 *vnrm,
                                                                 unsigned long long *counters) {
  __shared__ uint32_t s_base[DVX_MAX_TREES + 1];
  for (int i = threadIdx.x; i < (int)p.n_trees; i += blockDim.x) s_base[i] = trees[i].base;
  __syncthreads();
  uint32_t g = blockIdx.x * blockDim.x + threadIdx.x;
  uint32_t npairs = 0, vis = 0;
  int t = 0, x0 = 0, y0 = 0, x1 = -1, y1 = -1;
  float rel[3] = {0.f, 0.f, 0.f}, s = 0.f;
  bool ok = false;
  if (g < p.v_total) {
    t = find_tree(s_base, p.n_trees, g);
    ok = voxel_rect(p, trees[t], trees[t].code[g - s_base[t]], rel, s, x0, y0, x1, y1);
  }
  const bool big = ok && rect_tiles(x0, y0, x1, y1) > BIG_TILES;
  if (ok && !big) npairs = count_pairs(p, octmask, t, x0, y0, x1, y1);
  for (uint32_t bm = __ballot_sync(0xffffffffu, big); bm; bm &= bm - 1) {
    const int src = __ffs(bm) - 1;
    const uint32_t c = count_pairs_warp(p, octmask, src, t, x0, y0, x1, y1);
    if ((int)(threadIdx.x & 31) == src) npairs = c;
  }
  if (g < p.v_total) {
    const TreeFrame &T = trees[t];
    const uint32_t v = g - s_base[t];
    if (npairs == 0) {
      pxrect[g] = make_ushort4(0xFFFF, 0xFFFF, 0, 0);
    } else {
      vis = 1;
      pxrect[g] = make_ushort4((unsigned short)x0, (unsigned short)y0, (unsigned short)x1, (unsigned short)y1);
      // O7 / R8: one colour per voxel per camera, direction camera origin -> voxel centre in the tree's frame
      float dx = rel[0] + 0.5f * s, dy = rel[1] + 0.5f * s, dz = rel[2] + 0.5f * s;
      float inv = rsqrtf(dx * dx + dy * dy + dz * dz);
      float Y[16];
      dvx_sh_basis(dx * inv, dy * inv, dz * inv, Y, (int)T.n_sh);
      float acc[3] = {0.5f, 0.5f, 0.5f};
      const float *k = T.sh + (size_t)v * T.n_sh * 3;
      if (T.n_sh == 16) {
        const float4 *k4 = reinterpret_cast<const float4 *>(k);
        float kk[48];
#pragma unroll
        for (int i = 0; i < 12; ++i) {
          float4 q = __ldg(k4 + i);
          kk[4 * i] = q.x; kk[4 * i + 1] = q.y; kk[4 * i + 2] = q.z; kk[4 * i + 3] = q.w;
        }
#pragma unroll
        for (int i = 0; i < 16; ++i) {
          acc[0] += Y[i] * kk[3 * i]; acc[1] += Y[i] * kk[3 * i + 1]; acc[2] += Y[i] * kk[3 * i + 2];
        }
      } else {
        for (int i = 0; i < (int)T.n_sh; ++i) {
          acc[0] += Y[i] * __ldg(k + 3 * i); acc[1] += Y[i] * __ldg(k + 3 * i + 1); acc[2] += Y[i] * __ldg(k + 3 * i + 2);
        }
      }
      FrameVox fv;
      fv.rel[0] = rel[0]; fv.rel[1] = rel[1]; fv.rel[2] = rel[2]; fv.s = s;
      uint32_t meta = 0;
#pragma unroll
      for (int ch = 0; ch < 3; ++ch) {
        if (!(acc[ch] > 0.f)) { meta |= 1u << ch; acc[ch] = 0.f; }
        fv.rgb[ch] = acc[ch];
      }
      fv.meta = meta | (npairs << 8);  // bits 8-31: this voxel's pair count (step 2 allocates its slots from it)
      fvox[g] = fv;
      if (NRM) {  // O11 / R22: world-frame voxel normal, only when a normal map was requested
        const float4 *gp = reinterpret_cast<const float4 *>(T.geo + (size_t)v * 8);
        const float4 g0 = __ldg(gp), g1 = __ldg(gp + 1);
        const float gg[8] = {g0.x, g0.y, g0.z, g0.w, g1.x, g1.y, g1.z, g1.w};
        float gr[3];
        dvx_centre_gradient(gg, gr);
        const float den = fmaxf(sqrtf(gr[0] * gr[0] + gr[1] * gr[1] + gr[2] * gr[2]), DVX_NRM_EPS);
        const float nl[3] = {-gr[0] / den, -gr[1] / den, -gr[2] / den};
        vnrm[g] = make_float4(T.R[0] * nl[0] + T.R[1] * nl[1] + T.R[2] * nl[2], T.R[3] * nl[0] + T.R[4] * nl[1] + T.R[5] * nl[2],
                              T.R[6] * nl[0] + T.R[7] * nl[1] + T.R[8] * nl[2], 0.f);
      }
    }
  }
  // warp-aggregated totals
  for (int o = 16; o > 0; o >>= 1) {
    npairs += __shfl_xor_sync(0xffffffffu, npairs, o);
    vis += __shfl_xor_sync(0xffffffffu, vis, o);
  }
  if ((threadIdx.x & 31) == 0 && (npairs | vis)) {
    atomicAdd(&counters[CNT_PAIRS], (unsigned long long)npairs);
    atomicAdd(&counters[CNT_VVIS], (unsigned long long)vis);
  }
}

// ------------------------------------------------------------------ step 2: key generation
// key = ((tile * 8 + q) << rank_bits) | (base_tree + rank_q(v)); value = global voxel id.  The octree is not a key field of
// its own: base_tree (the octree's first global voxel id) puts the ranks of all octrees into one number space of
// bits_for(v_total) bits, so the key is tile | octant | combined rank = 39 bits for config 3 (5 radix passes) instead of
// tile | tree | octant | rank = 42 (6 passes).  Within a tile the sorted order is (octant, tree, rank); every
// (tile, tree, octant) bucket is still one contiguous run, found by ranges_kernel.
// Every key is unique, so the order in which pairs are emitted does not matter: slots are handed out with one
// warp-aggregated atomic per warp from the per-voxel pair counts step 1 left in fvox.meta.  Voxels with a large
// footprint are emitted by the whole warp, 32 tiles per step.
__device__ __forceinline__ void emit_tile(const FrameParams &p, const TreeFrame &T, uint32_t tile, int t, uint32_t v, uint32_t g,
                                          uint32_t m, unsigned long long pos, uint64_t *keys, uint32_t *vals) {
  while (m) {
    const int q = __ffs(m) - 1;
    m &= m - 1;
    keys[pos] = (((uint64_t)tile * 8u + q) << p.rank_bits) | (uint64_t)(T.base + __ldg(T.rank + (size_t)q * T.n_voxels + v));
    vals[pos] = g;
    ++pos;
  }
}

__global__ void __launch_bounds__(PRE_THREADS) emit_pairs_kernel(FrameParams p, const TreeFrame *trees,
                                                                 const uint8_t *octmask, const ushort4 *pxrect,
                                                                 const FrameVox *fvox, uint64_t *keys, uint32_t *vals,
                                                                 unsigned long long capacity,
                                                                 unsigned long long *counters) {
  __shared__ uint32_t s_base[DVX_MAX_TREES + 1];
  for (int i = threadIdx.x; i < (int)p.n_trees; i += blockDim.x) s_base[i] = trees[i].base;
  __syncthreads();
  uint32_t g = blockIdx.x * blockDim.x + threadIdx.x;
  const int lane = threadIdx.x & 31;
  uint32_t n = 0;
  int t = 0;
  ushort4 r = make_ushort4(0xFFFF, 0xFFFF, 0, 0);
  if (g < p.v_total) {
    r = pxrect[g];
    if (r.x <= r.z) {
      t = find_tree(s_base, p.n_trees, g);
      n = fvox[g].meta >> 8;
    }
  }
  // warp exclusive scan of n, one atomic for the warp
  uint32_t inc = n;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    uint32_t x = __shfl_up_sync(0xffffffffu, inc, o);
    if (lane >= o) inc += x;
  }
  uint32_t total = __shfl_sync(0xffffffffu, inc, 31);
  if (total == 0) return;
  unsigned long long wbase = 0;
  if (lane == 31) wbase = atomicAdd(&counters[CNT_EMIT], (unsigned long long)total);
  wbase = __shfl_sync(0xffffffffu, wbase, 31);
  if (wbase + total > capacity) {
    if (lane == 0) atomicOr((unsigned int *)&counters[CNT_OVERFLOW], 1u);
    return;
  }
  unsigned long long pos = wbase + (inc - n);
  const bool big = n && rect_tiles(r.x, r.y, r.z, r.w) > BIG_TILES;
  if (n && !big) {
    const TreeFrame &T = trees[t];
    const uint32_t v = g - s_base[t];
    for (int ty = r.y >> 4; ty <= (r.w >> 4); ++ty)
      for (int tx = r.x >> 4; tx <= (r.z >> 4); ++tx) {
        const uint32_t tile = ty * p.tiles_x + tx;
        const uint32_t m = octmask[(size_t)tile * p.n_trees + t];
        emit_tile(p, T, tile, t, v, g, m, pos, keys, vals);
        pos += __popc(m);
      }
  }
  for (uint32_t bm = __ballot_sync(0xffffffffu, big); bm; bm &= bm - 1) {
    const int src = __ffs(bm) - 1;
    const int bt = __shfl_sync(0xffffffffu, t, src);
    const uint32_t bg = __shfl_sync(0xffffffffu, g, src);
    const int tx0 = __shfl_sync(0xffffffffu, (int)r.x, src) >> 4, ty0 = __shfl_sync(0xffffffffu, (int)r.y, src) >> 4;
    const int tx1 = __shfl_sync(0xffffffffu, (int)r.z, src) >> 4, ty1 = __shfl_sync(0xffffffffu, (int)r.w, src) >> 4;
    unsigned long long bpos = __shfl_sync(0xffffffffu, pos, src);
    const TreeFrame &T = trees[bt];
    const uint32_t v = bg - s_base[bt];
    const int w = tx1 - tx0 + 1, nt = w * (ty1 - ty0 + 1);
    for (int i0 = 0; i0 < nt; i0 += 32) {
      const int i = i0 + lane;
      uint32_t tile = 0, m = 0;
      if (i < nt) {
        tile = (ty0 + i / w) * p.tiles_x + tx0 + i % w;
        m = octmask[(size_t)tile * p.n_trees + bt];
      }
      uint32_t c = __popc(m), ci = c;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        uint32_t x = __shfl_up_sync(0xffffffffu, ci, o);
        if (lane >= o) ci += x;
      }
      emit_tile(p, T, tile, bt, v, bg, m, bpos + (ci - c), keys, vals);
      bpos += __shfl_sync(0xffffffffu, ci, 31);
    }
  }
}

// range[bucket] = [begin, end) in the sorted pair array, by boundary detection (buffers pre-zeroed: empty = [0,0)); bucket =
// (tile * n_trees + tree) * 8 + octant, with the tree recovered from the combined rank by a search over the trees' bases.
// tile_cost[tile] (pre-zeroed) receives the tile's pair count as sum(end) - sum(begin) over its buckets, in u32 arithmetic.
__device__ __forceinline__ uint32_t bucket_of(uint64_t key, uint32_t rank_bits, const uint32_t *s_base, int n_trees) {
  const uint32_t tq = (uint32_t)(key >> rank_bits), comb = (uint32_t)(key & ((1ull << rank_bits) - 1ull));
  int lo = 0;                         // last tree whose base <= comb
  if (n_trees > 1 && comb >= s_base[1]) {   // most pairs belong to the static octree (tree 0): one compare
#pragma unroll
    for (int step = 64; step >= 1; step >>= 1) {   // branch-free: n_trees <= 65
      const int m = lo + step;
      if (m < n_trees && s_base[m] <= comb) lo = m;
    }
  }
  return ((tq >> 3) * (uint32_t)n_trees + (uint32_t)lo) * 8u + (tq & 7u);
}
__global__ void ranges_kernel(const uint64_t *keys, uint64_t n, uint32_t rank_bits, const TreeFrame *trees, uint32_t n_trees,
                              uint32_t *range_beg, uint32_t *range_end, uint32_t *tile_cost) {
  __shared__ uint32_t s_base[DVX_MAX_TREES + 1];
  for (int i = threadIdx.x; i < (int)n_trees; i += blockDim.x) s_base[i] = trees[i].base;
  __syncthreads();
  const uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int lane = threadIdx.x & 31;
  const bool valid = i < n;
  // one search per element; the neighbours' buckets come by shuffle, only the warp's edge lanes look at a second key
  const uint32_t b = valid ? bucket_of(keys[i], rank_bits, s_base, (int)n_trees) : 0xFFFFFFFFu;
  uint32_t prev = __shfl_up_sync(0xffffffffu, b, 1), next = __shfl_down_sync(0xffffffffu, b, 1);
  if (!valid) return;
  if (lane == 0) prev = i == 0 ? 0xFFFFFFFFu : bucket_of(keys[i - 1], rank_bits, s_base, (int)n_trees);
  if (lane == 31) next = i + 1 == n ? 0xFFFFFFFFu : bucket_of(keys[i + 1], rank_bits, s_base, (int)n_trees);
  const bool first = prev != b, last = next != b;
  if (first) range_beg[b] = (uint32_t)i;
  if (last) range_end[b] = (uint32_t)(i + 1);
  if (tile_cost && (first || last)) {
    const uint32_t tile = b / (n_trees * 8u);
    if (first && last) atomicAdd(tile_cost + tile, 1u);
    else atomicAdd(tile_cost + tile, first ? 0u - (uint32_t)i : (uint32_t)(i + 1));
  }
}

// Launch order of the compositing CTAs: tiles by descending pair count (longest processing time first), so that the heavy
// tiles do not end up as the kernel's tail.  One CTA; the cost is quantised to 12 bits (relative to the heaviest tile) and
// sorted by a stable two-pass LSD counting sort (6 bits each), so equal-cost tiles keep raster order and the result is
// deterministic.  A warp ranks ORDER_ROUNDS x 32 consecutive tiles against its own digit counters (no block barrier inside),
// so a 1920x1080 frame (8160 tiles) is one chunk per pass: 28.8 -> 7 us.
// tile_order holds 2 n_tiles entries: the second half is the intermediate order, the first half the result.
constexpr int ORDER_THREADS = 1024, ORDER_DIGITS = 64, ORDER_ROUNDS = 8;
__device__ __forceinline__ uint32_t order_key(uint32_t cost, float scale) {  // key 0 = the most expensive tiles
  return 4095u - min(4095u, (uint32_t)((float)cost * scale));
}
__global__ void __launch_bounds__(ORDER_THREADS) tile_order_kernel(const uint32_t *tile_cost, uint32_t n_tiles, uint32_t *tile_order) {
  __shared__ uint32_t s_cnt[32][ORDER_DIGITS + 1];  // column ORDER_DIGITS: lanes past the end
  __shared__ uint32_t s_base[ORDER_DIGITS];
  __shared__ uint32_t s_warp[32];
  __shared__ uint32_t s_max;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  uint32_t mx = 0;
  for (uint32_t t = tid; t < n_tiles; t += ORDER_THREADS) mx = max(mx, tile_cost[t]);
  mx = __reduce_max_sync(0xffffffffu, mx);
  if (lane == 0) s_warp[warp] = mx;
  __syncthreads();
  if (warp == 0) {
    mx = __reduce_max_sync(0xffffffffu, s_warp[lane]);
    if (lane == 0) s_max = mx;
  }
  __syncthreads();
  const float scale = 4096.0f / ((float)s_max + 1.0f);
  for (int pass = 0; pass < 2; ++pass) {
    const uint32_t shift = 6u * pass;
    const uint32_t *src = pass ? tile_order + n_tiles : nullptr;  // pass 0 reads the tiles in raster order
    uint32_t *dst = pass ? tile_order : tile_order + n_tiles;
    if (tid < ORDER_DIGITS) s_base[tid] = 0;
    __syncthreads();
    for (uint32_t t0 = 0; t0 < n_tiles; t0 += ORDER_THREADS) {  // digit histogram, one shared-memory atomic per (warp, digit)
      const uint32_t t = t0 + tid;
      const uint32_t dig = t < n_tiles ? (order_key(tile_cost[t], scale) >> shift) & 63u : (uint32_t)ORDER_DIGITS;
      const uint32_t same = __match_any_sync(0xffffffffu, dig);
      if (dig != ORDER_DIGITS && (same & ((1u << lane) - 1u)) == 0u) atomicAdd(&s_base[dig], __popc(same));
    }
    __syncthreads();
    if (warp == 0) {  // exclusive scan of the 64 digit counts
      const uint32_t a = s_base[2 * lane], b = s_base[2 * lane + 1];
      uint32_t inc = a + b;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const uint32_t x = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += x;
      }
      s_base[2 * lane] = inc - a - b;
      s_base[2 * lane + 1] = inc - b;
    }
    for (uint32_t c0 = 0; c0 < n_tiles; c0 += ORDER_THREADS * ORDER_ROUNDS) {
      for (int i = tid; i < 32 * (ORDER_DIGITS + 1); i += ORDER_THREADS) (&s_cnt[0][0])[i] = 0;
      __syncthreads();
      uint32_t tl[ORDER_ROUNDS], dg[ORDER_ROUNDS], of[ORDER_ROUNDS];
#pragma unroll
      for (int r = 0; r < ORDER_ROUNDS; ++r) {  // chunk order = (warp, round, lane): consecutive entries of src
        const uint32_t idx = c0 + (uint32_t)(warp * ORDER_ROUNDS + r) * 32u + lane;
        tl[r] = idx < n_tiles ? (src ? src[idx] : idx) : 0xFFFFFFFFu;
      }
#pragma unroll
      for (int r = 0; r < ORDER_ROUNDS; ++r)  // all gathers in flight before the first ranking round
        dg[r] = tl[r] != 0xFFFFFFFFu ? (order_key(tile_cost[tl[r]], scale) >> shift) & 63u : (uint32_t)ORDER_DIGITS;
#pragma unroll
      for (int r = 0; r < ORDER_ROUNDS; ++r) {
        const uint32_t same = __match_any_sync(0xffffffffu, dg[r]);
        const uint32_t rank = __popc(same & ((1u << lane) - 1u));
        const uint32_t before = s_cnt[warp][dg[r]];
        of[r] = before + rank;
        __syncwarp();
        if (rank == 0) s_cnt[warp][dg[r]] = before + __popc(same);
        __syncwarp();
      }
      __syncthreads();
      if (tid < ORDER_DIGITS) {
        uint32_t run = s_base[tid];
        for (int w = 0; w < 32; ++w) { const uint32_t v = s_cnt[w][tid]; s_cnt[w][tid] = run; run += v; }
        s_base[tid] = run;
      }
      __syncthreads();
#pragma unroll
      for (int r = 0; r < ORDER_ROUNDS; ++r)
        if (dg[r] != ORDER_DIGITS) dst[s_cnt[warp][dg[r]] + of[r]] = tl[r];
      __syncthreads();
    }
    __threadfence_block();
  }
}

// ------------------------------------------------------------------ step 5b: dL/dk_{v,i} = Y_i(dir_v) dL/drgb_v
// SH degree 3 (the configured case): four threads per voxel, thread j owns coefficients 4j..4j+3 = 12 consecutive floats,
// so a quad reads and writes the voxel's 192 contiguous bytes with 16-byte accesses.  Other degrees: one thread per voxel.
__global__ void __launch_bounds__(PRE_THREADS) sh_backward_kernel(FrameParams p, const TreeFrame *trees,
                                                                  const FrameVox *fvox, const float *drgb) {
  __shared__ uint32_t s_base[DVX_MAX_TREES + 1];
  for (int i = threadIdx.x; i < (int)p.n_trees; i += blockDim.x) s_base[i] = trees[i].base;
  __syncthreads();
  const uint32_t gt = blockIdx.x * blockDim.x + threadIdx.x;
  const uint32_t g = gt >> 2, part = gt & 3u;
  if (g >= p.v_total) return;
  // drgb was zeroed before the compositing backward: a voxel no ray composited (culled, hidden, or off screen) still holds zeros
  float4 d = reinterpret_cast<const float4 *>(drgb)[g];
  if (d.x == 0.f && d.y == 0.f && d.z == 0.f) return;
  int t = find_tree(s_base, p.n_trees, g);
  const TreeFrame &T = trees[t];
  if (!T.dsh) return;
  if (T.n_sh != 16 && part != 0) return;
  FrameVox fv = fvox[g];
  float dx = fv.rel[0] + 0.5f * fv.s, dy = fv.rel[1] + 0.5f * fv.s, dz = fv.rel[2] + 0.5f * fv.s;
  float inv = rsqrtf(dx * dx + dy * dy + dz * dz);
  float Y[16];
  dvx_sh_basis(dx * inv, dy * inv, dz * inv, Y, (int)T.n_sh);
  float gch[3] = {(fv.meta & 1u) ? 0.f : d.x, (fv.meta & 2u) ? 0.f : d.y, (fv.meta & 4u) ? 0.f : d.z};
  float *out = T.dsh + (size_t)(g - s_base[t]) * T.n_sh * 3;
  if (T.n_sh == 16) {
    float y[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) y[k] = part == 0 ? Y[k] : part == 1 ? Y[4 + k] : part == 2 ? Y[8 + k] : Y[12 + k];
    float v[12];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      v[3 * k] = y[k] * gch[0]; v[3 * k + 1] = y[k] * gch[1]; v[3 * k + 2] = y[k] * gch[2];
    }
    float4 *o4 = reinterpret_cast<float4 *>(out) + 3 * part;
#pragma unroll
    for (int k = 0; k < 3; ++k) {
      float4 x = o4[k];
      x.x += v[4 * k]; x.y += v[4 * k + 1]; x.z += v[4 * k + 2]; x.w += v[4 * k + 3];
      o4[k] = x;
    }
  } else {
    for (int i = 0; i < (int)T.n_sh; ++i) {
      out[3 * i] += Y[i] * gch[0];
      out[3 * i + 1] += Y[i] * gch[1];
      out[3 * i + 2] += Y[i] * gch[2];
    }
  }
}

// ------------------------------------------------------------------ step 5c: dL/dgeo through the voxel normal (R22)
// dnrm[v] = sum over pixels of T alpha g_N (world frame).  n = -g / max(|g|, eps): dn/dg = -(I - n n^T)/|g| above eps,
// -I/eps below; g is linear in the corners with weights +-1/4.  One thread per voxel, after the compositing replay.
__global__ void __launch_bounds__(PRE_THREADS) normal_backward_kernel(FrameParams p, const TreeFrame *trees, const float *dnrm) {
  __shared__ uint32_t s_base[DVX_MAX_TREES + 1];
  for (int i = threadIdx.x; i < (int)p.n_trees; i += blockDim.x) s_base[i] = trees[i].base;
  __syncthreads();
  const uint32_t g = blockIdx.x * blockDim.x + threadIdx.x;
  if (g >= p.v_total) return;
  const float4 d = reinterpret_cast<const float4 *>(dnrm)[g];   // zeroed before the compositing backward, like drgb
  if (d.x == 0.f && d.y == 0.f && d.z == 0.f) return;
  const int t = find_tree(s_base, p.n_trees, g);
  const TreeFrame &T = trees[t];
  if (!T.dgeo) return;
  const uint32_t v = g - s_base[t];
  const float4 *gp = reinterpret_cast<const float4 *>(T.geo + (size_t)v * 8);
  const float4 g0 = __ldg(gp), g1 = __ldg(gp + 1);
  const float gg[8] = {g0.x, g0.y, g0.z, g0.w, g1.x, g1.y, g1.z, g1.w};
  float gr[3];
  dvx_centre_gradient(gg, gr);
  const float gn = sqrtf(gr[0] * gr[0] + gr[1] * gr[1] + gr[2] * gr[2]);
  const float gl[3] = {T.R[0] * d.x + T.R[3] * d.y + T.R[6] * d.z, T.R[1] * d.x + T.R[4] * d.y + T.R[7] * d.z,
                       T.R[2] * d.x + T.R[5] * d.y + T.R[8] * d.z};  // R^T dL/dn_world
  float dg[3];
  if (gn > DVX_NRM_EPS) {
    const float nl[3] = {-gr[0] / gn, -gr[1] / gn, -gr[2] / gn};
    const float dot = nl[0] * gl[0] + nl[1] * gl[1] + nl[2] * gl[2];
#pragma unroll
    for (int a = 0; a < 3; ++a) dg[a] = -(gl[a] - nl[a] * dot) / gn;
  } else {
#pragma unroll
    for (int a = 0; a < 3; ++a) dg[a] = -gl[a] / DVX_NRM_EPS;
  }
  float4 *o = reinterpret_cast<float4 *>(T.dgeo + (size_t)v * 8);
  float4 o0 = o[0], o1 = o[1];
  const float qx = 0.25f * dg[0], qy = 0.25f * dg[1], qz = 0.25f * dg[2];
  o0.x += -qx - qy - qz; o0.y += -qx - qy + qz; o0.z += -qx + qy - qz; o0.w += -qx + qy + qz;
  o1.x += qx - qy - qz;  o1.y += qx - qy + qz;  o1.z += qx + qy - qz;  o1.w += qx + qy + qz;
  o[0] = o0; o[1] = o1;
}

// The gradient pointers of a backward call go into the frame's tree table by a one-block kernel with the table in its
// parameters - not by one small host-to-device copy per octree: those queue on the copy engine behind whatever image copy is in
// flight there (the host-buffer entry points) and each costs a driver round trip.
__global__ void patch_grads_kernel(TreeFrame *trees, uint32_t n_trees, const __grid_constant__ DvxGradTable tbl,
                                   const unsigned long long *counters, unsigned long long *rec_last, unsigned long long npix) {
  const uint32_t t = threadIdx.x;
  if (t < n_trees) { trees[t].dgeo = tbl.dgeo[t]; trees[t].dsh = tbl.dsh[t]; }
  if (t == 0 && rec_last && counters) { rec_last[0] = counters[CNT_REC_CHUNKS]; rec_last[1] = npix; }
}
__global__ void publish_rec_kernel(const unsigned long long *counters, unsigned long long *rec_last, unsigned long long npix) {
  rec_last[0] = counters[CNT_REC_CHUNKS];
  rec_last[1] = npix;
}

inline unsigned blocks_for(uint64_t n, int threads) { return (unsigned)((n + threads - 1) / threads); }

}  // namespace

void dvx_rank_keys_launch(const uint64_t *code, uint32_t n, int q, uint64_t *keys, uint32_t *vals, cudaStream_t st) {
  if (n) { DVX_COUNT_LAUNCH(1); rank_keys_kernel<<<blocks_for(n, 256), 256, 0, st>>>(code, n, (uint64_t)q * 0x249249249249ull, keys, vals); }
}
void dvx_rank_scatter_launch(const uint32_t *perm, uint32_t n, uint32_t *rank, cudaStream_t st) {
  if (n) { DVX_COUNT_LAUNCH(1); rank_scatter_kernel<<<blocks_for(n, 256), 256, 0, st>>>(perm, n, rank); }
}
void dvx_validate_launch(const uint64_t *skeys, const uint32_t *perm, const uint64_t *code, uint32_t n,
                         uint32_t *bad_flag, cudaStream_t st) {
  if (n) { DVX_COUNT_LAUNCH(1); validate_kernel<<<blocks_for(n, 256), 256, 0, st>>>(skeys, perm, code, n, bad_flag); }
}
void dvx_tree_setup_launch(const FrameParams &p, TreeFrame *trees, unsigned long long *counters, const unsigned long long *rec_last,
                           cudaStream_t st) {
  { DVX_COUNT_LAUNCH(1); tree_setup_kernel<<<1, 128, 0, st>>>(p, trees, counters, rec_last); }
}
void dvx_tile_masks_launch(const FrameParams &p, const TreeFrame *trees, uint8_t *octmask, unsigned long long *actor_mask,
                           cudaStream_t st) {
  { DVX_COUNT_LAUNCH(1); tile_masks_kernel<<<blocks_for(p.n_tiles, 128), 128, 0, st>>>(p, trees, octmask, actor_mask); }
}
void dvx_normal_backward_launch(const FrameParams &p, const TreeFrame *trees, const float *dnrm, cudaStream_t st) {
  if (p.v_total) {
    DVX_COUNT_LAUNCH(1);
    normal_backward_kernel<<<blocks_for(p.v_total, PRE_THREADS), PRE_THREADS, 0, st>>>(p, trees, dnrm);
  }
}
void dvx_preprocess_launch(const FrameParams &p, const TreeFrame *trees, const uint8_t *octmask, FrameVox *fvox,
                           ushort4 *pxrect, float4 *vnrm, unsigned long long *counters, cudaStream_t st) {
  if (!p.v_total) return;
  DVX_COUNT_LAUNCH(1);
  if (vnrm) preprocess_kernel<true><<<blocks_for(p.v_total, PRE_THREADS), PRE_THREADS, 0, st>>>(p, trees, octmask, fvox, pxrect, vnrm, counters);
  else preprocess_kernel<false><<<blocks_for(p.v_total, PRE_THREADS), PRE_THREADS, 0, st>>>(p, trees, octmask, fvox, pxrect, vnrm, counters);
}
void dvx_emit_pairs_launch(const FrameParams &p, const TreeFrame *trees, const uint8_t *octmask, const ushort4 *pxrect,
                           const FrameVox *fvox, uint64_t *keys, uint32_t *vals, unsigned long long capacity,
                           unsigned long long *counters, cudaStream_t st) {
    if (p.v_total) { DVX_COUNT_LAUNCH(1); emit_pairs_kernel<<<blocks_for(p.v_total, PRE_THREADS), PRE_THREADS, 0, st>>>(p, trees, octmask, pxrect, fvox, keys, vals,
                                                                                   capacity, counters); }
}
void dvx_ranges_launch(const uint64_t *keys, uint64_t n, uint32_t rank_bits, const TreeFrame *trees, uint32_t n_trees,
                       uint32_t *range_beg, uint32_t *range_end, uint32_t *tile_cost, cudaStream_t st) {
  if (n) { DVX_COUNT_LAUNCH(1); ranges_kernel<<<blocks_for(n, 256), 256, 0, st>>>(keys, n, rank_bits, trees, n_trees, range_beg, range_end, tile_cost); }
}
void dvx_tile_order_launch(const uint32_t *tile_cost, uint32_t n_tiles, uint32_t *tile_order, cudaStream_t st) {
  if (n_tiles) { DVX_COUNT_LAUNCH(1); tile_order_kernel<<<1, ORDER_THREADS, 0, st>>>(tile_cost, n_tiles, tile_order); }
}
void dvx_sh_backward_launch(const FrameParams &p, const TreeFrame *trees, const FrameVox *fvox, const float *drgb,
                            cudaStream_t st) {
    if (p.v_total) { DVX_COUNT_LAUNCH(1); sh_backward_kernel<<<blocks_for(4ull * p.v_total, PRE_THREADS), PRE_THREADS, 0, st>>>(p, trees, fvox, drgb); }
}
void dvx_patch_grads_launch(TreeFrame *trees, uint32_t n_trees, const DvxGradTable &tbl, const unsigned long long *counters,
                            unsigned long long *rec_last, unsigned long long npix, cudaStream_t st) {
  DVX_COUNT_LAUNCH(1);
  patch_grads_kernel<<<1, DVX_MAX_TREES, 0, st>>>(trees, n_trees, tbl, counters, rec_last, npix);
}
void dvx_publish_rec_launch(const unsigned long long *counters, unsigned long long *rec_last, unsigned long long npix, cudaStream_t st) {
  DVX_COUNT_LAUNCH(1);
  publish_rec_kernel<<<1, 1, 0, st>>>(counters, rec_last, npix);
}
