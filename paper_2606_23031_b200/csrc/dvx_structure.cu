// dvx_structure.cu - widening row N4: LiDAR-guided structure operations of the static octree
// (PAPER.md:87-93): proximity-based subdivision rounds, the Eq. 1 soft density prior per grid point, pruning.
//
// All three are one-off / once-per-thousand-iterations operations, so the kernels favour exactness over speed: the
// geometry (voxel boxes, grid-point positions, point distances) is evaluated in fp64 with explicitly rounded operations in
// the order reading R26 states, so that the integer decisions (split / keep) are reproducible bit for bit.
//
// The LiDAR cloud is binned once into a uniform cell grid (dvx_cloud): cell index per point, ONE radix sort of
// (cell, point) pairs (the step-2 sort), the points gathered into cell order, and a sorted list of the occupied cells with
// their start offsets.  A query visits the cells its search box overlaps (binary search per cell) - or, when that box
// holds more cells than are occupied at all, walks the occupied-cell list instead.
#include "dvx_internal.cuh"

namespace {

constexpr int ST_THREADS = 256;

struct CloudView {
  double origin[3];
  double cell;
  uint32_t dims[3];
  uint32_t n_cells;            // occupied
  const uint64_t *cell_key;    // [n_cells] ascending linear cell index
  const uint32_t *cell_start;  // [n_cells + 1]
  const float4 *pts;           // [n] in cell order
};

__device__ __forceinline__ unsigned long long enc_f(float f) {  // order-preserving float -> uint
  uint32_t u = __float_as_uint(f);
  return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}

// ---- cloud build
__global__ void __launch_bounds__(ST_THREADS) cloud_bounds_kernel(const float *__restrict__ pts, uint64_t n, uint32_t *mm) {
  const uint64_t i = (uint64_t)blockIdx.x * ST_THREADS + threadIdx.x;
  uint32_t lo[3] = {0xFFFFFFFFu, 0xFFFFFFFFu, 0xFFFFFFFFu}, hi[3] = {0u, 0u, 0u};
  if (i < n)
    for (int a = 0; a < 3; ++a) lo[a] = hi[a] = (uint32_t)enc_f(pts[3 * i + a]);
  for (int a = 0; a < 3; ++a) {
    lo[a] = __reduce_min_sync(0xffffffffu, lo[a]);
    hi[a] = __reduce_max_sync(0xffffffffu, hi[a]);
  }
  __shared__ uint32_t s_mm[6];  // one set of global atomics per block, not per warp
  if (threadIdx.x < 6) s_mm[threadIdx.x] = threadIdx.x < 3 ? 0xFFFFFFFFu : 0u;
  __syncthreads();
  if ((threadIdx.x & 31) == 0)
    for (int a = 0; a < 3; ++a) {
      atomicMin(s_mm + a, lo[a]);
      atomicMax(s_mm + 3 + a, hi[a]);
    }
  __syncthreads();
  if (threadIdx.x < 3) atomicMin(mm + threadIdx.x, s_mm[threadIdx.x]);
  else if (threadIdx.x < 6) atomicMax(mm + threadIdx.x, s_mm[threadIdx.x]);
}

__device__ __forceinline__ int cell_of(double x, double origin, double cell) {
  return (int)fmin(fmax(floor(__ddiv_rn(__dsub_rn(x, origin), cell)), -1.0e9), 1.0e9);
}

__global__ void __launch_bounds__(ST_THREADS) cloud_keys_kernel(const float *__restrict__ pts, uint64_t n, CloudView c,
                                                                uint64_t *__restrict__ keys, uint32_t *__restrict__ vals) {
  const uint64_t i = (uint64_t)blockIdx.x * ST_THREADS + threadIdx.x;
  if (i >= n) return;
  uint64_t k[3];
  for (int a = 0; a < 3; ++a) {
    int ci = cell_of((double)pts[3 * i + a], c.origin[a], c.cell);
    ci = ci < 0 ? 0 : (ci >= (int)c.dims[a] ? (int)c.dims[a] - 1 : ci);
    k[a] = (uint64_t)ci;
  }
  keys[i] = (k[2] * c.dims[1] + k[1]) * c.dims[0] + k[0];
  vals[i] = (uint32_t)i;
}

__global__ void __launch_bounds__(ST_THREADS) cloud_gather_kernel(const float *__restrict__ pts, const uint32_t *__restrict__ perm,
                                                                  uint64_t n, float4 *__restrict__ out) {
  const uint64_t i = (uint64_t)blockIdx.x * ST_THREADS + threadIdx.x;
  if (i >= n) return;
  const uint32_t s = perm[i];
  out[i] = make_float4(pts[3 * (size_t)s], pts[3 * (size_t)s + 1], pts[3 * (size_t)s + 2], 0.f);
}

__global__ void __launch_bounds__(ST_THREADS) cloud_cells_kernel(const uint64_t *__restrict__ skeys,
                                                                 const uint32_t *__restrict__ excl, uint64_t n,
                                                                 uint64_t *__restrict__ cell_key,
                                                                 uint32_t *__restrict__ cell_start) {
  const uint64_t i = (uint64_t)blockIdx.x * ST_THREADS + threadIdx.x;
  if (i >= n) return;
  const bool head = i == 0 || skeys[i] != skeys[i - 1];
  const uint32_t c = excl[i] + (head ? 1u : 0u) - 1u;
  if (head) {
    cell_key[c] = skeys[i];
    cell_start[c] = (uint32_t)i;
  }
  if (i == n - 1) cell_start[c + 1] = (uint32_t)n;
}

// ---- queries
__device__ __forceinline__ int find_cell(const CloudView &c, uint64_t key) {
  int lo = 0, hi = (int)c.n_cells - 1;
  while (lo <= hi) {
    const int mid = (lo + hi) >> 1;
    const uint64_t k = __ldg(c.cell_key + mid);
    if (k == key) return mid;
    if (k < key) lo = mid + 1;
    else hi = mid - 1;
  }
  return -1;
}

__device__ __forceinline__ uint32_t lower_cell(const CloudView &c, uint64_t key) {  // first occupied cell with key >= `key`
  uint32_t lo = 0, hi = c.n_cells;
  while (lo < hi) {
    const uint32_t mid = (lo + hi) >> 1;
    if (__ldg(c.cell_key + mid) < key) lo = mid + 1;
    else hi = mid;
  }
  return lo;
}

// lattice coordinate -> octree frame, in R26's order of operations: (centre - side/2) + X * (side / 65536)
__device__ __forceinline__ double lattice_pos(double center, double side, uint32_t X) {
  return __dadd_rn(__dsub_rn(center, __dmul_rn(0.5, side)), __dmul_rn((double)X, __ddiv_rn(side, 65536.0)));
}

__device__ __forceinline__ uint64_t compact3s(uint64_t x) {
  x &= 0x1249249249249249ull;
  x = (x ^ (x >> 2)) & 0x10c30c30c30c30c3ull;
  x = (x ^ (x >> 4)) & 0x100f00f00f00f00full;
  x = (x ^ (x >> 8)) & 0x001f0000ff0000ffull;
  x = (x ^ (x >> 16)) & 0x001f00000000ffffull;
  x = (x ^ (x >> 32)) & 0x00000000001fffffull;
  return x;
}

// squared distance from point p to the closed box [lo, hi] (0 inside), R26 order: ((gx^2 + gy^2) + gz^2)
__device__ __forceinline__ double box_dist2(const double lo[3], const double hi[3], float4 p) {
  const double q[3] = {(double)p.x, (double)p.y, (double)p.z};
  double s = 0.0;
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    const double g = fmax(fmax(__dsub_rn(lo[a], q[a]), __dsub_rn(q[a], hi[a])), 0.0);
    s = a == 0 ? __dmul_rn(g, g) : __dadd_rn(s, __dmul_rn(g, g));
  }
  return s;
}

// min over the cloud's points of box_dist2, restricted to the cells overlapping the box inflated by `reach`; lanes of the
// warp share the cells.  early = stop as soon as a point within reach is found (returns any value <= reach^2 then).
// G = lanes that share one query (32: a warp per leaf; 8: four grid points per warp, for queries whose search box has only
// a handful of rows); early exits need G = 32 (the warp-wide vote).
template <int G>
__device__ double warp_min_box_dist2(const CloudView &c, const double lo[3], const double hi[3], double reach, bool early) {
  const int lane = threadIdx.x & (G - 1);
  int c0[3], c1[3];
  bool empty = c.n_cells == 0;
  for (int a = 0; a < 3; ++a) {
    // a relative slack of 1e-9 (fp64 rounds at 1e-16) keeps a point at exactly `reach` on a cell boundary inside the range
    const double eps = 1e-9 * (fabs(lo[a]) + fabs(hi[a]) + reach + c.cell);
    c0[a] = cell_of(lo[a] - reach - eps, c.origin[a], c.cell);
    c1[a] = cell_of(hi[a] + reach + eps, c.origin[a], c.cell);
    c0[a] = max(c0[a], 0);
    c1[a] = min(c1[a], (int)c.dims[a] - 1);
    if (c1[a] < c0[a]) empty = true;
  }
  double best = 1.0e300;
  // an empty search box does not return here: it has no rows below and falls through to the shuffles (with G < 32 the other
  // groups of the warp go on, and a full-mask shuffle needs every lane)
  const double reach2 = reach * reach;
  const uint64_t nx = empty ? 0 : (uint64_t)(c1[0] - c0[0] + 1), ny = empty ? 0 : (uint64_t)(c1[1] - c0[1] + 1),
                 nz = empty ? 0 : (uint64_t)(c1[2] - c0[2] + 1);
  const uint64_t range = nx * ny * nz;
  // the occupied cells of the z-slab [c0z, c1z] are one contiguous run of the sorted cell list: when that run is shorter
  // than the search box has cells (coarse leaves, sparse clouds), walk the run instead of probing every cell of the box
  const uint64_t plane = (uint64_t)c.dims[0] * c.dims[1];
  uint32_t run_lo = 0, run_hi = 0xFFFFFFFFu;
  if (range > 256) {  // small boxes (fine leaves, grid points) are probed cell by cell without looking at the run
    run_lo = lower_cell(c, (uint64_t)c0[2] * plane);
    run_hi = lower_cell(c, (uint64_t)(c1[2] + 1) * plane);
  }
  const bool by_list = range > (uint64_t)(run_hi - run_lo);
  if (by_list) {
    const uint64_t total = (uint64_t)(run_hi - run_lo);
    for (uint64_t base = 0; base < total; base += G) {
      const uint64_t i = base + lane;
      int idx = -1;
      if (i < total) {
        const uint64_t key = __ldg(c.cell_key + run_lo + i);
        const int cx = (int)(key % c.dims[0]), cy = (int)((key / c.dims[0]) % c.dims[1]), cz = (int)(key / ((uint64_t)c.dims[0] * c.dims[1]));
        if (cx >= c0[0] && cx <= c1[0] && cy >= c0[1] && cy <= c1[1] && cz >= c0[2] && cz <= c1[2]) idx = (int)(run_lo + i);
      }
      if (idx >= 0) {
        const uint32_t b = __ldg(c.cell_start + idx), e = __ldg(c.cell_start + idx + 1);
        for (uint32_t j = b; j < e; ++j) {
          const double d2 = box_dist2(lo, hi, __ldg(c.pts + j));
          best = fmin(best, d2);
          if (early && d2 <= reach2) break;
        }
      }
      if (G == 32 && early && __any_sync(0xffffffffu, best <= reach2)) break;
    }
  } else {
    // lane = one x-row of the search box: its occupied cells are ONE contiguous run of the sorted cell list (keys are
    // (z * ny + y) * nx + x), found by one binary search per row instead of one per cell, and their points are one
    // contiguous range of the binned cloud
    const uint64_t rows = ny * nz;
    for (uint64_t base = 0; base < rows; base += G) {
      const uint64_t i = base + lane;
      if (i < rows) {
        const int cy = c0[1] + (int)(i % ny), cz = c0[2] + (int)(i / ny);
        const uint64_t row = ((uint64_t)cz * c.dims[1] + cy) * c.dims[0];
        const uint32_t i0 = lower_cell(c, row + (uint64_t)c0[0]);
        uint32_t i1 = i0;
        while (i1 < c.n_cells && __ldg(c.cell_key + i1) <= row + (uint64_t)c1[0]) ++i1;
        if (i1 > i0) {
          const uint32_t b = __ldg(c.cell_start + i0), e = __ldg(c.cell_start + i1);
          for (uint32_t j = b; j < e; ++j) {
            const double d2 = box_dist2(lo, hi, __ldg(c.pts + j));
            best = fmin(best, d2);
            if (early && d2 <= reach2) break;
          }
        }
      }
      if (G == 32 && early && __any_sync(0xffffffffu, best <= reach2)) break;
    }
  }
  for (int o = G / 2; o > 0; o >>= 1) {
    const double other = __hiloint2double(__shfl_xor_sync(0xffffffffu, __double2hiint(best), o),
                                          __shfl_xor_sync(0xffffffffu, __double2loint(best), o));
    best = fmin(best, other);
  }
  return best;
}

// Eq. 1 per grid point (warp = grid point): v_far + (v_close - v_far) exp(-2 d^2 / s^2); points beyond `reach` cannot change
// the fp32 result (the caller picks reach so that (v_close - v_far) exp(-2 reach^2 / s^2) is below half an ulp of v_far)
__global__ void __launch_bounds__(ST_THREADS) density_prior_kernel(CloudView c, const uint64_t *__restrict__ code,
                                                                   const uint32_t *__restrict__ offsets,
                                                                   const uint32_t *__restrict__ slots, uint32_t n_points,
                                                                   double cx, double cy, double cz, double side, double s_min,
                                                                   double reach, double v_close, double v_far,
                                                                   float *__restrict__ density) {
  // eight lanes per grid point (its search box has about 3 x 3 rows); a point index beyond the end keeps its lanes in the
  // warp's shuffles with a clamped, harmless query
  const uint64_t pg = ((uint64_t)blockIdx.x * ST_THREADS + threadIdx.x) >> 3;  // 64-bit: n_points * 8 threads may exceed 2^32
  const bool live = pg < n_points;
  const uint32_t p = live ? (uint32_t)pg : n_points - 1u;
  const uint32_t slot = __ldg(slots + __ldg(offsets + p));
  const uint64_t cd = __ldg(code + (slot >> 3));
  const uint32_t cn = slot & 7u, level = (uint32_t)(cd >> 48) & 31u;
  const uint64_t path = cd & 0xFFFFFFFFFFFFull;
  const uint32_t size = 1u << (DVX_MAX_LEVEL - level);
  const uint32_t X = (uint32_t)compact3s(path >> 2) + ((cn >> 2) & 1u) * size;
  const uint32_t Y = (uint32_t)compact3s(path >> 1) + ((cn >> 1) & 1u) * size;
  const uint32_t Z = (uint32_t)compact3s(path) + (cn & 1u) * size;
  const double q[3] = {lattice_pos(cx, side, X), lattice_pos(cy, side, Y), lattice_pos(cz, side, Z)};
  const double d2 = warp_min_box_dist2<8>(c, q, q, reach, false);
  if (live && (threadIdx.x & 7) == 0) {
    const double v = d2 > reach * reach ? v_far : v_far + (v_close - v_far) * exp(-2.0 * d2 / (s_min * s_min));
    density[p] = (float)v;
  }
}

// R26 (warp = leaf): flag = some point within `threshold` of the closed box, and level < max_level
__global__ void __launch_bounds__(ST_THREADS) near_flags_kernel(CloudView c, const uint64_t *__restrict__ code, uint32_t n_voxels,
                                                                double cx, double cy, double cz, double side,
                                                                double threshold, uint32_t max_level,
                                                                uint32_t *__restrict__ count, uint8_t *__restrict__ split) {
  const uint32_t v = (uint32_t)(((uint64_t)blockIdx.x * ST_THREADS + threadIdx.x) >> 5);  // 64-bit: n_voxels * 32 threads exceeds 2^32
  if (v >= n_voxels) return;
  const uint64_t cd = __ldg(code + v);
  const uint32_t level = (uint32_t)(cd >> 48) & 31u;
  const uint64_t path = cd & 0xFFFFFFFFFFFFull;
  const uint32_t size = 1u << (DVX_MAX_LEVEL - level);
  const uint32_t X = (uint32_t)compact3s(path >> 2), Y = (uint32_t)compact3s(path >> 1), Z = (uint32_t)compact3s(path);
  const double lo[3] = {lattice_pos(cx, side, X), lattice_pos(cy, side, Y), lattice_pos(cz, side, Z)};
  const double hi[3] = {lattice_pos(cx, side, X + size), lattice_pos(cy, side, Y + size), lattice_pos(cz, side, Z + size)};
  bool near = false;
  if (level < max_level) {
    const double d2 = warp_min_box_dist2<32>(c, lo, hi, threshold, true);
    near = __dsqrt_rn(d2) <= threshold;  // R26 compares the distance, not its square
  }
  if ((threadIdx.x & 31) == 0) {
    count[v] = near ? 8u : 1u;
    if (split) split[v] = near ? 1 : 0;
  }
}

// offsets [V+1] = exclusive scan of the counts (1 or 8) followed by a 0; a split leaf writes its 8 children in octant order 4x+2y+z
__global__ void __launch_bounds__(ST_THREADS) expand_kernel(const uint64_t *__restrict__ code, uint32_t n_voxels,
                                                            const uint32_t *__restrict__ offsets,
                                                            uint64_t *__restrict__ out) {
  const uint32_t v = blockIdx.x * ST_THREADS + threadIdx.x;
  if (v >= n_voxels) return;
  const uint32_t at = offsets[v];
  const uint32_t cnt = offsets[v + 1] - at;
  const uint64_t cd = code[v];
  if (cnt == 1) {
    out[at] = cd;
    return;
  }
  const uint64_t level = (cd >> 48) & 31ull, path = cd & 0xFFFFFFFFFFFFull;
  const uint64_t shift = 45ull - 3ull * level;
  for (uint64_t o = 0; o < 8; ++o) out[at + o] = ((level + 1ull) << 48) | path | (o << shift);
}

// R29: parameters of the leaves after a subdivision round.  count[v] = 8 or 1 from the split flags; offsets = their
// exclusive scan; thread = input leaf.  A child's corner c of octant o samples the parent's trilinear raw density at
// u = (o + b) / 2 (each u_a in {0, 1/2, 1}), evaluated in fp64 from the fp32 corners and rounded once; SH rows are copied.
__global__ void __launch_bounds__(ST_THREADS) split_counts_kernel(const uint8_t *__restrict__ split, uint32_t n_voxels,
                                                                  uint32_t *__restrict__ count) {
  const uint32_t v = blockIdx.x * ST_THREADS + threadIdx.x;
  if (v < n_voxels) count[v] = split[v] ? 8u : 1u;
}
__global__ void __launch_bounds__(ST_THREADS) subdivide_fill_kernel(const uint32_t *__restrict__ offsets, uint32_t n_voxels,
                                                                    const float *__restrict__ geo_in, const float *__restrict__ sh_in,
                                                                    uint32_t sh_floats, float *__restrict__ geo_out,
                                                                    float *__restrict__ sh_out) {
  const uint32_t v = blockIdx.x * ST_THREADS + threadIdx.x;
  if (v >= n_voxels) return;
  const uint32_t at = offsets[v], cnt = offsets[v + 1] - at;
  const float4 a = __ldg(reinterpret_cast<const float4 *>(geo_in) + 2 * (size_t)v);
  const float4 b = __ldg(reinterpret_cast<const float4 *>(geo_in) + 2 * (size_t)v + 1);
  const double g[8] = {a.x, a.y, a.z, a.w, b.x, b.y, b.z, b.w};
  const float *sh_src = sh_in ? sh_in + (size_t)v * sh_floats : nullptr;
  for (uint32_t o = 0; o < cnt; ++o) {
    float outv[8];
    if (cnt == 1) {
#pragma unroll
      for (int c = 0; c < 8; ++c) outv[c] = (float)g[c];
    } else {
#pragma unroll
      for (int c = 0; c < 8; ++c) {
        const double ux = 0.5 * (double)(((o >> 2) & 1u) + ((c >> 2) & 1)), uy = 0.5 * (double)(((o >> 1) & 1u) + ((c >> 1) & 1)),
                     uz = 0.5 * (double)((o & 1u) + (c & 1));
        double val = 0.0;
#pragma unroll
        for (int pc = 0; pc < 8; ++pc) {
          const double w = ((pc & 4) ? ux : 1.0 - ux) * ((pc & 2) ? uy : 1.0 - uy) * ((pc & 1) ? uz : 1.0 - uz);
          val += w * g[pc];
        }
        outv[c] = (float)val;
      }
    }
    float4 *go = reinterpret_cast<float4 *>(geo_out) + 2 * (size_t)(at + o);
    go[0] = make_float4(outv[0], outv[1], outv[2], outv[3]);
    go[1] = make_float4(outv[4], outv[5], outv[6], outv[7]);
    if (sh_src && sh_out) {
      float *so = sh_out + (size_t)(at + o) * sh_floats;
      for (uint32_t i = 0; i < sh_floats; ++i) so[i] = __ldg(sh_src + i);
    }
  }
}

// R28: keep = max corner >= threshold
__global__ void __launch_bounds__(ST_THREADS) prune_flags_kernel(const float *__restrict__ geo, uint32_t n_voxels, float threshold,
                                                                 uint32_t *__restrict__ keep) {
  const uint32_t v = blockIdx.x * ST_THREADS + threadIdx.x;
  if (v >= n_voxels) return;
  const float4 a = __ldg(reinterpret_cast<const float4 *>(geo) + 2 * (size_t)v);
  const float4 b = __ldg(reinterpret_cast<const float4 *>(geo) + 2 * (size_t)v + 1);
  const float m = fmaxf(fmaxf(fmaxf(a.x, a.y), fmaxf(a.z, a.w)), fmaxf(fmaxf(b.x, b.y), fmaxf(b.z, b.w)));
  keep[v] = m >= threshold ? 1u : 0u;
}

__global__ void __launch_bounds__(ST_THREADS) prune_scatter_kernel(const uint64_t *__restrict__ code, uint32_t n_voxels,
                                                                   const uint32_t *__restrict__ offsets,
                                                                   uint64_t *__restrict__ code_out, uint32_t *__restrict__ index_out) {
  const uint32_t v = blockIdx.x * ST_THREADS + threadIdx.x;
  if (v >= n_voxels) return;
  const uint32_t at = offsets[v];
  const uint32_t nxt = offsets[v + 1];
  if (nxt != at) {
    code_out[at] = code[v];
    if (index_out) index_out[at] = v;
  }
}

inline unsigned st_blocks(uint64_t n) { return (unsigned)((n + ST_THREADS - 1) / ST_THREADS); }

CloudView make_view(const DvxCloudData &d) {
  CloudView c;
  for (int a = 0; a < 3; ++a) { c.origin[a] = d.origin[a]; c.dims[a] = d.dims[a]; }
  c.cell = d.cell; c.n_cells = d.n_cells; c.cell_key = d.cell_key; c.cell_start = d.cell_start; c.pts = d.pts;
  return c;
}

}  // namespace

void dvx_cloud_bounds_launch(const float *pts, uint64_t n, uint32_t *minmax6, cudaStream_t st) {
  DVX_COUNT_LAUNCH(1);
  cloud_bounds_kernel<<<st_blocks(n), ST_THREADS, 0, st>>>(pts, n, minmax6);
}
void dvx_cloud_keys_launch(const float *pts, uint64_t n, const DvxCloudData &d, uint64_t *keys, uint32_t *vals, cudaStream_t st) {
  DVX_COUNT_LAUNCH(1);
  cloud_keys_kernel<<<st_blocks(n), ST_THREADS, 0, st>>>(pts, n, make_view(d), keys, vals);
}
void dvx_cloud_gather_launch(const float *pts, const uint32_t *perm, uint64_t n, float4 *out, cudaStream_t st) {
  DVX_COUNT_LAUNCH(1);
  cloud_gather_kernel<<<st_blocks(n), ST_THREADS, 0, st>>>(pts, perm, n, out);
}
void dvx_cloud_cells_launch(const uint64_t *skeys, const uint32_t *excl, uint64_t n, uint64_t *cell_key, uint32_t *cell_start,
                            cudaStream_t st) {
  DVX_COUNT_LAUNCH(1);
  cloud_cells_kernel<<<st_blocks(n), ST_THREADS, 0, st>>>(skeys, excl, n, cell_key, cell_start);
}
void dvx_density_prior_launch(const DvxCloudData &d, const uint64_t *code, const uint32_t *offsets, const uint32_t *slots,
                              uint32_t n_points, const double center[3], double side, double s_min, double reach,
                              double v_close, double v_far, float *density, cudaStream_t st) {
  DVX_COUNT_LAUNCH(1);
  density_prior_kernel<<<st_blocks((uint64_t)n_points * 8), ST_THREADS, 0, st>>>(make_view(d), code, offsets, slots, n_points,
                                                                                 center[0], center[1], center[2], side, s_min,
                                                                                 reach, v_close, v_far, density);
}
void dvx_near_flags_launch(const DvxCloudData &d, const uint64_t *code, uint32_t n_voxels, const double center[3], double side,
                           double threshold, uint32_t max_level, uint32_t *count, uint8_t *split, cudaStream_t st) {
  DVX_COUNT_LAUNCH(1);
  near_flags_kernel<<<st_blocks((uint64_t)n_voxels * 32), ST_THREADS, 0, st>>>(make_view(d), code, n_voxels, center[0], center[1],
                                                                              center[2], side, threshold, max_level, count, split);
}
void dvx_expand_launch(const uint64_t *code, uint32_t n_voxels, const uint32_t *offsets, uint64_t *out, cudaStream_t st) {
  DVX_COUNT_LAUNCH(1);
  expand_kernel<<<st_blocks(n_voxels), ST_THREADS, 0, st>>>(code, n_voxels, offsets, out);
}
void dvx_prune_flags_launch(const float *geo, uint32_t n_voxels, float threshold, uint32_t *keep, cudaStream_t st) {
  DVX_COUNT_LAUNCH(1);
  prune_flags_kernel<<<st_blocks(n_voxels), ST_THREADS, 0, st>>>(geo, n_voxels, threshold, keep);
}
void dvx_prune_scatter_launch(const uint64_t *code, uint32_t n_voxels, const uint32_t *offsets, uint64_t *code_out,
                              uint32_t *index_out, cudaStream_t st) {
  DVX_COUNT_LAUNCH(1);
  prune_scatter_kernel<<<st_blocks(n_voxels), ST_THREADS, 0, st>>>(code, n_voxels, offsets, code_out, index_out);
}

void dvx_split_counts_launch(const uint8_t *split, uint32_t n_voxels, uint32_t *count, cudaStream_t st) {
  if (n_voxels) { DVX_COUNT_LAUNCH(1); split_counts_kernel<<<(n_voxels + ST_THREADS - 1) / ST_THREADS, ST_THREADS, 0, st>>>(split, n_voxels, count); }
}
void dvx_subdivide_fill_launch(const uint32_t *offsets, uint32_t n_voxels, const float *geo_in, const float *sh_in, uint32_t sh_floats,
                               float *geo_out, float *sh_out, cudaStream_t st) {
  if (n_voxels) {
    DVX_COUNT_LAUNCH(1);
    subdivide_fill_kernel<<<(n_voxels + ST_THREADS - 1) / ST_THREADS, ST_THREADS, 0, st>>>(offsets, n_voxels, geo_in, sh_in, sh_floats, geo_out, sh_out);
  }
}
