// dvx_grid.cu - widening row N2: shared grid-point corner densities and the optimizer step.
//
// The rasterizer reads a [V][8] corner record per voxel; training optimises ONE raw density per lattice
// point that neighbouring voxels share (reading R23).  Three tables tie the two views together, built once per leaf set
// like the step-0 rank tables:  point_of[V][8] (corner slot -> grid point),  slots[8V] + offsets[G+1] (grid point ->
// its corner slots, CSR).  They fall out of ONE radix sort of the 8V corner keys (51-bit Morton key of the corner's
// level-16 lattice coordinate): runs of equal keys are the grid points, and the sorted payload is the CSR slot list.
//
// The optimizer step (reading R24: Adam) is one kernel per parameter KIND (all octrees of a scene in one launch), HBM-bound:
//   grid_adam_kernel : thread = grid point.  GATHERS its <= 8 corner gradients (fixed order, so the step is
//                      deterministic and needs no atomics) and does the Adam update of its density.
//   grid_write_kernel: thread = voxel.  Rebuilds the [V][8] corner record the next forward reads from the grid-point
//                      densities (gathers from a mostly L2-resident array, two 16-byte stores) and zeroes the voxel's
//                      gradient record.  (One kernel doing both from the grid-point side - 16 scattered 4-byte stores per
//                      point - ran at 35 % of the HBM peak, 0.34 ms on config 3; the two passes take 0.20 ms, 58 %.)
//   adam_kernel      : plain elementwise Adam + gradient zeroing for the SH coefficients (float4 lanes).
// Keeping dL/dgeo as the [V][8] accumulation target of the backward pass (two 16-byte reductions per voxel run) and
// summing per grid point here, once per step, replaces the scatter-add "fused into the backward atomics" that SURVEY.md
// sketches: 8 scalar reductions per run would quadruple the reduction instructions of a kernel that is issue-bound.
#include "dvx_internal.cuh"

#include <cstring>

namespace {

constexpr int GRID_THREADS = 256;

__device__ __forceinline__ uint64_t compact3(uint64_t x) {  // every third bit -> low 21 bits
  x &= 0x1249249249249249ull;
  x = (x ^ (x >> 2)) & 0x10c30c30c30c30c3ull;
  x = (x ^ (x >> 4)) & 0x100f00f00f00f00full;
  x = (x ^ (x >> 8)) & 0x001f0000ff0000ffull;
  x = (x ^ (x >> 16)) & 0x001f00000000ffffull;
  x = (x ^ (x >> 32)) & 0x00000000001fffffull;
  return x;
}
__device__ __forceinline__ uint64_t spread3(uint64_t x) {  // low 21 bits -> every third bit
  x &= 0x1fffffull;
  x = (x | (x << 32)) & 0x001f00000000ffffull;
  x = (x | (x << 16)) & 0x001f0000ff0000ffull;
  x = (x | (x << 8)) & 0x100f00f00f00f00full;
  x = (x | (x << 4)) & 0x10c30c30c30c30c3ull;
  x = (x | (x << 2)) & 0x1249249249249249ull;
  return x;
}

// slot s = 8 v + c  ->  key = Morton51(lattice coordinate of corner c of voxel v), value = s
__global__ void __launch_bounds__(GRID_THREADS) corner_keys_kernel(const uint64_t *__restrict__ code, uint64_t n_slots,
                                                                   uint64_t *__restrict__ keys, uint32_t *__restrict__ vals) {
  const uint64_t s = (uint64_t)blockIdx.x * GRID_THREADS + threadIdx.x;
  if (s >= n_slots) return;
  const uint64_t cd = __ldg(code + (s >> 3));
  const uint32_t c = (uint32_t)s & 7u;
  const uint32_t level = (uint32_t)(cd >> 48) & 31u;
  const uint64_t path = cd & 0xFFFFFFFFFFFFull;  // left-aligned: already the level-16 Morton number of the min corner
  const uint64_t size = 1ull << (DVX_MAX_LEVEL - level);
  const uint64_t X = compact3(path >> 2) + ((c >> 2) & 1u) * size;
  const uint64_t Y = compact3(path >> 1) + ((c >> 1) & 1u) * size;
  const uint64_t Z = compact3(path) + (c & 1u) * size;
  keys[s] = (spread3(X) << 2) | (spread3(Y) << 1) | spread3(Z);
  vals[s] = (uint32_t)s;
}

__global__ void __launch_bounds__(GRID_THREADS) grid_heads_kernel(const uint64_t *__restrict__ skeys, uint64_t n,
                                                                  uint32_t *__restrict__ flag) {
  const uint64_t i = (uint64_t)blockIdx.x * GRID_THREADS + threadIdx.x;
  if (i >= n) return;
  flag[i] = (i == 0 || skeys[i] != skeys[i - 1]) ? 1u : 0u;
}

// excl = exclusive scan of the head flags.  n_points = excl[n-1] + head(n-1).
__global__ void grid_count_kernel(const uint64_t *__restrict__ skeys, const uint32_t *__restrict__ excl, uint64_t n,
                                  uint32_t *n_points) {
  const bool head = n == 1 || skeys[n - 1] != skeys[n - 2];
  *n_points = excl[n - 1] + (head ? 1u : 0u);
}

__global__ void __launch_bounds__(GRID_THREADS) grid_tables_kernel(const uint64_t *__restrict__ skeys,
                                                                   const uint32_t *__restrict__ svals,
                                                                   const uint32_t *__restrict__ excl, uint64_t n,
                                                                   uint32_t *__restrict__ point_of,
                                                                   uint32_t *__restrict__ offsets,
                                                                   uint32_t *__restrict__ slots) {
  const uint64_t i = (uint64_t)blockIdx.x * GRID_THREADS + threadIdx.x;
  if (i >= n) return;
  const bool head = i == 0 || skeys[i] != skeys[i - 1];
  const uint32_t p = excl[i] + (head ? 1u : 0u) - 1u;
  const uint32_t s = svals[i];
  point_of[s] = p;
  slots[i] = s;  // stable sort of ascending payloads: ascending within a run
  if (head) offsets[p] = (uint32_t)i;
  if (i == n - 1) offsets[p + 1] = (uint32_t)n;
}

__global__ void __launch_bounds__(GRID_THREADS) grid_gather_kernel(const float *__restrict__ density,
                                                                   const uint32_t *__restrict__ point_of, uint64_t n_slots,
                                                                   float *__restrict__ geo) {
  const uint64_t s = (uint64_t)blockIdx.x * GRID_THREADS + threadIdx.x;
  if (s >= n_slots) return;
  geo[s] = __ldg(density + point_of[s]);
}

__global__ void __launch_bounds__(GRID_THREADS) grid_reduce_kernel(const float *__restrict__ dgeo,
                                                                   const uint32_t *__restrict__ offsets,
                                                                   const uint32_t *__restrict__ slots, uint32_t n_points,
                                                                   float *__restrict__ ddensity) {
  const uint32_t p = blockIdx.x * GRID_THREADS + threadIdx.x;
  if (p >= n_points) return;
  const uint32_t b = offsets[p], e = offsets[p + 1];
  float g = 0.f;
  for (uint32_t i = b; i < e; ++i) g += __ldg(dgeo + slots[i]);
  ddensity[p] = g;
}

struct AdamConst {
  float b1, b2, omb1, omb2;  // beta, 1 - beta
  float step_size;           // lr / (1 - b1^t)
  float inv_sqrt_bc2;        // 1 / sqrt(1 - b2^t)
  float eps;
};

// Kingma & Ba, Algorithm 1:  p -= lr * mhat / (sqrt(vhat) + eps)  =  step_size * m / (sqrt(v) * inv_sqrt_bc2 + eps)
__device__ __forceinline__ void adam_update(const AdamConst &h, float g, float &p, float &m, float &v) {
  m = fmaf(h.b1, m, h.omb1 * g);
  v = fmaf(h.b2, v, h.omb2 * g * g);
  const float denom = fmaf(sqrtf(v), h.inv_sqrt_bc2, h.eps);
  p -= h.step_size * (m / denom);
}

// One launch serves up to ADAM_BATCH parameter arrays (the static octree and the actor octrees of a scene): a block finds
// its array by a short scan of the block prefix held in the kernel parameters.  Ten launches of a few hundred blocks each
// cost ten latency chains (9 us apiece measured); batched they hide inside the static octree's launch.
constexpr int ADAM_BATCH = 32;

struct GridAdamBatch {
  uint32_t block_start[ADAM_BATCH + 1];
  const uint32_t *offsets[ADAM_BATCH];
  const uint32_t *slots[ADAM_BATCH];
  float *density[ADAM_BATCH], *m[ADAM_BATCH], *v[ADAM_BATCH], *dgeo[ADAM_BATCH], *geo[ADAM_BATCH];
  uint32_t n_points[ADAM_BATCH];
  int n;
};
struct GridWriteBatch {   // second pass of the grid step: thread = voxel
  uint32_t block_start[ADAM_BATCH + 1];
  const uint32_t *point_of[ADAM_BATCH];
  const float *density[ADAM_BATCH];
  float *dgeo[ADAM_BATCH], *geo[ADAM_BATCH];
  uint32_t n_voxels[ADAM_BATCH];
  int n;
};

constexpr int DVX_GA_MINB = 8;  // 32 registers, 64 warps per SM: the kernel waits on scattered 4-byte accesses
__global__ void __launch_bounds__(GRID_THREADS, DVX_GA_MINB) grid_adam_kernel(const __grid_constant__ AdamConst h,
                                                                 const __grid_constant__ GridAdamBatch B) {
  int e = 0;
  while (e + 1 < B.n && blockIdx.x >= B.block_start[e + 1]) ++e;
  const uint32_t p = (blockIdx.x - B.block_start[e]) * GRID_THREADS + threadIdx.x;
  if (p >= B.n_points[e]) return;
  const uint32_t *__restrict__ offsets = B.offsets[e];
  const uint32_t *__restrict__ slots = B.slots[e];
  float *__restrict__ dgeo = B.dgeo[e];
  float *__restrict__ geo = B.geo[e];
  const uint32_t b = offsets[p], end = offsets[p + 1];
  uint32_t sl[8];
  float gs[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) sl[i] = b + i < end ? __ldg(slots + b + i) : 0xFFFFFFFFu;
#pragma unroll
  for (int i = 0; i < 8; ++i) gs[i] = sl[i] != 0xFFFFFFFFu ? dgeo[sl[i]] : 0.f;  // all eight loads in flight together
  float g = 0.f;
#pragma unroll
  for (int i = 0; i < 8; ++i) g += gs[i];  // ascending slot order: deterministic
  float pv = B.density[e][p], mv = B.m[e][p], vv = B.v[e][p];
  adam_update(h, g, pv, mv, vv);
  B.density[e][p] = pv;
  B.m[e][p] = mv;
  B.v[e][p] = vv;
}

// Second pass (thread = voxel): the 32-byte corner record the next forward reads is rebuilt from the grid-point densities
// (eight 4-byte gathers from an array that mostly sits in L2) and written with two 16-byte stores, and the voxel's gradient
// record is zeroed the same way - instead of 16 scattered 4-byte stores per grid point in the first pass.
__global__ void __launch_bounds__(GRID_THREADS) grid_write_kernel(const __grid_constant__ GridWriteBatch B) {
  int e = 0;
  while (e + 1 < B.n && blockIdx.x >= B.block_start[e + 1]) ++e;
  const uint32_t v = (blockIdx.x - B.block_start[e]) * GRID_THREADS + threadIdx.x;
  if (v >= B.n_voxels[e]) return;
  const uint4 *po = reinterpret_cast<const uint4 *>(B.point_of[e]) + 2 * (size_t)v;
  const uint4 a = __ldg(po), b = __ldg(po + 1);
  const float *__restrict__ d = B.density[e];
  const float4 g0 = make_float4(d[a.x], d[a.y], d[a.z], d[a.w]), g1 = make_float4(d[b.x], d[b.y], d[b.z], d[b.w]);
  float4 *go = reinterpret_cast<float4 *>(B.geo[e]) + 2 * (size_t)v;
  go[0] = g0; go[1] = g1;
  float4 *dg = reinterpret_cast<float4 *>(B.dgeo[e]) + 2 * (size_t)v;
  dg[0] = make_float4(0.f, 0.f, 0.f, 0.f); dg[1] = make_float4(0.f, 0.f, 0.f, 0.f);
}

// elementwise Adam: a block owns ADAM_CHUNK consecutive floats of one array (4 float4 per thread, 16 loads in flight),
// the last block of an array also its scalar tail; zeroes the gradient
constexpr int ADAM_V4 = 4;
constexpr int ADAM_CHUNK = GRID_THREADS * ADAM_V4 * 4;  // 4096 floats

struct AdamBatch {
  uint32_t block_start[ADAM_BATCH + 1];
  float *p[ADAM_BATCH], *m[ADAM_BATCH], *v[ADAM_BATCH], *g[ADAM_BATCH];
  uint64_t n[ADAM_BATCH];
  int count;
};

__global__ void __launch_bounds__(GRID_THREADS) adam_kernel(const __grid_constant__ AdamConst h,
                                                            const __grid_constant__ AdamBatch B) {
  int e = 0;
  while (e + 1 < B.count && blockIdx.x >= B.block_start[e + 1]) ++e;
  const uint64_t n = B.n[e], n4 = n >> 2;
  float4 *__restrict__ p4 = reinterpret_cast<float4 *>(B.p[e]);
  float4 *__restrict__ m4 = reinterpret_cast<float4 *>(B.m[e]);
  float4 *__restrict__ v4 = reinterpret_cast<float4 *>(B.v[e]);
  float4 *__restrict__ g4 = reinterpret_cast<float4 *>(B.g[e]);
  const uint64_t base = (uint64_t)(blockIdx.x - B.block_start[e]) * (GRID_THREADS * ADAM_V4) + threadIdx.x;
  float4 gp[ADAM_V4], pp[ADAM_V4], mp[ADAM_V4], vp[ADAM_V4];
#pragma unroll
  for (int k = 0; k < ADAM_V4; ++k) {
    const uint64_t i = base + (uint64_t)k * GRID_THREADS;
    if (i < n4) {
      gp[k] = g4[i];
      pp[k] = p4[i];
      mp[k] = m4[i];
      vp[k] = v4[i];
    }
  }
#pragma unroll
  for (int k = 0; k < ADAM_V4; ++k) {
    const uint64_t i = base + (uint64_t)k * GRID_THREADS;
    if (i < n4) {
      adam_update(h, gp[k].x, pp[k].x, mp[k].x, vp[k].x);
      adam_update(h, gp[k].y, pp[k].y, mp[k].y, vp[k].y);
      adam_update(h, gp[k].z, pp[k].z, mp[k].z, vp[k].z);
      adam_update(h, gp[k].w, pp[k].w, mp[k].w, vp[k].w);
      p4[i] = pp[k];
      m4[i] = mp[k];
      v4[i] = vp[k];
      g4[i] = make_float4(0.f, 0.f, 0.f, 0.f);
    }
  }
  if (blockIdx.x + 1 == B.block_start[e + 1]) {  // scalar tail (n mod 4 floats) by the array's last block
    const uint64_t t = (n4 << 2) + threadIdx.x;
    if (t < n) {
      float pv = B.p[e][t], mv = B.m[e][t], vv = B.v[e][t];
      adam_update(h, B.g[e][t], pv, mv, vv);
      B.p[e][t] = pv;
      B.m[e][t] = mv;
      B.v[e][t] = vv;
      B.g[e][t] = 0.f;
    }
  }
}

AdamConst adam_const(float lr, float beta1, float beta2, float eps, uint32_t step) {
  AdamConst h;
  h.b1 = beta1;
  h.b2 = beta2;
  h.omb1 = (float)(1.0 - (double)beta1);
  h.omb2 = (float)(1.0 - (double)beta2);
  h.step_size = (float)((double)lr / (1.0 - pow((double)beta1, (double)step)));
  h.inv_sqrt_bc2 = (float)(1.0 / sqrt(1.0 - pow((double)beta2, (double)step)));
  h.eps = eps;
  return h;
}

inline unsigned blocks_for(uint64_t n) { return (unsigned)((n + GRID_THREADS - 1) / GRID_THREADS); }

}  // namespace

void dvx_corner_keys_launch(const uint64_t *code, uint64_t n_slots, uint64_t *keys, uint32_t *vals, cudaStream_t st) {
  DVX_COUNT_LAUNCH(1);
  corner_keys_kernel<<<blocks_for(n_slots), GRID_THREADS, 0, st>>>(code, n_slots, keys, vals);
}
void dvx_grid_heads_launch(const uint64_t *skeys, uint64_t n, uint32_t *flag, cudaStream_t st) {
  DVX_COUNT_LAUNCH(1);
  grid_heads_kernel<<<blocks_for(n), GRID_THREADS, 0, st>>>(skeys, n, flag);
}
void dvx_grid_count_launch(const uint64_t *skeys, const uint32_t *excl, uint64_t n, uint32_t *n_points, cudaStream_t st) {
  DVX_COUNT_LAUNCH(1);
  grid_count_kernel<<<1, 1, 0, st>>>(skeys, excl, n, n_points);
}
void dvx_grid_tables_launch(const uint64_t *skeys, const uint32_t *svals, const uint32_t *excl, uint64_t n,
                            uint32_t *point_of, uint32_t *offsets, uint32_t *slots, cudaStream_t st) {
  DVX_COUNT_LAUNCH(1);
  grid_tables_kernel<<<blocks_for(n), GRID_THREADS, 0, st>>>(skeys, svals, excl, n, point_of, offsets, slots);
}
void dvx_grid_gather_launch(const float *density, const uint32_t *point_of, uint64_t n_slots, float *geo, cudaStream_t st) {
  DVX_COUNT_LAUNCH(1);
  grid_gather_kernel<<<blocks_for(n_slots), GRID_THREADS, 0, st>>>(density, point_of, n_slots, geo);
}
void dvx_grid_reduce_launch(const float *dgeo, const uint32_t *offsets, const uint32_t *slots, uint32_t n_points,
                            float *ddensity, cudaStream_t st) {
  DVX_COUNT_LAUNCH(1);
  grid_reduce_kernel<<<blocks_for(n_points), GRID_THREADS, 0, st>>>(dgeo, offsets, slots, n_points, ddensity);
}
void dvx_grid_adam_launch(float lr, float beta1, float beta2, float eps, uint32_t step, uint32_t n,
                          const DvxGridAdamItem *items, cudaStream_t st) {
  const AdamConst h = adam_const(lr, beta1, beta2, eps, step);
  for (uint32_t at = 0; at < n;) {
    GridAdamBatch B;
    memset(&B, 0, sizeof(B));
    uint32_t blocks = 0;
    const uint32_t first = at;
    while (at < n && B.n < ADAM_BATCH) {
      const DvxGridAdamItem &it = items[at++];
      if (it.n_points == 0) continue;
      const int e = B.n++;
      B.block_start[e] = blocks;
      blocks += blocks_for(it.n_points);
      B.offsets[e] = it.offsets; B.slots[e] = it.slots; B.n_points[e] = it.n_points;
      B.density[e] = it.density; B.m[e] = it.m; B.v[e] = it.v; B.dgeo[e] = it.dgeo; B.geo[e] = it.geo;
    }
    if (B.n == 0) continue;
    B.block_start[B.n] = blocks;
    DVX_COUNT_LAUNCH(1);
    grid_adam_kernel<<<blocks, GRID_THREADS, 0, st>>>(h, B);
    GridWriteBatch Wb;
    memset(&Wb, 0, sizeof(Wb));
    uint32_t wblocks = 0;
    for (uint32_t j = first; j < at; ++j) {
      const DvxGridAdamItem &it = items[j];
      if (it.n_points == 0 || it.n_voxels == 0) continue;
      const int e = Wb.n++;
      Wb.block_start[e] = wblocks;
      wblocks += blocks_for(it.n_voxels);
      Wb.point_of[e] = it.point_of; Wb.density[e] = it.density; Wb.dgeo[e] = it.dgeo; Wb.geo[e] = it.geo; Wb.n_voxels[e] = it.n_voxels;
    }
    Wb.block_start[Wb.n] = wblocks;
    if (wblocks) { DVX_COUNT_LAUNCH(1); grid_write_kernel<<<wblocks, GRID_THREADS, 0, st>>>(Wb); }
  }
}
void dvx_adam_launch(float lr, float beta1, float beta2, float eps, uint32_t step, uint32_t n, const DvxAdamItem *items,
                     cudaStream_t st) {
  const AdamConst h = adam_const(lr, beta1, beta2, eps, step);
  for (uint32_t at = 0; at < n;) {
    AdamBatch B;
    memset(&B, 0, sizeof(B));
    uint64_t blocks = 0;
    while (at < n && B.count < ADAM_BATCH) {
      const DvxAdamItem &it = items[at];
      if (it.n == 0) { ++at; continue; }
      const uint64_t nb = (it.n + ADAM_CHUNK - 1) / ADAM_CHUNK;
      if (blocks + nb > 0x7FFFFFFFull) break;  // grid.x limit: the rest goes into the next launch
      ++at;
      const int e = B.count++;
      B.block_start[e] = (uint32_t)blocks;
      blocks += nb;
      B.p[e] = it.p; B.m[e] = it.m; B.v[e] = it.v; B.g[e] = it.g; B.n[e] = it.n;
    }
    if (B.count == 0) break;  // a single array beyond 2^31 blocks (2^43 floats) is rejected by the caller
    B.block_start[B.count] = (uint32_t)blocks;
    DVX_COUNT_LAUNCH(1);
    adam_kernel<<<(unsigned)blocks, GRID_THREADS, 0, st>>>(h, B);
  }
}
