// dvx_grid.cu - widening row N2: shared grid-point corner densities and the optimizer step.
//
// The rasterizer reads a [V][8] corner record per voxel; training optimises ONE raw density per lattice
// point that neighbouring voxels share (reading R23).  Three tables tie the two views together, built once per leaf set
// like the step-0 rank tables:  point_of[V][8] (corner slot -> grid point),  slots[8V] + offsets[G+1] (grid point ->
// its corner slots, CSR).  They fall out of ONE radix sort of the 8V corner keys (51-bit Morton key of the corner's
// level-16 lattice coordinate): runs of equal keys are the grid points, and the sorted payload is the CSR slot list.
//
// The optimizer step (reading R24: Adam) is one kernel per parameter array and is purely HBM-bound:
//   grid_adam_kernel : thread = grid point.  GATHERS its <= 8 corner gradients (fixed order, so the step is
//                      deterministic and needs no atomics), Adam, writes the new density back into every corner slot of
//                      the [V][8] record the next forward reads, and zeroes the gradients it consumed.
//   adam_kernel      : plain elementwise Adam + gradient zeroing for the SH coefficients (float4 lanes).
// Keeping dL/dgeo as the [V][8] accumulation target of the backward pass (two 16-byte reductions per voxel run) and
// summing per grid point here, once per step, replaces the scatter-add "fused into the backward atomics" that SURVEY.md
// sketches: 8 scalar reductions per run would quadruple the reduction instructions of a kernel that is issue-bound.
#include "dvx_internal.cuh"

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

__global__ void __launch_bounds__(GRID_THREADS) grid_adam_kernel(AdamConst h, const uint32_t *__restrict__ offsets,
                                                                 const uint32_t *__restrict__ slots, uint32_t n_points,
                                                                 float *__restrict__ density, float *__restrict__ m,
                                                                 float *__restrict__ v, float *__restrict__ dgeo,
                                                                 float *__restrict__ geo) {
  const uint32_t p = blockIdx.x * GRID_THREADS + threadIdx.x;
  if (p >= n_points) return;
  const uint32_t b = offsets[p], e = offsets[p + 1];
  uint32_t sl[8];
  float gs[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    sl[i] = b + i < e ? __ldg(slots + b + i) : 0xFFFFFFFFu;
  }
#pragma unroll
  for (int i = 0; i < 8; ++i) gs[i] = sl[i] != 0xFFFFFFFFu ? dgeo[sl[i]] : 0.f;  // all eight loads in flight together
  float g = 0.f;
#pragma unroll
  for (int i = 0; i < 8; ++i) g += gs[i];  // ascending slot order: deterministic
  float pv = density[p], mv = m[p], vv = v[p];
  adam_update(h, g, pv, mv, vv);
  density[p] = pv;
  m[p] = mv;
  v[p] = vv;
#pragma unroll
  for (int i = 0; i < 8; ++i)
    if (sl[i] != 0xFFFFFFFFu) {
      geo[sl[i]] = pv;
      dgeo[sl[i]] = 0.f;
    }
}

// elementwise Adam over n floats, float4 lanes + scalar tail; zeroes the gradient
__global__ void __launch_bounds__(GRID_THREADS) adam_kernel(AdamConst h, uint64_t n, float *__restrict__ p,
                                                            float *__restrict__ m, float *__restrict__ v,
                                                            float *__restrict__ g) {
  const uint64_t n4 = n >> 2;
  const uint64_t stride = (uint64_t)gridDim.x * GRID_THREADS;
  for (uint64_t i = (uint64_t)blockIdx.x * GRID_THREADS + threadIdx.x; i < n4; i += stride) {
    float4 gp = reinterpret_cast<float4 *>(g)[i];
    float4 pp = reinterpret_cast<float4 *>(p)[i];
    float4 mp = reinterpret_cast<float4 *>(m)[i];
    float4 vp = reinterpret_cast<float4 *>(v)[i];
    adam_update(h, gp.x, pp.x, mp.x, vp.x);
    adam_update(h, gp.y, pp.y, mp.y, vp.y);
    adam_update(h, gp.z, pp.z, mp.z, vp.z);
    adam_update(h, gp.w, pp.w, mp.w, vp.w);
    reinterpret_cast<float4 *>(p)[i] = pp;
    reinterpret_cast<float4 *>(m)[i] = mp;
    reinterpret_cast<float4 *>(v)[i] = vp;
    reinterpret_cast<float4 *>(g)[i] = make_float4(0.f, 0.f, 0.f, 0.f);
  }
  const uint64_t t = (n4 << 2) + (uint64_t)blockIdx.x * GRID_THREADS + threadIdx.x;
  if (t < n) {
    float pv = p[t], mv = m[t], vv = v[t];
    adam_update(h, g[t], pv, mv, vv);
    p[t] = pv;
    m[t] = mv;
    v[t] = vv;
    g[t] = 0.f;
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
void dvx_grid_adam_launch(float lr, float beta1, float beta2, float eps, uint32_t step, const uint32_t *offsets,
                          const uint32_t *slots, uint32_t n_points, float *density, float *m, float *v, float *dgeo,
                          float *geo, cudaStream_t st) {
  DVX_COUNT_LAUNCH(1);
  grid_adam_kernel<<<blocks_for(n_points), GRID_THREADS, 0, st>>>(adam_const(lr, beta1, beta2, eps, step), offsets, slots,
                                                                 n_points, density, m, v, dgeo, geo);
}
void dvx_adam_launch(float lr, float beta1, float beta2, float eps, uint32_t step, uint64_t n, float *p, float *m, float *v,
                     float *g, cudaStream_t st) {
  // grid-stride over float4 lanes; 148 SMs x 8 resident blocks of 256 threads
  uint64_t want = ((n >> 2) + GRID_THREADS - 1) / GRID_THREADS;
  if (want < 1) want = 1;
  const uint64_t cap = 148ull * 8ull * 4ull;
  DVX_COUNT_LAUNCH(1);
  adam_kernel<<<(unsigned)(want < cap ? want : cap), GRID_THREADS, 0, st>>>(adam_const(lr, beta1, beta2, eps, step), n, p, m,
                                                                           v, g);
}
