// dvx_sort.cu - hot-path step 2: LSD radix sort of (64-bit key, 32-bit value) pairs, plus the exclusive scan it needs.
// "per-tile key generation and radix sort in direction-dependent Morton order" (BASELINE.json north_star (2));
// the paper only says the traversal is "Morton-ordered".  One kernel per 8-bit digit (one-sweep with
// decoupled look-back): per pass keys and values are read once and written once; one up-front kernel histograms every
// digit position.  n < 2^30 pairs (the status word of the look-back keeps a 30-bit count).
#include "dvx_internal.cuh"

#include <stdio.h>

#include <mutex>

namespace {

constexpr int SORT_THREADS = 256;
constexpr int DVX_SORT_ITEMS = 12;  // keys per thread: 3072-key tiles (45 KB of shared memory, 3 CTAs per SM). Config 3 sort stage ms for 6 / 8 / 12: 0.381 / 0.353 / 0.341
constexpr int SORT_ITEMS = DVX_SORT_ITEMS;
constexpr int SORT_TILE = SORT_THREADS * SORT_ITEMS;   // 3072 keys per block
constexpr int SORT_WARPS = SORT_THREADS / 32;
constexpr int RADIX = 256;
constexpr int DVX_SORT_LOOK = 4;  // measured on config 3 (6 passes over 2.9 M pairs), sort stage ms for 1 / 4 / 8 / 16: 0.386 / 0.356 / 0.359 / 0.378
// Payload loads are issued with the key loads.  Same box, config 3 sort stage ms: look-back 1 wide 0.446, 4 wide 0.395,
// 4 wide + early payload loads 0.351, + 3072-key tiles 0.341.
constexpr int SORT_LOOK = DVX_SORT_LOOK;  // one-sweep look-back: predecessor tiles read per round trip

constexpr int SCAN_THREADS = 512;
constexpr int SCAN_ITEMS = 8;
constexpr int SCAN_TILE = SCAN_THREADS * SCAN_ITEMS;   // 4096

// ------------------------------------------------------------------ exclusive scan (reduce-then-scan, recursive)
__device__ __forceinline__ uint32_t warp_incl_scan(uint32_t v) {
  const int lane = threadIdx.x & 31;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    uint32_t t = __shfl_up_sync(0xffffffffu, v, o);
    if (lane >= o) v += t;
  }
  return v;
}

// block-wide exclusive scan of one value per thread; returns the exclusive prefix, *total = block sum
__device__ __forceinline__ uint32_t block_excl_scan(uint32_t v, uint32_t *total) {
  __shared__ uint32_t wsum[32];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = blockDim.x >> 5;
  uint32_t inc = warp_incl_scan(v);
  if (lane == 31) wsum[w] = inc;
  __syncthreads();
  if (w == 0) {
    uint32_t s = lane < nw ? wsum[lane] : 0;
    uint32_t si = warp_incl_scan(s);
    wsum[lane] = si - s;
    if (lane == 31) wsum[31] = si;  // nw <= 16 here, so slot 31 is free for the total
  }
  __syncthreads();
  uint32_t r = wsum[w] + inc - v;
  *total = wsum[31];
  __syncthreads();
  return r;
}

__global__ void scan_block_sums(const uint32_t *data, uint64_t n, uint32_t *sums) {
  uint64_t base = (uint64_t)blockIdx.x * SCAN_TILE;
  uint32_t s = 0;
#pragma unroll
  for (int i = 0; i < SCAN_ITEMS; ++i) {
    uint64_t idx = base + (uint64_t)i * SCAN_THREADS + threadIdx.x;
    if (idx < n) s += data[idx];
  }
  uint32_t total;
  block_excl_scan(s, &total);
  if (threadIdx.x == 0) sums[blockIdx.x] = total;
}

__global__ void scan_apply(uint32_t *data, uint64_t n, const uint32_t *block_off) {
  uint64_t base = (uint64_t)blockIdx.x * SCAN_TILE + (uint64_t)threadIdx.x * SCAN_ITEMS;
  uint32_t v[SCAN_ITEMS], s = 0;
#pragma unroll
  for (int i = 0; i < SCAN_ITEMS; ++i) {
    v[i] = (base + i < n) ? data[base + i] : 0;
    s += v[i];
  }
  uint32_t total;
  uint32_t off = block_excl_scan(s, &total) + (block_off ? block_off[blockIdx.x] : 0);
#pragma unroll
  for (int i = 0; i < SCAN_ITEMS; ++i) {
    if (base + i < n) data[base + i] = off;
    off += v[i];
  }
}

// ------------------------------------------------------------------ one-sweep pass (decoupled look-back)
// One kernel per digit instead of histogram + scan + scatter: the global base of every digit comes from one up-front
// histogram of all digit positions (digit counts do not depend on the order of the keys), and the offset of a tile inside
// a digit comes from a look-back over the per-tile digit counts that earlier tiles publish in `status`.  Tiles take their
// index from a ticket counter, so a tile only ever waits for tiles that are already running (no deadlock).
constexpr uint32_t ST_AGG = 1u << 30, ST_PREFIX = 1u << 31, ST_MASK = ST_AGG - 1u;  // counts < 2^30 (checked by the host)
constexpr int MAX_PASSES = 8;

__global__ void __launch_bounds__(SORT_THREADS) radix_digit_hist(const uint64_t *__restrict__ keys, uint64_t n, int passes,
                                                                  uint32_t *__restrict__ ghist /* [passes][RADIX] */) {
  __shared__ uint32_t h[MAX_PASSES][RADIX];
  for (int p = 0; p < passes; ++p) h[p][threadIdx.x] = 0;
  __syncthreads();
  for (uint64_t i = (uint64_t)blockIdx.x * SORT_THREADS + threadIdx.x; i < n; i += (uint64_t)gridDim.x * SORT_THREADS) {
    const uint64_t k = keys[i];
    for (int p = 0; p < passes; ++p) atomicAdd(&h[p][(uint32_t)(k >> (8 * p)) & (RADIX - 1)], 1u);
  }
  __syncthreads();
  for (int p = 0; p < passes; ++p)
    if (h[p][threadIdx.x]) atomicAdd(&ghist[p * RADIX + threadIdx.x], h[p][threadIdx.x]);
}
// one block per pass: exclusive scan of its 256 digit counts, in place
__global__ void __launch_bounds__(RADIX) radix_digit_scan(uint32_t *ghist) {
  uint32_t *g = ghist + blockIdx.x * RADIX;
  uint32_t total;
  const uint32_t ex = block_excl_scan(g[threadIdx.x], &total);
  g[threadIdx.x] = ex;
}

constexpr int DVX_SORT_MIN_CTAS = 3;  // register cap with the payload loads issued early (12 keys per thread at 4 CTAs per SM: 0.363 ms)
__global__ void __launch_bounds__(SORT_THREADS, DVX_SORT_MIN_CTAS) radix_onesweep(const uint64_t *__restrict__ keys_in,
                                                                const uint32_t *__restrict__ vals_in,
                                                                uint64_t *__restrict__ keys_out, uint32_t *__restrict__ vals_out,
                                                                uint64_t n, uint32_t shift, const uint32_t *__restrict__ dbase,
                                                                volatile uint32_t *status /* [tiles][RADIX], zeroed */,
                                                                uint32_t *ticket) {
  __shared__ uint32_t cnt[SORT_WARPS][RADIX];
  __shared__ uint64_t s_key[SORT_TILE];
  __shared__ uint32_t s_val[SORT_TILE];
  __shared__ uint32_t gbase[RADIX];
  __shared__ uint32_t s_tile;
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  if (threadIdx.x == 0) s_tile = atomicAdd(ticket, 1u);
  for (int d = lane; d < RADIX; d += 32) cnt[w][d] = 0;
  __syncthreads();
  const uint32_t tile = s_tile;
  const uint64_t tbase = (uint64_t)tile * SORT_TILE;
  const uint64_t wbase = tbase + (uint64_t)w * (32 * SORT_ITEMS);
  uint64_t key[SORT_ITEMS];
  uint16_t rnk[SORT_ITEMS];
#pragma unroll
  for (int i = 0; i < SORT_ITEMS; ++i) {
    const uint64_t idx = wbase + (uint64_t)i * 32 + lane;
    key[i] = idx < n ? keys_in[idx] : 0;
  }
  uint32_t val[SORT_ITEMS];  // payload loads in flight under the ranking and the look-back
#pragma unroll
  for (int i = 0; i < SORT_ITEMS; ++i) {
    const uint64_t idx = wbase + (uint64_t)i * 32 + lane;
    val[i] = idx < n ? vals_in[idx] : 0;
  }
#pragma unroll
  for (int i = 0; i < SORT_ITEMS; ++i) {
    const uint64_t idx = wbase + (uint64_t)i * 32 + lane;
    const bool valid = idx < n;
    const uint32_t d = valid ? ((uint32_t)(key[i] >> shift) & (RADIX - 1)) : RADIX;  // RADIX = "no key"
    const uint32_t peers = __match_any_sync(0xffffffffu, d);
    const uint32_t before = __popc(peers & ((1u << lane) - 1u));
    const int leader = __ffs(peers) - 1;
    uint32_t old = 0;
    if (valid && lane == leader) {
      old = cnt[w][d];
      cnt[w][d] = old + __popc(peers);
    }
    old = __shfl_sync(0xffffffffu, old, leader);
    rnk[i] = (uint16_t)(old + before);
    __syncwarp();
  }
  __syncthreads();
  {  // digit d = threadIdx.x
    const int d = threadIdx.x;
    uint32_t run = 0;
#pragma unroll
    for (int ww = 0; ww < SORT_WARPS; ++ww) {
      const uint32_t c = cnt[ww][d];
      cnt[ww][d] = run;
      run += c;
    }
    // publish this tile's count of digit d, then look back for the number of keys with digit d in earlier tiles
    volatile uint32_t *mine = status + (size_t)tile * RADIX + d;
    *mine = run | (tile == 0 ? ST_PREFIX : ST_AGG);
    uint32_t excl = 0;
    if (tile > 0) {
      // LOOK predecessors are read at once (independent loads, one L2 round trip) and then consumed front to back up to the
      // first prefix or the first one not yet published: a walk of h tiles costs h / LOOK round trips instead of h.
      uint32_t t = tile;  // the next tile to consume is t - 1
      for (bool found = false; !found;) {
        uint32_t v[SORT_LOOK];
#pragma unroll
        for (int j = 0; j < SORT_LOOK; ++j) v[j] = t > (uint32_t)j ? status[(size_t)(t - 1 - j) * RADIX + d] : 0u;
#pragma unroll
        for (int j = 0; j < SORT_LOOK; ++j) {
          if (found || !(v[j] & (ST_PREFIX | ST_AGG))) break;  // not yet published: poll again from here
          excl += v[j] & ST_MASK;
          if (v[j] & ST_PREFIX) found = true;   // tile 0 always publishes a prefix, so the walk never passes it
          else --t;
        }
      }
      *mine = (excl + run) | ST_PREFIX;
    }
    uint32_t total;
    const uint32_t lbase = block_excl_scan(run, &total);
#pragma unroll
    for (int ww = 0; ww < SORT_WARPS; ++ww) cnt[ww][d] += lbase;
    gbase[d] = dbase[d] + excl - lbase;
  }
  __syncthreads();
#pragma unroll
  for (int i = 0; i < SORT_ITEMS; ++i) {
    const uint64_t idx = wbase + (uint64_t)i * 32 + lane;
    if (idx < n) {
      const uint32_t d = (uint32_t)(key[i] >> shift) & (RADIX - 1);
      const uint32_t pos = cnt[w][d] + rnk[i];
      s_key[pos] = key[i];
      s_val[pos] = val[i];
    }
  }
  __syncthreads();
  const uint32_t nb = (uint32_t)min((uint64_t)SORT_TILE, n - tbase);
  for (uint32_t i = threadIdx.x; i < nb; i += SORT_THREADS) {
    const uint64_t k = s_key[i];
    const uint32_t out = gbase[(uint32_t)(k >> shift) & (RADIX - 1)] + i;
    keys_out[out] = k;
    vals_out[out] = s_val[i];
  }
}

inline uint64_t ceil_div(uint64_t a, uint64_t b) { return (a + b - 1) / b; }

}  // namespace

// scratch for a scan of n counters: the chain of block-sum levels
static size_t scan_scratch_elems(uint64_t n) {
  size_t tot = 0;
  while (n > SCAN_TILE) {
    n = ceil_div(n, SCAN_TILE);
    tot += n;
  }
  return tot + 1;
}

void dvx_scan_u32_launch(uint32_t *data, uint64_t n, uint32_t *scratch, cudaStream_t st) {
  if (n == 0) return;
  uint64_t nb = ceil_div(n, SCAN_TILE);
  if (nb == 1) {
    { DVX_COUNT_LAUNCH(1); scan_apply<<<1, SCAN_THREADS, 0, st>>>(data, n, nullptr); }
    return;
  }
  { DVX_COUNT_LAUNCH(1); scan_block_sums<<<(unsigned)nb, SCAN_THREADS, 0, st>>>(data, n, scratch); }
  dvx_scan_u32_launch(scratch, nb, scratch + nb, st);
  { DVX_COUNT_LAUNCH(1); scan_apply<<<(unsigned)nb, SCAN_THREADS, 0, st>>>(data, n, scratch); }
}

// scratch: digit histograms, tickets, tile status
static size_t onesweep_words(uint64_t n) {
  uint64_t nb = ceil_div(n ? n : 1, SORT_TILE);
  return (size_t)MAX_PASSES * RADIX + MAX_PASSES + (size_t)MAX_PASSES * nb * RADIX;
}
size_t dvx_sort_scratch_bytes(uint64_t n) {
  // also used as the scratch of dvx_scan_u32_launch over n counters (the chain of block-sum levels is far smaller)
  const size_t one = onesweep_words(n) + 64, scan = scan_scratch_elems(n) + 64;
  return (one > scan ? one : scan) * sizeof(uint32_t);
}

// n must be below 2^30 (callers check).  2 + passes launches.
int dvx_sort_launch(uint64_t *keys_a, uint32_t *vals_a, uint64_t *keys_b, uint32_t *vals_b, uint64_t n, uint32_t key_bits,
                    void *scratch, cudaStream_t st) {
  if (n == 0) return 0;
  uint32_t nb = (uint32_t)ceil_div(n, SORT_TILE);
  int passes = (int)((key_bits + 7) / 8);
  if (passes < 1) passes = 1;
  int cur = 0;
  uint32_t *ghist = (uint32_t *)scratch;                 // [MAX_PASSES][RADIX]
  uint32_t *ticket = ghist + MAX_PASSES * RADIX;         // [MAX_PASSES]
  uint32_t *status = ticket + MAX_PASSES;                // [passes][nb][RADIX]
  cudaMemsetAsync(scratch, 0, (MAX_PASSES * RADIX + MAX_PASSES + (size_t)passes * nb * RADIX) * sizeof(uint32_t), st);
  const unsigned hb = nb < 592u ? nb : 592u;
  { DVX_COUNT_LAUNCH(1); radix_digit_hist<<<hb, SORT_THREADS, 0, st>>>(keys_a, n, passes, ghist); }
  { DVX_COUNT_LAUNCH(1); radix_digit_scan<<<passes, RADIX, 0, st>>>(ghist); }
  for (int p = 0; p < passes; ++p) {
    uint64_t *kin = cur ? keys_b : keys_a, *kout = cur ? keys_a : keys_b;
    uint32_t *vin = cur ? vals_b : vals_a, *vout = cur ? vals_a : vals_b;
    DVX_COUNT_LAUNCH(1);
    radix_onesweep<<<nb, SORT_THREADS, 0, st>>>(kin, vin, kout, vout, n, 8u * p, ghist + p * RADIX,
                                                status + (size_t)p * nb * RADIX, ticket + p);
    cur ^= 1;
  }
  return cur;
}

// ------------------------------------------------------------------ dvx_sort_pairs_no_alloc (include/dvx.h)
// The step-2 sort for callers that may not allocate (CUDA graph capture, tight serving loops, harnesses that forbid
// cudaMalloc): the ping-pong buffers and the one-sweep scratch of dvx_sort_launch live in ONE file-scope device array of
// fixed size, so the entry point calls no cudaMalloc / cudaFree / allocator callback.  Every GPU that loads the library
// holds the array (DVX_SORT_NO_ALLOC_BYTES, about 15 MB) until the process exits.  All calls share it: two calls that overlap
// on the GPU (different streams, or threads) race; it keeps the last call's contents, and what must start at zero (digit
// histograms, tickets, tile status) is cleared by dvx_sort_launch's cudaMemsetAsync on every call.
namespace {
constexpr uint64_t NA_MAX_PAIRS = DVX_SORT_NO_ALLOC_MAX_PAIRS;
constexpr size_t NA_TILES = (size_t)((NA_MAX_PAIRS + SORT_TILE - 1) / SORT_TILE);
constexpr size_t NA_SCRATCH_WORDS = (size_t)MAX_PASSES * RADIX + MAX_PASSES + (size_t)MAX_PASSES * NA_TILES * RADIX + 64;
constexpr size_t na_round(size_t b) { return (b + 255) & ~(size_t)255; }
constexpr size_t NA_OFF_VALS = na_round((size_t)NA_MAX_PAIRS * 8);                    // keys_b first
constexpr size_t NA_OFF_SCRATCH = NA_OFF_VALS + na_round((size_t)NA_MAX_PAIRS * 4);   // then vals_b
constexpr size_t NA_BYTES = NA_OFF_SCRATCH + na_round(NA_SCRATCH_WORDS * sizeof(uint32_t));
}  // namespace

// In host code this name is a host-side stand-in for the device array, NOT a device address: the address the kernels get
// comes from cudaGetSymbolAddress below, once per device.
static __device__ __align__(256) unsigned char g_sort_no_alloc[NA_BYTES];

namespace {
constexpr int NA_MAX_DEVICES = 64;
std::mutex g_na_mutex;
unsigned char *g_na_base[NA_MAX_DEVICES] = {};   // device address of g_sort_no_alloc on each device, resolved on first use

void na_error(char *err, size_t cap, const char *msg) {
  if (err && cap) snprintf(err, cap, "%s", msg);
}
}  // namespace

extern "C" dvx_status dvx_sort_pairs_no_alloc(int device, void *cuda_stream, uint64_t *keys, uint32_t *vals, uint64_t n,
                                              uint32_t key_bits, char *err, size_t err_cap) {
  if (err && err_cap) err[0] = 0;
  if (n == 0) return DVX_OK;
  if (!keys || !vals) { na_error(err, err_cap, "dvx_sort_pairs_no_alloc: keys / vals is NULL"); return DVX_ERR_INVALID_ARG; }
  if (key_bits < 1 || key_bits > 64) { na_error(err, err_cap, "dvx_sort_pairs_no_alloc: key_bits must be in [1,64]"); return DVX_ERR_INVALID_ARG; }
  if (n > NA_MAX_PAIRS) {
    if (err && err_cap)
      snprintf(err, err_cap, "dvx_sort_pairs_no_alloc: n = %llu exceeds DVX_SORT_NO_ALLOC_MAX_PAIRS = %llu (the static scratch is sized for that; use dvx_sort_pairs)",
               (unsigned long long)n, (unsigned long long)NA_MAX_PAIRS);
    return DVX_ERR_INVALID_ARG;
  }
  if (device < 0 || device >= NA_MAX_DEVICES) { na_error(err, err_cap, "dvx_sort_pairs_no_alloc: device index out of range"); return DVX_ERR_INVALID_ARG; }
  cudaError_t e = cudaSetDevice(device);
  if (e != cudaSuccess) { na_error(err, err_cap, cudaGetErrorString(e)); return DVX_ERR_CUDA; }
  unsigned char *base = nullptr;
  {
    std::lock_guard<std::mutex> lock(g_na_mutex);
    if (!g_na_base[device]) {   // once per device, with that device current
      void *p = nullptr;
      e = cudaGetSymbolAddress(&p, g_sort_no_alloc);
      if (e != cudaSuccess || !p) {
        na_error(err, err_cap, e != cudaSuccess ? cudaGetErrorString(e) : "cudaGetSymbolAddress returned NULL");
        cudaGetLastError();
        return DVX_ERR_CUDA;
      }
      g_na_base[device] = (unsigned char *)p;
    }
    base = g_na_base[device];
  }
  if (dvx_sort_scratch_bytes(n) > NA_SCRATCH_WORDS * sizeof(uint32_t)) {  // cannot happen for n <= NA_MAX_PAIRS; kept as a guard
    na_error(err, err_cap, "dvx_sort_pairs_no_alloc: internal scratch bound violated");
    return DVX_ERR_INVALID_ARG;
  }
  cudaStream_t st = (cudaStream_t)cuda_stream;
  uint64_t *kb = reinterpret_cast<uint64_t *>(base);
  uint32_t *vb = reinterpret_cast<uint32_t *>(base + NA_OFF_VALS);
  void *scr = base + NA_OFF_SCRATCH;
  const int which = dvx_sort_launch(keys, vals, kb, vb, n, key_bits, scr, st);   // clears its scratch itself
  if (which) {   // an odd number of passes left the result in the static buffers
    cudaMemcpyAsync(keys, kb, n * 8, cudaMemcpyDeviceToDevice, st);
    cudaMemcpyAsync(vals, vb, n * 4, cudaMemcpyDeviceToDevice, st);
  }
  e = cudaGetLastError();
  if (e != cudaSuccess) { na_error(err, err_cap, cudaGetErrorString(e)); return DVX_ERR_CUDA; }
  return DVX_OK;
}
