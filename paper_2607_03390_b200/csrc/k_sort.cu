// k_sort.cu -- A6: stable LSD radix sort of (uint32 key, uint32 value) pairs, onesweep style: one
// histogram kernel for all digits, then one scatter kernel per 8-bit digit in which every tile obtains its
// global offsets from its predecessors through decoupled look-back (a single pass over the data per
// digit: 8 B read + 8 B written per item).  The item count lives in device memory.
//
// The path sorts by tile|depth ("for each tile, sorts its intersected Gaussians by depth from
// front to back") in two levels that give exactly the order of one stable sort on the 64-bit key
// (tile << 32 | bits(depth)) with ties by ascending Gaussian index (R28):
//   (1) the N_v visible Gaussians are sorted by bits(depth) (4 digits, N_v items), then
//   (2) their (tile, Gaussian) pairs, emitted in that order, are sorted stably by tile id (ceil(log2 T / 8)
//       digits, P items).  At config 3 (P ~ 70 N_v) this moves ~40 B per pair instead of ~150 B.
#include "tgs_internal.cuh"

namespace {

constexpr int SORT_THREADS = 256;
constexpr int SORT_WARPS = SORT_THREADS / 32;
constexpr int SORT_IPT = 8;
constexpr int SORT_TILE = SORT_THREADS * SORT_IPT;   // 2048 pairs per tile
constexpr int SORT_CTAS_PER_SM = 5;
constexpr int LOOKBACK_BATCH = 4;                    // predecessor descriptors fetched per look-back step
constexpr int RADIX = 256;
constexpr uint32_t FLAG_AGG = 1u << 30, FLAG_PREFIX = 2u << 30, FLAG_MASK = 3u << 30, VALUE_MASK = ~FLAG_MASK;
constexpr uint32_t LOOKBACK_WATCHDOG = 1u << 26;

__device__ __forceinline__ uint32_t ld_volatile(const uint32_t* p) { return *reinterpret_cast<const volatile uint32_t*>(p); }
__device__ __forceinline__ void st_volatile(uint32_t* p, uint32_t v) { *reinterpret_cast<volatile uint32_t*>(p) = v; }

// ---- histogram of every digit + reset of the look-back descriptors of the tiles this frame will use
__global__ void __launch_bounds__(256) k_sort_hist(const uint32_t* __restrict__ keys, const uint32_t* __restrict__ n_ptr,
                                                   uint32_t* __restrict__ hist, uint32_t* __restrict__ desc, int passes,
                                                   uint32_t tiles_cap) {
  __shared__ uint32_t s_hist[4 * RADIX];
  const uint32_t n = *n_ptr;
  for (int i = threadIdx.x; i < passes * RADIX; i += blockDim.x) s_hist[i] = 0;
  __syncthreads();
  const uint32_t num_tiles = (n + SORT_TILE - 1) / SORT_TILE;
  for (uint32_t tile = blockIdx.x; tile < num_tiles; tile += gridDim.x) {
    for (int p = 0; p < passes; ++p) desc[((size_t)p * tiles_cap + tile) * RADIX + threadIdx.x] = 0;
    const uint32_t base = tile * SORT_TILE;
#pragma unroll 4
    for (int i = 0; i < SORT_IPT; ++i) {
      const uint32_t idx = base + i * 256 + threadIdx.x;
      if (idx < n) {
        const uint32_t k = keys[idx];
        for (int p = 0; p < passes; ++p) atomicAdd(&s_hist[p * RADIX + (uint32_t)((k >> (8 * p)) & 255u)], 1u);
      }
    }
  }
  __syncthreads();
  for (int i = threadIdx.x; i < passes * RADIX; i += blockDim.x)
    if (s_hist[i]) atomicAdd(&hist[i], s_hist[i]);
}

// ---- exclusive scan of each digit's 256-bin histogram (one CTA, one warp per digit)
__global__ void __launch_bounds__(256) k_sort_scan_hist(uint32_t* __restrict__ hist, int passes) {
  const uint32_t lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  if ((int)wid >= passes) return;
  uint32_t* h = hist + wid * RADIX;
  uint32_t run = 0;
  for (int c = 0; c < RADIX; c += 32) {
    const uint32_t v = h[c + lane];
    uint32_t incl = v;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) { const uint32_t o = __shfl_up_sync(0xffffffffu, incl, d); if (lane >= (uint32_t)d) incl += o; }
    h[c + lane] = run + incl - v;
    run += __shfl_sync(0xffffffffu, incl, 31);
  }
}

// ---- one digit: rank within the tile (warp match + per-warp counters), look-back, scatter through smem
struct SortSmem {
  uint32_t keys[SORT_TILE];
  uint32_t vals[SORT_TILE];
  uint32_t warp_hist[SORT_WARPS][RADIX];
  uint32_t gbase[RADIX];        // global index of block-sorted position p is gbase[digit] + p
  uint32_t scan_tmp[SORT_WARPS];
  uint32_t tile;
};

__global__ void __launch_bounds__(SORT_THREADS, SORT_CTAS_PER_SM) k_onesweep(const uint32_t* __restrict__ keys_in, const uint32_t* __restrict__ vals_in,
                                                           uint32_t* __restrict__ keys_out, uint32_t* __restrict__ vals_out,
                                                           const uint32_t* __restrict__ n_ptr, uint32_t* __restrict__ ticket,
                                                           uint32_t* __restrict__ error_flag, const uint32_t* __restrict__ hist_scan,
                                                           uint32_t* __restrict__ desc, int pass) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  SortSmem& sm = *reinterpret_cast<SortSmem*>(smem_raw);
  const uint32_t n = *n_ptr;
  const uint32_t num_tiles = (n + SORT_TILE - 1) / SORT_TILE;
  const uint32_t lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  const uint32_t lt_mask = (1u << lane) - 1u;
  const int shift = 8 * pass;
  while (true) {
    if (threadIdx.x == 0) sm.tile = atomicAdd(ticket, 1u);
    __syncthreads();
    const uint32_t tile = sm.tile;
    if (tile >= num_tiles) break;
    for (int i = threadIdx.x; i < SORT_WARPS * RADIX; i += SORT_THREADS) (&sm.warp_hist[0][0])[i] = 0;
    const uint32_t base = tile * SORT_TILE + wid * (32 * SORT_IPT);
    uint32_t key[SORT_IPT];
#pragma unroll
    for (int i = 0; i < SORT_IPT; ++i) {
      const uint32_t idx = base + i * 32 + lane;
      key[i] = idx < n ? keys_in[idx] : 0xffffffffu;     // padding sorts (stably) behind every real key of the tile
    }
    __syncthreads();
    uint32_t rank[SORT_IPT];
#pragma unroll
    for (int i = 0; i < SORT_IPT; ++i) {
      const uint32_t d = (uint32_t)(key[i] >> shift) & 255u;
      const uint32_t m = __match_any_sync(0xffffffffu, d);
      const uint32_t prev = sm.warp_hist[wid][d];
      __syncwarp();
      if ((m & lt_mask) == 0) sm.warp_hist[wid][d] = prev + __popc(m);
      __syncwarp();
      rank[i] = prev + __popc(m & lt_mask);
    }
    __syncthreads();
    // per digit (thread d): exclusive offsets of the warps, tile count
    const uint32_t d = threadIdx.x;
    uint32_t cnt = 0;
#pragma unroll
    for (int w = 0; w < SORT_WARPS; ++w) { const uint32_t t = sm.warp_hist[w][d]; sm.warp_hist[w][d] = cnt; cnt += t; }
    // exclusive scan of cnt over the 256 digits
    uint32_t incl = cnt;
#pragma unroll
    for (int s = 1; s < 32; s <<= 1) { const uint32_t o = __shfl_up_sync(0xffffffffu, incl, s); if (lane >= (uint32_t)s) incl += o; }
    if (lane == 31) sm.scan_tmp[wid] = incl;
    __syncthreads();
    uint32_t loff = incl - cnt;
#pragma unroll
    for (int w = 0; w < SORT_WARPS; ++w) if ((uint32_t)w < wid) loff += sm.scan_tmp[w];
    // decoupled look-back, one digit per thread (descriptor rows are 1 KB, read coalesced)
    uint32_t* my = desc + (size_t)tile * RADIX + d;
    uint32_t excl = 0;
    if (tile > 0) {
      st_volatile(my, FLAG_AGG | cnt);
      uint32_t polls = 0;
      int t = (int)tile - 1;
      bool done = false;
      while (!done) {                       // LOOKBACK_BATCH independent loads in flight per step instead of one
        uint32_t v[LOOKBACK_BATCH];
#pragma unroll
        for (int i = 0; i < LOOKBACK_BATCH; ++i) v[i] = (t - i >= 0) ? ld_volatile(desc + (size_t)(t - i) * RADIX + d) : FLAG_PREFIX;
#pragma unroll
        for (int i = 0; i < LOOKBACK_BATCH; ++i) {
          if (done) break;
          if ((v[i] & FLAG_MASK) == 0) { if (++polls > LOOKBACK_WATCHDOG) { *error_flag = 2; done = true; } break; }   // not ready: poll again from here
          excl += v[i] & VALUE_MASK;
          --t;
          if ((v[i] & FLAG_MASK) == FLAG_PREFIX) done = true;
        }
      }
    }
    st_volatile(my, FLAG_PREFIX | (excl + cnt));
    sm.gbase[d] = hist_scan[d] + excl - loff;
    // stash loff where the scatter can read it: add it to every warp's exclusive offset
#pragma unroll
    for (int w = 0; w < SORT_WARPS; ++w) sm.warp_hist[w][d] += loff;
    __syncthreads();
    // block-sorted positions; keys through smem
#pragma unroll
    for (int i = 0; i < SORT_IPT; ++i) {
      const uint32_t dg = (uint32_t)(key[i] >> shift) & 255u;
      rank[i] += sm.warp_hist[wid][dg];
      sm.keys[rank[i]] = key[i];
    }
#pragma unroll
    for (int i = 0; i < SORT_IPT; ++i) {
      const uint32_t idx = base + i * 32 + lane;
      if (idx < n) sm.vals[rank[i]] = vals_in[idx];
    }
    __syncthreads();
    const uint32_t valid = min((uint32_t)SORT_TILE, n - tile * SORT_TILE);
#pragma unroll 4
    for (int i = 0; i < SORT_IPT; ++i) {
      const uint32_t p = i * SORT_THREADS + threadIdx.x;
      if (p < valid) {
        const uint32_t k = sm.keys[p];
        const uint32_t o = sm.gbase[(uint32_t)(k >> shift) & 255u] + p;
        keys_out[o] = k;
        vals_out[o] = sm.vals[p];
      }
    }
    __syncthreads();
  }
}

}  // namespace

uint32_t sort_tile_items() { return SORT_TILE; }

int tile_sort_passes(int n_tiles) {
  int tile_bits = 1;
  while ((1 << tile_bits) < n_tiles) ++tile_bits;
  return (tile_bits + 7) / 8;
}

// Sorts n = *n_ptr items on digits [0, passes) of the key.  keys/vals are ping-pong pairs; returns the index
// (0/1) of the buffers holding the result.  `tickets` points at `passes` zeroed counters, `hist` at 4*256 words.
int launch_sort(cudaStream_t s, uint32_t* const keys[2], uint32_t* const vals[2], const uint32_t* n_ptr, int passes,
                uint32_t* hist, uint32_t* desc, uint32_t tiles_cap, uint32_t* tickets, uint32_t* error_flag, int num_sms) {
  static bool attr_set = false;
  if (!attr_set) {
    cudaFuncSetAttribute(k_onesweep, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(SortSmem));
    attr_set = true;
  }
  cudaMemsetAsync(hist, 0, 4 * RADIX * sizeof(uint32_t), s);
  k_sort_hist<<<num_sms * 4, 256, 0, s>>>(keys[0], n_ptr, hist, desc, passes, tiles_cap);
  k_sort_scan_hist<<<1, 256, 0, s>>>(hist, passes);
  int cur = 0;
  for (int p = 0; p < passes; ++p) {
    k_onesweep<<<num_sms * SORT_CTAS_PER_SM, SORT_THREADS, sizeof(SortSmem), s>>>(keys[cur], vals[cur], keys[cur ^ 1], vals[cur ^ 1], n_ptr, tickets + p,
                                                                   error_flag, hist + p * RADIX, desc + (size_t)p * tiles_cap * RADIX, p);
    cur ^= 1;
  }
  return cur;
}
