// scan.cuh -- single-pass prefix sums across the work chunks of a persistent grid: block-wide exclusive scan of
// per-thread sums + decoupled look-back over the chunks' descriptors, 32 predecessor descriptors per step.
// A descriptor is (epoch << 34 | state << 32 | value), state 1 = aggregate, 2 = inclusive prefix; `epoch` is the
// frame number, so descriptors written by earlier frames read as "not ready" and nothing is ever zeroed.
// Chunks must be handed out in ticket order (atomic counter), so that every predecessor of a chunk is held by a
// CTA that is already running.  NOT shared with oracle/.
#pragma once
#include <stdint.h>

namespace tgs_scan {

constexpr uint32_t LOOKBACK_WATCHDOG = 1u << 26;   // polls before a look-back gives up and flags an error

__device__ __forceinline__ unsigned long long ld_volatile64(const unsigned long long* p) {
  return *reinterpret_cast<const volatile unsigned long long*>(p);
}
__device__ __forceinline__ void st_volatile64(unsigned long long* p, unsigned long long v) {
  *reinterpret_cast<volatile unsigned long long*>(p) = v;
}

// Exclusive prefix over all earlier chunks of this chunk's `total` (call from warp 0, all 32 lanes).
// desc[chunk] is published as "aggregate" first and "inclusive prefix" at the end.
// publish = false: the caller has already published the aggregate with publish_aggregate (deferred look-back).
__device__ __forceinline__ void publish_aggregate(uint32_t total, uint32_t chunk, unsigned long long* __restrict__ desc, uint32_t epoch) {
  const unsigned long long tag = (unsigned long long)epoch << 34;
  st_volatile64(&desc[chunk], tag | ((chunk > 0 ? 1ull : 2ull) << 32) | total);      // chunk 0: its aggregate is its prefix
}

__device__ __forceinline__ uint32_t lookback_warp(uint32_t total, uint32_t chunk, unsigned long long* __restrict__ desc,
                                                  uint32_t* error_flag, uint32_t epoch, bool publish = true) {
  const unsigned long long tag = (unsigned long long)epoch << 34;
  const uint32_t lane = threadIdx.x & 31;
  uint32_t excl = 0;
  if (chunk > 0) {
    if (publish && lane == 0) st_volatile64(&desc[chunk], tag | (1ull << 32) | total);   // aggregate available
    int base = (int)chunk - 1;
    uint32_t polls = 0;
    while (true) {
      const int t = base - (int)lane;
      const unsigned long long d = t >= 0 ? ld_volatile64(&desc[t]) : (tag | (2ull << 32));   // "prefix 0" before chunk 0
      const uint32_t st = (d >> 34) == (unsigned long long)epoch ? (uint32_t)(d >> 32) & 3u : 0u;
      const uint32_t ready = __ballot_sync(0xffffffffu, st != 0), pref = __ballot_sync(0xffffffffu, st == 2);
      const int first = pref ? __ffs(pref) - 1 : 31;
      const uint32_t span = first == 31 ? 0xffffffffu : ((2u << first) - 1u);         // lanes 0..first
      if ((ready & span) != span) { if (++polls > LOOKBACK_WATCHDOG) { if (lane == 0) *error_flag = 1; break; } continue; }
      excl += __reduce_add_sync(0xffffffffu, (int)lane <= first ? (uint32_t)d : 0u);
      if (pref) break;
      base -= 32;
    }
  }
  if (lane == 0) st_volatile64(&desc[chunk], tag | (2ull << 32) | (excl + total));     // inclusive prefix available
  return excl;
}

// Block-wide exclusive scan of `tsum` (one value per thread, THREADS threads) + look-back across chunks.
// Returns the global exclusive prefix of this thread's value; *incl_total = inclusive prefix of the whole chunk.
// s_warp: THREADS/32 words, s_excl: 1 word of shared memory.  Contains two __syncthreads.
template <int THREADS>
__device__ __forceinline__ uint32_t chunk_scan(uint32_t tsum, uint32_t chunk, unsigned long long* __restrict__ desc, uint32_t* s_warp,
                                               uint32_t* s_excl, uint32_t* error_flag, uint32_t* incl_total, uint32_t epoch) {
  const uint32_t lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  uint32_t incl = tsum;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) { const uint32_t o = __shfl_up_sync(0xffffffffu, incl, d); if (lane >= (uint32_t)d) incl += o; }
  if (lane == 31) s_warp[wid] = incl;
  __syncthreads();
  uint32_t wbase = 0, total = 0;
#pragma unroll
  for (int w = 0; w < THREADS / 32; ++w) { const uint32_t t = s_warp[w]; if ((uint32_t)w < wid) wbase += t; total += t; }
  if (wid == 0) {
    const uint32_t excl = lookback_warp(total, chunk, desc, error_flag, epoch);
    if (lane == 0) *s_excl = excl;
  }
  __syncthreads();
  *incl_total = *s_excl + total;
  return *s_excl + wbase + (incl - tsum);
}

}  // namespace tgs_scan
