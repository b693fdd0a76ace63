// k_bin.cu -- integer work around the sort (A5, A7): compaction of the Gaussians that emit pairs,
// pair offsets (single-pass scan with decoupled look-back) fused with the (tile, Gaussian) pair emission
// in depth order, per-tile ranges, and the reconstruction of the 64-bit tile|depth keys for the tests.
// PAPER.md:L61 ("Gaussians that intersect with multiple tiles are duplicated ... sorts its intersected
// Gaussians by depth from front to back"), L123 (only Gaussians intersecting T_selected are sorted).
//
// Problem sizes that are not known on the host (number of emitting Gaussians, number of pairs P) are read
// from device memory; the kernels run as persistent grids pulling work tickets, so a frame needs no host
// round trip.
#include "tgs_internal.cuh"
#include "decide_math.cuh"   // this file is compiled with -fmad=false: k_emit repeats k_count_color's tile test

namespace {

constexpr uint32_t LOOKBACK_WATCHDOG = 1u << 26;   // polls before a look-back gives up and flags an error

__device__ __forceinline__ unsigned long long ld_volatile64(const unsigned long long* p) {
  return *reinterpret_cast<const volatile unsigned long long*>(p);
}
__device__ __forceinline__ void st_volatile64(unsigned long long* p, unsigned long long v) {
  *reinterpret_cast<volatile unsigned long long*>(p) = v;
}

constexpr int SCAN_THREADS = 256;
constexpr int SCAN_IPT = 4;
constexpr int SCAN_TILE = SCAN_THREADS * SCAN_IPT;   // items per tile

// Block-wide exclusive scan of per-thread sums + decoupled look-back across tiles.
// Returns the exclusive prefix of this thread's first item; *incl_total = inclusive prefix of the tile.
__device__ __forceinline__ uint32_t tile_scan(uint32_t tsum, uint32_t tile, unsigned long long* __restrict__ desc,
                                              uint32_t* s_warp, uint32_t* s_excl, uint32_t* error_flag, uint32_t* incl_total) {
  const uint32_t lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  uint32_t incl = tsum;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) { const uint32_t o = __shfl_up_sync(0xffffffffu, incl, d); if (lane >= (uint32_t)d) incl += o; }
  if (lane == 31) s_warp[wid] = incl;
  __syncthreads();
  uint32_t wbase = 0, total = 0;
#pragma unroll
  for (int w = 0; w < SCAN_THREADS / 32; ++w) { const uint32_t t = s_warp[w]; if ((uint32_t)w < wid) wbase += t; total += t; }
  if (wid == 0) {   // warp-parallel decoupled look-back: 32 predecessor descriptors per step
    uint32_t excl = 0;
    if (tile > 0) {
      if (lane == 0) st_volatile64(&desc[tile], (1ull << 32) | total);   // aggregate available
      int base = (int)tile - 1;
      uint32_t polls = 0;
      while (true) {
        const int t = base - (int)lane;
        const unsigned long long d = t >= 0 ? ld_volatile64(&desc[t]) : (2ull << 32);   // "prefix 0" before tile 0
        const uint32_t st = (uint32_t)(d >> 32);
        const uint32_t ready = __ballot_sync(0xffffffffu, st != 0), pref = __ballot_sync(0xffffffffu, st == 2);
        const int first = pref ? __ffs(pref) - 1 : 31;
        const uint32_t span = first == 31 ? 0xffffffffu : ((2u << first) - 1u);         // lanes 0..first
        if ((ready & span) != span) { if (++polls > LOOKBACK_WATCHDOG) { if (lane == 0) *error_flag = 1; break; } continue; }
        excl += __reduce_add_sync(0xffffffffu, (int)lane <= first ? (uint32_t)d : 0u);
        if (pref) break;
        base -= 32;
      }
    }
    if (lane == 0) {
      st_volatile64(&desc[tile], (2ull << 32) | (excl + total));       // inclusive prefix available
      *s_excl = excl;
    }
  }
  __syncthreads();
  *incl_total = *s_excl + total;
  return *s_excl + wbase + (incl - tsum);
}

// ================================================================== A5a: compaction
// Gaussians with tiles_touched > 0, in ascending index order: ckeys = bits(depth), cvals = index.
__global__ void __launch_bounds__(SCAN_THREADS) k_compact(uint32_t n, const uint32_t* __restrict__ tiles_touched,
                                                          const float4* __restrict__ rec_uvdo, unsigned long long* __restrict__ desc,
                                                          uint32_t* __restrict__ ckeys, uint32_t* __restrict__ cvals,
                                                          Counters* __restrict__ counters) {
  __shared__ uint32_t s_tile, s_warp[SCAN_THREADS / 32], s_excl;
  const uint32_t num_tiles = (n + SCAN_TILE - 1) / SCAN_TILE;
  while (true) {
    __syncthreads();
    if (threadIdx.x == 0) s_tile = atomicAdd(&counters->ticket_compact, 1u);
    __syncthreads();
    const uint32_t tile = s_tile;
    if (tile >= num_tiles) break;
    const uint32_t g0 = tile * SCAN_TILE + threadIdx.x * SCAN_IPT;
    uint32_t c[SCAN_IPT];
    if (g0 + SCAN_IPT <= n) {
      const uint4 v = *reinterpret_cast<const uint4*>(tiles_touched + g0);
      c[0] = v.x; c[1] = v.y; c[2] = v.z; c[3] = v.w;
    } else {
#pragma unroll
      for (int i = 0; i < SCAN_IPT; ++i) c[i] = (g0 + i < n) ? tiles_touched[g0 + i] : 0u;
    }
    const uint32_t tsum = (c[0] != 0) + (c[1] != 0) + (c[2] != 0) + (c[3] != 0);
    uint32_t incl_total;
    uint32_t off = tile_scan(tsum, tile, desc, s_warp, &s_excl, &counters->error, &incl_total);
    if (tile == num_tiles - 1 && threadIdx.x == 0) counters->n_emit = incl_total;
#pragma unroll
    for (int i = 0; i < SCAN_IPT; ++i)
      if (c[i]) { ckeys[off] = __float_as_uint(rec_uvdo[g0 + i].z); cvals[off] = g0 + i; ++off; }
  }
}

// ================================================================== A5b: offsets + pair emission in depth order
// items = the emitting Gaussians in depth order (sorted_g); the pair lists of consecutive items are
// consecutive, so after the stable sort by tile every tile's list is in (depth, index) order.
__global__ void __launch_bounds__(SCAN_THREADS) k_scan_offsets(FrameConst fc, const uint32_t* __restrict__ sorted_g,
                                                               const uint32_t* __restrict__ tiles_touched,
                                                               unsigned long long* __restrict__ desc, uint32_t* __restrict__ offsets,
                                                               Counters* __restrict__ counters) {
  __shared__ uint32_t s_tile, s_warp[SCAN_THREADS / 32], s_excl;
  const uint32_t n = counters->n_emit;
  const uint32_t num_tiles = (n + SCAN_TILE - 1) / SCAN_TILE;
  if (n == 0) { if (blockIdx.x == 0 && threadIdx.x == 0) counters->n_pairs = 0; return; }
  while (true) {
    __syncthreads();
    if (threadIdx.x == 0) s_tile = atomicAdd(&counters->ticket_scan, 1u);
    __syncthreads();
    const uint32_t tile = s_tile;
    if (tile >= num_tiles) break;
    const uint32_t i0 = tile * SCAN_TILE + threadIdx.x * SCAN_IPT;
    uint32_t c[SCAN_IPT];
#pragma unroll
    for (int i = 0; i < SCAN_IPT; ++i) c[i] = (i0 + i < n) ? tiles_touched[sorted_g[i0 + i]] : 0u;
    const uint32_t tsum = c[0] + c[1] + c[2] + c[3];
    uint32_t incl_total;
    uint32_t off = tile_scan(tsum, tile, desc, s_warp, &s_excl, &counters->error, &incl_total);
    if (tile == num_tiles - 1 && threadIdx.x == 0) {
      if (incl_total > fc.max_pairs) { counters->overflow = 1; counters->n_pairs = 0; }
      else counters->n_pairs = incl_total;
    }
#pragma unroll
    for (int i = 0; i < SCAN_IPT; ++i) { if (i0 + i < n) offsets[i0 + i] = off; off += c[i]; }
  }
}

// One warp per emitting Gaussian, items dealt round-robin to the warps of the grid: in depth order the nearest
// Gaussians -- the ones covering hundreds or thousands of tiles -- are neighbours, and this spreads them over all SMs.
// Pairs are written in the oracle's order (ty ascending, then tx) at offsets[i].
__global__ void __launch_bounds__(256) k_emit(FrameConst fc, const uint32_t* __restrict__ sorted_g, const uint32_t* __restrict__ offsets,
                                              const uint2* __restrict__ rec_rect, const float4* __restrict__ rec_uvdo,
                                              const float4* __restrict__ rec_conic, const uint32_t* __restrict__ sel_bits,
                                              uint32_t* __restrict__ keys, uint32_t* __restrict__ vals,
                                              const Counters* __restrict__ counters) {
  if (counters->overflow) return;
  const uint32_t n = counters->n_emit;
  const uint32_t lane = threadIdx.x & 31;
  const uint32_t nwarps = gridDim.x * (blockDim.x >> 5);
  for (uint32_t i = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5); i < n; i += nwarps) {
    const uint32_t g = sorted_g[i];
    uint32_t off = offsets[i];
    const uint2 r = rec_rect[g];
    const uint32_t x_lo = r.x & 0xffffu, x_hi = r.x >> 16, y_lo = r.y & 0xffffu, y_hi = r.y >> 16;
    const uint32_t w = x_hi - x_lo, area = w * (y_hi - y_lo);
    float4 uv, cn;
    if (fc.exact_tiles) { uv = rec_uvdo[g]; cn = rec_conic[g]; }
    for (uint32_t base = 0; base < area; base += 32) {
      const uint32_t idx = base + lane;
      const uint32_t ry = idx / w, ty = y_lo + ry, tx = x_lo + (idx - ry * w);
      const uint32_t t = ty * fc.cam.TX + tx;
      bool sel = idx < area && (fc.all_tiles || ((sel_bits[t >> 5] >> (t & 31)) & 1u));
      if (sel && fc.exact_tiles) sel = tile_alpha_reach(uv.x, uv.y, cn.x, cn.y, cn.z, cn.w, tx, ty, fc.cam.W, fc.cam.H);   // R39
      const uint32_t bal = __ballot_sync(0xffffffffu, sel);
      if (sel) {
        const uint32_t p = off + __popc(bal & ((1u << lane) - 1u));
        keys[p] = t;
        vals[p] = g;
      }
      off += __popc(bal);
    }
  }
}

// ================================================================== A7: per-tile ranges
__global__ void __launch_bounds__(256) k_ranges(const uint32_t* __restrict__ keys, const Counters* __restrict__ counters,
                                                uint2* __restrict__ ranges, int n_tiles) {
  const uint32_t n = counters->n_pairs;
  for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
    const uint32_t t = keys[i];
    if (t >= (uint32_t)n_tiles) continue;
    if (i == 0) ranges[t].x = 0;
    else {
      const uint32_t p = keys[i - 1];
      if (p != t) { ranges[t].x = i; if (p < (uint32_t)n_tiles) ranges[p].y = i; }
    }
    if (i == n - 1) ranges[t].y = n;
  }
}

// test-only: the 64-bit sort keys tile << 32 | bits(depth) of the sorted pair list
__global__ void __launch_bounds__(256) k_keys64(const uint32_t* __restrict__ keys, const uint32_t* __restrict__ vals,
                                                const float4* __restrict__ rec_uvdo, uint32_t n, uint64_t* __restrict__ out) {
  const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) out[i] = ((uint64_t)keys[i] << 32) | __float_as_uint(rec_uvdo[vals[i]].z);
}

}  // namespace

uint32_t scan_tile_items() { return SCAN_TILE; }

void launch_compact(cudaStream_t s, const FrameConst& fc, DevBuffers& b, int num_sms) {
  const uint32_t num_tiles = (fc.n + SCAN_TILE - 1) / SCAN_TILE;
  cudaMemsetAsync(b.scan_desc, 0, (size_t)(num_tiles + 1) * sizeof(uint64_t), s);
  const uint32_t grid = num_tiles < (uint32_t)(num_sms * 4) ? num_tiles : (uint32_t)(num_sms * 4);
  k_compact<<<grid ? grid : 1, SCAN_THREADS, 0, s>>>(fc.n, b.tiles_touched, b.rec_uvdo, (unsigned long long*)b.scan_desc, b.ckeys[0],
                                                    b.cvals[0], b.counters);
}

void launch_scan_emit(cudaStream_t s, const FrameConst& fc, DevBuffers& b, int sorted_g_idx, int num_sms) {
  const uint32_t num_tiles = (fc.n + SCAN_TILE - 1) / SCAN_TILE;   // upper bound (n_emit <= N)
  cudaMemsetAsync(b.scan_desc, 0, (size_t)(num_tiles + 1) * sizeof(uint64_t), s);
  const uint32_t grid = num_tiles < (uint32_t)(num_sms * 4) ? num_tiles : (uint32_t)(num_sms * 4);
  k_scan_offsets<<<grid ? grid : 1, SCAN_THREADS, 0, s>>>(fc, b.cvals[sorted_g_idx], b.tiles_touched, (unsigned long long*)b.scan_desc,
                                                         b.offsets, b.counters);
  k_emit<<<num_sms * 8, 256, 0, s>>>(fc, b.cvals[sorted_g_idx], b.offsets, b.rec_rect, b.rec_uvdo, b.rec_conic, b.sel_bits, b.keys[0], b.vals[0], b.counters);
}

void launch_ranges(cudaStream_t s, const FrameConst& fc, DevBuffers& b, int sorted_idx, int num_sms) {
  cudaMemsetAsync(b.ranges, 0, (size_t)fc.n_tiles * sizeof(uint2), s);
  k_ranges<<<num_sms * 8, 256, 0, s>>>(b.keys[sorted_idx], b.counters, b.ranges, fc.n_tiles);
}

void launch_keys64(cudaStream_t s, DevBuffers& b, int sorted_idx, uint32_t n, uint64_t* out) {
  if (n) k_keys64<<<(n + 255) / 256, 256, 0, s>>>(b.keys[sorted_idx], b.vals[sorted_idx], b.rec_uvdo, n, out);
}
