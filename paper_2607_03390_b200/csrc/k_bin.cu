// k_bin.cu -- integer work of the path: A5 pair offsets (single-pass scan with decoupled look-back)
// fused with tile|depth key emission, A6 onesweep-style LSD radix sort (one histogram pass + one
// scatter pass per 8-bit digit, decoupled look-back between tiles), A7 per-tile ranges.
// PAPER.md:L61 ("Gaussians that intersect with multiple tiles are duplicated ... sorts its intersected
// Gaussians by depth from front to back"), L123 (only Gaussians intersecting T_selected are sorted).
//
// Every kernel here takes its problem size (N is host-known, P = number of pairs is not) from device
// memory and runs as a persistent grid that pulls work tickets, so a frame needs no host round trip.
#include "tgs_internal.cuh"

namespace {

constexpr uint32_t LOOKBACK_WATCHDOG = 1u << 26;   // polls before a look-back gives up and flags an error

__device__ __forceinline__ unsigned long long ld_volatile64(const unsigned long long* p) {
  return *reinterpret_cast<const volatile unsigned long long*>(p);
}

// ================================================================== A5: scan + key emission
constexpr int SCAN_THREADS = 256;
constexpr int SCAN_IPT = 4;
constexpr int SCAN_TILE = SCAN_THREADS * SCAN_IPT;   // Gaussians per tile
constexpr uint32_t BIG_SPLAT = 48;                   // pairs above which a Gaussian is emitted by a whole warp

// emits the pairs of one Gaussian, in the oracle's order (ty ascending, then tx), by one warp
__device__ __forceinline__ void emit_warp(const FrameConst& fc, uint32_t g, uint32_t off, const uint2 r, uint32_t dbits,
                                          const uint32_t* __restrict__ sel_bits, uint64_t* __restrict__ keys,
                                          uint32_t* __restrict__ vals, uint32_t lane) {
  const uint32_t x_lo = r.x & 0xffffu, x_hi = r.x >> 16, y_lo = r.y & 0xffffu, y_hi = r.y >> 16;
  for (uint32_t ty = y_lo; ty < y_hi; ++ty)
    for (uint32_t tx0 = x_lo; tx0 < x_hi; tx0 += 32) {
      const uint32_t tx = tx0 + lane;
      const uint32_t t = ty * fc.cam.TX + tx;
      const bool sel = tx < x_hi && (fc.all_tiles || ((sel_bits[t >> 5] >> (t & 31)) & 1u));
      const uint32_t bal = __ballot_sync(0xffffffffu, sel);
      if (sel) {
        const uint32_t p = off + __popc(bal & ((1u << lane) - 1u));
        keys[p] = ((uint64_t)t << 32) | dbits;
        vals[p] = g;
      }
      off += __popc(bal);
    }
}

__global__ void __launch_bounds__(SCAN_THREADS) k_scan_emit(FrameConst fc, const uint32_t* __restrict__ tiles_touched,
                                                            const uint2* __restrict__ rec_rect, const float4* __restrict__ rec_uvdo,
                                                            const uint32_t* __restrict__ sel_bits, unsigned long long* __restrict__ desc,
                                                            uint32_t* __restrict__ offsets, uint64_t* __restrict__ keys,
                                                            uint32_t* __restrict__ vals, Counters* __restrict__ counters) {
  __shared__ uint32_t s_tile, s_warp[SCAN_THREADS / 32], s_excl, s_nbig;
  __shared__ uint2 s_big[SCAN_TILE];
  const uint32_t lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  const uint32_t num_tiles = (fc.n + SCAN_TILE - 1) / SCAN_TILE;
  while (true) {
    if (threadIdx.x == 0) { s_tile = atomicAdd(&counters->ticket_scan, 1u); s_nbig = 0; }
    __syncthreads();
    const uint32_t tile = s_tile;
    if (tile >= num_tiles) break;
    const uint32_t g0 = tile * SCAN_TILE + threadIdx.x * SCAN_IPT;
    uint32_t c[SCAN_IPT];
    if (g0 + SCAN_IPT <= fc.n) {
      const uint4 v = *reinterpret_cast<const uint4*>(tiles_touched + g0);
      c[0] = v.x; c[1] = v.y; c[2] = v.z; c[3] = v.w;
    } else {
#pragma unroll
      for (int i = 0; i < SCAN_IPT; ++i) c[i] = (g0 + i < fc.n) ? tiles_touched[g0 + i] : 0u;
    }
    const uint32_t tsum = c[0] + c[1] + c[2] + c[3];
    uint32_t incl = tsum;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) { const uint32_t o = __shfl_up_sync(0xffffffffu, incl, d); if (lane >= (uint32_t)d) incl += o; }
    if (lane == 31) s_warp[wid] = incl;
    __syncthreads();
    uint32_t wbase = 0, total = 0;
#pragma unroll
    for (int w = 0; w < SCAN_THREADS / 32; ++w) { const uint32_t t = s_warp[w]; if ((uint32_t)w < wid) wbase += t; total += t; }
    // decoupled look-back over the previous tiles (thread 0)
    if (threadIdx.x == 0) {
      uint32_t excl = 0;
      if (tile > 0) {
        *reinterpret_cast<volatile unsigned long long*>(&desc[tile]) = (1ull << 32) | total;   // aggregate available
        __threadfence();
        uint32_t polls = 0;
        for (int t = (int)tile - 1; t >= 0;) {
          const unsigned long long d = ld_volatile64(&desc[t]);
          const uint32_t st = (uint32_t)(d >> 32);
          if (st == 0) { if (++polls > LOOKBACK_WATCHDOG) { counters->error = 1; break; } continue; }
          excl += (uint32_t)d;
          if (st == 2) break;
          --t;
        }
      }
      *reinterpret_cast<volatile unsigned long long*>(&desc[tile]) = (2ull << 32) | (excl + total);   // inclusive prefix available
      s_excl = excl;
      if (tile == num_tiles - 1) {
        const uint32_t P = excl + total;
        if (P > fc.max_pairs) { counters->overflow = 1; counters->n_pairs = 0; }
        else counters->n_pairs = P;
      }
    }
    __syncthreads();
    uint32_t off = s_excl + wbase + (incl - tsum);
#pragma unroll
    for (int i = 0; i < SCAN_IPT; ++i) {
      const uint32_t g = g0 + i;
      if (g < fc.n) offsets[g] = off;
      if (c[i]) {
        if ((unsigned long long)off + c[i] <= fc.max_pairs) {
          if (c[i] >= BIG_SPLAT) s_big[atomicAdd(&s_nbig, 1u)] = make_uint2(g, off);
          else {
            const uint2 r = rec_rect[g];
            const uint32_t dbits = __float_as_uint(rec_uvdo[g].z);
            const uint32_t x_lo = r.x & 0xffffu, x_hi = r.x >> 16, y_lo = r.y & 0xffffu, y_hi = r.y >> 16;
            uint32_t p = off;
            for (uint32_t ty = y_lo; ty < y_hi; ++ty)
              for (uint32_t tx = x_lo; tx < x_hi; ++tx) {
                const uint32_t t = ty * fc.cam.TX + tx;
                if (fc.all_tiles || ((sel_bits[t >> 5] >> (t & 31)) & 1u)) { keys[p] = ((uint64_t)t << 32) | dbits; vals[p] = g; ++p; }
              }
          }
        }
        off += c[i];
      }
    }
    __syncthreads();
    const uint32_t nbig = s_nbig;
    for (uint32_t j = wid; j < nbig; j += SCAN_THREADS / 32) {
      const uint2 e = s_big[j];
      emit_warp(fc, e.x, e.y, rec_rect[e.x], __float_as_uint(rec_uvdo[e.x].z), sel_bits, keys, vals, lane);
    }
    __syncthreads();
  }
}

// ================================================================== A7: per-tile ranges
__global__ void __launch_bounds__(256) k_ranges(const uint64_t* __restrict__ keys, const Counters* __restrict__ counters,
                                                uint2* __restrict__ ranges, int n_tiles) {
  const uint32_t n = counters->n_pairs;
  for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
    const uint32_t t = (uint32_t)(keys[i] >> 32);
    if (t >= (uint32_t)n_tiles) continue;
    if (i == 0) ranges[t].x = 0;
    else {
      const uint32_t p = (uint32_t)(keys[i - 1] >> 32);
      if (p != t) { ranges[t].x = i; if (p < (uint32_t)n_tiles) ranges[p].y = i; }
    }
    if (i == n - 1) ranges[t].y = n;
  }
}

}  // namespace

uint32_t scan_tile_items() { return SCAN_TILE; }

void launch_scan_emit(cudaStream_t s, const FrameConst& fc, DevBuffers& b, int num_sms) {
  const uint32_t num_tiles = (fc.n + SCAN_TILE - 1) / SCAN_TILE;
  cudaMemsetAsync(b.scan_desc, 0, (size_t)num_tiles * sizeof(uint64_t), s);
  const uint32_t grid = num_tiles < (uint32_t)(num_sms * 4) ? num_tiles : (uint32_t)(num_sms * 4);
  k_scan_emit<<<grid ? grid : 1, SCAN_THREADS, 0, s>>>(fc, b.tiles_touched, b.rec_rect, b.rec_uvdo, b.sel_bits,
                                                      (unsigned long long*)b.scan_desc, b.offsets, b.keys[0], b.vals[0], b.counters);
}

void launch_ranges(cudaStream_t s, const FrameConst& fc, DevBuffers& b, int sorted_idx, int num_sms) {
  cudaMemsetAsync(b.ranges, 0, (size_t)fc.n_tiles * sizeof(uint2), s);
  k_ranges<<<num_sms * 8, 256, 0, s>>>(b.keys[sorted_idx], b.counters, b.ranges, fc.n_tiles);
}
