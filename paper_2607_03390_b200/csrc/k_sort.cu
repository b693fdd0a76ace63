// k_sort.cu -- A6: stable LSD radix sort of (uint32 key, uint32 value) pairs, onesweep style: one scatter kernel
// per 8-bit digit in which every tile obtains its global offsets from its predecessors through decoupled
// look-back (a single pass over the data per digit: 8 B read + 8 B written per item).  The item count lives in
// device memory.  The digit histograms are accumulated by the kernels that PRODUCE the keys (k_preprocess: depth
// bits of the visible Gaussians; k_bin: tile ids of the pairs), so a sort is nothing but its scatter passes.
//
// The path sorts by tile|depth ("for each tile, sorts its intersected Gaussians by depth from
// front to back") in two levels that give exactly the order of one stable sort on the 64-bit key
// (tile << 32 | bits(depth)) with ties by ascending Gaussian index (R28):
//   (1) the N_v visible Gaussians are sorted by bits(depth) (4 digits, N_v items), then
//   (2) their (tile, Gaussian) pairs, emitted in that order, are sorted stably by tile id (ceil(log2 T / 8)
//       digits, P items).  At config 3 (P ~ 25 N_v) this moves ~36 B per pair instead of ~150 B.
//
// Look-back descriptors are (epoch << 34 | flag << 32 | count): tagged with the frame number, never zeroed.
#include "tgs_internal.cuh"
#include "bin_params.cuh"
#include "scan.cuh"

namespace {

constexpr int SORT_THREADS = 256;
constexpr int SORT_WARPS = SORT_THREADS / 32;
constexpr int SORT_IPT_SMALL = 8;     // depth sort (N_v ~ 0.1-0.3 M): 2048-item tiles, more tiles in flight
constexpr int SORT_IPT_BIG = 16;      // tile sort (millions of pairs): 4096-pair tiles halve the per-tile overhead (scans, look-back): -7 %
constexpr int SORT_CTAS_PER_SM = 2;
constexpr int RADIX = 256;
constexpr unsigned long long FLAG_AGG = 1ull << 32, FLAG_PREFIX = 2ull << 32;
constexpr uint32_t LOOKBACK_WATCHDOG = 1u << 26;

__device__ __forceinline__ unsigned long long ld_volatile64(const unsigned long long* p) {
  return *reinterpret_cast<const volatile unsigned long long*>(p);
}
__device__ __forceinline__ void st_volatile64(unsigned long long* p, unsigned long long v) {
  *reinterpret_cast<volatile unsigned long long*>(p) = v;
}

template <int SORT_IPT>
struct SortSmem {
  uint32_t keys[SORT_THREADS * SORT_IPT];
  uint32_t vals[SORT_THREADS * SORT_IPT];
  uint32_t warp_hist[SORT_WARPS][RADIX];
  uint32_t gbase[RADIX];        // global index of block-sorted position p is gbase[digit] + p
  uint32_t hbase[RADIX];        // exclusive scan of the digit histogram of the whole input
  uint32_t scan_tmp[SORT_WARPS];
  uint32_t tile;
};

// one digit: rank within the tile (warp match + per-warp counters), look-back, scatter through smem
template <int LB_BATCH, int CTAS_PER_SM, int SORT_IPT>
__global__ void __launch_bounds__(SORT_THREADS, CTAS_PER_SM) k_onesweep(
    const uint32_t* __restrict__ keys_in, const uint32_t* __restrict__ vals_in, uint32_t* __restrict__ keys_out,
    uint32_t* __restrict__ vals_out, const uint32_t* __restrict__ n_ptr, uint32_t* __restrict__ ticket, uint32_t* __restrict__ error_flag,
    const uint32_t* __restrict__ hist, unsigned long long* __restrict__ desc, int shift, int nbits, uint32_t epoch,
    uint2* __restrict__ ranges) {
  TGS_PDL_WAIT();
  TGS_PDL_TRIGGER();
  constexpr int SORT_TILE = SORT_THREADS * SORT_IPT;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  SortSmem<SORT_IPT>& sm = *reinterpret_cast<SortSmem<SORT_IPT>*>(smem_raw);
  const uint32_t n = *n_ptr;
  const uint32_t num_tiles = (n + SORT_TILE - 1) / SORT_TILE;
  const uint32_t lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  const uint32_t lt_mask = (1u << lane) - 1u;
  const unsigned long long tag = (unsigned long long)epoch << 34;
  if (blockIdx.x >= num_tiles) return;
  {   // exclusive scan of this digit's 256-bin histogram (thread d = bin d)
    const uint32_t h = hist[threadIdx.x];
    uint32_t incl = h;
#pragma unroll
    for (int s = 1; s < 32; s <<= 1) { const uint32_t o = __shfl_up_sync(0xffffffffu, incl, s); if (lane >= (uint32_t)s) incl += o; }
    if (lane == 31) sm.scan_tmp[wid] = incl;
    __syncthreads();
    uint32_t off = incl - h;
#pragma unroll
    for (int w = 0; w < SORT_WARPS; ++w) if ((uint32_t)w < wid) off += sm.scan_tmp[w];
    sm.hbase[threadIdx.x] = off;
  }
  while (true) {
    __syncthreads();
    if (threadIdx.x == 0) sm.tile = atomicAdd(ticket, 1u);
    __syncthreads();
    const uint32_t tile = sm.tile;
    if (tile >= num_tiles) break;
    for (int i = threadIdx.x; i < SORT_WARPS * RADIX; i += SORT_THREADS) (&sm.warp_hist[0][0])[i] = 0;
    sm.gbase[threadIdx.x] = 0;                            // doubles as the tile's digit histogram until the look-back
    const uint32_t base = tile * SORT_TILE + wid * (32 * SORT_IPT);
    uint32_t key[SORT_IPT], val[SORT_IPT];
#pragma unroll
    for (int i = 0; i < SORT_IPT; ++i) {
      const uint32_t idx = base + i * 32 + lane;
      key[i] = idx < n ? keys_in[idx] : 0xffffffffu;     // padding sorts (stably) behind every real key of the tile
    }
#pragma unroll
    for (int i = 0; i < SORT_IPT; ++i) {                 // values: loaded now so that their latency overlaps the ranking
      const uint32_t idx = base + i * 32 + lane;
      val[i] = idx < n ? vals_in[idx] : 0u;
    }
    __syncthreads();
    // The tile's digit counts are published as its look-back AGGREGATE before the (long) ranking: by the time a
    // successor looks back, its predecessors' aggregates are there and nobody spins.
#pragma unroll
    for (int i = 0; i < SORT_IPT; ++i) atomicAdd(&sm.gbase[(uint32_t)(key[i] >> shift) & 255u], 1u);
    __syncthreads();
    unsigned long long* my = desc + (size_t)tile * RADIX + threadIdx.x;
    {
      uint32_t c = sm.gbase[threadIdx.x];
      if (threadIdx.x == 255u) c -= SORT_TILE - min((uint32_t)SORT_TILE, n - tile * SORT_TILE);   // padding keys all have digit 255
      if (tile > 0) st_volatile64(my, tag | FLAG_AGG | c);
    }
    uint32_t rank[SORT_IPT], mt[SORT_IPT];
#pragma unroll
    for (int i = 0; i < SORT_IPT; ++i) {      // lanes of the warp with the same digit, from one ballot per bit: match.any
      const uint32_t dg = (uint32_t)(key[i] >> shift) & 255u;   // costs a step per distinct value, and these digits are mostly distinct
      uint32_t m = 0xffffffffu;
      for (int bit = 0; bit < nbits; ++bit) {
        const bool on = (dg >> bit) & 1u;
        const uint32_t bal = __ballot_sync(0xffffffffu, on);
        m &= on ? bal : ~bal;
      }
      if (nbits < 8) {                     // padding keys (digit 255) must not join real keys whose low bits are all set
        const bool pad = dg >> nbits;
        const uint32_t bal = __ballot_sync(0xffffffffu, pad);
        m &= pad ? bal : ~bal;
      }
      mt[i] = m;
    }
#pragma unroll
    for (int i = 0; i < SORT_IPT; ++i) {
      const uint32_t d = (uint32_t)(key[i] >> shift) & 255u;
      const uint32_t m = mt[i];
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
    // decoupled look-back, one digit per thread (descriptor rows are 2 KB, read coalesced); 4 predecessors per step
    // at first, LB_BATCH per step when the chain is long (a small input starts all its tiles at once: nobody has a
    // prefix yet, so the instance used for the few visible Gaussians walks 32 at a time)
    uint32_t excl = 0;
    if (tile > 0) {
      uint32_t polls = 0;
      int t = (int)tile - 1;
      bool done = false;
      int batch = 4;
      while (!done) {
        unsigned long long v[LB_BATCH];
#pragma unroll
        for (int i = 0; i < LB_BATCH; ++i)
          if (i < batch) v[i] = (t - i >= 0) ? ld_volatile64(desc + (size_t)(t - i) * RADIX + d) : (tag | FLAG_PREFIX);
#pragma unroll
        for (int i = 0; i < LB_BATCH; ++i) {
          if (done || i >= batch) break;
          const bool mine = (v[i] >> 34) == (unsigned long long)epoch;
          const uint32_t fl = mine ? (uint32_t)(v[i] >> 32) & 3u : 0u;
          if (fl == 0) { __nanosleep(64); if (++polls > LOOKBACK_WATCHDOG) { *error_flag = 2; done = true; } break; }   // not ready: poll again from here
          excl += (uint32_t)v[i];
          --t;
          if (fl == 2) done = true;
        }
        batch = LB_BATCH;
      }
    }
    st_volatile64(my, tag | FLAG_PREFIX | (excl + cnt));
    sm.gbase[d] = sm.hbase[d] + excl - loff;
    // stash loff where the scatter can read it: add it to every warp's exclusive offset
#pragma unroll
    for (int w = 0; w < SORT_WARPS; ++w) sm.warp_hist[w][d] += loff;
    __syncthreads();
    // block-sorted positions through smem
#pragma unroll
    for (int i = 0; i < SORT_IPT; ++i) {
      const uint32_t dg = (uint32_t)(key[i] >> shift) & 255u;
      rank[i] += sm.warp_hist[wid][dg];
      sm.keys[rank[i]] = key[i];
      sm.vals[rank[i]] = val[i];
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
        if (ranges) {
          // A7 in the last pass (the keys are the tile ids, now fully sorted): ranges[t] = {~start, end}, zero = empty.
          // Inside a digit segment of this tile the neighbours in shared memory are the neighbours of the final list,
          // so a change of tile id is a boundary; at the ends of a segment the neighbour belongs to another tile of the
          // sort, so start / end are candidates combined by atomicMax (max of ~o = min of o).
          const uint32_t dg = (uint32_t)(k >> shift) & 255u;
          const uint32_t kp = p > 0 ? sm.keys[p - 1] : 0xffffffffu;
          const bool seg_first = p == 0 || ((uint32_t)(kp >> shift) & 255u) != dg;
          bool seg_last = p + 1 >= valid;
          if (!seg_last) seg_last = ((uint32_t)(sm.keys[p + 1] >> shift) & 255u) != dg;
          // every update is an atomicMax (a tile's range may be touched by several CTAs: no plain store ever meets an
          // atomic on the same word)
          if (seg_first) atomicMax(&ranges[k].x, ~o);
          else if (kp != k) { atomicMax(&ranges[k].x, ~o); atomicMax(&ranges[kp].y, o); }
          if (seg_last) atomicMax(&ranges[k].y, o + 1u);
        }
      }
    }
  }
}

}  // namespace

uint32_t sort_tile_items() { return SORT_THREADS * SORT_IPT_SMALL; }   // capacity of the descriptor arrays: the smaller tile

// Per-device function attributes (dynamic shared memory above 48 KB); tgs_create calls this for the context's device.
void sort_prepare_device() {
  cudaFuncSetAttribute(k_onesweep<4, SORT_CTAS_PER_SM, SORT_IPT_BIG>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(SortSmem<SORT_IPT_BIG>));
  cudaFuncSetAttribute(k_onesweep<32, 2, SORT_IPT_SMALL>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(SortSmem<SORT_IPT_SMALL>));
}

int tile_sort_passes(int n_tiles) {
  int tile_bits = 1;
  while ((1 << tile_bits) < n_tiles) ++tile_bits;
  return (tile_bits + 7) / 8;
}

// Sorts n = *n_ptr items on the low `key_bits` bits of the key, 8 bits per pass.  keys/vals are ping-pong pairs;
// returns the index (0/1) of the buffers holding the result.  `hist` = [passes][256] digit histograms of the keys
// (filled by the producer of the keys), `tickets` = one zeroed counter per pass, `desc` = [passes][tiles_cap][256].
int launch_sort(cudaStream_t s, uint32_t* const keys[2], uint32_t* const vals[2], const uint32_t* n_ptr, int key_bits,
                const uint32_t* hist, uint64_t* desc, uint32_t tiles_cap, uint32_t* tickets, uint32_t* error_flag, uint32_t epoch,
                int num_sms, bool small_input, uint2* ranges) {
  const int passes = (key_bits + 7) / 8;
  int cur = 0;
  for (int p = 0; p < passes; ++p) {
    const int nbits = key_bits - 8 * p < 8 ? key_bits - 8 * p : 8;
    unsigned long long* d = (unsigned long long*)desc + (size_t)p * tiles_cap * RADIX;
    if (small_input)
      TGS_LAUNCH((k_onesweep<32, 2, SORT_IPT_SMALL>), num_sms * 2, SORT_THREADS, sizeof(SortSmem<SORT_IPT_SMALL>), s, keys[cur], vals[cur], keys[cur ^ 1], vals[cur ^ 1], n_ptr, tickets + p,
                                                                           error_flag, hist + p * RADIX, d, 8 * p, nbits, epoch, p == passes - 1 ? ranges : (uint2*)nullptr);
    else
      TGS_LAUNCH((k_onesweep<4, SORT_CTAS_PER_SM, SORT_IPT_BIG>), num_sms * SORT_CTAS_PER_SM, SORT_THREADS, sizeof(SortSmem<SORT_IPT_BIG>), s, 
          keys[cur], vals[cur], keys[cur ^ 1], vals[cur ^ 1], n_ptr, tickets + p, error_flag, hist + p * RADIX, d, 8 * p, nbits, epoch, p == passes - 1 ? ranges : (uint2*)nullptr);
    cur ^= 1;
  }
  return cur;
}

// ------------------------------------------------------------------------------------------------------------------
// Depth sort of the visible Gaussians as ONE launch.  The four onesweep launches above spend 10-14 us
// each on ~140 co-resident tiles: a launch, a prologue and a look-back chain per digit for 2 MB of data.  Here one
// persistent grid of at most one CTA per SM keeps the four passes inside one kernel:
//  * tile t (2048 consecutive items of the current buffer) belongs to CTA t mod gridDim.x for all passes;
//  * the digit counts of every tile for pass p are the rows of a matrix H[p][tile][256] in global memory.  H[0] is filled
//    by k_compact_vis (it knows position and key of every item it writes); H[p + 1] is filled by the scatter of pass p,
//    which knows where each item lands (destination tile = position / 2048) and its next digit: one RED per item.
//    So a pass needs no counting phase of its own, and the offset of (tile, digit) is the digit's global base (the
//    histograms k_preprocess accumulates, as before) plus a column sum over the rows of the earlier tiles;
//  * between two passes all CTAs meet at a grid barrier (all CTAs are resident: the grid is not larger than the number
//    of SMs and nothing this kernel waits for comes from a later launch).  Rows of H[p] are cleared by their tile's CTA
//    after the barrier that ends pass p, so the matrices are all zero again when the kernel ends.
// Data written by other CTAs of this launch are read with ld.global.cg (no stale L1 lines, no non-coherent path).
// The result (buffer index 0, stable, ties in input order) is bit-identical to launch_sort's.
namespace {

constexpr int FUSED_IPT = SORT_IPT_SMALL;
constexpr int FUSED_TILE = SORT_THREADS * FUSED_IPT;
constexpr int FUSED_CTAS_PER_SM = 2;            // the grid: every CTA is resident (grid barriers)
constexpr uint32_t FUSED_MLP = 16;             // 16-byte loads in flight per thread in the column sums
constexpr uint32_t BARRIER_WATCHDOG = 1u << 22;

// Arrival is a release (the CTA's earlier writes, ordered before it by the bar.sync, are visible to whoever acquires the
// count), the poll an acquire: no separate fences.
__device__ __forceinline__ void grid_barrier(uint32_t* ctr, uint32_t expect, uint32_t* error_flag) {
  __syncthreads();
  if (threadIdx.x == 0) {
    asm volatile("red.release.gpu.global.add.u32 [%0], 1;" ::"l"(ctr) : "memory");
    uint32_t polls = 0, v;
    while (true) {
      asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(ctr) : "memory");
      if (v >= expect) break;
      if (++polls > BARRIER_WATCHDOG) { *error_flag = 3; break; }
    }
  }
  __syncthreads();
}

template <int CTAS_PER_SM>
__global__ void __launch_bounds__(SORT_THREADS, CTAS_PER_SM) k_depth_sort_fused(uint32_t* keys0, uint32_t* vals0, uint32_t* keys1, uint32_t* vals1,
                                                                      const uint32_t* __restrict__ hist, uint32_t* H, uint32_t tiles_cap, Counters* counters,
                                                                      int exact, uint32_t epoch, const float4* __restrict__ rec_bin,
                                                                      uint4* __restrict__ bin_params, uint32_t* __restrict__ area_prefix,
                                                                      uint32_t* __restrict__ chunk_first, unsigned long long* __restrict__ scan_desc,
                                                                      unsigned long long max_tests, volatile uint32_t* __restrict__ host_overflow) {
  TGS_PDL_WAIT();
  extern __shared__ __align__(16) unsigned char smem_raw[];
  SortSmem<FUSED_IPT>& sm = *reinterpret_cast<SortSmem<FUSED_IPT>*>(smem_raw);
  const uint32_t n = counters->n_visible;
  uint32_t* const barrier_ctr = &counters->ticket_sort[0];
  uint32_t* const error_flag = &counters->error;
  if (n == 0) {                                                 // uniform over the grid
    if (blockIdx.x == 0 && threadIdx.x == 0) { counters->n_tests = 0; counters->n_pairs = 0; }
    return;
  }
  const uint32_t num_tiles = (n + FUSED_TILE - 1) / FUSED_TILE;
  const uint32_t lane = threadIdx.x & 31, wid = threadIdx.x >> 5, d = threadIdx.x;
  const uint32_t lt_mask = (1u << lane) - 1u;
  constexpr uint32_t MLP = CTAS_PER_SM == 1 ? 20u : FUSED_MLP;   // 16-byte loads in flight per thread in the column sums (registers permitting)
  uint32_t hv[4];                                               // the four global digit histograms (thread d = bin d): one round trip, not four
#pragma unroll
  for (int p = 0; p < 4; ++p) hv[p] = hist[p * RADIX + d];
#pragma unroll 1
  for (int pass = 0; pass < 4; ++pass) {
    const int shift = 8 * pass;
    const uint32_t* kin = (pass & 1) ? keys1 : keys0;
    const uint32_t* vin = (pass & 1) ? vals1 : vals0;
    uint32_t* kout = (pass & 1) ? keys0 : keys1;
    uint32_t* vout = (pass & 1) ? vals0 : vals1;
    const uint32_t* Hp = H + (size_t)pass * tiles_cap * RADIX;
    uint32_t* Hn = pass < 3 ? H + (size_t)(pass + 1) * tiles_cap * RADIX : nullptr;
    {   // exclusive scan of this digit's global histogram (thread d = bin d)
      const uint32_t h = pass == 0 ? hv[0] : pass == 1 ? hv[1] : pass == 2 ? hv[2] : hv[3];
      uint32_t incl = h;
#pragma unroll
      for (int s = 1; s < 32; s <<= 1) { const uint32_t o = __shfl_up_sync(0xffffffffu, incl, s); if (lane >= (uint32_t)s) incl += o; }
      __syncthreads();
      if (lane == 31) sm.scan_tmp[wid] = incl;
      __syncthreads();
      uint32_t off = incl - h;
#pragma unroll
      for (int w = 0; w < SORT_WARPS; ++w) if ((uint32_t)w < wid) off += sm.scan_tmp[w];
      sm.hbase[d] = off;
    }
    for (uint32_t tile = blockIdx.x; tile < num_tiles; tile += gridDim.x) {
      __syncthreads();
      for (int i = threadIdx.x; i < SORT_WARPS * RADIX; i += SORT_THREADS) (&sm.warp_hist[0][0])[i] = 0;
      const uint32_t base = tile * FUSED_TILE + wid * (32 * FUSED_IPT);
      uint32_t key[FUSED_IPT], val[FUSED_IPT];
#pragma unroll
      for (int i = 0; i < FUSED_IPT; ++i) {
        const uint32_t idx = base + i * 32 + lane;
        key[i] = idx < n ? __ldcg(kin + idx) : 0xffffffffu;     // padding sorts (stably) behind every real key of the tile
      }
#pragma unroll
      for (int i = 0; i < FUSED_IPT; ++i) {
        const uint32_t idx = base + i * 32 + lane;
        val[i] = idx < n ? __ldcg(vin + idx) : 0u;
      }
      // Offset of (tile, digit) inside the digit = the counts of the earlier tiles: column sums over the first `tile` rows of
      // Hp.  64 threads cover a row with 16-byte loads, the four 64-thread groups take every fourth row, 16 loads in flight
      // per thread; the four partial sums per column meet in shared memory (sm.keys is free until the scatter).
      {
        const uint32_t q = threadIdx.x & 63u, r0 = threadIdx.x >> 6;
        uint4 acc = make_uint4(0u, 0u, 0u, 0u);
        const uint4* Hq = reinterpret_cast<const uint4*>(Hp) + q;
        for (uint32_t t0 = r0; t0 < tile; t0 += 4u * MLP) {
          uint4 v[MLP];
#pragma unroll
          for (uint32_t j = 0; j < MLP; ++j) { const uint32_t t = t0 + 4u * j; v[j] = t < tile ? __ldcg(Hq + (size_t)t * (RADIX / 4)) : make_uint4(0u, 0u, 0u, 0u); }
#pragma unroll
          for (uint32_t j = 0; j < MLP; ++j) { acc.x += v[j].x; acc.y += v[j].y; acc.z += v[j].z; acc.w += v[j].w; }
        }
        reinterpret_cast<uint4*>(sm.keys)[r0 * 64u + q] = acc;    // [4][256] partial column sums
      }
      __syncthreads();
      uint32_t rank[FUSED_IPT];
#pragma unroll
      for (int i = 0; i < FUSED_IPT; ++i) {
        const uint32_t dg = (uint32_t)(key[i] >> shift) & 255u;
        uint32_t m = 0xffffffffu;
#pragma unroll
        for (int bit = 0; bit < 8; ++bit) {
          const bool on = (dg >> bit) & 1u;
          const uint32_t bal = __ballot_sync(0xffffffffu, on);
          m &= on ? bal : ~bal;
        }
        const uint32_t prev = sm.warp_hist[wid][dg];
        __syncwarp();
        if ((m & lt_mask) == 0) sm.warp_hist[wid][dg] = prev + __popc(m);
        __syncwarp();
        rank[i] = prev + __popc(m & lt_mask);
      }
      __syncthreads();
      uint32_t cnt = 0;
#pragma unroll
      for (int w = 0; w < SORT_WARPS; ++w) { const uint32_t t = sm.warp_hist[w][d]; sm.warp_hist[w][d] = cnt; cnt += t; }
      uint32_t incl = cnt;
#pragma unroll
      for (int s = 1; s < 32; s <<= 1) { const uint32_t o = __shfl_up_sync(0xffffffffu, incl, s); if (lane >= (uint32_t)s) incl += o; }
      if (lane == 31) sm.scan_tmp[wid] = incl;
      __syncthreads();
      uint32_t loff = incl - cnt;
#pragma unroll
      for (int w = 0; w < SORT_WARPS; ++w) if ((uint32_t)w < wid) loff += sm.scan_tmp[w];
      const uint32_t col = sm.keys[d] + sm.keys[256 + d] + sm.keys[512 + d] + sm.keys[768 + d];
      sm.gbase[d] = sm.hbase[d] + col - loff;
#pragma unroll
      for (int w = 0; w < SORT_WARPS; ++w) sm.warp_hist[w][d] += loff;
      __syncthreads();
#pragma unroll
      for (int i = 0; i < FUSED_IPT; ++i) {
        const uint32_t dg = (uint32_t)(key[i] >> shift) & 255u;
        const uint32_t r = rank[i] + sm.warp_hist[wid][dg];
        sm.keys[r] = key[i];
        sm.vals[r] = val[i];
      }
      __syncthreads();
      const uint32_t valid = min((uint32_t)FUSED_TILE, n - tile * FUSED_TILE);
#pragma unroll 4
      for (int i = 0; i < FUSED_IPT; ++i) {
        const uint32_t p = i * SORT_THREADS + threadIdx.x;
        if (p < valid) {
          const uint32_t k = sm.keys[p];
          const uint32_t o = sm.gbase[(uint32_t)(k >> shift) & 255u] + p;
          kout[o] = k;
          vout[o] = sm.vals[p];
          if (Hn) atomicAdd(Hn + (size_t)(o / FUSED_TILE) * RADIX + ((k >> (shift + 8)) & 255u), 1u);
        }
      }
    }
    // the barrier after the last pass only protects H[3] (later tiles may still be summing its columns); a consumer of the
    // sorted list that lives in this kernel would need it anyway
    grid_barrier(barrier_ctr, (uint32_t)(pass + 1) * gridDim.x, error_flag);
    // nobody reads H[pass] any more: every CTA has summed its columns before it arrived
    for (uint32_t tile = blockIdx.x; tile < num_tiles; tile += gridDim.x) const_cast<uint32_t*>(Hp)[(size_t)tile * RADIX + d] = 0u;
  }
  // ---- A5a on the sorted list (what k_scan_area does in the multi-launch pipeline, k_bin.cu): the records k_bin reads, in
  // sorted order; area_prefix[i] = tests of the Gaussians before position i; chunk_first[k] = position of the Gaussian that
  // holds test k * BIN_CHUNK.  One tile = 8 consecutive positions per thread; the prefix across the tiles is a decoupled
  // look-back over one descriptor per tile (every tile is resident or finished).
  if (counters->area_sum > max_tests) {                         // the tests do not fit the binning's index space: frame invalid
    if (blockIdx.x == 0 && threadIdx.x == 0) { counters->n_tests = 0; counters->n_pairs = 0; counters->overflow = 1; *host_overflow = 1u; __threadfence_system(); }
    return;
  }
  // Only now may the next kernel of the stream (k_bin) be scheduled: its CTAs would otherwise sit in their
  // griddepcontrol.wait for this whole kernel and keep the kernels of the side streams (SH colours, T^oc, selection) off the SMs.
  TGS_PDL_TRIGGER();
  uint32_t* s_warp = sm.scan_tmp;
  uint32_t* s_excl = &sm.tile;
  for (uint32_t tile = blockIdx.x; tile < num_tiles; tile += gridDim.x) {
    __syncthreads();
    const uint32_t i0 = tile * FUSED_TILE + threadIdx.x * FUSED_IPT;
    // everything A5a needs of a Gaussian is one 32-byte record (rec_bin, k_preprocess): one sector per Gaussian, all eight
    // fetched together; positions behind the end of the list read record 0 and store nothing
    uint32_t g[FUSED_IPT], a[FUSED_IPT];
#pragma unroll
    for (int j = 0; j < FUSED_IPT; ++j) g[j] = i0 + j < n ? __ldcg(vals0 + i0 + j) : 0u;
    float4 r0[FUSED_IPT], r1[FUSED_IPT];
#pragma unroll
    for (int j = 0; j < FUSED_IPT; ++j) { r0[j] = rec_bin[2 * (size_t)g[j]]; r1[j] = rec_bin[2 * (size_t)g[j] + 1]; }
    uint32_t tsum = 0;
#pragma unroll
    for (int j = 0; j < FUSED_IPT; ++j) {
      const GaussParams P = make_params_bin(g[j], r0[j], r1[j], exact != 0, &a[j]);
      if (i0 + j < n) store_params(bin_params + 3 * (size_t)(i0 + j), P); else a[j] = 0u;
      tsum += a[j];
    }
    uint32_t incl_total;
    uint32_t off = tgs_scan::chunk_scan<SORT_THREADS>(tsum, tile, scan_desc, s_warp, s_excl, error_flag, &incl_total, epoch);
    if (tile == num_tiles - 1 && threadIdx.x == 0) { counters->n_tests = incl_total; area_prefix[n] = incl_total; }
#pragma unroll
    for (int j = 0; j < FUSED_IPT; ++j) {
      if (i0 + j >= n) break;
      area_prefix[i0 + j] = off;
      const unsigned long long end = (unsigned long long)off + a[j];
      for (unsigned long long kb = ((unsigned long long)off + BIN_CHUNK - 1) / BIN_CHUNK; kb * BIN_CHUNK < end; ++kb) chunk_first[kb] = i0 + j;
      off += a[j];
    }
  }
}

}  // namespace

uint32_t depth_sort_fused_tile_items() { return FUSED_TILE; }
uint32_t depth_sort_fused_ctas_per_sm() { return FUSED_CTAS_PER_SM; }
size_t depth_sort_fused_words(uint32_t tiles_cap) { return (size_t)4 * RADIX * (size_t)tiles_cap; }

// The depth sort (result in buffer 0, bit-identical to launch_sort(..., key_bits = 32)) and A5a (k_scan_area) as one launch.
// b.dsort_H = [4][tiles_cap][256] zeroed counters whose first matrix the producer of the list has filled (k_compact_vis).
void launch_depth_sort_fused(cudaStream_t s, const FrameConst& fc, DevBuffers& b, unsigned long long max_tests, uint32_t* host_overflow, int num_sms,
                             uint32_t n_hint) {
  // one CTA per SM while that gives every tile its own CTA: the second CTA of an SM only becomes resident when the kernels of
  // the side streams (SH colours) leave it the registers, and every CTA has to arrive at the barriers
  // (A cooperative launch, which would make the driver start the grid only when all of it fits, was tried: with
  // cudaLaunchAttributeCooperative the kernel read a visible count of zero on this driver, with or without the programmatic
  // launch attribute, so the plain launch stays.  Within a context nothing can keep these CTAs off the SMs for good; two
  // contexts rendering on one device at the same time could each hold part of the SMs -- the barrier's watchdog then flags
  // the frame (TGS_E_CUDA from tgs_get_stats) instead of hanging.  include/tgs.h says so.)
  const uint32_t tiles_hint = (n_hint + FUSED_TILE - 1) / FUSED_TILE + 2;     // a few tiles more only give a few CTAs a second tile
#define FUSED_LAUNCH(CPS)                                                                                                                                    \
  TGS_LAUNCH((k_depth_sort_fused<CPS>), num_sms * (CPS), SORT_THREADS, sizeof(SortSmem<FUSED_IPT>), s, b.ckeys[0], b.cvals[0], b.ckeys[1], b.cvals[1],              \
             (const uint32_t*)b.sort_hist, b.dsort_H, b.dsort_tiles_cap, b.counters, fc.exact_tiles, fc.epoch, (const float4*)b.rec_bin,                                     \
             b.bin_params, b.area_prefix, b.chunk_first, (unsigned long long*)b.scan_desc, max_tests, (volatile uint32_t*)host_overflow)
  if (tiles_hint <= (uint32_t)num_sms) FUSED_LAUNCH(1);      // (the instance without a register cap is also the faster one)
  else FUSED_LAUNCH(FUSED_CTAS_PER_SM);
#undef FUSED_LAUNCH
}

// ------------------------------------------------------------------------------------------------------------------
// tgs_sort_pairs_static (include/tgs.h): the same scatter passes as a call that allocates nothing.  Every byte of scratch
// lives in the file-scope array below; the kernels get its DEVICE address, which host code obtains once per device with
// cudaGetSymbolAddress (in host code the array's name is only a stand-in for the symbol, not a pointer a kernel could use).
// The array is shared by all calls on a device and keeps the last call's contents: histograms / tickets / the error word
// are cleared by every call, the descriptors are tagged with (call number * 4 + pass) and never cleared, the ping-pong
// buffers are written before they are read.  Calls that overlap on the GPU race (documented in the header).
#include <cstddef>
#include <cstdio>
#include <mutex>

namespace {

constexpr uint32_t STATIC_MAX_ITEMS = TGS_SORT_STATIC_MAX_ITEMS;
constexpr uint32_t STATIC_SMALL_MAX = 1u << 18;      // up to here the 2048-item instance (more tiles in flight), above it the 4096-item one
constexpr uint32_t STATIC_MAX_TILES = 256;           // = 2^20 / 4096 >= 2^18 / 2048
static_assert(STATIC_MAX_ITEMS / (SORT_THREADS * SORT_IPT_BIG) <= STATIC_MAX_TILES && STATIC_SMALL_MAX / (SORT_THREADS * SORT_IPT_SMALL) <= STATIC_MAX_TILES, "descriptor rows");

struct StaticSortScratch {
  uint32_t hist[4][RADIX];                                // cleared by every call, filled by k_static_hist
  uint32_t tickets[4];                                    // cleared by every call
  uint32_t error;                                         // cleared by every call; 2 = a look-back gave up
  uint32_t n;                                             // written by k_static_hist (k_onesweep reads its item count from device memory)
  uint32_t pad[58];
  unsigned long long desc[STATIC_MAX_TILES * RADIX];      // one region for all passes: the tag tells the passes and the calls apart
  uint32_t tmp_keys[STATIC_MAX_ITEMS];                    // destination of every other pass
  uint32_t tmp_vals[STATIC_MAX_ITEMS];
};
static_assert(sizeof(StaticSortScratch) == TGS_SORT_STATIC_SCRATCH_BYTES, "tgs.h states the size");
static_assert(offsetof(StaticSortScratch, desc) == 4352 && offsetof(StaticSortScratch, desc) % 256 == 0, "head");

static __device__ __align__(256) unsigned char g_static_sort_scratch[sizeof(StaticSortScratch)];

// digit histograms of the low `passes` bytes of the keys (in the path the producer of the keys counts them; here nobody has)
__global__ void __launch_bounds__(256) k_static_hist(const uint32_t* __restrict__ keys, uint32_t n, int passes, StaticSortScratch* __restrict__ sc) {
  __shared__ uint32_t h[4][RADIX];
  for (int i = threadIdx.x; i < 4 * RADIX; i += 256) (&h[0][0])[i] = 0;
  __syncthreads();
  for (uint32_t i = blockIdx.x * 256u + threadIdx.x; i < n; i += gridDim.x * 256u) {
    const uint32_t k = keys[i];
    for (int p = 0; p < passes; ++p) atomicAdd(&h[p][(k >> (8 * p)) & 255u], 1u);
  }
  __syncthreads();
  for (int i = threadIdx.x; i < passes * RADIX; i += 256) {
    const uint32_t v = (&h[0][0])[i];
    if (v) atomicAdd(&sc->hist[0][0] + i, v);
  }
  if (blockIdx.x == 0 && threadIdx.x == 0) sc->n = n;
}

struct StaticSortDev {
  StaticSortScratch* ptr = nullptr;   // device address of g_static_sort_scratch on this device
  int num_sms = 0;
  uint32_t call = 0;                  // descriptor tag = call * 4 + pass, kept below 2^30 (the tag field of a descriptor)
};
constexpr int STATIC_MAX_DEVICES = 64;
StaticSortDev g_static_dev[STATIC_MAX_DEVICES];
std::mutex g_static_mutex;
thread_local char g_static_err[256] = "";

int static_fail(int code, const char* what, cudaError_t e = cudaSuccess) {
  if (e != cudaSuccess) snprintf(g_static_err, sizeof(g_static_err), "tgs_sort_pairs_static: %s: %s", what, cudaGetErrorString(e));
  else snprintf(g_static_err, sizeof(g_static_err), "tgs_sort_pairs_static: %s", what);
  return code;
}

bool ranges_overlap(const void* a, const void* b, size_t bytes) {
  const uintptr_t x = (uintptr_t)a, y = (uintptr_t)b;
  return x < y + bytes && y < x + bytes;
}

}  // namespace

extern "C" const char* tgs_static_last_error(void) { return g_static_err; }

extern "C" int tgs_sort_pairs_static(int cuda_device, void* cuda_stream, const uint32_t* keys_in, const uint32_t* vals_in, uint32_t* keys_out,
                                     uint32_t* vals_out, uint32_t n, int key_bytes, uint32_t* status) {
  g_static_err[0] = 0;
  if (n > STATIC_MAX_ITEMS) {
    snprintf(g_static_err, sizeof(g_static_err), "tgs_sort_pairs_static: n = %u exceeds the maximum of %u items (TGS_SORT_STATIC_MAX_ITEMS): the static scratch array has a fixed size",
             n, STATIC_MAX_ITEMS);
    return TGS_E_INVALID_ARG;
  }
  if (key_bytes < 1 || key_bytes > 4) return static_fail(TGS_E_INVALID_ARG, "key_bytes must be 1..4");
  if (cuda_device < 0 || cuda_device >= STATIC_MAX_DEVICES) return static_fail(TGS_E_INVALID_ARG, "bad device index");
  if (n > 0) {
    if (!keys_in || !vals_in || !keys_out || !vals_out) return static_fail(TGS_E_INVALID_ARG, "null buffer");
    const size_t bytes = (size_t)n * 4;
    if (ranges_overlap(keys_in, keys_out, bytes) || ranges_overlap(keys_in, vals_out, bytes) || ranges_overlap(vals_in, keys_out, bytes) ||
        ranges_overlap(vals_in, vals_out, bytes) || ranges_overlap(keys_out, vals_out, bytes))
      return static_fail(TGS_E_INVALID_ARG, "output buffers overlap the inputs or each other");
  }
  cudaStream_t s = (cudaStream_t)cuda_stream;
  cudaError_t e;
  int prev_device = -1;
  if ((e = cudaGetDevice(&prev_device)) != cudaSuccess) return static_fail(TGS_E_CUDA, "cudaGetDevice", e);
  if ((e = cudaSetDevice(cuda_device)) != cudaSuccess) return static_fail(TGS_E_CUDA, "cudaSetDevice", e);
  struct Restore { int d; ~Restore() { if (d >= 0) cudaSetDevice(d); } } restore{prev_device == cuda_device ? -1 : prev_device};

  std::lock_guard<std::mutex> lock(g_static_mutex);
  StaticSortDev& d = g_static_dev[cuda_device];
  if (!d.ptr) {   // set-up, once per device, with that device current
    StaticSortScratch* p = nullptr;
    if ((e = cudaGetSymbolAddress((void**)&p, g_static_sort_scratch)) != cudaSuccess || !p) return static_fail(TGS_E_CUDA, "cudaGetSymbolAddress(g_static_sort_scratch)", e);
    int sms = 0;
    if ((e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, cuda_device)) != cudaSuccess || sms <= 0) return static_fail(TGS_E_CUDA, "cudaDeviceGetAttribute", e);
    if ((e = cudaFuncSetAttribute(k_onesweep<4, SORT_CTAS_PER_SM, SORT_IPT_BIG>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(SortSmem<SORT_IPT_BIG>))) != cudaSuccess ||
        (e = cudaFuncSetAttribute(k_onesweep<32, 2, SORT_IPT_SMALL>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(SortSmem<SORT_IPT_SMALL>))) != cudaSuccess)
      return static_fail(TGS_E_CUDA, "cudaFuncSetAttribute", e);
    d.num_sms = sms;
    d.ptr = p;      // last: a failed set-up is tried again by the next call
  }
  StaticSortScratch* sc = d.ptr;
  if (status && (e = cudaMemsetAsync(status, 0, 4, s)) != cudaSuccess) return static_fail(TGS_E_CUDA, "cudaMemsetAsync(status)", e);
  if (n == 0) return TGS_OK;
  if (++d.call >= (1u << 28)) {   // the tags wrap: forget the old ones (static device memory starts as zeros, and tag 0..3 is never used)
    d.call = 1;
    if ((e = cudaMemsetAsync(sc->desc, 0, sizeof(sc->desc), s)) != cudaSuccess) return static_fail(TGS_E_CUDA, "cudaMemsetAsync(desc)", e);
  }
  if ((e = cudaMemsetAsync(sc, 0, offsetof(StaticSortScratch, desc), s)) != cudaSuccess) return static_fail(TGS_E_CUDA, "cudaMemsetAsync(head)", e);
  const int passes = key_bytes;
  const uint32_t hist_blocks = (n + 256u * 16u - 1u) / (256u * 16u);
  k_static_hist<<<hist_blocks < (uint32_t)d.num_sms * 4u ? hist_blocks : (uint32_t)d.num_sms * 4u, 256, 0, s>>>(keys_in, n, passes, sc);
  ++g_tgs_launches;
  const bool small_input = n <= STATIC_SMALL_MAX;
  const uint32_t* src_k = keys_in;
  const uint32_t* src_v = vals_in;
  for (int p = 0; p < passes; ++p) {
    const bool to_out = ((passes - 1 - p) & 1) == 0;      // the last pass writes the caller's buffers, the passes before it alternate
    uint32_t* dst_k = to_out ? keys_out : sc->tmp_keys;
    uint32_t* dst_v = to_out ? vals_out : sc->tmp_vals;
    const uint32_t tag = d.call * 4u + (uint32_t)p;
    if (small_input)
      k_onesweep<32, 2, SORT_IPT_SMALL><<<d.num_sms * 2, SORT_THREADS, sizeof(SortSmem<SORT_IPT_SMALL>), s>>>(
          src_k, src_v, dst_k, dst_v, &sc->n, &sc->tickets[p], &sc->error, &sc->hist[p][0], sc->desc, 8 * p, 8, tag, (uint2*)nullptr);
    else
      k_onesweep<4, SORT_CTAS_PER_SM, SORT_IPT_BIG><<<d.num_sms * SORT_CTAS_PER_SM, SORT_THREADS, sizeof(SortSmem<SORT_IPT_BIG>), s>>>(
          src_k, src_v, dst_k, dst_v, &sc->n, &sc->tickets[p], &sc->error, &sc->hist[p][0], sc->desc, 8 * p, 8, tag, (uint2*)nullptr);
    ++g_tgs_launches;
    src_k = dst_k;
    src_v = dst_v;
  }
  if (status && (e = cudaMemcpyAsync(status, &sc->error, 4, cudaMemcpyDeviceToDevice, s)) != cudaSuccess) return static_fail(TGS_E_CUDA, "cudaMemcpyAsync(status)", e);
  if ((e = cudaGetLastError()) != cudaSuccess) return static_fail(TGS_E_CUDA, "kernel launch", e);
  return TGS_OK;
}
