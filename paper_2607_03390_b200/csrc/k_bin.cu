// k_bin.cu -- A5 + A7: which (Gaussian, tile) pairs exist, in which order, and where each tile's list starts.
// PAPER.md:L61 ("Gaussians that intersect with multiple tiles are duplicated ... sorts its intersected
// Gaussians by depth from front to back"), L123 (only Gaussians intersecting T_selected are sorted).
//
// The visible Gaussians arrive sorted by (depth, index).  Every (Gaussian, tile of its test rect) combination -- the
// test rect is the part of the 3-sigma rect that k_preprocess could not rule out -- is one TEST; the tests of all
// Gaussians, in that order and row-major inside a rect, form one flat index space (k_scan_area: prefix sums of the
// rect areas).  k_bin cuts that space into equal chunks -- so a screen-filling Gaussian is spread over many CTAs
// instead of stalling one warp -- evaluates each test once (tile selected, L123, and reached with alpha >= 1/255,
// R39), ranks the passing tests with a single-pass scan (decoupled look-back over the chunks) and writes the pairs
// (tile id, Gaussian) in exactly the oracle's emission order; the stable sort by tile id that follows (k_sort.cu)
// then leaves every tile's list in (depth, index) order.  The same kernel counts the pairs per Gaussian and the
// digit histograms of the tile sort; k_colour_all evaluates SH -> RGB (L61 "color c_i"; R5) of the visible Gaussians.
//
// Compiled with -fmad=false: the tile test is decision arithmetic (decide_math.cuh).
// Problem sizes that are not known on the host (visible Gaussians, tests, pairs) are read from device memory, so a
// frame needs no host round trip.
#include "tgs_internal.cuh"
#include "bin_params.cuh"
#include "decide_math.cuh"
#include "scan.cuh"

namespace {

constexpr int SCAN_THREADS = 256;
constexpr int SCAN_IPT = 2;          // 8 (2048-Gaussian tiles, a shorter look-back) measured slower: +20 us, the gathers of a tile are serial per thread
constexpr int SCAN_TILE = SCAN_THREADS * SCAN_IPT;

constexpr int BIN_CTAS_PER_SM = 8;

constexpr int BIN_PCAP = 192;           // Gaussians of a chunk staged in shared memory (the rest is read from global)

// ================================================================== A5a: flat test space
// area_prefix[i] = number of tests of the Gaussians before position i of the sorted visible list (area_prefix[n] =
// all tests); chunk_first[k] = position of the Gaussian that contains test k * BIN_CHUNK.
__global__ void __launch_bounds__(SCAN_THREADS) k_scan_area(FrameConst fc, const uint32_t* __restrict__ sorted_g,
                                                            const float4* __restrict__ rec_bin, unsigned long long* __restrict__ desc,
                                                            uint32_t* __restrict__ area_prefix, uint32_t* __restrict__ chunk_first,
                                                            uint4* __restrict__ bin_params,
                                                            Counters* __restrict__ counters, unsigned long long max_tests,
                                                            volatile uint32_t* __restrict__ host_overflow) {
  TGS_PDL_WAIT();
  TGS_PDL_TRIGGER();
  __shared__ uint32_t s_tile, s_warp[SCAN_THREADS / 32], s_excl;
  const uint32_t n = counters->n_visible;
  if (n == 0 || counters->area_sum > max_tests) {
    if (blockIdx.x == 0 && threadIdx.x == 0) {
      counters->n_tests = 0; counters->n_pairs = 0;
      if (n) { counters->overflow = 1; *host_overflow = 1u; __threadfence_system(); }
    }
    return;
  }
  const uint32_t num_tiles = (n + SCAN_TILE - 1) / SCAN_TILE;
  while (true) {
    __syncthreads();
    if (threadIdx.x == 0) s_tile = atomicAdd(&counters->ticket_scan, 1u);
    __syncthreads();
    const uint32_t tile = s_tile;
    if (tile >= num_tiles) break;
    const uint32_t i0 = tile * SCAN_TILE + threadIdx.x * SCAN_IPT;
    uint32_t a[SCAN_IPT];
#pragma unroll
    for (int j = 0; j < SCAN_IPT; ++j) {
      a[j] = 0;
      if (i0 + j < n) {
        const uint32_t g = sorted_g[i0 + j];
        const float4 r0 = rec_bin[2 * (size_t)g], r1 = rec_bin[2 * (size_t)g + 1];      // one 32-byte sector per Gaussian
        store_params(bin_params + 3 * (size_t)(i0 + j), make_params_bin(g, r0, r1, fc.exact_tiles != 0, &a[j]));
      }
    }
    uint32_t tsum = 0;
#pragma unroll
    for (int j = 0; j < SCAN_IPT; ++j) tsum += a[j];
    uint32_t incl_total;
    uint32_t off = tgs_scan::chunk_scan<SCAN_THREADS>(tsum, tile, desc, s_warp, &s_excl, &counters->error, &incl_total, fc.epoch);
    if (tile == num_tiles - 1 && threadIdx.x == 0) { counters->n_tests = incl_total; area_prefix[n] = incl_total; }
#pragma unroll
    for (int j = 0; j < SCAN_IPT; ++j) {
      if (i0 + j >= n) break;
      area_prefix[i0 + j] = off;
      const unsigned long long end = (unsigned long long)off + a[j];
      for (unsigned long long kb = ((unsigned long long)off + BIN_CHUNK - 1) / BIN_CHUNK; kb * BIN_CHUNK < end; ++kb) chunk_first[kb] = i0 + j;
      off += a[j];
    }
  }
}

__device__ __forceinline__ void sh_basis(int deg, float x, float y, float z, float* Y) {   // R5
  Y[0] = 0.28209479177387814f;
  if (deg < 1) return;
  Y[1] = -0.4886025119029199f * y; Y[2] = 0.4886025119029199f * z; Y[3] = -0.4886025119029199f * x;
  if (deg < 2) return;
  const float xx = x * x, yy = y * y, zz = z * z, xy = x * y, yz = y * z, xz = x * z;
  Y[4] = 1.0925484305920792f * xy; Y[5] = -1.0925484305920792f * yz;
  Y[6] = 0.31539156525252005f * (2.0f * zz - xx - yy);
  Y[7] = -1.0925484305920792f * xz; Y[8] = 0.5462742152960396f * (xx - yy);
  if (deg < 3) return;
  Y[9] = -0.5900435899266435f * y * (3.0f * xx - yy);
  Y[10] = 2.890611442640554f * xy * z;
  Y[11] = -0.4570457994644658f * y * (4.0f * zz - xx - yy);
  Y[12] = 0.3731763325901154f * z * (2.0f * zz - 3.0f * xx - 3.0f * yy);
  Y[13] = -0.4570457994644658f * x * (4.0f * zz - xx - yy);
  Y[14] = 1.445305721320277f * z * (xx - yy);
  Y[15] = -0.5900435899266435f * x * (xx - 3.0f * yy);
}

template <int DEG>
__device__ __forceinline__ void sh_colour(const FrameConst& fc, uint32_t g, const float4* __restrict__ cull4, const float* __restrict__ sh,
                                          float4* __restrict__ rec_rgb) {
  constexpr int K = (DEG + 1) * (DEG + 1);
  const float4 c4 = cull4[g];
  float dx = c4.x - fc.cam.campos[0], dy = c4.y - fc.cam.campos[1], dz = c4.z - fc.cam.campos[2];
  const float inv = 1.0f / sqrtf(dx * dx + dy * dy + dz * dz);
  dx *= inv; dy *= inv; dz *= inv;
  float Y[K];
  sh_basis(DEG, dx, dy, dz, Y);
  float cr = 0.5f, cg = 0.5f, cb = 0.5f;
  const float* p = sh + (size_t)g * K * 3;
  if constexpr (K % 4 == 0) {            // K*3 floats = 3K/4 float4, 16 B aligned
    const float4* p4 = reinterpret_cast<const float4*>(p);
    float buf[K * 3];
#pragma unroll
    for (int i = 0; i < K * 3 / 4; ++i) {
      const float4 t = __ldg(p4 + i);
      buf[4 * i] = t.x; buf[4 * i + 1] = t.y; buf[4 * i + 2] = t.z; buf[4 * i + 3] = t.w;
    }
#pragma unroll
    for (int kk = 0; kk < K; ++kk) { cr += Y[kk] * buf[3 * kk]; cg += Y[kk] * buf[3 * kk + 1]; cb += Y[kk] * buf[3 * kk + 2]; }
  } else {
#pragma unroll
    for (int kk = 0; kk < K; ++kk) { cr += Y[kk] * p[3 * kk]; cg += Y[kk] * p[3 * kk + 1]; cb += Y[kk] * p[3 * kk + 2]; }
  }
  rec_rgb[g] = make_float4(fmaxf(cr, 0.0f), fmaxf(cg, 0.0f), fmaxf(cb, 0.0f), 0.0f);
}

// ================================================================== A5b: tests -> pairs, counts
// The tile test is box_qmin(...) <= tau in the oracle's fp32 operation order (4 IEEE divisions).  Most tests are far
// from the threshold, so each is first evaluated in fast arithmetic (reciprocals of A and C once per Gaussian, FMAs):
// with M = A dx^2 + C t^2 (>= |2B dx t|, the form is positive semi-definite) every edge value of either evaluation is
// within a few 2^-24 * 2M of the exact one, hence the two agree unless |best - tau| <= 1e-5 * max M; only in that band
// (a fraction of a percent of the tests) the exact sequence is run.  The decision is always the oracle's.
// fast evaluation of one box edge: dx fixed, t free in [lo, hi]; q = A dx^2 + 2B dx t + C t^2 at the clamped optimum
__device__ __forceinline__ void edge_fast(float A, float B2, float C, float k, float dx, float lo, float hi, float& best, float& Mmax) {
  const float t = fminf(fmaxf(k * dx, lo), hi);
  const float s1 = (A * dx) * dx, s2 = (C * t) * t;
  best = fminf(best, fmaf(B2 * dx, t, s1 + s2));
  Mmax = fmaxf(Mmax, s1 + s2);
}

__device__ __forceinline__ bool tile_reach(const GaussParams& P, uint32_t tx, uint32_t ty, int W, int H) {
  if (!(P.tau >= 0.0f)) return false;
  const float x0 = (float)(tx * 16u), x1 = (float)min((int)(tx * 16u + 15u), W - 1);
  const float y0 = (float)(ty * 16u), y1 = (float)min((int)(ty * 16u + 15u), H - 1);
  if (P.u >= x0 && P.u <= x1 && P.v >= y0 && P.v <= y1) return true;
  const float xl = x0 - P.u, xh = x1 - P.u, yl = y0 - P.v, yh = y1 - P.v, B2 = 2.0f * P.B;
  float best = 3.0e38f, Mmax = 0.0f;
  edge_fast(P.A, B2, P.C, P.kC, xl, yl, yh, best, Mmax);
  edge_fast(P.A, B2, P.C, P.kC, xh, yl, yh, best, Mmax);
  edge_fast(P.C, B2, P.A, P.kA, yl, xl, xh, best, Mmax);
  edge_fast(P.C, B2, P.A, P.kA, yh, xl, xh, best, Mmax);
  const float margin = 1.0e-5f * Mmax;
  if (best < P.tau - margin) return true;
  if (best > P.tau + margin) return false;
  return box_qmin(P.u, P.v, P.A, P.B, P.C, x0, x1, y0, y1) <= P.tau;       // the oracle's sequence decides
}

// ---- k_bin: tests, ranks (single-pass scan with decoupled look-back over the chunks) and pairs of one chunk
// TileT: uint16_t when every tile id fits (T <= 65536: up to 4K images), which lets 8 CTAs share an SM; else uint32_t, 7
template <typename TileT>
struct BinSmem {
  uint32_t prefix[BIN_CHUNK + 2];       // area_prefix of the Gaussians of this chunk (+ sentinel)
  TileT st_tile[2][BIN_CHUNK];          // passing tests of a chunk, in order: tile id (double buffered: pipeline)
  uint32_t st_g[2][BIN_CHUNK];          //                                      Gaussian
  GaussParams gp[BIN_PCAP];
  uint32_t warp[BIN_THREADS / 32];
  uint32_t excl, chunk;
  uint32_t hist[sizeof(TileT) == 2 ? 2 : 3][256];   // digit histograms of the tile ids of the emitted pairs (for the tile sort)
};

// 8 CTAs per SM (7 with 32-bit tile staging) is what the persistent grid is sized for: the register cap that goes with
// it (64) must hold, or the eighth CTA of every SM starts only when another one has run out of tickets.
// LATER: the instance for the second and later slabs (dead-Gaussian skip through the summed-area table, early return when
// every tile has finished); ALL: every tile is selected and alive (R / P frames, first slab), so no bit is looked up and
// the evaluated tests need no counting.  The first-slab instances compile to round 1's kernel.
template <typename TileT, bool LATER, bool ALL>
__global__ void __launch_bounds__(BIN_THREADS, sizeof(TileT) == 2 ? BIN_CTAS_PER_SM : BIN_CTAS_PER_SM - 1) k_bin(FrameConst fc, const uint4* __restrict__ bin_params, const uint32_t* __restrict__ area_prefix,
                                                     const uint32_t* __restrict__ chunk_first,
                                                     const uint32_t* __restrict__ live_bits, unsigned long long* __restrict__ desc_all,
                                                     uint32_t* __restrict__ keys,
                                                     uint32_t* __restrict__ vals, uint32_t* __restrict__ tile_hist,
                                                     Counters* __restrict__ counters, volatile uint32_t* __restrict__ host_overflow, int slab,
                                                     const uint32_t* __restrict__ live_sat) {
  TGS_PDL_WAIT();
  TGS_PDL_TRIGGER();
  __shared__ BinSmem<TileT> sm;
  const uint32_t n = counters->n_visible, total_tests = counters->n_tests;
  // pairs <= tests: with the tests inside the capacity no slab can overflow, and the host need not wait for the end of the
  // frame to know it (2 = cannot be ruled out yet).  (Here and not in k_scan_area: a system fence inside that kernel's loop
  // cost it 4 us even when never executed.)
  if (!LATER && blockIdx.x == 0 && threadIdx.x == 0 && total_tests > fc.max_pairs) { *host_overflow = 2u; __threadfence_system(); }
  const uint32_t all_chunks = (uint32_t)(((unsigned long long)total_tests + BIN_CHUNK - 1) / BIN_CHUNK);
  // this slab's range of chunks; inside the slab the chunks are numbered from 0 for the look-back
  const uint32_t c_lo = LATER ? (uint32_t)(((unsigned long long)all_chunks * fc.slab_bound[slab]) >> 10) : 0u;
  const uint32_t c_hi = (uint32_t)(((unsigned long long)all_chunks * fc.slab_bound[slab + 1]) >> 10);
  uint32_t num_chunks = c_hi - c_lo;
  unsigned long long* desc = desc_all + c_lo;
  if (LATER) {      // every selected tile has finished in the earlier slabs: nothing left to bin (n_pairs_slab stays 0)
    uint32_t fin = 0;
    for (int j = 0; j < slab; ++j) fin += counters->n_finished[j];
    if (fin >= counters->n_sel) num_chunks = 0;
  }
  const uint32_t tid = threadIdx.x, lane = tid & 31;
  const int TX = fc.cam.TX;
  const bool exact = fc.exact_tiles != 0;
  constexpr int NH = sizeof(TileT) == 2 ? 2 : 3;      // digits of a tile id (ids up to 2^24 with 32-bit staging)
  for (int i = tid; i < NH * 256; i += BIN_THREADS) (&sm.hist[0][0])[i] = 0;
  // Software pipeline over the chunks of this CTA: the tests of chunk k+1 run BEFORE the look-back of chunk k.  A chunk
  // publishes its aggregate right after its tests; by the time its CTA has tested another chunk, the predecessors'
  // aggregates are there, so the look-back does not spin on stragglers (profiles/r1c: 41 % of the warp samples of the
  // unpipelined kernel sat at the barrier behind a polling warp 0).  Passing tests wait in a double-buffered stage.
  uint32_t pend = 0xffffffffu, pend_total = 0, it = 0;
  uint32_t n_eval = 0;                  // tests whose tile was alive, i.e. that were really evaluated (statistics)
  while (true) {
    __syncthreads();
    if (tid == 0) sm.chunk = atomicAdd(&counters->ticket_bin[slab], 1u);
    __syncthreads();
    const uint32_t chunk = sm.chunk;                                 // within the slab
    const bool have = chunk < num_chunks;
    const uint32_t buf = it & 1u;
    uint32_t total = 0;
    if (have) {
      const uint32_t gchunk = c_lo + chunk;                          // in the flat test space
      const uint32_t cbase = gchunk * BIN_CHUNK;
      const uint32_t tend = (total_tests - cbase < (uint32_t)BIN_CHUNK) ? total_tests : cbase + BIN_CHUNK;
      const uint32_t i_first = chunk_first[gchunk];
      const uint32_t i_last = (gchunk + 1 < all_chunks) ? chunk_first[gchunk + 1] : n - 1;
      const uint32_t m = i_last - i_first + 1;                     // <= BIN_CHUNK + 1
      for (uint32_t i = tid; i <= m; i += BIN_THREADS) sm.prefix[i] = area_prefix[i_first + i];
      {   // the chunk's parameters are one contiguous block of the sorted array: coalesced 16 B copies
        const uint32_t nq = 3u * (m < (uint32_t)BIN_PCAP ? m : (uint32_t)BIN_PCAP);
        const uint4* src = bin_params + 3 * (size_t)i_first;
        uint4* dst = reinterpret_cast<uint4*>(sm.gp);
        for (uint32_t i = tid; i < nq; i += BIN_THREADS) dst[i] = src[i];
      }
      __syncthreads();
      bool chunk_alive = true;
      if (LATER) {
        // Later slabs: most tiles have finished.  A Gaussian whose test rect holds no live tile -- four look-ups in the
        // summed-area table of the live tiles (k_live_sat) -- has all its tests skipped without looking at them.
        const uint32_t mm = m < (uint32_t)BIN_PCAP ? m : (uint32_t)BIN_PCAP;
        const uint32_t SW = (uint32_t)TX + 1u;
        bool alive_here = m > (uint32_t)BIN_PCAP;                  // Gaussians beyond the staged ones are not looked up: alive
        for (uint32_t l = tid; l < mm; l += BIN_THREADS) {
          GaussParams& Gp = sm.gp[l];
          const uint32_t x0 = Gp.lo & 0xffffu, y0 = Gp.lo >> 16, w = Gp.w, h = (sm.prefix[l + 1] - sm.prefix[l]) / (w ? w : 1u);
          const uint32_t cnt = (live_sat[(y0 + h) * SW + x0 + w] - live_sat[y0 * SW + x0 + w]) - (live_sat[(y0 + h) * SW + x0] - live_sat[y0 * SW + x0]);
          Gp.pad = cnt ? 0u : 1u;                                  // pad = 1: dead
          alive_here = alive_here || cnt != 0u;
        }
        // a chunk none of whose Gaussians can reach a live tile (most chunks of a later slab) is not enumerated at all
        chunk_alive = __syncthreads_or(alive_here ? 1 : 0) != 0;
      }
      // -------------------------------------------------------------- tests
      const uint32_t t0 = cbase + tid * BIN_IPT;
      uint32_t mask = 0, tl[BIN_IPT], gg[BIN_IPT];
      if (t0 < tend && (!LATER || chunk_alive)) {
        uint32_t lo = 0, hi = m;                                   // largest li with prefix[li] <= t0
        while (hi - lo > 1) { const uint32_t mid = (lo + hi) >> 1; if (sm.prefix[mid] <= t0) lo = mid; else hi = mid; }
        uint32_t li = lo, end, rx, ry, x_lo, y_lo;
        GaussParams G;
        auto load = [&](uint32_t l, uint32_t t) {
          G = l < (uint32_t)BIN_PCAP ? sm.gp[l] : load_params(bin_params + 3 * (size_t)(i_first + l));
          end = sm.prefix[l + 1];
          const uint32_t local = t - sm.prefix[l];
          ry = local / G.w; rx = local - ry * G.w;
          x_lo = G.lo & 0xffffu; y_lo = G.lo >> 16;
        };
        load(li, t0);
#pragma unroll
        for (int k = 0; k < BIN_IPT; ++k) {
          const uint32_t t = t0 + k;
          if (t < tend) {
            if (t >= end) { do { ++li; } while (sm.prefix[li + 1] <= t); load(li, t); }
            const uint32_t tx = x_lo + rx, ty = y_lo + ry, tile = ty * TX + tx;
            // selected (L123) and not yet finished (slabs); G.pad: no live tile in this Gaussian's rect at all (later slabs)
            bool pass = ALL || ((!LATER || !G.pad) && ((live_bits[tile >> 5] >> (tile & 31)) & 1u));
            if (!ALL) n_eval += pass ? 1u : 0u;
            if (pass && exact) pass = tile_reach(G, tx, ty, fc.cam.W, fc.cam.H);                           // R39
            if (pass) mask |= 1u << k;
            tl[k] = tile; gg[k] = G.g;
            if (++rx == G.w) { rx = 0; ++ry; }
          }
        }
      }
      // -------------------------------------------------------------- chunk-local ranks, stage, publish the aggregate
      const uint32_t cnt = __popc(mask);
      uint32_t incl = cnt;
#pragma unroll
      for (int d = 1; d < 32; d <<= 1) { const uint32_t o = __shfl_up_sync(0xffffffffu, incl, d); if (lane >= (uint32_t)d) incl += o; }
      if (lane == 31) sm.warp[tid >> 5] = incl;
      __syncthreads();
      uint32_t lpos = incl - cnt;
#pragma unroll
      for (int w = 0; w < BIN_THREADS / 32; ++w) { const uint32_t t = sm.warp[w]; if ((uint32_t)w < (tid >> 5)) lpos += t; total += t; }
      if (tid == 0) tgs_scan::publish_aggregate(total, chunk, desc, fc.epoch);
#pragma unroll
      for (int k = 0; k < BIN_IPT; ++k)
        if ((mask >> k) & 1u) { sm.st_tile[buf][lpos] = (TileT)tl[k]; sm.st_g[buf][lpos] = gg[k]; ++lpos; }
    }
    // ---------------------------------------------------------------- finish the chunk tested one round ago
    if (pend != 0xffffffffu) {
      if (tid < 32) {
        const uint32_t e = tgs_scan::lookback_warp(pend_total, pend, desc, &counters->error, fc.epoch, false);
        if (lane == 0) sm.excl = e;
      }
      __syncthreads();
      const uint32_t cexcl = sm.excl, ctotal = pend_total, incl_total = cexcl + ctotal, pbuf = buf ^ 1u;
      const bool overflow = incl_total > fc.max_pairs;
      if (pend == num_chunks - 1 && tid == 0) {
        if (overflow) { counters->overflow = 1; counters->n_pairs_slab[slab] = 0; *host_overflow = 1u; __threadfence_system(); }
        else { counters->n_pairs_slab[slab] = incl_total; counters->n_pairs += incl_total; }   // slabs run one after the other
      }
      if (!overflow)
        for (uint32_t p0 = 0; p0 < ctotal; p0 += BIN_THREADS) {
          const uint32_t p = p0 + tid;
          const bool in = p < ctotal;
          const uint32_t tile = in ? (uint32_t)sm.st_tile[pbuf][p] : 0xffffffffu;
          if (in) { keys[cexcl + p] = tile; vals[cexcl + p] = sm.st_g[pbuf][p]; atomicAdd(&sm.hist[0][tile & 255u], 1u); }
          // upper digit: consecutive pairs are consecutive tiles of one Gaussian, so it comes in runs: one atomic per run
          const uint32_t hi = tile >> 8, prev = __shfl_up_sync(0xffffffffu, hi, 1);
          const uint32_t heads = __ballot_sync(0xffffffffu, lane == 0 || hi != prev);
          if (in && ((heads >> lane) & 1u)) {
            const uint32_t above = heads & ~((2u << lane) - 1u);               // heads of later runs
            const uint32_t run = (above ? (uint32_t)__ffs(above) - 1u : 32u) - lane;
            atomicAdd(&sm.hist[1][hi & 255u], run);
          }
          if (NH == 3 && in) atomicAdd(&sm.hist[NH - 1][(tile >> 16) & 255u], 1u);
        }
    }
    if (!have) break;
    pend = chunk; pend_total = total; ++it;
  }
  __syncthreads();
  for (int i = tid; i < NH * 256; i += BIN_THREADS) { const uint32_t h = (&sm.hist[0][0])[i]; if (h) atomicAdd(&tile_hist[i], h); }
  if (ALL) {          // every test of the slab was evaluated
    if (blockIdx.x == 0 && tid == 0 && num_chunks) {
      const unsigned long long t_hi = (unsigned long long)c_hi * BIN_CHUNK;
      atomicAdd(&counters->n_tests_eval, (t_hi < total_tests ? t_hi : (unsigned long long)total_tests) - (unsigned long long)c_lo * BIN_CHUNK);
    }
  } else {
    n_eval = __reduce_add_sync(0xffffffffu, n_eval);
    if (lane == 0 && n_eval) atomicAdd(&counters->n_tests_eval, (unsigned long long)n_eval);
  }
}

// ================================================================== A5c: SH -> RGB (L61 "color c_i"; R5)
// One thread per visible Gaussian of the compacted visible list (index order, k_compact_vis): every lane works and the
// 12 K bytes of a Gaussian are read as K 3/4 independent 16-byte loads.  Needs neither the sorted list nor the pair
// counts, so it runs on its own stream beside the depth sort, which leaves most SMs idle.  (A variant that waited for
// k_bin and skipped Gaussians without pairs read fewer SH bytes on S frames but could only run beside the tile sort,
// whose CTAs fill the register file: no overlap, 20-47 us on the critical path.)
template <int DEG>
__global__ void __launch_bounds__(128) k_colour_all(FrameConst fc, const uint32_t* __restrict__ vis_list, const Counters* __restrict__ counters,
                                                    const float4* __restrict__ cull4, const float* __restrict__ sh, float4* __restrict__ rec_rgb) {
  TGS_PDL_WAIT();
  TGS_PDL_TRIGGER();
  const uint32_t nv = counters->n_visible;
  for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < nv; i += gridDim.x * blockDim.x) sh_colour<DEG>(fc, vis_list[i], cull4, sh, rec_rgb);
}

// ================================================================== A7: per-tile ranges
// Written by the last pass of the tile sort (k_sort.cu) as {~start, end}, all zero for a tile without pairs.
// test-only: the plain {start, end} form the oracle reports ({0, 0} for an empty tile)
__global__ void __launch_bounds__(256) k_ranges_decode(const uint2* __restrict__ ranges, int n_tiles, uint2* __restrict__ out) {
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t < n_tiles) { const uint2 r = ranges[t]; out[t] = r.y ? make_uint2(~r.x, r.y) : make_uint2(0u, 0u); }
}

// test-only: pairs per Gaussian (the oracle's record.tiles_touched), counted from the pair list
__global__ void __launch_bounds__(256) k_count_pairs(const uint32_t* __restrict__ vals, uint32_t n, uint32_t* __restrict__ out) {
  const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) atomicAdd(&out[vals[i]], 1u);
}

// test-only: the 64-bit sort keys tile << 32 | bits(depth) of the sorted pair list
__global__ void __launch_bounds__(256) k_keys64(const uint32_t* __restrict__ keys, const uint32_t* __restrict__ vals,
                                                const float4* __restrict__ rec_b1, uint32_t n, uint64_t* __restrict__ out) {
  const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) out[i] = ((uint64_t)keys[i] << 32) | __float_as_uint(rec_b1[2 * (size_t)vals[i]].z);
}

}  // namespace

uint32_t scan_tile_items() { return SCAN_TILE; }
uint32_t bin_chunk_items() { return BIN_CHUNK; }

// Summed-area table of the live tiles, (TY + 1) x (TX + 1) with a zero border: sat[y][x] = live tiles with ty < y, tx < x.
// One CTA: a thread per tile row (prefix along x), then a thread per column (prefix along y); 8 K entries at 1080p, built
// in shared memory (SMEM = true; grids beyond 48 KB fall back to global memory) and copied out coalesced.
template <bool SMEM>
__global__ void __launch_bounds__(1024) k_live_sat(int TX, int TY, const uint32_t* __restrict__ live_bits, uint32_t* __restrict__ sat,
                                                   const Counters* __restrict__ counters, int slab) {
  TGS_PDL_WAIT();
  TGS_PDL_TRIGGER();
  {   // every selected tile finished in the earlier slabs (the usual case once the split has settled): k_bin will not look at the table
    uint32_t fin = 0;
    for (int j = 0; j < slab; ++j) fin += counters->n_finished[j];
    if (fin >= counters->n_sel) return;
  }
  extern __shared__ uint32_t s_sat[];
  uint32_t* const w = SMEM ? s_sat : sat;
  const int SW = TX + 1;
  for (int x = threadIdx.x; x <= TX; x += blockDim.x) w[x] = 0;
  {   // rows: one warp per tile row, 32 tiles per step, prefix by ballot + popc
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
    for (int y = wid; y < TY; y += nw) {
      uint32_t carry = 0;
      if (lane == 0) w[(y + 1) * SW] = 0;
      for (int x0 = 0; x0 < TX; x0 += 32) {
        const int x = x0 + lane, t = y * TX + x;
        const bool live = x < TX && ((live_bits[t >> 5] >> (t & 31)) & 1u);
        const uint32_t bal = __ballot_sync(0xffffffffu, live);
        if (x < TX) w[(y + 1) * SW + x + 1] = carry + __popc(bal & (0xffffffffu >> (31 - lane)));
        carry += __popc(bal);
      }
    }
  }
  __syncthreads();
  for (int x = threadIdx.x + 1; x <= TX; x += blockDim.x) {
    uint32_t run = 0;
    for (int y = 1; y <= TY; ++y) { run += w[y * SW + x]; w[y * SW + x] = run; }
  }
  if (SMEM) {
    __syncthreads();
    const int n = SW * (TY + 1);
    for (int i = threadIdx.x; i < n; i += blockDim.x) sat[i] = s_sat[i];
  }
}

// sorted_g_idx: which of cvals[] holds the visible Gaussians in (depth, index) order
unsigned long long bin_max_tests(uint32_t bin_chunks_cap) { return (unsigned long long)(bin_chunks_cap - 2) * BIN_CHUNK; }

void launch_bin(cudaStream_t s, const FrameConst& fc, DevBuffers& b, int sorted_g_idx, uint32_t bin_chunks_cap, int num_sms,
                uint32_t* host_overflow, int slab) {
  if (slab == 0 && !fc.dsort_fused) {            // fused: k_depth_sort_fused has done A5a
    const uint32_t scan_tiles = (fc.n + SCAN_TILE - 1) / SCAN_TILE;   // upper bound (n_visible <= N)
    const unsigned long long max_tests = bin_max_tests(bin_chunks_cap);
    const uint32_t* sorted_g = b.cvals[sorted_g_idx];
    uint32_t grid = scan_tiles < (uint32_t)(num_sms * 4) ? scan_tiles : (uint32_t)(num_sms * 4);
    TGS_LAUNCH((k_scan_area), grid ? grid : 1, SCAN_THREADS, 0, s, fc, sorted_g, (const float4*)b.rec_bin, (unsigned long long*)b.scan_desc, b.area_prefix, b.chunk_first,
                                                        b.bin_params, b.counters, max_tests, (volatile uint32_t*)host_overflow);
  }
  if (slab > 0) {
    const size_t sat_bytes = (size_t)(fc.cam.TX + 1) * (fc.cam.TY + 1) * sizeof(uint32_t);
    if (sat_bytes <= 48 * 1024) TGS_LAUNCH((k_live_sat<true>), 1, 1024, sat_bytes, s, fc.cam.TX, fc.cam.TY, (const uint32_t*)b.live_bits, b.live_sat, (const Counters*)b.counters, slab);
    else TGS_LAUNCH((k_live_sat<false>), 1, 1024, 0, s, fc.cam.TX, fc.cam.TY, (const uint32_t*)b.live_bits, b.live_sat, (const Counters*)b.counters, slab);
  }
  uint32_t* hist = b.sort_hist + (1 + slab) * 4 * 256;
#define BIN_LAUNCH(T, CPS, LATER_, ALL_)                                                                                              \
  TGS_LAUNCH((k_bin<T, LATER_, ALL_>), num_sms * (CPS), BIN_THREADS, 0, s, fc, b.bin_params, b.area_prefix, b.chunk_first, b.live_bits,   \
             (unsigned long long*)b.bin_desc, b.keys[0], b.vals[0], hist, b.counters, (volatile uint32_t*)host_overflow, slab, (const uint32_t*)b.live_sat)
  const bool all = slab == 0 && fc.all_tiles != 0;
  if (fc.n_tiles <= 65536) {
    if (slab > 0) BIN_LAUNCH(uint16_t, BIN_CTAS_PER_SM, true, false);
    else if (all) BIN_LAUNCH(uint16_t, BIN_CTAS_PER_SM, false, true);
    else BIN_LAUNCH(uint16_t, BIN_CTAS_PER_SM, false, false);
  } else {
    if (slab > 0) BIN_LAUNCH(uint32_t, BIN_CTAS_PER_SM - 1, true, false);
    else if (all) BIN_LAUNCH(uint32_t, BIN_CTAS_PER_SM - 1, false, true);
    else BIN_LAUNCH(uint32_t, BIN_CTAS_PER_SM - 1, false, false);
  }
#undef BIN_LAUNCH
}

void launch_colour_all(cudaStream_t s, const FrameConst& fc, DevBuffers& b, int num_sms) {
#define LAUNCH(D) TGS_LAUNCH((k_colour_all<D>), num_sms * 16, 128, 0, s, fc, b.vis_list, (const Counters*)b.counters, b.cull4, b.sh, b.rec_rgb)
  switch (fc.sh_degree) {
    case 0: LAUNCH(0); break;
    case 1: LAUNCH(1); break;
    case 2: LAUNCH(2); break;
    default: LAUNCH(3); break;
  }
#undef LAUNCH
}

void launch_ranges_decode(cudaStream_t s, const DevBuffers& b, int n_tiles, uint2* out) {
  k_ranges_decode<<<(n_tiles + 255) / 256, 256, 0, s>>>(b.ranges, n_tiles, out);
}

void launch_count_pairs(cudaStream_t s, DevBuffers& b, int sorted_idx, uint32_t n_pairs, uint32_t n) {
  cudaMemsetAsync(b.tiles_touched, 0, (size_t)n * 4, s);
  if (n_pairs) k_count_pairs<<<(n_pairs + 255) / 256, 256, 0, s>>>(b.vals[sorted_idx], n_pairs, b.tiles_touched);
}

// test-only: the records the oracle reports per Gaussian, put together from what the path keeps -- rec_bin {u, v, A, B | C, tau,
// ..}, the blend record rec_b1 {.., .., d, rad}, the scene's opacity (g2): which = 0 {u, v, d, o}, 1 {A, B, C, tau}, 2 the
// 3-sigma rect as {x_lo | x_hi << 16, y_lo | y_hi << 16} (uint2 per Gaussian), recomputed with the function k_preprocess
// decides with.  Entries of Gaussians that are not visible in the current frame are stale.
__global__ void __launch_bounds__(256) k_debug_record(uint32_t n, int which, float TXf, float TYf, const float4* __restrict__ rec_bin,
                                                      const float4* __restrict__ rec_b1, const float4* __restrict__ g2, float4* __restrict__ out) {
  const uint32_t g = blockIdx.x * blockDim.x + threadIdx.x;
  if (g >= n) return;
  const float4 q0 = rec_bin[2 * (size_t)g], q1 = rec_bin[2 * (size_t)g + 1], b1 = rec_b1[2 * (size_t)g];
  if (which == 0) out[g] = make_float4(q0.x, q0.y, b1.z, g2[2 * (size_t)g + 1].z);
  else if (which == 1) out[g] = make_float4(q0.z, q0.w, q1.x, q1.y);
  else {
    uint32_t x_lo, x_hi, y_lo, y_hi;
    tile_rect(q0.x, q0.y, b1.w, TXf, TYf, x_lo, x_hi, y_lo, y_hi);
    reinterpret_cast<uint2*>(out)[g] = make_uint2(x_lo | (x_hi << 16), y_lo | (y_hi << 16));
  }
}
void launch_debug_record(cudaStream_t s, const FrameConst& fc, const DevBuffers& b, uint32_t n, int which, float4* out) {
  if (n) k_debug_record<<<(n + 255) / 256, 256, 0, s>>>(n, which, (float)fc.cam.TX, (float)fc.cam.TY, (const float4*)b.rec_bin, (const float4*)b.rec_b1,
                                                        (const float4*)b.g2, out);
}

__global__ void __launch_bounds__(256) k_debug_flags(uint32_t n, const uint8_t* __restrict__ flags, uint32_t* __restrict__ out) {
  const uint32_t g = blockIdx.x * blockDim.x + threadIdx.x;
  if (g < n) out[g] = flags[g];
}
void launch_debug_flags(cudaStream_t s, const DevBuffers& b, uint32_t n, uint32_t* out) {
  if (n) k_debug_flags<<<(n + 255) / 256, 256, 0, s>>>(n, (const uint8_t*)b.rec_flags, out);
}

void launch_keys64(cudaStream_t s, DevBuffers& b, int sorted_idx, uint32_t n, uint64_t* out) {
  if (n) k_keys64<<<(n + 255) / 256, 256, 0, s>>>(b.keys[sorted_idx], b.vals[sorted_idx], b.rec_b1, n, out);
}
