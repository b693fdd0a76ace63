// k_decide.cu -- kernels whose fp32 arithmetic DECIDES integers (cull masks, nearest pixels, tile
// rects, sort-key depth bits, tile selection).  Compiled with -fmad=false: every +,-,*,/,sqrt is one
// IEEE rounding in the order written, so the decisions are reproducible bit for bit (DESIGN.md §2 R33).
// All of these kernels are HBM- or latency-bound; the lost FMA contraction costs nothing measurable.
//
// A1 forward warp (Eq.3), A2 depth fill + correspondence + T^um (L121),
// A3 preprocess + AFC + TOC + newly-visible + T^oc (L61, L109-113, L119), A4 tile selection (L117-123),
// A5a count + SH colour, F reduction (L109).
#include <cstddef>

#include "tgs_internal.cuh"
#include "decide_math.cuh"

namespace {

__device__ __forceinline__ uint32_t warp_sum(uint32_t v) { return __reduce_add_sync(0xffffffffu, v); }

// order-preserving float <-> uint key (for atomicMin / atomicMax on signed floats)
__device__ __forceinline__ uint32_t f2key(float f) {
  const uint32_t b = __float_as_uint(f);
  return (b & 0x80000000u) ? ~b : (b | 0x80000000u);
}
__device__ __forceinline__ float key2f(uint32_t k) {
  return __uint_as_float((k & 0x80000000u) ? (k & 0x7fffffffu) : ~k);
}

// ------------------------------------------------------------------ load-time repack
// Sigma = R S S^T R^T, quaternion (w,x,y,z) normalised; tau = 2 ln(255 o) (L119, R18).
__global__ void __launch_bounds__(256) k_repack(uint32_t n, const float* __restrict__ means, const float* __restrict__ scales,
                                                const float* __restrict__ quats, const float* __restrict__ opacity,
                                                float4* __restrict__ cull4, float4* __restrict__ g2) {
  const uint32_t g = blockIdx.x * blockDim.x + threadIdx.x;
  if (g >= n) return;
  const float o = opacity[g];
  // cull record: mean + the largest scale (bounds the screen extent without the covariance, see k_preprocess)
  cull4[g] = make_float4(means[3 * g], means[3 * g + 1], means[3 * g + 2],
                         fmaxf(fabsf(scales[3 * g]), fmaxf(fabsf(scales[3 * g + 1]), fabsf(scales[3 * g + 2]))));
  float w = quats[4 * g], x = quats[4 * g + 1], y = quats[4 * g + 2], z = quats[4 * g + 3];
  const float nrm = sqrtf(((w * w + x * x) + y * y) + z * z);
  w /= nrm; x /= nrm; y /= nrm; z /= nrm;
  const float R[9] = {1.0f - 2.0f * (y * y + z * z), 2.0f * (x * y - w * z), 2.0f * (x * z + w * y),
                      2.0f * (x * y + w * z), 1.0f - 2.0f * (x * x + z * z), 2.0f * (y * z - w * x),
                      2.0f * (x * z - w * y), 2.0f * (y * z + w * x), 1.0f - 2.0f * (x * x + y * y)};
  float Mx[9];
#pragma unroll
  for (int i = 0; i < 3; ++i)
#pragma unroll
    for (int k = 0; k < 3; ++k) Mx[i * 3 + k] = R[i * 3 + k] * scales[3 * g + k];
#define SIG(i, j) ((Mx[(i) * 3] * Mx[(j) * 3] + Mx[(i) * 3 + 1] * Mx[(j) * 3 + 1]) + Mx[(i) * 3 + 2] * Mx[(j) * 3 + 2])
  // second-stage record, 32 B: Sigma (xx,xy,xz,yy,yz,zz), opacity, tau
  g2[2 * (size_t)g] = make_float4(SIG(0, 0), SIG(0, 1), SIG(0, 2), SIG(1, 1));
  g2[2 * (size_t)g + 1] = make_float4(SIG(1, 2), SIG(2, 2), o, (float)(2.0 * log(255.0 * (double)o)));
#undef SIG
}

// ------------------------------------------------------------------ per-frame init
// counters <- 0; sort histograms <- 0; tile_flags <- 0;
// S frames: D^min <- INVALID bits, sigma^max <- 0; R / P frames: rendered_next <- 0;
// R frames: F <- (+inf, +inf, -inf, -inf).
__global__ void __launch_bounds__(256) k_frame_init(FrameConst fc, Counters* counters, uint32_t* tile_flags, uint2* warp_tgb,
                                                    uint32_t* rendered_next_words, uint32_t n_words,
                                                    uint32_t* sort_hist, uint2* ranges, uint8_t* tile_mask, uint32_t* tile_order, uint32_t* sel_bits,
                                                    uint32_t* live_bits, uint32_t* F_key, int reset_F) {
  TGS_PDL_WAIT();
  TGS_PDL_TRIGGER();
  const uint32_t tid = blockIdx.x * blockDim.x + threadIdx.x, nth = gridDim.x * blockDim.x;
  // R / P frames select every tile and carry no T^oc / T^um flags: the outputs of k_select are written here
  const bool trivial_sel = fc.ftype != TGS_FRAME_S;
  if (tid < sizeof(Counters) / 4) ((uint32_t*)counters)[tid] = (trivial_sel && tid == offsetof(Counters, n_sel) / 4) ? (uint32_t)fc.n_tiles : 0u;
  if (reset_F && tid < 4) F_key[tid] = (tid < 2) ? 0xff800000u /* key(+inf) */ : 0x007fffffu /* key(-inf) */;
  for (uint32_t i = tid; i < (uint32_t)fc.n_tiles; i += nth) {
    tile_flags[i] = 0; ranges[i] = make_uint2(0u, 0u);
    if (trivial_sel) { tile_mask[i] = 4; tile_order[i] = i; if ((i & 31u) == 0u) { sel_bits[i >> 5] = 0xffffffffu; live_bits[i >> 5] = 0xffffffffu; } }
  }
  if (tid < (1 + TGS_MAX_SLABS) * 4 * 256) sort_hist[tid] = 0;
  if (fc.do_tgb) {
    const uint32_t px = (uint32_t)(fc.tg.W * fc.tg.H);
    for (uint32_t i = tid; i < px; i += nth) warp_tgb[i] = make_uint2(TGS_INVALID_BITS, 0u);
  }
  if (rendered_next_words)
    for (uint32_t i = tid; i < n_words; i += nth) rendered_next_words[i] = 0;
}

// ------------------------------------------------------------------ A1 forward warp
// One thread per reference pixel.  Nearest-pixel splat (R14) with atomicMin on the depth bits (positive
// floats order like their bit patterns) and atomicMax on the sigma bits: min depth and max sigma are kept
// independently (L91, L97; R15), so the result does not depend on the order of arrival.
__global__ void __launch_bounds__(256) k_warp(FrameConst fc, const float* __restrict__ prior_depth,
                                              const float* __restrict__ prior_sigma, uint2* __restrict__ warp_tgb) {
  TGS_PDL_WAIT();
  const int x = blockIdx.x * 32 + (threadIdx.x & 31), y = blockIdx.y * 8 + (threadIdx.x >> 5);
  const CamConst& kc = fc.cam;
  const TgbGrid& k = fc.tg;
  if (x >= k.W || y >= k.H) return;
  float D, sg;
  if (k.ds == 1) { D = prior_depth[(size_t)y * kc.W + x]; sg = prior_sigma[(size_t)y * kc.W + x]; }
  else {                                                          // R43: 2x2 block, nearest valid depth / largest sigma
    D = TGS_DEPTH_INVALID; sg = 0.0f;
#pragma unroll
    for (int j = 0; j < 2; ++j)
#pragma unroll
      for (int i = 0; i < 2; ++i) {
        const int xx = 2 * x + i, yy = 2 * y + j;
        if (xx >= kc.W || yy >= kc.H) continue;
        const float v = prior_depth[(size_t)yy * kc.W + xx];
        if (!(v < 1.0e38f)) continue;
        D = fminf(D, v); sg = fmaxf(sg, prior_sigma[(size_t)yy * kc.W + xx]);
      }
  }
  if (!(D < 1.0e38f)) return;                                   // R11
  const float* M = fc.M;
  const float rx = ((float)x - k.cx) / k.fx, ry = ((float)y - k.cy) / k.fy;
  const float Px = D * rx, Py = D * ry, Pz = D;
  const float X = ((M[0] * Px + M[1] * Py) + M[2] * Pz) + M[3];
  const float Y = ((M[4] * Px + M[5] * Py) + M[6] * Pz) + M[7];
  const float Z = ((M[8] * Px + M[9] * Py) + M[10] * Pz) + M[11];
  if (!(Z > kc.znear)) return;
  const float u = (k.fx * X) / Z + k.cx, v = (k.fy * Y) / Z + k.cy;
  const float fu = floorf(u + 0.5f), fv = floorf(v + 0.5f);
  if (!(fu >= 0.0f && fu < k.Wf && fv >= 0.0f && fv < k.Hf)) return;
  const size_t q = (size_t)(int)fv * k.W + (int)fu;
  const float s = sg * fabsf((M[8] * rx + M[9] * ry) + M[10]);   // R13
  atomicMin(&warp_tgb[q].x, __float_as_uint(Z));       // {D^min, sigma^max} interleaved: one 8-byte word per TOC lookup
  if (s > 0.0f) atomicMax(&warp_tgb[q].y, __float_as_uint(s));
}

// ------------------------------------------------------------------ A2 depth fill + correspondence + T^um
// One CTA per tile, one thread per pixel.  D' = D^min with isolated holes filled by the mean of the 8
// neighbours (L121; R19).  matched <=> D' valid, back-projected z > z_near and the nearest reference pixel
// is inside the image (R20).  Tile in T^um <=> any in-image pixel unmatched (R22).
__global__ void __launch_bounds__(256) k_fill_corr(FrameConst fc, const float2* __restrict__ warp_tgb, float* __restrict__ fill_depth,
                                                   uint32_t* __restrict__ tile_flags) {
  TGS_PDL_WAIT();
  const TgbGrid& k = fc.tg;
  const float znear = fc.cam.znear;
  const int edge = TGS_TILE / k.ds;                              // a tile is edge x edge grid pixels (R43)
  const int lx = threadIdx.x % edge, ly = threadIdx.x / edge;
  const int x = blockIdx.x * edge + lx, y = blockIdx.y * edge + ly;
  const bool inside = ly < edge && x < k.W && y < k.H;
  bool unmatched = false;
  if (inside) {
    const float2* wd = warp_tgb;
    float D = wd[(size_t)y * k.W + x].x;
    if (!(D < 1.0e38f) && x > 0 && y > 0 && x < k.W - 1 && y < k.H - 1) {
      const float n0 = wd[(size_t)(y - 1) * k.W + x - 1].x, n1 = wd[(size_t)(y - 1) * k.W + x].x, n2 = wd[(size_t)(y - 1) * k.W + x + 1].x;
      const float n3 = wd[(size_t)y * k.W + x - 1].x, n4 = wd[(size_t)y * k.W + x + 1].x;
      const float n5 = wd[(size_t)(y + 1) * k.W + x - 1].x, n6 = wd[(size_t)(y + 1) * k.W + x].x, n7 = wd[(size_t)(y + 1) * k.W + x + 1].x;
      if (n0 < 1.0e38f && n1 < 1.0e38f && n2 < 1.0e38f && n3 < 1.0e38f && n4 < 1.0e38f && n5 < 1.0e38f && n6 < 1.0e38f && n7 < 1.0e38f)
        D = (((((((n0 + n1) + n2) + n3) + n4) + n5) + n6) + n7) * 0.125f;
    }
    fill_depth[(size_t)y * k.W + x] = D;
    unmatched = true;
    if (D < 1.0e38f) {
      const float* M = fc.Minv;
      const float rx = ((float)x - k.cx) / k.fx, ry = ((float)y - k.cy) / k.fy;
      const float Px = D * rx, Py = D * ry, Pz = D;
      const float X = ((M[0] * Px + M[1] * Py) + M[2] * Pz) + M[3];
      const float Y = ((M[4] * Px + M[5] * Py) + M[6] * Pz) + M[7];
      const float Z = ((M[8] * Px + M[9] * Py) + M[10] * Pz) + M[11];
      if (Z > znear) {
        const float xs = (k.fx * X) / Z + k.cx, ys = (k.fy * Y) / Z + k.cy;
        const float fu = floorf(xs + 0.5f), fv = floorf(ys + 0.5f);
        if (fu >= 0.0f && fu < k.Wf && fv >= 0.0f && fv < k.Hf) unmatched = false;
      }
    }
  }
  const int any = __syncthreads_or(unmatched ? 1 : 0);
  if (threadIdx.x == 0 && any) atomicOr(&tile_flags[blockIdx.y * fc.cam.TX + blockIdx.x], 2u);   // bit1 = T^um (k_preprocess ORs bit0 concurrently)
}

}  // namespace

namespace {

// T^oc test of one (newly visible Gaussian, tile) pair: max alpha over the tile's pixel-centre box >= 1/255
// <=> box_qmin <= tau (L119, R18).  The mark is an OR, so the order of evaluation does not matter.
__device__ __forceinline__ void mark_oc_tile(const CamConst& k, float u, float v, float A, float B, float C, float tau, uint32_t txx,
                                             uint32_t tyy, uint32_t* __restrict__ tile_flags, Counters* __restrict__ counters) {
  const uint32_t t = tyy * k.TX + txx;
  if (*reinterpret_cast<volatile uint32_t*>(&tile_flags[t]) & 1u) return;
  const float bx0 = (float)(txx * TGS_TILE), bx1 = (float)min((int)(txx * TGS_TILE + TGS_TILE - 1), k.W - 1);
  const float by0 = (float)(tyy * TGS_TILE), by1 = (float)min((int)(tyy * TGS_TILE + TGS_TILE - 1), k.H - 1);
  if (box_qmin(u, v, A, B, C, bx0, bx1, by0, by1) <= tau)
    if (!(atomicOr(&tile_flags[t], 1u) & 1u)) atomicAdd(&counters->n_oc_marked, 1u);
}

// Newly visible Gaussians with rects of more than 4 tiles (queued by k_preprocess): one CTA per Gaussian, threads
// over the tiles of the rect (a near Gaussian covers thousands).  Stops as soon as every tile carries the mark.
__global__ void __launch_bounds__(128) k_mark_oc(FrameConst fc, const uint32_t* __restrict__ nv_queue, const float4* __restrict__ rec_bin,
                                                 uint32_t* __restrict__ tile_flags, Counters* __restrict__ counters) {
  TGS_PDL_WAIT();
  TGS_PDL_TRIGGER();
  const CamConst& k = fc.cam;
  const uint32_t nq = counters->n_nv_queue;
  for (uint32_t j = blockIdx.x; j < nq; j += gridDim.x) {
    if (*reinterpret_cast<volatile uint32_t*>(&counters->n_oc_marked) >= (uint32_t)fc.n_tiles) break;
    const uint32_t g = nv_queue[j];
    const float4 q0 = rec_bin[2 * (size_t)g], q1 = rec_bin[2 * (size_t)g + 1];      // {u, v, A, B}, {C, tau, test rect}: one sector
    const float4 r0 = make_float4(q0.x, q0.y, 0.0f, 0.0f), r1 = make_float4(q0.z, q0.w, q1.x, q1.y);
    const uint2 r = make_uint2(__float_as_uint(q1.z), __float_as_uint(q1.w));
    const uint32_t x_lo = r.x & 0xffffu, x_hi = r.x >> 16, y_lo = r.y & 0xffffu, y_hi = r.y >> 16;
    const uint32_t w = x_hi - x_lo, area = w * (y_hi - y_lo);
    for (uint32_t i = threadIdx.x; i < area; i += blockDim.x) {
      const uint32_t ry = i / w;
      mark_oc_tile(k, r0.x, r0.y, r1.x, r1.y, r1.z, r1.w, x_lo + (i - ry * w), y_lo + ry, tile_flags, counters);
    }
  }
}

// ------------------------------------------------------------------ A3 preprocess (+AFC +TOC +newly-visible +T^oc)
// Persistent grid; a work item is a chunk of 2048 consecutive Gaussians (ticket order): two phase-A passes of 1024, 4 per thread.
//  phase A (all Gaussians, 16 B each): near cull, projection of the mean, AFC, TOC + newly-visible lookups in the
//          warped TGB, and a conservative off-screen test; the survivors are compacted in shared memory;
//  phase B (survivors only, +32 B each): EWA covariance, conic, radius, rect, records, T^oc marks of small rects;
//  phase C: the visible Gaussians of the chunk go, compacted, to the chunk's own 2048 slots of a staging list, and the
//          chunk's count to pre_cnt; the CTA that finishes last scans the counts; k_compact_vis then closes the gaps.
//          The list the depth sort works on is thus in ascending index order (equal depths stay in index order
//          through the stable sort, R28) and no chunk waits for another one.
// SH (the bulk of the scene bytes) is not touched here at all.  Order of the tests and of every fp32 operation of a
// decision: DESIGN.md §2 (O3), identical to what the oracle states.
//
// Off-screen test (an early-out, never a different decision): with s = the largest scale, lambda_max(Sigma') <=
// |J|_F^2 s^2 + 0.3 and |J row|^2 <= (f/z)^2 (1 + lim^2) because the Jacobian's x/z, y/z are clamped to +-lim (R3), so
// r <= 3 sqrt(lambda_b + 0.32) + 1.  A Gaussian whose centre is further outside the tile grid than this bound has an
// empty rect.  It is only applied when lambda_b <= 1e4: then det(Sigma') >= 0.3 (a + c) - rounding(1e-6 a c) > 0, so
// the Gaussian cannot be one the full computation would have flagged DEGENERATE instead of EMPTY.
constexpr int PRE_THREADS = 256;
constexpr int PRE_IPT = 4;
constexpr int PRE_SUB = 2;                 // phase A passes per work item: phases B / C then run on the survivors of all of them
constexpr int PRE_EPT = PRE_IPT * PRE_SUB; // list entries per thread in phase C
constexpr int PRE_CHUNK = PRE_THREADS * PRE_IPT * PRE_SUB;
static_assert(PRE_CHUNK <= 4096, "12-bit local index in PreSmem::list");

struct PreSmem {
  uint16_t list[PRE_CHUNK];     // survivors of phase A: local index | newly-visible << 15 | visible << 14
  uint32_t depth[PRE_CHUNK];    // bits(d) of the visible survivors (indexed like list)
  uint32_t warp[PRE_THREADS / 32];
  uint32_t excl, chunk, nsurv;
  uint32_t stat[8];
  unsigned long long area;
  uint32_t hist[4][256];        // digit histograms of the depth keys of the visible Gaussians (for the depth sort)
};

__global__ void __launch_bounds__(PRE_THREADS, 4) k_preprocess(FrameConst fc, const float4* __restrict__ cull4, const float4* __restrict__ g2,
                                                               const uint8_t* __restrict__ rendered, const float2* __restrict__ warp_tgb,
                                                               const uint32_t* __restrict__ F_key,
                                                               float4* __restrict__ rec_bin,
                                                               uint8_t* __restrict__ rec_flags,
                                                               float4* __restrict__ rec_b0, float4* __restrict__ rec_b1,
                                                               uint32_t* __restrict__ tile_flags, uint32_t* __restrict__ nv_queue,
                                                               uint32_t* __restrict__ vis_keys,
                                                               uint32_t* __restrict__ vis_vals, uint2* __restrict__ pre_cnt,
                                                               uint32_t* __restrict__ depth_hist, Counters* __restrict__ counters) {
  TGS_PDL_WAIT();
  TGS_PDL_TRIGGER();
  __shared__ PreSmem sm;
  const CamConst& k = fc.cam;
  const float* V = k.V;
  const uint32_t tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  const uint32_t num_chunks = (fc.n + PRE_CHUNK - 1) / PRE_CHUNK;
  float F0 = 0.f, F1 = 0.f, F2 = 0.f, F3 = 0.f;
  if (fc.do_afc) { F0 = key2f(F_key[0]); F1 = key2f(F_key[1]); F2 = key2f(F_key[2]); F3 = key2f(F_key[3]); }
  const uint32_t ds_shift = fc.tg.ds == 2 ? 1u : 0u;
  const float offx = 1.0f + k.limx * k.limx, offy = 1.0f + k.limy * k.limy;
  const float xmax = (float)(k.TX * TGS_TILE) + 2.0f, ymax = (float)(k.TY * TGS_TILE) + 2.0f;
  uint32_t st_near = 0, st_afc = 0, st_toc = 0, st_deg = 0, st_empty = 0, st_nv = 0;
  unsigned long long st_area = 0;
  if (tid < 8) sm.stat[tid] = 0;
  if (tid == 0) sm.area = 0;
  for (int i = tid; i < 4 * 256; i += PRE_THREADS) (&sm.hist[0][0])[i] = 0;
  while (true) {
    __syncthreads();
    if (tid == 0) sm.chunk = atomicAdd(&counters->ticket_pre, 1u);
    __syncthreads();
    const uint32_t chunk = sm.chunk;
    if (chunk >= num_chunks) break;
    const uint32_t base = chunk * PRE_CHUNK;
    // ---------------------------------------------------------------- phase A
    uint32_t total = 0;
   for (int sub = 0; sub < PRE_SUB; ++sub) {
    const uint32_t g0 = base + (uint32_t)sub * (PRE_THREADS * PRE_IPT) + tid * PRE_IPT;
    float4 c4[PRE_IPT];
#pragma unroll
    for (int j = 0; j < PRE_IPT; ++j) c4[j] = (g0 + j < fc.n) ? cull4[g0 + j] : make_float4(0.f, 0.f, 0.f, 0.f);
    uint32_t rend4 = 0;
    if (fc.do_tgb && g0 < fc.n) rend4 = *reinterpret_cast<const uint32_t*>(rendered + g0);   // g0 % 4 == 0; padded allocation
    uint32_t surv = 0;      // 4 x {bit0 survivor, bit1 newly visible}
    uint32_t cf[PRE_IPT] = {0u, 0u, 0u, 0u};   // flags of the Gaussians culled in phase A (survivors: written in phase B)
#pragma unroll
    for (int j = 0; j < PRE_IPT; ++j) {
      const uint32_t g = g0 + j;
      if (g >= fc.n) continue;
      const float x = c4[j].x, y = c4[j].y, z = c4[j].z;
      const float tx = ((V[0] * x + V[1] * y) + V[2] * z) + V[3];
      const float ty = ((V[4] * x + V[5] * y) + V[6] * z) + V[7];
      const float tz = ((V[8] * x + V[9] * y) + V[10] * z) + V[11];
      if (!(tz > k.znear)) { cf[j] = TGS_CULL_NEAR; ++st_near; continue; }                 // L61, R4
      const float u = (k.fx * tx) / tz + k.cx, v = (k.fy * ty) / tz + k.cy;
      if (fc.do_afc) {                                                                            // L109-111
        const float nx = (2.0f * u + 1.0f) / k.Wf - 1.0f, ny = (2.0f * v + 1.0f) / k.Hf - 1.0f;
        if (!(F0 <= nx && nx <= F2 && F1 <= ny && ny <= F3)) { cf[j] = TGS_CULL_AFC; ++st_afc; continue; }
      }
      uint32_t fl = 0;
      const float fu = floorf(u + 0.5f), fv = floorf(v + 0.5f);
      const bool centre_in = fu >= 0.0f && fu < k.Wf && fv >= 0.0f && fv < k.Hf;
      if (fc.do_tgb && !((rend4 >> (8 * j)) & 0xffu) && centre_in) {                              // L113, L119
        const uint32_t q = ((uint32_t)(int)fv >> ds_shift) * (uint32_t)fc.tg.W + ((uint32_t)(int)fu >> ds_shift);   // R43: block of the nearest pixel
        const float2 Ds = warp_tgb[q];                                // {D^min, sigma^max}: one 8-byte word per lookup
        const float D = Ds.x, s = Ds.y;
        if (fc.do_toc && tz > D + fc.lambda2 * s) { cf[j] = TGS_CULL_TOC; ++st_toc; continue; }
        if (tz <= D - fc.lambda1 * s) fl = 2u;
      }
      if (!centre_in) {                                                                           // provably empty rect
        const float kx = k.fx / tz, ky = k.fy / tz;
        const float lam_b = (((kx * kx) * offx + (ky * ky) * offy) * (c4[j].w * c4[j].w)) * 1.02f + 0.7f;
        if (lam_b <= 1.0e4f) {
          const float rb = 3.03f * sqrtf(lam_b) + 3.0f;
          if (u + rb < -17.0f || v + rb < -17.0f || u - rb > xmax || v - rb > ymax) { cf[j] = TGS_CULL_EMPTY; ++st_empty; continue; }
        }
      }
      surv |= (1u | fl) << (2 * j);
      asm volatile("prefetch.global.L2 [%0];" ::"l"(g2 + 2 * (size_t)g));   // phase B reads the covariance of this survivor
    }
    // one byte per Gaussian (the flags fit in seven bits): 4 N bytes a frame less to write than with words
    if (g0 + PRE_IPT <= fc.n) *reinterpret_cast<uchar4*>(rec_flags + g0) = make_uchar4((uint8_t)cf[0], (uint8_t)cf[1], (uint8_t)cf[2], (uint8_t)cf[3]);
    else
      for (int j = 0; j < PRE_IPT; ++j) if (g0 + j < fc.n) rec_flags[g0 + j] = (uint8_t)cf[j];
    // survivors -> sm.list, in ascending index order
    const uint32_t ns_t = (surv & 1u) + ((surv >> 2) & 1u) + ((surv >> 4) & 1u) + ((surv >> 6) & 1u);
    uint32_t incl = ns_t;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) { const uint32_t o = __shfl_up_sync(0xffffffffu, incl, d); if (lane >= (uint32_t)d) incl += o; }
    if (lane == 31) sm.warp[wid] = incl;
    __syncthreads();
    uint32_t pos = total + incl - ns_t, sub_total = 0;
#pragma unroll
    for (int w = 0; w < PRE_THREADS / 32; ++w) { const uint32_t t = sm.warp[w]; if ((uint32_t)w < wid) pos += t; sub_total += t; }
#pragma unroll
    for (int j = 0; j < PRE_IPT; ++j)
      if ((surv >> (2 * j)) & 1u) sm.list[pos++] = (uint16_t)((sub * (PRE_THREADS * PRE_IPT) + tid * PRE_IPT + j) | (((surv >> (2 * j + 1)) & 1u) << 15));
    total += sub_total;
    __syncthreads();
   }
    // ---------------------------------------------------------------- phase B
    for (uint32_t i = tid; i < total; i += PRE_THREADS) {
      const uint32_t e = sm.list[i];
      const uint32_t g = base + (e & 0xfffu);
      const uint32_t fl = (e >> 15) ? TGS_NEWLY_VISIBLE : 0u;
      const float4 c = cull4[g];
      const float4 ga = g2[2 * (size_t)g], gb = g2[2 * (size_t)g + 1];
      const float x = c.x, y = c.y, z = c.z;
      const float tx = ((V[0] * x + V[1] * y) + V[2] * z) + V[3];
      const float ty = ((V[4] * x + V[5] * y) + V[6] * z) + V[7];
      const float tz = ((V[8] * x + V[9] * y) + V[10] * z) + V[11];
      const float u = (k.fx * tx) / tz + k.cx, v = (k.fy * ty) / tz + k.cy;
      const float S0 = ga.x, S1 = ga.y, S2 = ga.z, S3 = ga.w, S4 = gb.x, S5 = gb.y, opac = gb.z, tau = gb.w;
      const float rxz = tx / tz, ryz = ty / tz;
      const float jx = fminf(k.limx, fmaxf(-k.limx, rxz)) * tz;
      const float jy = fminf(k.limy, fmaxf(-k.limy, ryz)) * tz;
      const float j00 = k.fx / tz, j02 = -(k.fx * jx) / (tz * tz);
      const float j11 = k.fy / tz, j12 = -(k.fy * jy) / (tz * tz);
      const float T00 = j00 * V[0] + j02 * V[8], T01 = j00 * V[1] + j02 * V[9], T02 = j00 * V[2] + j02 * V[10];
      const float T10 = j11 * V[4] + j12 * V[8], T11 = j11 * V[5] + j12 * V[9], T12 = j11 * V[6] + j12 * V[10];
      const float a0 = (S0 * T00 + S1 * T01) + S2 * T02;
      const float a1 = (S1 * T00 + S3 * T01) + S4 * T02;
      const float a2 = (S2 * T00 + S4 * T01) + S5 * T02;
      const float q0 = (S0 * T10 + S1 * T11) + S2 * T12;
      const float q1 = (S1 * T10 + S3 * T11) + S4 * T12;
      const float q2 = (S2 * T10 + S4 * T11) + S5 * T12;
      const float a = ((T00 * a0 + T01 * a1) + T02 * a2) + 0.3f;
      const float b = (T10 * a0 + T11 * a1) + T12 * a2;
      const float cc = ((T10 * q0 + T11 * q1) + T12 * q2) + 0.3f;
      const float det = a * cc - b * b;
      if (!(det > 0.0f)) { rec_flags[g] = (uint8_t)TGS_CULL_DEGENERATE; ++st_deg; continue; }
      const float A = cc / det, B = -b / det, C = a / det;
      const float mid = 0.5f * (a + cc);
      const float lam = mid + sqrtf(fmaxf(0.1f, mid * mid - det));
      const float rad = ceilf(3.0f * sqrtf(lam));
      const float TXf = (float)k.TX, TYf = (float)k.TY;
      uint32_t x_lo, x_hi, y_lo, y_hi;
      tile_rect(u, v, rad, TXf, TYf, x_lo, x_hi, y_lo, y_hi);
      if (!(x_hi > x_lo && y_hi > y_lo)) { rec_flags[g] = (uint8_t)TGS_CULL_EMPTY; ++st_empty; continue; }
      rec_flags[g] = (uint8_t)(fl | TGS_VISIBLE);
      if (fl) ++st_nv;
      // Test rect (never a different decision): the tiles of the 3-sigma rect that can reach alpha >= 1/255 lie inside the
      // bounding box of the ellipse q <= tau, |dx| <= sqrt(tau a), |dy| <= sqrt(tau c) (min over dy of q = dx^2 / a).  A tile
      // wholly outside that box, enlarged by 1 %, has q_min >= 1.02 tau in exact arithmetic, and the fp32 evaluation of the
      // oracle differs from it by at most ~1e-6 (18 kappa + 1700) -- below 0.02 tau when cond(Sigma') <= 400 and tau >= 0.5
      // (DESIGN.md §7).  Otherwise, and when the box would be empty, the whole rect is kept (or one tile of it).
      // exact_tiles = 0 (tgs.h): "intersect" = every tile of the 3-sigma rect, so the test rect IS the rect.
      uint32_t tx_lo = x_lo, tx_hi = x_hi, ty_lo = y_lo, ty_hi = y_hi;
      if (!fc.exact_tiles) {}
      else if (!(tau >= 0.0f)) { tx_hi = x_lo + 1u; ty_hi = y_lo + 1u; }         // o < 1/255: reaches nothing; one (failing) test
      else if (tau >= 0.5f && lam * lam <= 400.0f * det) {
        const float ex = sqrtf(tau * a) * 1.01f + 0.01f, ey = sqrtf(tau * cc) * 1.01f + 0.01f;
        const float fx_lo = ceilf((u - ex - 15.0f) / 16.0f), fx_hi = floorf((u + ex) / 16.0f) + 1.0f;
        const float fy_lo = ceilf((v - ey - 15.0f) / 16.0f), fy_hi = floorf((v + ey) / 16.0f) + 1.0f;
        const uint32_t nx_lo = (uint32_t)fminf(fmaxf(fx_lo, (float)x_lo), (float)x_hi), nx_hi = (uint32_t)fminf(fmaxf(fx_hi, (float)x_lo), (float)x_hi);
        const uint32_t ny_lo = (uint32_t)fminf(fmaxf(fy_lo, (float)y_lo), (float)y_hi), ny_hi = (uint32_t)fminf(fmaxf(fy_hi, (float)y_lo), (float)y_hi);
        if (nx_hi > nx_lo && ny_hi > ny_lo) { tx_lo = nx_lo; tx_hi = nx_hi; ty_lo = ny_lo; ty_hi = ny_hi; }
        else { tx_hi = x_lo + 1u; ty_hi = y_lo + 1u; }
      }
      rec_bin[2 * (size_t)g] = make_float4(u, v, A, B);           // what A5a gathers behind the depth sort, in one sector
      rec_bin[2 * (size_t)g + 1] = make_float4(C, tau, __uint_as_float(tx_lo | (tx_hi << 16)), __uint_as_float(ty_lo | (ty_hi << 16)));
      const uint32_t area = (tx_hi - tx_lo) * (ty_hi - ty_lo);
      st_area += area;
      // blend-side parameters: the quadratic form as a sum of two squares (no cancellation between its terms)
      rec_b0[2 * (size_t)g] = make_float4(u, v, -0.72134752f * A, -b / cc);        // b0 / b1 interleaved: one 32-byte sector per Gaussian, written whole
      rec_b1[2 * (size_t)g] = make_float4(-0.72134752f / cc, log2f(opac), tz, rad);            // (.w is not read by the blend: it serves the test-only views -- the 3-sigma rect is tile_rect(u, v, rad), the decision record {u, v, d, o | A, B, C, tau} is rec_bin + d + the scene's opacity)
      sm.list[i] = (uint16_t)(e | 0x4000u);
      sm.depth[i] = __float_as_uint(tz);
      if (fl && tau >= 0.0f) {                                                      // A4: T^oc (L119, R18)
        if (area > 4u) nv_queue[atomicAdd(&counters->n_nv_queue, 1u)] = g;         // larger rects: k_mark_oc
        else
          for (uint32_t tyy = ty_lo; tyy < ty_hi; ++tyy)
            for (uint32_t txx = tx_lo; txx < tx_hi; ++txx) mark_oc_tile(k, u, v, A, B, C, tau, txx, tyy, tile_flags, counters);
      }
    }
    __syncthreads();
    // ---------------------------------------------------------------- phase C: visible list, ascending index
    uint32_t nv_t = 0;
#pragma unroll
    for (int j = 0; j < PRE_EPT; ++j) { const uint32_t i = tid * PRE_EPT + j; if (i < total && (sm.list[i] & 0x4000u)) ++nv_t; }
    uint32_t vincl = nv_t;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) { const uint32_t o = __shfl_up_sync(0xffffffffu, vincl, d); if (lane >= (uint32_t)d) vincl += o; }
    if (lane == 31) sm.warp[wid] = vincl;
    __syncthreads();
    uint32_t off = vincl - nv_t, vtotal = 0;
#pragma unroll
    for (int w = 0; w < PRE_THREADS / 32; ++w) { const uint32_t t = sm.warp[w]; if ((uint32_t)w < wid) off += t; vtotal += t; }
    if (tid == 0) pre_cnt[chunk].x = vtotal;
    off += base;                                             // staging slots of this chunk
#pragma unroll
    for (int j = 0; j < PRE_EPT; ++j) {
      const uint32_t i = tid * PRE_EPT + j;
      if (i < total && (sm.list[i] & 0x4000u)) {
        const uint32_t key = sm.depth[i];
        vis_keys[off] = key; vis_vals[off] = base + (sm.list[i] & 0xfffu); ++off;
        atomicAdd(&sm.hist[0][key & 255u], 1u); atomicAdd(&sm.hist[1][(key >> 8) & 255u], 1u);
        atomicAdd(&sm.hist[2][(key >> 16) & 255u], 1u); atomicAdd(&sm.hist[3][key >> 24], 1u);
      }
    }
  }
  // ---- the last CTA to arrive: exclusive scan of the chunks' visible counts (pre_cnt = {count, offset}), N_v
  __threadfence();
  __syncthreads();
  if (tid == 0) sm.excl = (atomicAdd(&counters->pre_done, 1u) == gridDim.x - 1u) ? 1u : 0u;
  __syncthreads();
  if (sm.excl) {
    __threadfence();
    const uint32_t per = (num_chunks + PRE_THREADS - 1) / PRE_THREADS;
    const uint32_t c0 = tid * per, c1 = min(num_chunks, c0 + per);
    uint32_t sum = 0;
    for (uint32_t c = c0; c < c1; ++c) sum += *reinterpret_cast<volatile uint32_t*>(&pre_cnt[c].x);
    uint32_t incl = sum;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) { const uint32_t o = __shfl_up_sync(0xffffffffu, incl, d); if (lane >= (uint32_t)d) incl += o; }
    if (lane == 31) sm.warp[wid] = incl;
    __syncthreads();
    uint32_t off = incl - sum, tot = 0;
    for (int w = 0; w < PRE_THREADS / 32; ++w) { if ((uint32_t)w < wid) off += sm.warp[w]; tot += sm.warp[w]; }
    for (uint32_t c = c0; c < c1; ++c) { const uint32_t v = *reinterpret_cast<volatile uint32_t*>(&pre_cnt[c].x); pre_cnt[c].y = off; off += v; }
    if (tid == 0) counters->n_visible = tot;
    __syncthreads();
  }
  // statistics: one atomic per CTA and class
  st_near = warp_sum(st_near); st_afc = warp_sum(st_afc); st_toc = warp_sum(st_toc); st_deg = warp_sum(st_deg);
  st_empty = warp_sum(st_empty); st_nv = warp_sum(st_nv);
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) st_area += __shfl_xor_sync(0xffffffffu, st_area, d);
  if (lane == 0) {
    if (st_near) atomicAdd(&sm.stat[0], st_near);
    if (st_afc) atomicAdd(&sm.stat[1], st_afc);
    if (st_toc) atomicAdd(&sm.stat[2], st_toc);
    if (st_deg) atomicAdd(&sm.stat[3], st_deg);
    if (st_empty) atomicAdd(&sm.stat[4], st_empty);
    if (st_nv) atomicAdd(&sm.stat[6], st_nv);
    if (st_area) atomicAdd(&sm.area, st_area);
  }
  __syncthreads();
  for (int i = tid; i < 4 * 256; i += PRE_THREADS) { const uint32_t h = (&sm.hist[0][0])[i]; if (h) atomicAdd(&depth_hist[i], h); }
  if (tid == 0) {
    if (sm.stat[0]) atomicAdd(&counters->n_near, sm.stat[0]);
    if (sm.stat[1]) atomicAdd(&counters->n_afc, sm.stat[1]);
    if (sm.stat[2]) atomicAdd(&counters->n_toc, sm.stat[2]);
    if (sm.stat[3]) atomicAdd(&counters->n_degenerate, sm.stat[3]);
    if (sm.stat[4]) atomicAdd(&counters->n_empty, sm.stat[4]);
    if (sm.stat[6]) atomicAdd(&counters->n_newly_visible, sm.stat[6]);
    if (sm.area) atomicAdd(&counters->area_sum, sm.area);
  }
}

// Visible list: the chunks' runs from the staging list (2048 slots per chunk) to their offsets (ascending index order).
// The indices also go to `vis_list`, a copy the depth sort does not permute (SH colours).
__global__ void __launch_bounds__(128) k_compact_vis(uint32_t n, const uint2* __restrict__ pre_cnt, const uint32_t* __restrict__ st_keys,
                                                     const uint32_t* __restrict__ st_vals, uint32_t* __restrict__ vis_keys,
                                                     uint32_t* __restrict__ vis_vals, uint32_t* __restrict__ vis_list,
                                                     uint32_t* __restrict__ dsort_H0, uint32_t dsort_tile) {
  TGS_PDL_WAIT();
  TGS_PDL_TRIGGER();
  const uint32_t num_chunks = (n + PRE_CHUNK - 1) / PRE_CHUNK;
  for (uint32_t c = blockIdx.x; c < num_chunks; c += gridDim.x) {
    const uint2 cc = pre_cnt[c];
    for (uint32_t i = threadIdx.x; i < cc.x; i += blockDim.x) {
      const uint32_t g = st_vals[(size_t)c * PRE_CHUNK + i];
      const uint32_t key = st_keys[(size_t)c * PRE_CHUNK + i];
      vis_keys[cc.y + i] = key;
      vis_vals[cc.y + i] = g; vis_list[cc.y + i] = g;
      // one-launch depth sort (k_sort.cu): digit counts of its first pass, per sort tile
      if (dsort_H0) atomicAdd(dsort_H0 + (size_t)((cc.y + i) / dsort_tile) * 256u + (key & 255u), 1u);
    }
  }
}

// ------------------------------------------------------------------ A4 tile selection: T_sel = T^oc U T^um (L123)
// One CTA of 1024 threads, each owning a run of consecutive tiles (a multiple of 32, so a thread writes whole words
// of the bit set).  Builds the tile mask, the bit set used by the pair binning, and the work order of the blend
// kernel: selected tiles first (ascending id), then the tiles that are only stitched.
__global__ void __launch_bounds__(1024) k_select(FrameConst fc, const uint32_t* __restrict__ tile_flags, uint8_t* __restrict__ tile_mask,
                                                 uint32_t* __restrict__ sel_bits, uint32_t* __restrict__ live_bits, uint32_t* __restrict__ tile_order,
                                                 Counters* __restrict__ counters, volatile uint32_t* __restrict__ host_n_sel) {
  TGS_PDL_WAIT();
  TGS_PDL_TRIGGER();
  __shared__ uint32_t s_sel[32], s_oc[32], s_um[32];
  const int T = fc.n_tiles;
  const uint32_t lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  // a warp owns a run of consecutive 32-tile words; a lane owns one tile of a word (coalesced loads, ballots)
  const int words = (T + 31) / 32, wpw = (words + 31) / 32;
  const int w0 = min(words, (int)wid * wpw), w1 = min(words, w0 + wpw);
  uint32_t nsel = 0, noc = 0, num = 0;                     // warp-uniform
  for (int w = w0; w < w1; ++w) {
    const int t = w * 32 + (int)lane;
    const uint32_t f = t < T ? tile_flags[t] & 3u : 0u;
    const bool sel = t < T && (fc.all_tiles || f != 0);
    if (t < T) tile_mask[t] = (uint8_t)(f | (sel ? 4u : 0u));
    const uint32_t word = __ballot_sync(0xffffffffu, sel);
    if (lane == 0) { sel_bits[w] = word; live_bits[w] = word; }
    nsel += __popc(word);
    noc += __popc(__ballot_sync(0xffffffffu, (f & 1u) != 0)); num += __popc(__ballot_sync(0xffffffffu, (f & 2u) != 0));
  }
  if (lane == 0) { s_sel[wid] = nsel; s_oc[wid] = noc; s_um[wid] = num; }
  __syncthreads();
  uint32_t before = 0, total = 0, toc = 0, tum = 0;
#pragma unroll
  for (int w = 0; w < 32; ++w) { const uint32_t v = s_sel[w]; if ((uint32_t)w < wid) before += v; total += v; toc += s_oc[w]; tum += s_um[w]; }
  if (threadIdx.x == 0) {
    counters->n_sel = total; counters->n_sel_oc = toc; counters->n_sel_um = tum;
    // the eta rule needs this count on the host (A0): a zero-copy store into pinned host memory -- a D2H memcpy would
    // queue behind an image read-back in flight on the copy engine
    if (host_n_sel) { *host_n_sel = total; __threadfence_system(); }
  }
  // work order of the blend: the selected tiles in ascending id at [0, total), the others behind them in ascending id
  uint32_t ps = before;
  for (int w = w0; w < w1; ++w) {
    const int t = w * 32 + (int)lane;
    const bool sel = t < T && (fc.all_tiles || (tile_flags[t] & 3u) != 0);
    const uint32_t word = __ballot_sync(0xffffffffu, sel);
    const uint32_t rank = __popc(word & ((1u << lane) - 1u));
    if (t < T) {
      if (sel) tile_order[ps + rank] = (uint32_t)t;
      else tile_order[total + ((uint32_t)(w * 32) - ps) + (lane - rank)] = (uint32_t)t;     // unselected tiles before t: t - selected before t
    }
    ps += __popc(word);
  }
}

// ------------------------------------------------------------------ F_min / F_max over G_rendered (L109) + |G_rendered|
// Only visible Gaussians can have been blended: the reduction runs over the visible list, not over all N.
__global__ void __launch_bounds__(256) k_frustum(FrameConst fc, const uint32_t* __restrict__ vis_vals, const uint8_t* __restrict__ rendered_now,
                                                 const float4* __restrict__ rec_bin, uint32_t* __restrict__ F_key,
                                                 Counters* __restrict__ counters, int update_F) {
  TGS_PDL_WAIT();
  TGS_PDL_TRIGGER();
  uint32_t kmin_x = 0xffffffffu, kmin_y = 0xffffffffu, kmax_x = 0, kmax_y = 0, cnt = 0;
  const uint32_t nv = counters->n_visible;
  for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < nv; i += gridDim.x * blockDim.x) {
    const uint32_t g = vis_vals[i];
    if (!rendered_now[g]) continue;
    ++cnt;
    if (update_F) {
      const float4 r = rec_bin[2 * (size_t)g];                       // {u, v, A, B}
      const float nx = (2.0f * r.x + 1.0f) / fc.cam.Wf - 1.0f, ny = (2.0f * r.y + 1.0f) / fc.cam.Hf - 1.0f;
      const uint32_t kx = f2key(nx), ky = f2key(ny);
      kmin_x = min(kmin_x, kx); kmax_x = max(kmax_x, kx); kmin_y = min(kmin_y, ky); kmax_y = max(kmax_y, ky);
    }
  }
  __shared__ uint32_t s_red[5];
  if (threadIdx.x == 0) { s_red[0] = 0; s_red[1] = 0xffffffffu; s_red[2] = 0xffffffffu; s_red[3] = 0; s_red[4] = 0; }
  __syncthreads();
  cnt = warp_sum(cnt);
  kmin_x = __reduce_min_sync(0xffffffffu, kmin_x); kmin_y = __reduce_min_sync(0xffffffffu, kmin_y);
  kmax_x = __reduce_max_sync(0xffffffffu, kmax_x); kmax_y = __reduce_max_sync(0xffffffffu, kmax_y);
  if ((threadIdx.x & 31) == 0 && cnt) {
    atomicAdd(&s_red[0], cnt); atomicMin(&s_red[1], kmin_x); atomicMin(&s_red[2], kmin_y); atomicMax(&s_red[3], kmax_x); atomicMax(&s_red[4], kmax_y);
  }
  __syncthreads();
  if (threadIdx.x == 0 && s_red[0]) {
    atomicAdd(&counters->n_rendered, s_red[0]);
    if (update_F) { atomicMin(&F_key[0], s_red[1]); atomicMin(&F_key[1], s_red[2]); atomicMax(&F_key[2], s_red[3]); atomicMax(&F_key[3], s_red[4]); }
  }
}

}  // namespace

// ====================================================================== launchers
uint32_t preprocess_chunk_items() { return PRE_CHUNK; }

void launch_repack(cudaStream_t s, uint32_t n, int K, const float* means, const float* scales, const float* quats,
                   const float* opacity, const float* sh, DevBuffers& b) {
  if (!n) return;
  k_repack<<<(n + 255) / 256, 256, 0, s>>>(n, means, scales, quats, opacity, b.cull4, b.g2);
  cudaMemcpyAsync(b.sh, sh, (size_t)n * K * 3 * sizeof(float), cudaMemcpyDeviceToDevice, s);
}

void launch_frame_init(cudaStream_t s, const FrameConst& fc, DevBuffers& b, bool reset_F, uint8_t* rendered_next) {
  const uint32_t n_words = rendered_next ? (fc.n + 3) / 4 : 0;
  TGS_LAUNCH((k_frame_init), 592, 256, 0, s, fc, b.counters, b.tile_flags, (uint2*)b.warp_tgb,
                                   (uint32_t*)rendered_next, n_words, b.sort_hist, b.ranges, b.tile_mask, b.tile_order, b.sel_bits, b.live_bits,
                                   b.F_key, reset_F ? 1 : 0);
}

void launch_warp(cudaStream_t s, const FrameConst& fc, DevBuffers& b, const float* prior_depth, const float* prior_sigma) {
  dim3 grid((fc.tg.W + 31) / 32, (fc.tg.H + 7) / 8);
  TGS_LAUNCH((k_warp), grid, 256, 0, s, fc, prior_depth, prior_sigma, (uint2*)b.warp_tgb);
}

void launch_fill_corr(cudaStream_t s, const FrameConst& fc, DevBuffers& b) {
  dim3 grid(fc.cam.TX, fc.cam.TY);
  TGS_LAUNCH((k_fill_corr), grid, 256, 0, s, fc, (const float2*)b.warp_tgb, b.fill_depth, b.tile_flags);
}

void launch_preprocess(cudaStream_t s, const FrameConst& fc, DevBuffers& b, int num_sms) {
  const uint32_t chunks = (fc.n + PRE_CHUNK - 1) / PRE_CHUNK;
  const uint32_t grid = chunks < (uint32_t)(num_sms * 4) ? chunks : (uint32_t)(num_sms * 4);
  TGS_LAUNCH((k_preprocess), grid ? grid : 1, PRE_THREADS, 0, s, fc, b.cull4, b.g2, b.rendered, (const float2*)b.warp_tgb, b.F_key,
                                                       b.rec_bin, b.rec_flags, b.rec_b0, b.rec_b1, b.tile_flags, b.nv_queue,
                                                       b.ckeys[1], b.cvals[1], b.pre_cnt, b.sort_hist, b.counters);
  TGS_LAUNCH((k_compact_vis), num_sms * 8, 128, 0, s, fc.n, (const uint2*)b.pre_cnt, b.ckeys[1], b.cvals[1], b.ckeys[0], b.cvals[0], b.vis_list,
             fc.dsort_fused ? b.dsort_H : (uint32_t*)nullptr, depth_sort_fused_tile_items());
}

void launch_mark_oc(cudaStream_t s, const FrameConst& fc, DevBuffers& b, int num_sms) {
  TGS_LAUNCH((k_mark_oc), num_sms * 8, 128, 0, s, fc, b.nv_queue, (const float4*)b.rec_bin, b.tile_flags, b.counters);
}

void launch_select(cudaStream_t s, const FrameConst& fc, DevBuffers& b, uint32_t* host_n_sel) {
  TGS_LAUNCH((k_select), 1, 1024, 0, s, fc, b.tile_flags, b.tile_mask, b.sel_bits, b.live_bits, b.tile_order, b.counters, (volatile uint32_t*)host_n_sel);
}

// The frame's counters to pinned host memory by zero-copy stores (no copy engine: see k_select).
__global__ void __launch_bounds__(128) k_export_counters(const Counters* __restrict__ counters, volatile uint32_t* __restrict__ host) {
  TGS_PDL_WAIT();
  if (threadIdx.x < sizeof(Counters) / 4) host[threadIdx.x] = reinterpret_cast<const uint32_t*>(counters)[threadIdx.x];
  __threadfence_system();
}
void launch_export_counters(cudaStream_t s, const DevBuffers& b, Counters* host) {
  TGS_LAUNCH((k_export_counters), 1, 128, 0, s, (const Counters*)b.counters, (volatile uint32_t*)host);
}

void launch_frustum(cudaStream_t s, const FrameConst& fc, DevBuffers& b, const uint32_t* vis_vals, const uint8_t* rendered_now, bool update_F) {
  TGS_LAUNCH((k_frustum), 296, 256, 0, s, fc, vis_vals, rendered_now, (const float4*)b.rec_bin, b.F_key, b.counters, update_F ? 1 : 0);
}
