// k_decide.cu -- kernels whose fp32 arithmetic DECIDES integers (cull masks, nearest pixels, tile
// rects, sort-key depth bits, tile selection).  Compiled with -fmad=false: every +,-,*,/,sqrt is one
// IEEE rounding in the order written, so the decisions are reproducible bit for bit (DESIGN.md §2 R33).
// All of these kernels are HBM- or latency-bound; the lost FMA contraction costs nothing measurable.
//
// A1 forward warp (Eq.3), A2 depth fill + correspondence + T^um (L121),
// A3 preprocess + AFC + TOC + newly-visible + T^oc (L61, L109-113, L119), A4 tile selection (L117-123),
// A5a count + SH colour, F reduction (L109).
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
                                                float4* __restrict__ cull4, float* __restrict__ cov3d, float* __restrict__ tau) {
  const uint32_t g = blockIdx.x * blockDim.x + threadIdx.x;
  if (g >= n) return;
  const float o = opacity[g];
  cull4[g] = make_float4(means[3 * g], means[3 * g + 1], means[3 * g + 2], o);
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
  float* c = cov3d + 6 * (size_t)g;
  c[0] = SIG(0, 0); c[1] = SIG(0, 1); c[2] = SIG(0, 2); c[3] = SIG(1, 1); c[4] = SIG(1, 2); c[5] = SIG(2, 2);
#undef SIG
  tau[g] = (float)(2.0 * log(255.0 * (double)o));
}

// ------------------------------------------------------------------ per-frame init
// counters <- 0; tile_flags <- 0; S frames: D^min <- INVALID bits, sigma^max <- 0;
// R / P frames: rendered_next <- 0; R frames: F <- (+inf, +inf, -inf, -inf).
__global__ void __launch_bounds__(256) k_frame_init(FrameConst fc, Counters* counters, uint32_t* tile_flags, uint32_t* warp_depth,
                                                    uint32_t* warp_sigma, uint32_t* rendered_next_words, uint32_t n_words,
                                                    uint32_t* F_key, int reset_F) {
  const uint32_t tid = blockIdx.x * blockDim.x + threadIdx.x, nth = gridDim.x * blockDim.x;
  if (tid < sizeof(Counters) / 4) ((uint32_t*)counters)[tid] = 0;
  if (reset_F && tid < 4) F_key[tid] = (tid < 2) ? 0xff800000u /* key(+inf) */ : 0x007fffffu /* key(-inf) */;
  for (uint32_t i = tid; i < (uint32_t)fc.n_tiles; i += nth) tile_flags[i] = 0;
  if (fc.do_tgb) {
    const uint32_t px = (uint32_t)(fc.cam.W * fc.cam.H);
    for (uint32_t i = tid; i < px; i += nth) { warp_depth[i] = TGS_INVALID_BITS; warp_sigma[i] = 0; }
  }
  if (rendered_next_words)
    for (uint32_t i = tid; i < n_words; i += nth) rendered_next_words[i] = 0;
}

// ------------------------------------------------------------------ A1 forward warp
// One thread per reference pixel.  Nearest-pixel splat (R14) with atomicMin on the depth bits (positive
// floats order like their bit patterns) and atomicMax on the sigma bits: min depth and max sigma are kept
// independently (L91, L97; R15), so the result does not depend on the order of arrival.
__global__ void __launch_bounds__(256) k_warp(FrameConst fc, const float* __restrict__ prior_depth,
                                              const float* __restrict__ prior_sigma, uint32_t* __restrict__ warp_depth,
                                              uint32_t* __restrict__ warp_sigma) {
  const int x = blockIdx.x * 32 + (threadIdx.x & 31), y = blockIdx.y * 8 + (threadIdx.x >> 5);
  const CamConst& k = fc.cam;
  if (x >= k.W || y >= k.H) return;
  const float D = prior_depth[(size_t)y * k.W + x];
  if (!(D < 1.0e38f)) return;                                   // R11
  const float* M = fc.M;
  const float rx = ((float)x - k.cx) / k.fx, ry = ((float)y - k.cy) / k.fy;
  const float Px = D * rx, Py = D * ry, Pz = D;
  const float X = ((M[0] * Px + M[1] * Py) + M[2] * Pz) + M[3];
  const float Y = ((M[4] * Px + M[5] * Py) + M[6] * Pz) + M[7];
  const float Z = ((M[8] * Px + M[9] * Py) + M[10] * Pz) + M[11];
  if (!(Z > k.znear)) return;
  const float u = (k.fx * X) / Z + k.cx, v = (k.fy * Y) / Z + k.cy;
  const float fu = floorf(u + 0.5f), fv = floorf(v + 0.5f);
  if (!(fu >= 0.0f && fu < k.Wf && fv >= 0.0f && fv < k.Hf)) return;
  const size_t q = (size_t)(int)fv * k.W + (int)fu;
  const float s = prior_sigma[(size_t)y * k.W + x] * fabsf((M[8] * rx + M[9] * ry) + M[10]);   // R13
  atomicMin(&warp_depth[q], __float_as_uint(Z));
  if (s > 0.0f) atomicMax(&warp_sigma[q], __float_as_uint(s));
}

// ------------------------------------------------------------------ A2 depth fill + correspondence + T^um
// One CTA per tile, one thread per pixel.  D' = D^min with isolated holes filled by the mean of the 8
// neighbours (L121; R19).  matched <=> D' valid, back-projected z > z_near and the nearest reference pixel
// is inside the image (R20).  Tile in T^um <=> any in-image pixel unmatched (R22).
__global__ void __launch_bounds__(256) k_fill_corr(FrameConst fc, const float* __restrict__ warp_depth, float* __restrict__ fill_depth,
                                                   uint32_t* __restrict__ tile_flags) {
  const CamConst& k = fc.cam;
  const int lx = threadIdx.x & 15, ly = threadIdx.x >> 4;
  const int x = blockIdx.x * TGS_TILE + lx, y = blockIdx.y * TGS_TILE + ly;
  const bool inside = x < k.W && y < k.H;
  bool unmatched = false;
  if (inside) {
    const float* wd = warp_depth;
    float D = wd[(size_t)y * k.W + x];
    if (!(D < 1.0e38f) && x > 0 && y > 0 && x < k.W - 1 && y < k.H - 1) {
      const float n0 = wd[(size_t)(y - 1) * k.W + x - 1], n1 = wd[(size_t)(y - 1) * k.W + x], n2 = wd[(size_t)(y - 1) * k.W + x + 1];
      const float n3 = wd[(size_t)y * k.W + x - 1], n4 = wd[(size_t)y * k.W + x + 1];
      const float n5 = wd[(size_t)(y + 1) * k.W + x - 1], n6 = wd[(size_t)(y + 1) * k.W + x], n7 = wd[(size_t)(y + 1) * k.W + x + 1];
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
      if (Z > k.znear) {
        const float xs = (k.fx * X) / Z + k.cx, ys = (k.fy * Y) / Z + k.cy;
        const float fu = floorf(xs + 0.5f), fv = floorf(ys + 0.5f);
        if (fu >= 0.0f && fu < k.Wf && fv >= 0.0f && fv < k.Hf) unmatched = false;
      }
    }
  }
  const int any = __syncthreads_or(unmatched ? 1 : 0);
  if (threadIdx.x == 0 && any) tile_flags[blockIdx.y * k.TX + blockIdx.x] = 2u;   // bit1 = T^um (first writer of this word)
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

// Newly visible Gaussians with large rects (queued by k_preprocess): one warp per Gaussian, lanes over the tiles
// of the rect.  Stops as soon as every tile of the frame carries the T^oc mark.
__global__ void __launch_bounds__(256) k_mark_oc(FrameConst fc, const uint32_t* __restrict__ nv_queue, const float4* __restrict__ rec_uvdo,
                                                 const float4* __restrict__ rec_conic, const uint2* __restrict__ rec_rect,
                                                 uint32_t* __restrict__ tile_flags, Counters* __restrict__ counters) {
  const CamConst& k = fc.cam;
  const uint32_t lane = threadIdx.x & 31;
  const uint32_t nq = counters->n_nv_queue;
  while (true) {
    uint32_t j = 0;
    if (lane == 0) j = atomicAdd(&counters->ticket_mark, 1u);
    j = __shfl_sync(0xffffffffu, j, 0);
    if (j >= nq) break;
    if (*reinterpret_cast<volatile uint32_t*>(&counters->n_oc_marked) >= (uint32_t)fc.n_tiles) break;
    const uint32_t g = nv_queue[j];
    const float4 r0 = rec_uvdo[g], r1 = rec_conic[g];
    const uint2 r = rec_rect[g];
    const uint32_t x_lo = r.x & 0xffffu, x_hi = r.x >> 16, y_lo = r.y & 0xffffu, y_hi = r.y >> 16;
    const uint32_t w = x_hi - x_lo, area = w * (y_hi - y_lo);
    for (uint32_t i = lane; i < area; i += 32) mark_oc_tile(k, r0.x, r0.y, r1.x, r1.y, r1.z, r1.w, x_lo + i % w, y_lo + i / w, tile_flags, counters);
  }
}

// ------------------------------------------------------------------ A3 preprocess (+AFC +TOC +newly-visible +T^oc)
// One thread per Gaussian.  The 16 B cull record {mean, opacity} is read for all N; the 24 B covariance only
// for Gaussians that survive near / AFC / TOC; SH (the bulk of the bytes) is not touched here at all.
// Order of the tests and of every fp32 operation: DESIGN.md §2 (O3), identical to what the oracle states.
__global__ void __launch_bounds__(256) k_preprocess(FrameConst fc, const float4* __restrict__ cull4, const float* __restrict__ cov3d,
                                                    const float* __restrict__ tau_arr, const uint8_t* __restrict__ rendered,
                                                    const float* __restrict__ warp_depth, const float* __restrict__ warp_sigma,
                                                    const uint32_t* __restrict__ F_key, float4* __restrict__ rec_uvdo,
                                                    float4* __restrict__ rec_conic, uint2* __restrict__ rec_rect,
                                                    uint32_t* __restrict__ rec_flags, float4* __restrict__ rec_b0,
                                                    float4* __restrict__ rec_b1, uint32_t* __restrict__ tile_flags,
                                                    uint32_t* __restrict__ nv_queue, Counters* __restrict__ counters) {
  const uint32_t g = blockIdx.x * blockDim.x + threadIdx.x;
  const CamConst& k = fc.cam;
  const float* V = k.V;
  uint32_t flags = 0;
  if (g < fc.n) {
    const float4 c4 = cull4[g];
    const float x = c4.x, y = c4.y, z = c4.z;
    const float tx = ((V[0] * x + V[1] * y) + V[2] * z) + V[3];
    const float ty = ((V[4] * x + V[5] * y) + V[6] * z) + V[7];
    const float tz = ((V[8] * x + V[9] * y) + V[10] * z) + V[11];
    do {
      if (!(tz > k.znear)) { flags = TGS_CULL_NEAR; break; }                       // L61, R4
      const float u = (k.fx * tx) / tz + k.cx, v = (k.fy * ty) / tz + k.cy;
      if (fc.do_afc) {                                                             // L109-111
        const float F0 = key2f(F_key[0]), F1 = key2f(F_key[1]), F2 = key2f(F_key[2]), F3 = key2f(F_key[3]);
        const float nx = (2.0f * u + 1.0f) / k.Wf - 1.0f, ny = (2.0f * v + 1.0f) / k.Hf - 1.0f;
        if (!(F0 <= nx && nx <= F2 && F1 <= ny && ny <= F3)) { flags = TGS_CULL_AFC; break; }
      }
      uint32_t fl = 0;
      if (fc.do_tgb && !rendered[g]) {                                             // L113, L119
        const float fu = floorf(u + 0.5f), fv = floorf(v + 0.5f);
        if (fu >= 0.0f && fu < k.Wf && fv >= 0.0f && fv < k.Hf) {
          const size_t q = (size_t)(int)fv * k.W + (int)fu;
          const float D = warp_depth[q], s = warp_sigma[q];
          if (fc.do_toc && tz > D + fc.lambda2 * s) { flags = TGS_CULL_TOC; break; }
          if (tz <= D - fc.lambda1 * s) fl = TGS_NEWLY_VISIBLE;
        }
      }
      const float2 s01 = *reinterpret_cast<const float2*>(cov3d + 6 * (size_t)g);
      const float2 s23 = *reinterpret_cast<const float2*>(cov3d + 6 * (size_t)g + 2);
      const float2 s45 = *reinterpret_cast<const float2*>(cov3d + 6 * (size_t)g + 4);
      const float S0 = s01.x, S1 = s01.y, S2 = s23.x, S3 = s23.y, S4 = s45.x, S5 = s45.y;
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
      const float c = ((T10 * q0 + T11 * q1) + T12 * q2) + 0.3f;
      const float det = a * c - b * b;
      if (!(det > 0.0f)) { flags = TGS_CULL_DEGENERATE; break; }
      const float A = c / det, B = -b / det, C = a / det;
      const float mid = 0.5f * (a + c);
      const float lam = mid + sqrtf(fmaxf(0.1f, mid * mid - det));
      const float rad = ceilf(3.0f * sqrtf(lam));
      const float TXf = (float)k.TX, TYf = (float)k.TY;
      const uint32_t x_lo = (uint32_t)fminf(fmaxf(floorf((u - rad) / 16.0f), 0.0f), TXf);
      const uint32_t x_hi = (uint32_t)fminf(fmaxf(floorf((u + rad + 15.0f) / 16.0f), 0.0f), TXf);
      const uint32_t y_lo = (uint32_t)fminf(fmaxf(floorf((v - rad) / 16.0f), 0.0f), TYf);
      const uint32_t y_hi = (uint32_t)fminf(fmaxf(floorf((v + rad + 15.0f) / 16.0f), 0.0f), TYf);
      if (!(x_hi > x_lo && y_hi > y_lo)) { flags = TGS_CULL_EMPTY; break; }
      flags = fl | TGS_VISIBLE;
      const float tau = tau_arr[g];
      rec_uvdo[g] = make_float4(u, v, tz, c4.w);
      rec_conic[g] = make_float4(A, B, C, tau);
      rec_rect[g] = make_uint2(x_lo | (x_hi << 16), y_lo | (y_hi << 16));
      // blend-side parameters: the quadratic form as a sum of two squares (no cancellation between its terms)
      rec_b0[g] = make_float4(u, v, -0.72134752f * A, -b / c);
      rec_b1[g] = make_float4(-0.72134752f / c, log2f(c4.w), tz, 0.0f);
      if (fl && tau >= 0.0f) {                                                      // A4: T^oc (L119, R18)
        if ((x_hi - x_lo) * (y_hi - y_lo) > 16u) nv_queue[atomicAdd(&counters->n_nv_queue, 1u)] = g;   // large rect: k_mark_oc
        else
          for (uint32_t tyy = y_lo; tyy < y_hi; ++tyy)
            for (uint32_t txx = x_lo; txx < x_hi; ++txx) mark_oc_tile(k, u, v, A, B, C, tau, txx, tyy, tile_flags, counters);
      }
    } while (false);
    rec_flags[g] = flags;
  }
  // statistics: one atomic per warp and non-zero class
  const uint32_t lane = threadIdx.x & 31;
#define COUNT(bit, field)                                              \
  {                                                                    \
    const uint32_t m = __ballot_sync(0xffffffffu, (flags & (bit)) != 0); \
    if (m && lane == 0) atomicAdd(&counters->field, __popc(m));        \
  }
  COUNT(TGS_CULL_NEAR, n_near) COUNT(TGS_CULL_AFC, n_afc) COUNT(TGS_CULL_TOC, n_toc) COUNT(TGS_CULL_DEGENERATE, n_degenerate)
  COUNT(TGS_CULL_EMPTY, n_empty) COUNT(TGS_VISIBLE, n_visible)
  {
    const uint32_t m = __ballot_sync(0xffffffffu, (flags & (TGS_VISIBLE | TGS_NEWLY_VISIBLE)) == (TGS_VISIBLE | TGS_NEWLY_VISIBLE));
    if (m && lane == 0) atomicAdd(&counters->n_newly_visible, __popc(m));
  }
#undef COUNT
}

// ------------------------------------------------------------------ A4 tile selection: T_sel = T^oc U T^um (L123)
// One CTA.  Builds the tile mask, the bit set used by the pair counting, and the work order of the blend
// kernel: selected tiles first (ascending id), then the tiles that are only stitched.
__global__ void __launch_bounds__(1024) k_select(FrameConst fc, const uint32_t* __restrict__ tile_flags, uint8_t* __restrict__ tile_mask,
                                                 uint32_t* __restrict__ sel_bits, uint32_t* __restrict__ tile_order,
                                                 Counters* __restrict__ counters) {
  __shared__ uint32_t s_warp[32];
  __shared__ uint32_t s_base, s_noc, s_num;
  const int T = fc.n_tiles;
  const uint32_t lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  if (threadIdx.x == 0) { s_base = 0; s_noc = 0; s_num = 0; }
  __syncthreads();
  // pass 1: masks, bits, selected list
  for (int base = 0; base < T; base += 1024) {
    const int t = base + threadIdx.x;
    uint32_t f = 0; bool sel = false;
    if (t < T) {
      f = tile_flags[t] & 3u;
      sel = fc.all_tiles || f != 0;
      tile_mask[t] = (uint8_t)(f | (sel ? 4u : 0u));
    }
    const uint32_t bal = __ballot_sync(0xffffffffu, sel);
    if (lane == 0 && base + (int)(wid * 32) < T) sel_bits[(base >> 5) + wid] = bal;
    const uint32_t boc = __ballot_sync(0xffffffffu, (f & 1u) != 0), bum = __ballot_sync(0xffffffffu, (f & 2u) != 0);
    if (lane == 0) { s_warp[wid] = __popc(bal); if (boc) atomicAdd(&s_noc, __popc(boc)); if (bum) atomicAdd(&s_num, __popc(bum)); }
    __syncthreads();
    uint32_t before = s_base;
    for (uint32_t w = 0; w < wid; ++w) before += s_warp[w];
    if (sel) tile_order[before + __popc(bal & ((1u << lane) - 1u))] = (uint32_t)t;
    __syncthreads();
    if (threadIdx.x == 0) { uint32_t tot = 0; for (int w = 0; w < 32; ++w) tot += s_warp[w]; s_base += tot; }
    __syncthreads();
  }
  const uint32_t nsel = s_base;
  __syncthreads();
  if (threadIdx.x == 0) { counters->n_sel = nsel; counters->n_sel_oc = s_noc; counters->n_sel_um = s_num; s_base = nsel; }
  __syncthreads();
  // pass 2: the non-selected tiles follow
  for (int base = 0; base < T; base += 1024) {
    const int t = base + threadIdx.x;
    const bool ns = t < T && !(fc.all_tiles || (tile_flags[t] & 3u) != 0);
    const uint32_t bal = __ballot_sync(0xffffffffu, ns);
    if (lane == 0) s_warp[wid] = __popc(bal);
    __syncthreads();
    uint32_t before = s_base;
    for (uint32_t w = 0; w < wid; ++w) before += s_warp[w];
    if (ns) tile_order[before + __popc(bal & ((1u << lane) - 1u))] = (uint32_t)t;
    __syncthreads();
    if (threadIdx.x == 0) { uint32_t tot = 0; for (int w = 0; w < 32; ++w) tot += s_warp[w]; s_base += tot; }
    __syncthreads();
  }
}

// number of set bits of `bits` with index in [lo, hi)
__device__ __forceinline__ uint32_t popc_range(const uint32_t* __restrict__ bits, uint32_t lo, uint32_t hi) {
  uint32_t cnt = 0;
  uint32_t w = lo >> 5;
  const uint32_t wend = (hi - 1) >> 5;
  uint32_t m = 0xffffffffu << (lo & 31);
  for (; w < wend; ++w) { cnt += __popc(bits[w] & m); m = 0xffffffffu; }
  m &= 0xffffffffu >> (31 - ((hi - 1) & 31));
  return cnt + __popc(bits[w] & m);
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

// ------------------------------------------------------------------ A5a pair count + SH colour
// tiles_touched[g] = number of pairs this Gaussian emits (0 if invisible): the SELECTED tiles of its rect (L123)
// that it intersects (L61) -- with exact_tiles (R39) those where max alpha over the tile's pixel box >= 1/255,
// else every tile of the 3-sigma rect.  Rects of more than 4 tiles are counted by the whole warp (lanes over
// tiles): near Gaussians cover hundreds of tiles and would otherwise serialise one thread.
// SH -> RGB (L61 "color c_i"; R5) only for Gaussians that emit at least one pair: on S frames the 12K bytes
// of SH are read only for Gaussians that reach a selected tile.
template <int DEG>
__global__ void __launch_bounds__(256) k_count_color(FrameConst fc, const float4* __restrict__ cull4, const float* __restrict__ sh,
                                                     const uint32_t* __restrict__ rec_flags, const uint2* __restrict__ rec_rect,
                                                     const float4* __restrict__ rec_uvdo, const float4* __restrict__ rec_conic,
                                                     const uint32_t* __restrict__ sel_bits, uint32_t* __restrict__ tiles_touched,
                                                     float4* __restrict__ rec_rgb) {
  const uint32_t g = blockIdx.x * blockDim.x + threadIdx.x;
  const uint32_t lane = threadIdx.x & 31;
  const int TX = fc.cam.TX;
  uint32_t cnt = 0;
  const bool vis = g < fc.n && (rec_flags[g] & TGS_VISIBLE);
  uint32_t x_lo = 0, y_lo = 0, w = 0, area = 0;
  if (vis) {
    const uint2 r = rec_rect[g];
    x_lo = r.x & 0xffffu; y_lo = r.y & 0xffffu;
    w = (r.x >> 16) - x_lo; area = w * ((r.y >> 16) - y_lo);
  }
  if (!fc.exact_tiles) {
    if (vis) {
      if (fc.all_tiles) cnt = area;
      else
        for (uint32_t ty = y_lo; ty < y_lo + area / w; ++ty) cnt += popc_range(sel_bits, ty * TX + x_lo, ty * TX + x_lo + w);
    }
  } else {
    float4 uv = make_float4(0.f, 0.f, 0.f, 0.f), cn = make_float4(0.f, 0.f, 0.f, -1.f);
    if (vis) { uv = rec_uvdo[g]; cn = rec_conic[g]; }
    const bool big = area > 4u;
    if (vis && !big)
      for (uint32_t i = 0; i < area; ++i) {
        const uint32_t ty = y_lo + i / w, tx = x_lo + i % w, t = ty * TX + tx;
        if ((fc.all_tiles || ((sel_bits[t >> 5] >> (t & 31)) & 1u)) && tile_alpha_reach(uv.x, uv.y, cn.x, cn.y, cn.z, cn.w, tx, ty, fc.cam.W, fc.cam.H)) ++cnt;
      }
    uint32_t m = __ballot_sync(0xffffffffu, vis && big);
    while (m) {
      const int src = __ffs(m) - 1;
      m &= m - 1;
      const float su = __shfl_sync(0xffffffffu, uv.x, src), sv = __shfl_sync(0xffffffffu, uv.y, src);
      const float sA = __shfl_sync(0xffffffffu, cn.x, src), sB = __shfl_sync(0xffffffffu, cn.y, src);
      const float sC = __shfl_sync(0xffffffffu, cn.z, src), st = __shfl_sync(0xffffffffu, cn.w, src);
      const uint32_t sx = __shfl_sync(0xffffffffu, x_lo, src), sy = __shfl_sync(0xffffffffu, y_lo, src);
      const uint32_t sw = __shfl_sync(0xffffffffu, w, src), sa = __shfl_sync(0xffffffffu, area, src);
      uint32_t c = 0;
      if (st >= 0.0f)
        for (uint32_t i = lane; i < sa; i += 32) {
          const uint32_t ry = i / sw, ty = sy + ry, tx = sx + (i - ry * sw), t = ty * TX + tx;
          if ((fc.all_tiles || ((sel_bits[t >> 5] >> (t & 31)) & 1u)) && tile_alpha_reach(su, sv, sA, sB, sC, st, tx, ty, fc.cam.W, fc.cam.H)) ++c;
        }
      c = warp_sum(c);
      if ((int)lane == src) cnt = c;
    }
  }
  if (g >= fc.n) return;
  tiles_touched[g] = cnt;
  if (!cnt) return;
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

// ------------------------------------------------------------------ F_min / F_max over G_rendered (L109) + |G_rendered|
__global__ void __launch_bounds__(256) k_frustum(FrameConst fc, const uint8_t* __restrict__ rendered_now, const float4* __restrict__ rec_uvdo,
                                                 uint32_t* __restrict__ F_key, Counters* __restrict__ counters, int update_F) {
  uint32_t kmin_x = 0xffffffffu, kmin_y = 0xffffffffu, kmax_x = 0, kmax_y = 0, cnt = 0;
  for (uint32_t g = blockIdx.x * blockDim.x + threadIdx.x; g < fc.n; g += gridDim.x * blockDim.x) {
    if (!rendered_now[g]) continue;
    ++cnt;
    if (update_F) {
      const float4 r = rec_uvdo[g];
      const float nx = (2.0f * r.x + 1.0f) / fc.cam.Wf - 1.0f, ny = (2.0f * r.y + 1.0f) / fc.cam.Hf - 1.0f;
      const uint32_t kx = f2key(nx), ky = f2key(ny);
      kmin_x = min(kmin_x, kx); kmax_x = max(kmax_x, kx); kmin_y = min(kmin_y, ky); kmax_y = max(kmax_y, ky);
    }
  }
  cnt = warp_sum(cnt);
  kmin_x = __reduce_min_sync(0xffffffffu, kmin_x); kmin_y = __reduce_min_sync(0xffffffffu, kmin_y);
  kmax_x = __reduce_max_sync(0xffffffffu, kmax_x); kmax_y = __reduce_max_sync(0xffffffffu, kmax_y);
  if ((threadIdx.x & 31) == 0) {
    if (cnt) atomicAdd(&counters->n_rendered, cnt);
    if (update_F && cnt) {
      atomicMin(&F_key[0], kmin_x); atomicMin(&F_key[1], kmin_y); atomicMax(&F_key[2], kmax_x); atomicMax(&F_key[3], kmax_y);
    }
  }
}

}  // namespace

// ====================================================================== launchers
void launch_repack(cudaStream_t s, uint32_t n, int K, const float* means, const float* scales, const float* quats,
                   const float* opacity, const float* sh, DevBuffers& b) {
  if (!n) return;
  k_repack<<<(n + 255) / 256, 256, 0, s>>>(n, means, scales, quats, opacity, b.cull4, b.cov3d, b.tau);
  cudaMemcpyAsync(b.sh, sh, (size_t)n * K * 3 * sizeof(float), cudaMemcpyDeviceToDevice, s);
}

void launch_frame_init(cudaStream_t s, const FrameConst& fc, DevBuffers& b, bool reset_F, uint8_t* rendered_next) {
  const uint32_t n_words = rendered_next ? (fc.n + 3) / 4 : 0;
  k_frame_init<<<592, 256, 0, s>>>(fc, b.counters, b.tile_flags, (uint32_t*)b.warp_depth, (uint32_t*)b.warp_sigma,
                                   (uint32_t*)rendered_next, n_words, b.F_key, reset_F ? 1 : 0);
}

void launch_warp(cudaStream_t s, const FrameConst& fc, DevBuffers& b, const float* prior_depth, const float* prior_sigma) {
  dim3 grid((fc.cam.W + 31) / 32, (fc.cam.H + 7) / 8);
  k_warp<<<grid, 256, 0, s>>>(fc, prior_depth, prior_sigma, (uint32_t*)b.warp_depth, (uint32_t*)b.warp_sigma);
}

void launch_fill_corr(cudaStream_t s, const FrameConst& fc, DevBuffers& b) {
  dim3 grid(fc.cam.TX, fc.cam.TY);
  k_fill_corr<<<grid, 256, 0, s>>>(fc, b.warp_depth, b.fill_depth, b.tile_flags);
}

void launch_preprocess(cudaStream_t s, const FrameConst& fc, DevBuffers& b) {
  k_preprocess<<<(fc.n + 255) / 256, 256, 0, s>>>(fc, b.cull4, b.cov3d, b.tau, b.rendered, b.warp_depth, b.warp_sigma, b.F_key,
                                                  b.rec_uvdo, b.rec_conic, b.rec_rect, b.rec_flags, b.rec_b0, b.rec_b1, b.tile_flags, b.nv_queue, b.counters);
}

void launch_mark_oc(cudaStream_t s, const FrameConst& fc, DevBuffers& b, int num_sms) {
  k_mark_oc<<<num_sms * 4, 256, 0, s>>>(fc, b.nv_queue, b.rec_uvdo, b.rec_conic, b.rec_rect, b.tile_flags, b.counters);
}

void launch_select(cudaStream_t s, const FrameConst& fc, DevBuffers& b) {
  k_select<<<1, 1024, 0, s>>>(fc, b.tile_flags, b.tile_mask, b.sel_bits, b.tile_order, b.counters);
}

void launch_count_color(cudaStream_t s, const FrameConst& fc, DevBuffers& b) {
  const dim3 grid((fc.n + 255) / 256);
#define LAUNCH(D) k_count_color<D><<<grid, 256, 0, s>>>(fc, b.cull4, b.sh, b.rec_flags, b.rec_rect, b.rec_uvdo, b.rec_conic, b.sel_bits, b.tiles_touched, b.rec_rgb)
  switch (fc.sh_degree) {
    case 0: LAUNCH(0); break;
    case 1: LAUNCH(1); break;
    case 2: LAUNCH(2); break;
    default: LAUNCH(3); break;
  }
#undef LAUNCH
}

void launch_frustum(cudaStream_t s, const FrameConst& fc, DevBuffers& b, const uint8_t* rendered_now, bool update_F) {
  k_frustum<<<592, 256, 0, s>>>(fc, rendered_now, b.rec_uvdo, b.F_key, b.counters, update_F ? 1 : 0);
}
