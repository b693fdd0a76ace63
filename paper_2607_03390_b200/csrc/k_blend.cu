// k_blend.cu -- A8 front-to-back alpha blending of the selected tiles (+ Eq.1-2 depth moments and the
// G_rendered marks on R / P frames) fused with A9, the stitch of the non-selected tiles from the
// backward-warped TAB (Eq.4).  PAPER.md:L61 (alpha-blending), L73-84 (Eq.1-2), L103 (G_rendered),
// L101 + L125-128 (bilinear TAB, Eq.4).  Constants of R2: alpha <= 0.99, skip alpha < 1/255, stop when
// T(1-alpha) < 1e-4.
//
// One persistent grid; a work item is a tile of `tile_order` (selected tiles first).  A CTA is 16x16
// threads = one pixel each; the tile's sorted Gaussians are staged through shared memory in batches of
// 256 records, pre-scaled so that alpha = exp2(A' t^2 + D' dy^2 + log2 o), t = dx + k dy, is 7 FMA-pipe
// instructions + 1 MUFU.EX2: the form -1/2 delta^T Sigma'^-1 delta completed to two squares, which has no
// cancellation between terms (screen-filling anisotropic splats lose 1e-4 of alpha in the 3-term conic form).
// This kernel is FP32-pipe bound, not HBM bound.
#include "tgs_internal.cuh"

namespace {

constexpr int BLEND_THREADS = 256;
constexpr float ALPHA_MIN = 1.0f / 255.0f;
// log2(1/255) = -7.99435...; anything below this bound (with a safety gap far above the rounding of e and of
// ex2.approx) has alpha < 1/255 for sure, so the exact test on alpha is only evaluated near or above the threshold
constexpr float LOG2_ALPHA_MIN_LO = -7.9950f;

__device__ __forceinline__ float ex2_approx(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}

struct BlendSmem {
  float4 a[BLEND_THREADS];     // u, v, A', k
  float4 b[BLEND_THREADS];     // D', log2(o), d, r
  float2 c[BLEND_THREADS];     // g, b
  uint32_t id[BLEND_THREADS];  // Gaussian index (for the G_rendered marks)
  uint8_t contrib[BLEND_THREADS];   // G_rendered marks of the batch (benign same-value races)
  uint32_t work;
};

template <bool MARK, bool COUNT>
__global__ void __launch_bounds__(BLEND_THREADS) k_blend(FrameConst fc, const uint32_t* __restrict__ tile_order,
                                                         const uint2* __restrict__ ranges, const uint32_t* __restrict__ vals,
                                                         const float4* __restrict__ rec_b0, const float4* __restrict__ rec_b1,
                                                         const float4* __restrict__ rec_rgb, const float* __restrict__ prior_image,
                                                         const float* __restrict__ fill_depth, const float* __restrict__ warp_sigma,
                                                         float* __restrict__ image, float* __restrict__ depth, float* __restrict__ sigma,
                                                         uint8_t* __restrict__ rendered_next, Counters* __restrict__ counters) {
  __shared__ BlendSmem sm;
  const CamConst& k = fc.cam;
  const uint32_t lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  // a warp covers a 16x2 pixel strip of the tile
  const int lx = threadIdx.x & 15, ly = threadIdx.x >> 4;
  while (true) {
    __syncthreads();
    if (threadIdx.x == 0) sm.work = atomicAdd(&counters->ticket_blend, 1u);
    __syncthreads();
    const uint32_t w = sm.work;
    if (w >= (uint32_t)fc.n_tiles) break;
    const uint32_t tile = tile_order[w];
    const int px = (int)(tile % k.TX) * TGS_TILE + lx, py = (int)(tile / k.TX) * TGS_TILE + ly;
    const bool inside = px < k.W && py < k.H;
    const size_t pix = (size_t)py * k.W + px;
    if (w >= counters->n_sel) {
      // ------------------------------------------------ A9 stitch (Eq.4, second case)
      if (inside) {
        const float D = fill_depth[pix];
        const float* M = fc.Minv;
        const float rx = ((float)px - k.cx) / k.fx, ry = ((float)py - k.cy) / k.fy;
        const float Px = D * rx, Py = D * ry;
        const float X = M[0] * Px + M[1] * Py + M[2] * D + M[3];
        const float Y = M[4] * Px + M[5] * Py + M[6] * D + M[7];
        const float Z = M[8] * Px + M[9] * Py + M[10] * D + M[11];
        const float xs = k.fx * X / Z + k.cx, ys = k.fy * Y / Z + k.cy;
        const float x0 = floorf(xs), y0 = floorf(ys);
        const float wx = xs - x0, wy = ys - y0;
        const int ix0 = min(max((int)x0, 0), k.W - 1), ix1 = min(max((int)x0 + 1, 0), k.W - 1);
        const int iy0 = min(max((int)y0, 0), k.H - 1), iy1 = min(max((int)y0 + 1, 0), k.H - 1);
        const float* p00 = prior_image + ((size_t)iy0 * k.W + ix0) * 3;
        const float* p10 = prior_image + ((size_t)iy0 * k.W + ix1) * 3;
        const float* p01 = prior_image + ((size_t)iy1 * k.W + ix0) * 3;
        const float* p11 = prior_image + ((size_t)iy1 * k.W + ix1) * 3;
#pragma unroll
        for (int ch = 0; ch < 3; ++ch) {
          const float top = p00[ch] * (1.0f - wx) + p10[ch] * wx, bot = p01[ch] * (1.0f - wx) + p11[ch] * wx;
          image[pix * 3 + ch] = top * (1.0f - wy) + bot * wy;
        }
        depth[pix] = D;
        sigma[pix] = warp_sigma[pix];
      }
      continue;
    }
    // -------------------------------------------------- A8 blend
    const uint2 range = ranges[tile];
    const float fpx = (float)px, fpy = (float)py;
    float T = 1.0f, Cr = 0.0f, Cg = 0.0f, Cb = 0.0f;
    float Sw = 0.0f, S1 = 0.0f, S2 = 0.0f, d0 = 0.0f;      // Eq.1-2 moments, shifted by the first contributing depth
    bool done = !inside;
    uint32_t nint = 0;
    for (uint32_t start = range.x; start < range.y; start += BLEND_THREADS) {
      if (__syncthreads_count(done) == BLEND_THREADS) break;
      const uint32_t nb = min((uint32_t)BLEND_THREADS, range.y - start);
      if (threadIdx.x < nb) {
        const uint32_t g = vals[start + threadIdx.x];
        const float4 r0 = rec_b0[g], r1 = rec_b1[g], r2 = rec_rgb[g];
        sm.a[threadIdx.x] = r0;
        sm.b[threadIdx.x] = make_float4(r1.x, r1.y, r1.z, r2.x);
        sm.c[threadIdx.x] = make_float2(r2.y, r2.z);
        sm.id[threadIdx.x] = g;
      }
      if (MARK) sm.contrib[threadIdx.x] = 0;
      __syncthreads();
      if (!done) {
#pragma unroll 4
        for (uint32_t j = 0; j < nb; ++j) {
          if (COUNT) ++nint;
          const float4 ga = sm.a[j];
          const float4 gb = sm.b[j];
          const float dx = ga.x - fpx, dy = ga.y - fpy;
          const float t = fmaf(ga.w, dy, dx);
          const float e = fmaf(ga.z * t, t, fmaf(gb.x * dy, dy, gb.y));         // log2(o) + log2 of the falloff (<= log2 o)
          if (e < LOG2_ALPHA_MIN_LO) continue;                                  // surely alpha < 1/255: no MUFU
          const float alpha = fminf(0.99f, ex2_approx(e));
          if (alpha < ALPHA_MIN) continue;
          const float Tn = T * (1.0f - alpha);
          if (Tn < 1.0e-4f) { done = true; break; }
          const float wgt = alpha * T;
          const float2 gc = sm.c[j];
          Cr = fmaf(wgt, gb.w, Cr); Cg = fmaf(wgt, gc.x, Cg); Cb = fmaf(wgt, gc.y, Cb);
          if (Sw == 0.0f) d0 = gb.z;
          const float dd = gb.z - d0;
          Sw += wgt; S1 = fmaf(wgt, dd, S1); S2 = fmaf(wgt * dd, dd, S2);
          T = Tn;
          if (MARK) sm.contrib[j] = 1;
        }
      }
      if (MARK) {
        __syncthreads();
        if (threadIdx.x < nb && sm.contrib[threadIdx.x]) rendered_next[sm.id[threadIdx.x]] = 1;
      }
    }
    if (inside) {
      image[pix * 3 + 0] = Cr + T * fc.bg[0];
      image[pix * 3 + 1] = Cg + T * fc.bg[1];
      image[pix * 3 + 2] = Cb + T * fc.bg[2];
      if (Sw > 0.0f) {
        const float m1 = S1 / Sw;
        depth[pix] = d0 + m1;
        sigma[pix] = sqrtf(fmaxf(0.0f, S2 / Sw - m1 * m1));
      } else {
        depth[pix] = TGS_DEPTH_INVALID;
        sigma[pix] = 0.0f;
      }
    }
    if (COUNT) {
      nint = __reduce_add_sync(0xffffffffu, nint);
      if (lane == 0 && nint) atomicAdd(&counters->n_interactions, (unsigned long long)nint);
    }
    (void)wid;
  }
}

}  // namespace

void launch_blend(cudaStream_t s, const FrameConst& fc, DevBuffers& b, int sorted_idx, int out_idx, const float* prior_image,
                  uint8_t* rendered_next, int num_sms, bool count_interactions) {
  const int grid = num_sms * 4;
#define LAUNCH(M, C)                                                                                                          \
  k_blend<M, C><<<grid, BLEND_THREADS, 0, s>>>(fc, b.tile_order, b.ranges, b.vals[sorted_idx], b.rec_b0, b.rec_b1, b.rec_rgb, \
                                               prior_image, b.fill_depth, b.warp_sigma, b.image[out_idx], b.depth[out_idx],  \
                                               b.sigma[out_idx], rendered_next, b.counters)
  if (rendered_next) { if (count_interactions) LAUNCH(true, true); else LAUNCH(true, false); }
  else { if (count_interactions) LAUNCH(false, true); else LAUNCH(false, false); }
#undef LAUNCH
}
