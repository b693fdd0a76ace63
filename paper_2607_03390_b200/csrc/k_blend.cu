// k_blend.cu -- A8 front-to-back alpha blending of the selected tiles (+ Eq.1-2 depth moments and the
// G_rendered marks on R / P frames) fused with A9, the stitch of the non-selected tiles from the
// backward-warped TAB (Eq.4).  PAPER.md:L61 (alpha-blending), L73-84 (Eq.1-2), L103 (G_rendered),
// L101 + L125-128 (bilinear TAB, Eq.4).  Constants of R2: alpha <= 0.99, skip alpha < 1/255, stop when
// T(1-alpha) < 1e-4.
//
// One persistent grid; a work item is a tile of `tile_order` (selected tiles first).  A CTA is 64 threads
// = one 16x16 tile, each thread owning a run of 4 horizontally adjacent pixels, so that everything that depends
// only on the Gaussian and the row (two shared-memory loads, dy, D' dy^2 + log2 o, t at the first pixel) is paid once
// per 4 interactions: alpha_i = exp2(A' t_i^2 + D' dy^2 + log2 o), t_i = t_0 - i, is 3 FMA-pipe instructions per
// pixel + 5 per run.  The form is -1/2 delta^T Sigma'^-1 delta completed to two squares, which has no cancellation
// between terms (screen-filling anisotropic splats lose 1e-4 of alpha in the 3-term conic form).  The tile's
// sorted Gaussians are staged through shared memory in batches of 128 records.
// This kernel is FP32-pipe / issue bound, not HBM bound.
#include "tgs_internal.cuh"

namespace {

constexpr int BLEND_THREADS = 64;      // 16 rows x 4 runs of 4 pixels
constexpr int BLEND_BATCH = 128;
constexpr int PPT = 4;                 // pixels per thread
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
  float4 a[BLEND_BATCH];     // u, v, A', k
  float4 b[BLEND_BATCH];     // D', log2(o), d, r
  float2 c[BLEND_BATCH];     // g, b
  uint32_t id[BLEND_BATCH];  // Gaussian index (for the G_rendered marks)
  uint8_t contrib[BLEND_BATCH];   // G_rendered marks of the batch (benign same-value races)
  uint32_t work;
};

struct Pixel {               // per-pixel state of the front-to-back loop
  float T, Cr, Cg, Cb, Sw, S1, S2, d0;
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
  const uint32_t lane = threadIdx.x & 31;
  const int lx = (threadIdx.x & 3) * PPT, ly = threadIdx.x >> 2;
  const uint32_t n_sel = counters->n_sel;
  while (true) {
    __syncthreads();
    if (threadIdx.x == 0) sm.work = atomicAdd(&counters->ticket_blend, 1u);
    __syncthreads();
    const uint32_t w = sm.work;
    if (w >= (uint32_t)fc.n_tiles) break;
    const uint32_t tile = tile_order[w];
    const int px0 = (int)(tile % k.TX) * TGS_TILE + lx, py = (int)(tile / k.TX) * TGS_TILE + ly;
    const bool row_in = py < k.H;
    if (w >= n_sel) {
      // ------------------------------------------------ A9 stitch (Eq.4, second case)
#pragma unroll
      for (int i = 0; i < PPT; ++i) {
        const int px = px0 + i;
        if (!row_in || px >= k.W) continue;
        const size_t pix = (size_t)py * k.W + px;
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
    const float fpx = (float)px0, fpy = (float)py;
    Pixel p[PPT];
    bool alive[PPT];
#pragma unroll
    for (int i = 0; i < PPT; ++i) {
      p[i].T = 1.0f; p[i].Cr = p[i].Cg = p[i].Cb = 0.0f; p[i].Sw = p[i].S1 = p[i].S2 = p[i].d0 = 0.0f;
      alive[i] = row_in && px0 + i < k.W;
    }
    uint32_t nint = 0;
    for (uint32_t start = range.x; start < range.y; start += BLEND_BATCH) {
      const bool any_alive = alive[0] || alive[1] || alive[2] || alive[3];
      if (__syncthreads_count(any_alive) == 0) break;
      const uint32_t nb = min((uint32_t)BLEND_BATCH, range.y - start);
      for (uint32_t j = threadIdx.x; j < nb; j += BLEND_THREADS) {
        const uint32_t g = vals[start + j];
        const float4 r0 = rec_b0[g], r1 = rec_b1[g], r2 = rec_rgb[g];
        sm.a[j] = r0;
        sm.b[j] = make_float4(r1.x, r1.y, r1.z, r2.x);
        sm.c[j] = make_float2(r2.y, r2.z);
        sm.id[j] = g;
        if (MARK) sm.contrib[j] = 0;
      }
      __syncthreads();
      if (any_alive) {
#pragma unroll 2
        for (uint32_t j = 0; j < nb; ++j) {
          const float4 ga = sm.a[j];
          const float4 gb = sm.b[j];
          const float dy = ga.y - fpy;
          const float e1 = fmaf(gb.x * dy, dy, gb.y);                 // D' dy^2 + log2 o
          float t = fmaf(ga.w, dy, ga.x - fpx);                       // t at the first pixel of the run
          if (COUNT) nint += (uint32_t)alive[0] + (uint32_t)alive[1] + (uint32_t)alive[2] + (uint32_t)alive[3];
          bool hit[PPT];
          float e[PPT];
#pragma unroll
          for (int i = 0; i < PPT; ++i) {
            e[i] = fmaf(ga.z * t, t, e1);                             // log2(o) + log2 of the falloff
            hit[i] = alive[i] && e[i] >= LOG2_ALPHA_MIN_LO;           // else surely alpha < 1/255: no MUFU
            t -= 1.0f;
          }
          if (!(hit[0] || hit[1] || hit[2] || hit[3])) continue;
          const float2 gc = sm.c[j];
          bool marked = false;
#pragma unroll
          for (int i = 0; i < PPT; ++i) {
            if (!hit[i]) continue;
            const float alpha = fminf(0.99f, ex2_approx(e[i]));
            if (alpha < ALPHA_MIN) continue;
            const float Tn = p[i].T * (1.0f - alpha);
            if (Tn < 1.0e-4f) { alive[i] = false; continue; }
            const float wgt = alpha * p[i].T;
            p[i].Cr = fmaf(wgt, gb.w, p[i].Cr); p[i].Cg = fmaf(wgt, gc.x, p[i].Cg); p[i].Cb = fmaf(wgt, gc.y, p[i].Cb);
            if (p[i].Sw == 0.0f) p[i].d0 = gb.z;
            const float dd = gb.z - p[i].d0;
            p[i].Sw += wgt; p[i].S1 = fmaf(wgt, dd, p[i].S1); p[i].S2 = fmaf(wgt * dd, dd, p[i].S2);
            p[i].T = Tn;
            marked = true;
          }
          if (MARK && marked) sm.contrib[j] = 1;
          if (!(alive[0] || alive[1] || alive[2] || alive[3])) break;
        }
      }
      if (MARK) {
        __syncthreads();
        for (uint32_t j = threadIdx.x; j < nb; j += BLEND_THREADS)
          if (sm.contrib[j]) rendered_next[sm.id[j]] = 1;
      }
    }
#pragma unroll
    for (int i = 0; i < PPT; ++i) {
      const int px = px0 + i;
      if (!row_in || px >= k.W) continue;
      const size_t pix = (size_t)py * k.W + px;
      image[pix * 3 + 0] = p[i].Cr + p[i].T * fc.bg[0];
      image[pix * 3 + 1] = p[i].Cg + p[i].T * fc.bg[1];
      image[pix * 3 + 2] = p[i].Cb + p[i].T * fc.bg[2];
      if (p[i].Sw > 0.0f) {
        const float m1 = p[i].S1 / p[i].Sw;
        depth[pix] = p[i].d0 + m1;
        sigma[pix] = sqrtf(fmaxf(0.0f, p[i].S2 / p[i].Sw - m1 * m1));
      } else {
        depth[pix] = TGS_DEPTH_INVALID;
        sigma[pix] = 0.0f;
      }
    }
    if (COUNT) {
      nint = __reduce_add_sync(0xffffffffu, nint);
      if (lane == 0 && nint) atomicAdd(&counters->n_interactions, (unsigned long long)nint);
    }
  }
}

}  // namespace

void launch_blend(cudaStream_t s, const FrameConst& fc, DevBuffers& b, int sorted_idx, int out_idx, const float* prior_image,
                  uint8_t* rendered_next, int num_sms, bool count_interactions) {
  const int grid = num_sms * 16;
#define LAUNCH(M, C)                                                                                                          \
  k_blend<M, C><<<grid, BLEND_THREADS, 0, s>>>(fc, b.tile_order, b.ranges, b.vals[sorted_idx], b.rec_b0, b.rec_b1, b.rec_rgb, \
                                               prior_image, b.fill_depth, b.warp_sigma, b.image[out_idx], b.depth[out_idx],  \
                                               b.sigma[out_idx], rendered_next, b.counters)
  if (rendered_next) { if (count_interactions) LAUNCH(true, true); else LAUNCH(true, false); }
  else { if (count_interactions) LAUNCH(false, true); else LAUNCH(false, false); }
#undef LAUNCH
}
