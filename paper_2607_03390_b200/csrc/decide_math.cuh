// decide_math.cuh -- fp32 decision arithmetic shared by the kernels that take the tile test box-min q <= tau
// (T^oc marks in k_decide.cu, pair emission in k_bin.cu).  Only translation units compiled with
// -fmad=false may include it: every +,-,*,/ is one IEEE rounding in the order written (DESIGN.md §2 R33).
// NOT shared with oracle/.
#pragma once
#include <stdint.h>

// min over the tile's pixel-centre box [x0,x1]x[y0,y1] of A dx^2 + 2B dx dy + C dy^2 (R18):
// 0 if the centre is inside; else the min over the four edges, each with the unconstrained 1-D optimum clamped
// to the edge.
__device__ __forceinline__ float box_qmin(float u, float v, float A, float B, float C, float x0, float x1, float y0, float y1) {
  if (u >= x0 && u <= x1 && v >= y0 && v <= y1) return 0.0f;
  const float xl = x0 - u, xh = x1 - u, yl = y0 - v, yh = y1 - v;
  const float B2 = 2.0f * B;
  float best;
  {
    float t = -(B * xl) / C; t = fminf(fmaxf(t, yl), yh);
    best = ((A * xl) * xl + (B2 * xl) * t) + (C * t) * t;
    t = -(B * xh) / C; t = fminf(fmaxf(t, yl), yh);
    best = fminf(best, ((A * xh) * xh + (B2 * xh) * t) + (C * t) * t);
  }
  {
    float t = -(B * yl) / A; t = fminf(fmaxf(t, xl), xh);
    best = fminf(best, ((A * t) * t + (B2 * t) * yl) + (C * yl) * yl);
    t = -(B * yh) / A; t = fminf(fmaxf(t, xl), xh);
    best = fminf(best, ((A * t) * t + (B2 * t) * yh) + (C * yh) * yh);
  }
  return best;
}

// Does Gaussian (u, v, conic A B C, tau = 2 ln(255 o)) reach tile (tx, ty)?  max alpha over the tile's in-image
// pixel-centre box >= 1/255 (L119 for T^oc; R39 for "intersects", L61).
__device__ __forceinline__ bool tile_alpha_reach(float u, float v, float A, float B, float C, float tau, uint32_t tx, uint32_t ty, int W, int H) {
  const float x0 = (float)(tx * 16u), x1 = (float)min((int)(tx * 16u + 15u), W - 1);
  const float y0 = (float)(ty * 16u), y1 = (float)min((int)(ty * 16u + 15u), H - 1);
  return tau >= 0.0f && box_qmin(u, v, A, B, C, x0, x1, y0, y1) <= tau;
}

// Tiles [x_lo, x_hi) x [y_lo, y_hi) of the 3-sigma extent of a Gaussian at (u, v) with radius `rad` pixels (R3),
// clipped to the TX x TY tile grid.  k_preprocess decides with it; the test-only view of the rects recomputes it from the
// stored (u, v, rad) instead of reading a record nobody else needs.
__device__ __forceinline__ void tile_rect(float u, float v, float rad, float TXf, float TYf, uint32_t& x_lo, uint32_t& x_hi, uint32_t& y_lo, uint32_t& y_hi) {
  x_lo = (uint32_t)fminf(fmaxf(floorf((u - rad) / 16.0f), 0.0f), TXf);
  x_hi = (uint32_t)fminf(fmaxf(floorf((u + rad + 15.0f) / 16.0f), 0.0f), TXf);
  y_lo = (uint32_t)fminf(fmaxf(floorf((v - rad) / 16.0f), 0.0f), TYf);
  y_hi = (uint32_t)fminf(fmaxf(floorf((v + rad + 15.0f) / 16.0f), 0.0f), TYf);
}
