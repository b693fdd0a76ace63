// k_blend.cu -- A8 front-to-back alpha blending of the selected tiles (+ Eq.1-2 depth moments and the
// G_rendered marks on R / P frames) fused with A9, the stitch of the non-selected tiles from the
// backward-warped TAB (Eq.4).  PAPER.md:L61 (alpha-blending), L73-84 (Eq.1-2), L103 (G_rendered),
// L101 + L125-128 (bilinear TAB, Eq.4).  Constants of R2: alpha <= 0.99, skip alpha < 1/255, stop when
// T(1-alpha) < 1e-4.
//
// One persistent grid; a work item is a tile of `tile_order` (selected tiles first).  A CTA is 64 threads = one
// 16x16 tile.  The tile's sorted Gaussians stream through shared memory in batches of 128 records, double
// buffered with cp.async (the gather of batch b+1 overlaps the arithmetic of batch b).
//
// DENSE mode (all pixels of the tile): each thread owns a run of 4 horizontally adjacent pixels, so that what
// depends only on the Gaussian and the row (two shared-memory loads, dy, D' dy^2 + log2 o, t at the first pixel) is
// paid once per 4 interactions: alpha_i = exp2(A' t_i^2 + D' dy^2 + log2 o), t_i = t_0 - i.  The form is
// -1/2 delta^T Sigma'^-1 delta completed to two squares, which has no cancellation between terms (R36).
// SPARSE mode: a tile is finished only when its LAST pixel is saturated or the list ends, and in a cloud with gaps
// a few pixels per tile never saturate while most are done after a small part of the list.  When at most 64 pixels
// are still alive at a batch boundary, their states are compacted through shared memory to one pixel per thread
// (again at <= 32: one warp), so the rest of the list costs work in proportion to the pixels that still need it.
// This kernel is FP32-pipe / issue bound, not HBM bound.
#include "tgs_internal.cuh"
#include <type_traits>

namespace {

constexpr int PPT = 4;                 // pixels per thread (dense mode): a run of PPT horizontally adjacent pixels
constexpr int NQ = PPT / 2;            // packed pairs per thread
constexpr int RUNS = 16 / PPT;         // runs per tile row
constexpr int BLEND_THREADS = 256 / PPT;   // 16 rows x RUNS runs
constexpr int BLEND_WARPS = BLEND_THREADS / 32;
constexpr int BLEND_MIN_CTAS = PPT == 4 ? 10 : PPT == 8 ? 16 : 8;
constexpr int BLEND_BATCH = PPT == 8 ? 64 : 128;   // records per batch (two batches in flight per CTA)
constexpr int IDS_PER_THREAD = BLEND_BATCH / BLEND_THREADS;
constexpr int DENSE_GROUP = 8;         // records between two "whole warp finished" tests of the dense loop (divides BLEND_BATCH)
constexpr int DENSE_UNROLL = 8;
constexpr float ALPHA_MIN = 1.0f / 255.0f;
// log2(1/255) = -7.99435...; anything below this bound (with a safety gap far above the rounding of e and of
// ex2.approx) has alpha < 1/255 for sure, so the exact test on alpha is only evaluated near or above the threshold
constexpr float LOG2_ALPHA_MIN_LO = -7.9950f;
// log2(0.99) = -0.01449957...; a Gaussian with log2 o below this bound (1e-6 relative under 0.99, four times the error of
// ex2.approx) has alpha = o exp(q) < 0.99 at every pixel (q <= 0), so min(0.99, .) is the identity for it
constexpr float LOG2_O_NEVER_CLAMPED = -0.014501f;
// The skip test alpha >= 1/255 of the dense loop costs nothing: the exponent is biased by EX2_BIAS so that alpha = 1/255
// falls on 2^-126, the smallest normal number -- ex2.approx.ftz flushes every result below it to zero -- and the result is
// scaled back by EX2_SCALE = 2^-EX2_BIAS (the bias as rounded to fp32, so the scale is exact to 6e-8; the threshold sits at
// (1 - 5e-7) / 255).  Price: the biased exponent (~ -120) is rounded to 7.6e-6, alpha is good to 5e-6 relative instead of
// 3e-7 -- far inside the RGB tolerance and the margins the oracle attaches to the skip / stop decisions.
constexpr float EX2_BIAS = -118.00564575195312f;
constexpr float EX2_SCALE = 3.3360998530693856e+35f;
// The dense loop keeps the transmittance scaled, T' = EX2_SCALE T, so that the unscaled ex2 result beta = alpha / EX2_SCALE
// gives the weight alpha T = beta T' and the update T'(1 - alpha) = T' - EX2_SCALE (beta T') in two packed instructions
// (instead of scale, 1 - alpha, T (1 - alpha), alpha T); the stop test compares with 1e-4 EX2_SCALE.  Groups that hold a
// Gaussian with o > 0.99 take alpha = min(0.99, beta EX2_SCALE) and T' (1 - alpha) as written: next to the clamp 1 - alpha
// must be exact (two clamped Gaussians give T = 0.01^2 against the threshold 1e-4, R33).
constexpr float EX2_SCALE_INV = 2.997512208892664e-36f;    // 1 / EX2_SCALE
constexpr float T_STOP_SCALED = 3.3360997079982872e+31f;   // 1e-4f * EX2_SCALE

__device__ __forceinline__ float ex2_approx(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gmem_src) {
  const uint32_t d = (uint32_t)__cvta_generic_to_shared(smem_dst);
  asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

// T' -> T, sign kept (a finished pixel carries T' < 0); an untouched pixel is exactly 1 (write_pixel and the sparse mode test T == 1)
__device__ __forceinline__ float unscale_T(float t) { return fabsf(t) == EX2_SCALE ? copysignf(1.0f, t) : t * EX2_SCALE_INV; }

template <bool HALF>
struct BatchT {              // HALF: slot BLEND_BATCH is a null record (log2 o = -inf: alpha = 0 everywhere), the padding of the half-tile lists
  static constexpr int N = BLEND_BATCH + (HALF ? 1 : 0);
  float4 a[N];     // u, v, A', k
  float4 b[N];     // D', log2(o), d, -
  float4 c[N];     // r, g, b, -
  uint32_t id[N];  // Gaussian index (for the G_rendered marks)
  uint8_t contrib[BLEND_BATCH + (HALF ? 4 : 0)];   // G_rendered marks of the batch (benign same-value races)
};

struct Pixel {               // per-pixel state of the front-to-back loop; sum of the weights = 1 - T (telescoping)
  float T, Cr, Cg, Cb, S1, S2, d0;
};

template <bool HALF>
struct BlendSmemT {
  BatchT<HALF> bt[2];
  float st[BLEND_THREADS][7];      // pixel states in transit during a compaction
  uint16_t st_px[BLEND_THREADS];   // their pixel index inside the tile (ly * 16 + lx)
  uint32_t alive_cnt[2][BLEND_WARPS];   // [parity][warp] alive pixels
  uint32_t work;
  uint8_t wl[HALF ? BLEND_WARPS : 1][HALF ? BLEND_BATCH + DENSE_GROUP : 4];   // HALF: per warp, the records of the batch that can reach its half tile, in order
};

// one (pixel, Gaussian) interaction (sparse mode); returns false when the pixel is finished
__device__ __forceinline__ bool blend_one(Pixel& p, float e, float r, float g, float b, float d, bool& marked, uint32_t& nhit) {
  const float alpha = fminf(0.99f, ex2_approx(e));
  if (alpha < ALPHA_MIN) return true;
  const float Tn = p.T * (1.0f - alpha);
  if (Tn < 1.0e-4f) return false;
  const float wgt = alpha * p.T;
  p.Cr = fmaf(wgt, r, p.Cr); p.Cg = fmaf(wgt, g, p.Cg); p.Cb = fmaf(wgt, b, p.Cb);
  if (p.T == 1.0f) p.d0 = d;              // first contribution: the depth moments are taken about it (R30)
  const float dd = d - p.d0;
  p.S1 = fmaf(wgt, dd, p.S1); p.S2 = fmaf(wgt * dd, dd, p.S2);
  p.T = Tn;
  marked = true;
  ++nhit;
  return true;
}

__device__ __forceinline__ void write_pixel(const FrameConst& fc, const Pixel& p, size_t pix, float* __restrict__ image,
                                            float* __restrict__ depth, float* __restrict__ sigma) {
  image[pix * 3 + 0] = p.Cr + p.T * fc.bg[0];
  image[pix * 3 + 1] = p.Cg + p.T * fc.bg[1];
  image[pix * 3 + 2] = p.Cb + p.T * fc.bg[2];
  if (p.T < 1.0f) {
    const float Sw = 1.0f - p.T;
    const float m1 = p.S1 / Sw;
    depth[pix] = p.d0 + m1;
    sigma[pix] = sqrtf(fmaxf(0.0f, p.S2 / Sw - m1 * m1));
  } else {
    depth[pix] = TGS_DEPTH_INVALID;
    sigma[pix] = 0.0f;
  }
}

// The marking instances promise one CTA per SM less: ptxas still allocates 96 registers (10 CTAs per SM stay resident) but
// schedules the loop with fewer spills around the batch boundaries (P-frame blend 0.166 -> 0.162 ms).
// HALF: each warp (a 16 x 8 half tile) runs the dense loop only over the records of the batch that can reach its half with
// alpha >= 1/255: a conservative bound on the exponent over the half's pixel box (never skips a record that could reach;
// the result changes only by which records share a clamp group, i.e. by rounding), evaluated by the warp while the batch sits in shared memory.  Pays on scenes of small
// splats (config 4: 36 % of the (record, half tile) visits reach nothing; config 3: 0.5-7 %, where it is left off).
// SLABS: the instance for frames rendered in several front-to-back pieces (park / restore of pixel states, live tiles);
// one-piece frames run the instance without any of it, whose blend loop is register-allocated as in round 1.
template <bool MARK, bool COUNT, bool HALF, bool SLABS>
__global__ void __launch_bounds__(BLEND_THREADS, MARK ? BLEND_MIN_CTAS - 1 : BLEND_MIN_CTAS) k_blend(FrameConst fc, const uint32_t* __restrict__ tile_order,
                                                         uint2* __restrict__ ranges, const uint32_t* __restrict__ vals,
                                                         const float4* __restrict__ rec_b0, const float4* __restrict__ rec_b1,
                                                         const float4* __restrict__ rec_rgb, const float* __restrict__ prior_image,
                                                         const float* __restrict__ fill_depth, const float2* __restrict__ warp_tgb,
                                                         float* __restrict__ image, float* __restrict__ depth, float* __restrict__ sigma,
                                                         uint8_t* __restrict__ rendered_next, Counters* __restrict__ counters,
                                                         uint32_t* __restrict__ tile_flags, uint32_t* __restrict__ live_bits,
                                                         float* __restrict__ pix_state, int slab) {
  TGS_PDL_WAIT();
  TGS_PDL_TRIGGER();
  __shared__ BlendSmemT<HALF> sm;
  using Batch = BatchT<HALF>;
  const CamConst& k = fc.cam;
  const uint32_t tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  const int lx = (int)(tid % RUNS) * PPT, ly = (int)(tid / RUNS);
  const uint32_t n_sel = counters->n_sel;
  if constexpr (HALF) if (tid < 2) {
    Batch& Bn = sm.bt[tid];
    Bn.a[BLEND_BATCH] = make_float4(0.0f, 0.0f, 0.0f, 0.0f); Bn.b[BLEND_BATCH] = make_float4(0.0f, -INFINITY, 0.0f, 0.0f);
    Bn.c[BLEND_BATCH] = make_float4(0.0f, 0.0f, 0.0f, 0.0f); Bn.id[BLEND_BATCH] = 0u;
  }
  // Front-to-back slabs: this launch blends the pairs of slab `slab`.  A tile whose pixels have all
  // stopped is written out and leaves `live_bits` (the later slabs bin no pairs for it); a tile that is still alive at the
  // end of its list parks its pixel states in `pix_state` and goes on in the next slab; the last slab writes every tile.
  const bool last = !SLABS || slab == fc.n_slabs - 1;
  const uint32_t n_work = (!SLABS || slab == 0) ? (uint32_t)fc.n_tiles : n_sel;      // the stitched tiles are done with slab 0
  uint32_t zero_tile = 0xffffffffu;                                       // (thread 0) tile whose range is to be cleared for the next slab
  if (SLABS && slab > 0) {                                                // every selected tile finished in the earlier slabs: nothing to do
    uint32_t fin = 0;
    for (int j = 0; j < slab; ++j) fin += counters->n_finished[j];
    if (fin >= n_sel) return;
  }
  while (true) {
    __syncthreads();
    if (tid == 0) {
      if (SLABS && zero_tile != 0xffffffffu) { ranges[zero_tile] = make_uint2(0u, 0u); zero_tile = 0xffffffffu; }
      sm.work = atomicAdd(&counters->ticket_blend[slab], 1u);
    }
    __syncthreads();
    const uint32_t w = sm.work;
    if (w >= n_work) break;
    const uint32_t tile = tile_order[w];
    const int tile_x0 = (int)(tile % k.TX) * TGS_TILE, tile_y0 = (int)(tile / k.TX) * TGS_TILE;
    const int px0 = tile_x0 + lx, py = tile_y0 + ly;
    const bool row_in = py < k.H;
    if (w >= n_sel) {
      // ------------------------------------------------ A9 stitch (Eq.4, second case)
#pragma unroll
      for (int i = 0; i < PPT; ++i) {
        const int px = px0 + i;
        if (!row_in || px >= k.W) continue;
        const size_t pix = (size_t)py * k.W + px;
        const size_t tq = (size_t)(py / fc.tg.ds) * fc.tg.W + (size_t)(px / fc.tg.ds);   // TGB grid pixel (R43)
        const float D = fill_depth[tq];
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
        sigma[pix] = warp_tgb[tq].y;
      }
      continue;
    }
    // -------------------------------------------------- A8 blend
    if (SLABS && slab > 0 && !((live_bits[tile >> 5] >> (tile & 31u)) & 1u)) continue;      // finished (and written) in an earlier slab
    uint2 range = ranges[tile];                      // {~start, end}, zero for a tile without pairs (k_sort.cu, A7)
    range.x = range.y ? ~range.x : 0u;
    const uint32_t len = range.y - range.x, nb = (len + BLEND_BATCH - 1) / BLEND_BATCH;
    if (SLABS && len == 0u && !last) continue;       // nothing of this slab reaches the tile: its state, if any, stays parked
    if (SLABS && !last && tid == 0) zero_tile = tile;
    const bool restore = SLABS && slab > 0 && (tile_flags[tile] & 8u) != 0u;
    float* const st_base = pix_state + (size_t)tile * (7 * TGS_TILE * TGS_TILE);
    float fpx = (float)px0, fpy = (float)py;
    // dense mode: pixels (0,1) and (2,3) of the run as two packed pairs (fma.rn.f32x2 of sm_100); sparse mode: sp
    float2 T2[NQ], Cr2[NQ], Cg2[NQ], Cb2[NQ], S12[NQ], S22[NQ];
    // reference depth of the run's Eq.1-2 moments (R30): the depth of the first record that any of its PPT pixels
    // composites (`open` until then).  Per run, not per pixel: two compares / selects per record instead of two per pixel;
    // a pixel whose own first contribution comes later only has its moments taken about a slightly nearer depth
    float dref = 0.0f;
    bool open = true;
    Pixel sp;
    // dense mode keeps no alive flags: a finished pixel carries T < 0 (its |T| is the final transmittance), so that
    // T (1 - alpha) >= 1e-4 fails for it by itself; pixels outside the image start finished
    bool valid[PPT], salive = false;
#pragma unroll
    for (int q = 0; q < NQ; ++q) {
      Cr2[q] = Cg2[q] = Cb2[q] = S12[q] = S22[q] = make_float2(0.0f, 0.0f);
    }
#pragma unroll
    for (int i = 0; i < PPT; ++i) valid[i] = row_in && px0 + i < k.W;
#pragma unroll
    for (int q = 0; q < NQ; ++q) T2[q] = make_float2(valid[2 * q] ? EX2_SCALE : -EX2_SCALE, valid[2 * q + 1] ? EX2_SCALE : -EX2_SCALE);   // T' = EX2_SCALE T
    if (SLABS && restore) {
      // parked states, [field][pixel]: T' (scaled, negative = stopped, 0 = already written), Cr, Cg, Cb, S1, S2, d0
      static_assert(PPT == 4, "state layout: one float4 per thread and field");
      float f[7][PPT];
#pragma unroll
      for (int j = 0; j < 7; ++j) {
        const float4 t4 = reinterpret_cast<const float4*>(st_base + j * (TGS_TILE * TGS_TILE))[tid];
        f[j][0] = t4.x; f[j][1] = t4.y; f[j][2] = t4.z; f[j][3] = t4.w;
      }
      // common reference depth of the run's Eq.1-2 moments: that of its first pixel with a contribution; the moments of
      // pixels parked with another reference (sparse mode keeps one per pixel) are re-referenced (values, not decisions)
      bool have_ref = false;
#pragma unroll
      for (int i = 0; i < PPT; ++i) {
        if (f[0][i] == 0.0f) { valid[i] = false; f[0][i] = -EX2_SCALE; }
        else if (!have_ref && fabsf(f[0][i]) != EX2_SCALE) { have_ref = true; dref = f[6][i]; }
      }
      open = !have_ref;
#pragma unroll
      for (int i = 0; i < PPT; ++i) {
        if (valid[i] && fabsf(f[0][i]) != EX2_SCALE && f[6][i] != dref) {
          const float Sw = 1.0f - fabsf(f[0][i]) * EX2_SCALE_INV, dl = f[6][i] - dref;
          f[5][i] = fmaf(dl, fmaf(Sw, dl, 2.0f * f[4][i]), f[5][i]);
          f[4][i] = fmaf(Sw, dl, f[4][i]);
        }
      }
#pragma unroll
      for (int q = 0; q < NQ; ++q) {
        T2[q] = make_float2(f[0][2 * q], f[0][2 * q + 1]); Cr2[q] = make_float2(f[1][2 * q], f[1][2 * q + 1]);
        Cg2[q] = make_float2(f[2][2 * q], f[2][2 * q + 1]); Cb2[q] = make_float2(f[3][2 * q], f[3][2 * q + 1]);
        S12[q] = make_float2(f[4][2 * q], f[4][2 * q + 1]); S22[q] = make_float2(f[5][2 * q], f[5][2 * q + 1]);
      }
    }
    auto get_px = [&](int i) {
      Pixel r;
      const int q = i >> 1;
      if (i & 1) { r.T = unscale_T(T2[q].y); r.Cr = Cr2[q].y; r.Cg = Cg2[q].y; r.Cb = Cb2[q].y; r.S1 = S12[q].y; r.S2 = S22[q].y; r.d0 = dref; }
      else { r.T = unscale_T(T2[q].x); r.Cr = Cr2[q].x; r.Cg = Cg2[q].x; r.Cb = Cb2[q].x; r.S1 = S12[q].x; r.S2 = S22[q].x; r.d0 = dref; }
      return r;
    };
    auto count_alive = [&]() {
      uint32_t c = 0;
#pragma unroll
      for (int q = 0; q < NQ; ++q) c += (uint32_t)(T2[q].x > 0.0f) + (uint32_t)(T2[q].y > 0.0f);
      return c;
    };
    bool sparse = false, have = false;      // sparse mode: this thread owns pixel `spx` of the tile in p[0]
    uint32_t spx = 0, slots = TGS_TILE * TGS_TILE;
    uint32_t gid[IDS_PER_THREAD];
    auto load_ids = [&](uint32_t b) {
#pragma unroll
      for (int s = 0; s < IDS_PER_THREAD; ++s) {
        const uint32_t idx = range.x + b * BLEND_BATCH + tid + s * BLEND_THREADS;
        gid[s] = (b < nb && idx < range.y) ? vals[idx] : 0xffffffffu;
      }
    };
    auto issue = [&](uint32_t b) {
      Batch& B = sm.bt[b & 1];
#pragma unroll
      for (int s = 0; s < IDS_PER_THREAD; ++s) {
        const uint32_t j = tid + s * BLEND_THREADS;
        if (gid[s] != 0xffffffffu) {
          cp_async16(&B.a[j], rec_b0 + 2 * (size_t)gid[s]); cp_async16(&B.b[j], rec_b1 + 2 * (size_t)gid[s]); cp_async16(&B.c[j], rec_rgb + gid[s]);   // b0 / b1 interleaved: one sector
          B.id[j] = gid[s];
          if (MARK) B.contrib[j] = 0;
        } else {
          // padding behind the end of the list: log2 o = -inf gives alpha = 0 at every pixel, so the dense loop can run
          // in whole groups of DENSE_GROUP records without a bound check per record
          B.a[j] = make_float4(0.0f, 0.0f, 0.0f, 0.0f); B.b[j] = make_float4(0.0f, -INFINITY, 0.0f, 0.0f);
          B.c[j] = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
        }
      }
      cp_async_commit();
    };
    auto writeback_marks = [&](uint32_t b) {       // own slots of batch b
      const Batch& B = sm.bt[b & 1];
      const uint32_t cnt = min((uint32_t)BLEND_BATCH, len - b * BLEND_BATCH);
#pragma unroll
      for (int s = 0; s < IDS_PER_THREAD; ++s) {
        const uint32_t j = tid + s * BLEND_THREADS;
        if (j < cnt && B.contrib[j]) rendered_next[B.id[j]] = 1;
      }
    };
    load_ids(0); issue(0); load_ids(1);
    uint32_t nint = 0, nhit = 0, nslot = 0, nwrec = 0, nwdead = 0;
    int computed = -1;
    uint32_t nb_done = 0;                   // batches this tile went through (COUNT)
    for (uint32_t b = 0; b < nb; ++b) {
      const uint32_t na_t = sparse ? (uint32_t)(have && salive)
                                   : count_alive();
      const uint32_t na_w = __reduce_add_sync(0xffffffffu, na_t);
      if (lane == 0) sm.alive_cnt[b & 1][wid] = na_w;
      cp_async_wait_all();
      __syncthreads();
      uint32_t alive_before = 0, total_alive = 0;        // alive pixels in the warps before this one, in the tile
#pragma unroll
      for (int w_ = 0; w_ < BLEND_WARPS; ++w_) { const uint32_t a_ = sm.alive_cnt[b & 1][w_]; if ((uint32_t)w_ < wid) alive_before += a_; total_alive += a_; }
      if (MARK && b > 0) writeback_marks(b - 1);
      computed = -1;
      if (total_alive == 0) break;
      if (b + 1 < nb) issue(b + 1);
      load_ids(b + 2);
      // ---- compaction of the alive pixels to one per thread
      if ((total_alive <= BLEND_THREADS && slots > BLEND_THREADS) || (BLEND_THREADS > 32 && total_alive <= 32 && slots > 32)) {
        uint32_t incl = na_t;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) { const uint32_t o = __shfl_up_sync(0xffffffffu, incl, d); if (lane >= (uint32_t)d) incl += o; }
        uint32_t pos = alive_before + incl - na_t;
        if (!sparse) {
#pragma unroll
          for (int i = 0; i < PPT; ++i) {
            if (!valid[i]) continue;
            Pixel pi = get_px(i);
            const bool alive_i = pi.T > 0.0f;
            pi.T = fabsf(pi.T);
            if (alive_i) {
              float* s = sm.st[pos];
              s[0] = pi.T; s[1] = pi.Cr; s[2] = pi.Cg; s[3] = pi.Cb; s[4] = pi.S1; s[5] = pi.S2; s[6] = pi.d0;
              sm.st_px[pos] = (uint16_t)(ly * TGS_TILE + lx + i);
              ++pos;
            } else write_pixel(fc, pi, (size_t)py * k.W + px0 + i, image, depth, sigma);
          }
        } else if (have) {
          if (salive) {
            float* s = sm.st[pos];
            s[0] = sp.T; s[1] = sp.Cr; s[2] = sp.Cg; s[3] = sp.Cb; s[4] = sp.S1; s[5] = sp.S2; s[6] = sp.d0;
            sm.st_px[pos] = (uint16_t)spx;
          } else write_pixel(fc, sp, (size_t)(tile_y0 + (int)(spx >> 4)) * k.W + tile_x0 + (int)(spx & 15u), image, depth, sigma);
        }
        __syncthreads();
        sparse = true;
        have = tid < total_alive;
        salive = have;
        if (have) {
          const float* s = sm.st[tid];
          sp.T = s[0]; sp.Cr = s[1]; sp.Cg = s[2]; sp.Cb = s[3]; sp.S1 = s[4]; sp.S2 = s[5]; sp.d0 = s[6];
          spx = sm.st_px[tid];
          fpx = (float)(tile_x0 + (int)(spx & 15u)); fpy = (float)(tile_y0 + (int)(spx >> 4));
        }
        slots = total_alive <= 32 ? 32u : (uint32_t)BLEND_THREADS;
      }
      // ---- the batch
      const Batch& B = sm.bt[b & 1];
      Batch& Bw = sm.bt[b & 1];
      const uint32_t cnt = min((uint32_t)BLEND_BATCH, len - b * BLEND_BATCH);
      if (!sparse) {
        if (__any_sync(0xffffffffu, na_t != 0u)) {
          // branch-free: 85 % of the interactions of an alive pixel composite, so every pixel runs the whole update with
          // alpha forced to 0 where it is skipped (alpha < 1/255), stops (T (1 - alpha) < 1e-4) or is finished
          const float2 one2 = make_float2(1.0f, 1.0f), neg2 = make_float2(-1.0f, -1.0f);
          const float2 scale2 = make_float2(EX2_SCALE, EX2_SCALE), nscale2 = make_float2(-EX2_SCALE, -EX2_SCALE);
          // a group of DENSE_GROUP records; CLAMP = false: none of them can reach alpha = 0.99 (one FMNMX less per pixel)
          auto dense_group = [&](const uint32_t j0, auto clamp_tag) {
           constexpr bool CLAMP = decltype(clamp_tag)::value;
#pragma unroll(DENSE_UNROLL)
           for (uint32_t jj = 0; jj < DENSE_GROUP; ++jj) {
            const uint32_t j = HALF ? (uint32_t)sm.wl[wid][j0 + jj] : j0 + jj;
            const float4 ga = B.a[j];
            const float4 gb = B.b[j];
            const float4 gc = B.c[j];
            if (COUNT && j < cnt && j < (uint32_t)BLEND_BATCH) {
              nslot += PPT;
              nint += count_alive();
            }
            const float dy = ga.y - fpy;
            const float e1 = fmaf(gb.x * dy, dy, gb.y) + EX2_BIAS;      // D' dy^2 + log2 o (+ the bias of the free skip test)
            const float t0 = fmaf(ga.w, dy, ga.x - fpx);                // t at the first pixel of the run
            const float2 e12 = make_float2(e1, e1), A2 = make_float2(ga.z, ga.z);
            dref = open ? gb.z : dref;                                  // follows the list until the run's first contribution
            const float ddf = gb.z - dref;
            const float2 dd = make_float2(ddf, ddf), dd2 = make_float2(ddf * ddf, ddf * ddf);   // d - d_ref and its square
            float2 tt[NQ];
#pragma unroll
            for (int q = 0; q < NQ; ++q) tt[q] = __fadd2_rn(make_float2(t0, t0), make_float2(-(float)(2 * q), -(float)(2 * q + 1)));
            float2 wsum = make_float2(0.0f, 0.0f);
            bool reach_lane = false;                                    // (COUNT) alpha >= 1/255 at one of this lane's pixels
#pragma unroll
            for (int q = 0; q < NQ; ++q) {
              const float2 e = __ffma2_rn(__fmul2_rn(A2, tt[q]), tt[q], e12);     // log2(o) + log2 of the falloff
              const float2 be = make_float2(ex2_approx(e.x), ex2_approx(e.y));   // alpha / EX2_SCALE; 0 below 1/255: skip (R2)
              float2 wgt, Tn;                                                      // alpha T and T' (1 - alpha); Tn < 0 for a finished pixel
              if (CLAMP) {
                float2 al = __fmul2_rn(be, scale2);
                al.x = fminf(0.99f, al.x); al.y = fminf(0.99f, al.y);
                Tn = __fmul2_rn(T2[q], __ffma2_rn(al, neg2, one2));
                wgt = __fmul2_rn(al, __fmul2_rn(T2[q], make_float2(EX2_SCALE_INV, EX2_SCALE_INV)));
              } else {
                wgt = __fmul2_rn(be, T2[q]);
                Tn = __ffma2_rn(wgt, nscale2, T2[q]);
              }
              const bool bl0 = Tn.x >= T_STOP_SCALED, bl1 = Tn.y >= T_STOP_SCALED;   // else: stop (R2) or already finished
              wgt.x = bl0 ? wgt.x : 0.0f; wgt.y = bl1 ? wgt.y : 0.0f;                // 0 where nothing is composited
              if (COUNT) { nhit += (uint32_t)(wgt.x > 0.0f) + (uint32_t)(wgt.y > 0.0f); reach_lane = reach_lane || be.x > 0.0f || be.y > 0.0f; }
              T2[q].x = bl0 ? Tn.x : -fabsf(T2[q].x);                 // Tn = T' where alpha was skipped
              T2[q].y = bl1 ? Tn.y : -fabsf(T2[q].y);
              if (MARK) wsum = __fadd2_rn(wsum, wgt);
              Cr2[q] = __ffma2_rn(wgt, make_float2(gc.x, gc.x), Cr2[q]);
              Cg2[q] = __ffma2_rn(wgt, make_float2(gc.y, gc.y), Cg2[q]);
              Cb2[q] = __ffma2_rn(wgt, make_float2(gc.z, gc.z), Cb2[q]);
              S12[q] = __ffma2_rn(wgt, dd, S12[q]);
              S22[q] = __ffma2_rn(wgt, dd2, S22[q]);
            }
            if (COUNT && j < cnt && j < (uint32_t)BLEND_BATCH) {         // how many (record, half tile) visits reach no pixel of the half
              ++nwrec;
              if (!__any_sync(0xffffffffu, reach_lane)) ++nwdead;
            }
            if (MARK) {
              const bool hit = wsum.x + wsum.y > 0.0f;                  // some pixel of the run composited this record
              if (hit) Bw.contrib[j] = 1;
              open = open && !hit;
            } else {
              // without marks only `open` is needed: no pixel of the run has composited yet <=> every |T'| is still
              // EX2_SCALE (pixels outside the image carry -EX2_SCALE); min / compare run on the ALU pipe, which has slack
              float tm = fminf(fabsf(T2[0].x), fabsf(T2[0].y));
#pragma unroll
              for (int q = 1; q < NQ; ++q) tm = fminf(tm, fminf(fabsf(T2[q].x), fabsf(T2[q].y)));
              open = tm == EX2_SCALE;
            }
           }
          };
          uint32_t ncnt = cnt;
          if (HALF) {
            // this warp's list: records of the batch whose exponent can reach log2(1/255) somewhere in the half's pixel box.
            // e = l + A' t^2 + D' dy^2 (A', D' <= 0), t = dx + k dy: bounded by l + A' min|t|^2 + D' min|dy|^2 over the box
            const float bx0 = (float)tile_x0, bx1 = (float)(tile_x0 + TGS_TILE - 1);
            const float by0 = (float)(tile_y0 + (int)wid * (TGS_TILE / BLEND_WARPS)), by1 = by0 + (float)(TGS_TILE / BLEND_WARPS - 1);
            uint32_t nl = 0;
            for (uint32_t r0 = 0; r0 < cnt; r0 += 32) {
              const uint32_t r = r0 + lane;
              bool reach = false;
              if (r < cnt) {
                const float4 ga = B.a[r];
                const float4 gb = B.b[r];
                const float dxl = ga.x - bx1, dxh = ga.x - bx0, dyl = ga.y - by1, dyh = ga.y - by0;
                const float dym = dyl > 0.0f ? dyl : (dyh < 0.0f ? dyh : 0.0f);                  // min |dy| over the box
                const float ka = ga.w * dyl, kb = ga.w * dyh;
                const float tl = dxl + fminf(ka, kb), th = dxh + fmaxf(ka, kb);
                float tm = tl > 0.0f ? tl : (th < 0.0f ? -th : 0.0f);                            // min |t| over the box ...
                // ... less the rounding of t itself: for needle-like splats t is a small difference of large terms (the
                // dense loop's own t has the same absolute error), and A' is large, so the bound must not lean on it
                tm = fmaxf(0.0f, tm - 2.0e-6f * (fabsf(dxl) + fabsf(dxh) + fabsf(ka) + fabsf(kb)));
                const float eb = fmaf(ga.z * tm, tm, fmaf(gb.x * dym, dym, gb.y));
                reach = eb >= LOG2_ALPHA_MIN_LO - 0.05f;
              }
              const uint32_t m = __ballot_sync(0xffffffffu, reach);
              if (reach) sm.wl[wid][nl + __popc(m & ((1u << lane) - 1u))] = (uint8_t)r;
              nl += __popc(m);
            }
            if (lane < DENSE_GROUP) sm.wl[wid][nl + lane] = (uint8_t)BLEND_BATCH;               // pad the last group with the null record
            __syncwarp();
            ncnt = nl;
          }
          for (uint32_t j0 = 0; j0 < ncnt; j0 += DENSE_GROUP) {
           float lmax = B.b[HALF ? (uint32_t)sm.wl[wid][j0] : j0].y;
#pragma unroll
           for (uint32_t jj = 1; jj < DENSE_GROUP; ++jj) lmax = fmaxf(lmax, B.b[HALF ? (uint32_t)sm.wl[wid][j0 + jj] : j0 + jj].y);
           if (lmax > LOG2_O_NEVER_CLAMPED) dense_group(j0, std::true_type()); else dense_group(j0, std::false_type());
           float tmax = fmaxf(T2[0].x, T2[0].y);
#pragma unroll
           for (int q = 1; q < NQ; ++q) tmax = fmaxf(tmax, fmaxf(T2[q].x, T2[q].y));
           if (__all_sync(0xffffffffu, tmax < 0.0f)) break;
          }
        }
      } else if (__any_sync(0xffffffffu, salive)) {
        for (uint32_t j = 0; j < cnt; ++j) {
          if ((j & 15u) == 0u && !__any_sync(0xffffffffu, salive)) break;
          const float4 ga = B.a[j];
          const float4 gb = B.b[j];
          if (COUNT) nslot += 1;
          const float dx = ga.x - fpx, dy = ga.y - fpy;
          const float t = fmaf(ga.w, dy, dx);
          const float e1 = fmaf(gb.x * dy, dy, gb.y);
          const float e = fmaf(ga.z * t, t, e1);
          if (COUNT) nint += (uint32_t)salive;
          if (salive && e >= LOG2_ALPHA_MIN_LO) {
            const float4 gc = B.c[j];
            bool marked = false;
            salive = blend_one(sp, e, gc.x, gc.y, gc.z, gb.z, marked, nhit);
            if (MARK && marked) Bw.contrib[j] = 1;
          }
        }
      }
      computed = (int)b;
      if (COUNT) nb_done = b + 1u;
    }
    if (MARK && computed >= 0) { __syncthreads(); writeback_marks((uint32_t)computed); }
    // -------------------------------------------------- outputs, or the states parked for the next slab
    bool park = false;
    if (SLABS && !last) {
      const bool alive_t = sparse ? (have && salive) : (count_alive() != 0u);
      park = __syncthreads_or(alive_t ? 1 : 0) != 0;
    }
    if (SLABS && park) {
      float4* const st4 = reinterpret_cast<float4*>(st_base);
      constexpr int FS = TGS_TILE * TGS_TILE / 4;                     // float4 per field
      if (!sparse) {
        // a pixel outside the image is parked as "written" (it never is): T' = 0
        st4[0 * FS + tid] = make_float4(valid[0] ? T2[0].x : 0.0f, valid[1] ? T2[0].y : 0.0f, valid[2] ? T2[1].x : 0.0f, valid[3] ? T2[1].y : 0.0f);
        st4[1 * FS + tid] = make_float4(Cr2[0].x, Cr2[0].y, Cr2[1].x, Cr2[1].y);
        st4[2 * FS + tid] = make_float4(Cg2[0].x, Cg2[0].y, Cg2[1].x, Cg2[1].y);
        st4[3 * FS + tid] = make_float4(Cb2[0].x, Cb2[0].y, Cb2[1].x, Cb2[1].y);
        st4[4 * FS + tid] = make_float4(S12[0].x, S12[0].y, S12[1].x, S12[1].y);
        st4[5 * FS + tid] = make_float4(S22[0].x, S22[0].y, S22[1].x, S22[1].y);
        st4[6 * FS + tid] = make_float4(dref, dref, dref, dref);
      } else {
        // sparse mode: the pixels that were dropped at a compaction have been written; the others sit one per thread
        st4[tid] = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
        __syncthreads();
        if (have) {
          float* const sf = st_base;
          const float Ts = sp.T == 1.0f ? EX2_SCALE : sp.T * EX2_SCALE;
          sf[0 * 256 + spx] = salive ? Ts : -Ts;
          sf[1 * 256 + spx] = sp.Cr; sf[2 * 256 + spx] = sp.Cg; sf[3 * 256 + spx] = sp.Cb;
          sf[4 * 256 + spx] = sp.S1; sf[5 * 256 + spx] = sp.S2; sf[6 * 256 + spx] = sp.d0;
        }
      }
      if (tid == 0) { tile_flags[tile] |= 8u; atomicAdd(&counters->n_live_after[slab], 1u); }   // only this CTA touches the flag word while the blend runs
    } else {
      if (!sparse) {
#pragma unroll
        for (int i = 0; i < PPT; ++i)
          if (valid[i]) { Pixel pi = get_px(i); pi.T = fabsf(pi.T); write_pixel(fc, pi, (size_t)py * k.W + px0 + i, image, depth, sigma); }
      } else if (have) {
        write_pixel(fc, sp, (size_t)(tile_y0 + (int)(spx >> 4)) * k.W + tile_x0 + (int)(spx & 15u), image, depth, sigma);
      }
      if (SLABS && !last && tid == 0) { atomicAnd(&live_bits[tile >> 5], ~(1u << (tile & 31u))); atomicAdd(&counters->n_finished[slab], 1u); }   // finished: no pairs in the later slabs
    }
    if (COUNT) {
      nint = __reduce_add_sync(0xffffffffu, nint);
      if (lane == 0 && nint) atomicAdd(&counters->n_interactions, (unsigned long long)nint);
      nhit = __reduce_add_sync(0xffffffffu, nhit);
      nslot = __reduce_max_sync(0xffffffffu, nslot) * 32u;     // lanes that left the loop early still occupy the warp
      if (lane == 0) { atomicAdd(&counters->n_blended, (unsigned long long)nhit); atomicAdd(&counters->n_slots, (unsigned long long)nslot); }
      if (lane == 0 && nwrec) { atomicAdd(&counters->n_wrec, (unsigned long long)nwrec); atomicAdd(&counters->n_wrec_dead, (unsigned long long)nwdead); }
      if (tid == 0 && nb_done) atomicAdd(&counters->n_consumed, (unsigned long long)min(len, nb_done * BLEND_BATCH));
    }
  }
}

}  // namespace

void launch_blend(cudaStream_t s, const FrameConst& fc, DevBuffers& b, int sorted_idx, int out_idx, const float* prior_image,
                  uint8_t* rendered_next, int num_sms, bool count_interactions, int slab) {
  const int grid = num_sms * (PPT == 4 ? 12 : PPT == 8 ? 16 : 8);
#define LAUNCH(M, C, H, SL)                                                                                                     \
  TGS_LAUNCH((k_blend<M, C, H, SL>), grid, BLEND_THREADS, 0, s, fc, b.tile_order, b.ranges, b.vals[sorted_idx], b.rec_b0, b.rec_b1, b.rec_rgb, \
                                               prior_image, b.fill_depth, (const float2*)b.warp_tgb, b.image[out_idx], b.depth[out_idx],  \
                                               b.sigma[out_idx], rendered_next, b.counters, b.tile_flags, b.live_bits, b.pix_state, slab)
#define LAUNCH2(M, C) do { if (fc.n_slabs > 1) { if (fc.blend_half) LAUNCH(M, C, true, true); else LAUNCH(M, C, false, true); } \
                           else { if (fc.blend_half) LAUNCH(M, C, true, false); else LAUNCH(M, C, false, false); } } while (0)
  if (rendered_next) { if (count_interactions) LAUNCH2(true, true); else LAUNCH2(true, false); }
  else { if (count_interactions) LAUNCH2(false, true); else LAUNCH2(false, false); }
#undef LAUNCH2
#undef LAUNCH
}
