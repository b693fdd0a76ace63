// oracle/ora.cpp -- plain, slow, single-threaded CPU oracle of the TemporalGS hot path.
//
// TEST INFRASTRUCTURE ONLY (see ora.h).  Written from PAPER.md (arxiv/paper_2607_03390); every
// function cites the passage it follows as PAPER.md:L<line>.  "R<n>" = reading listed in DESIGN.md §2.
// Shares no code with the CUDA path.  Build: g++ -O2 -std=c++17 -ffp-contract=off -fno-fast-math.
//
// Precision policy (R33): arithmetic that DECIDES an integer (cull masks, nearest
// pixel, tile rect, sort key = bits(d), tile selection, matched flags) is evaluated in IEEE fp32
// with the operation order written here -- one rounding per +,-,*,/,sqrt, no contraction -- so the
// CUDA path can take the same decision bit for bit.  Arithmetic that only produces VALUES (SH
// colour, alpha blending, Eq.1-2 moments, bilinear taps) is fp64.
//
// Pins: tests/test_oracle_pins.py (P1-P11 of DESIGN.md §5).  Unpinned: image quality (PSNR) of S
// frames and the speed-up -- "parity unpinned" by the paper, reported only.
#include "ora.h"

#include <algorithm>
#include <chrono>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <limits>
#include <string>
#include <vector>

namespace {

constexpr int TILE = 16;                       // 16x16 tiles
constexpr double ALPHA_MIN = 1.0 / 255.0;      // PAPER.md:L119 (and R2)
constexpr double ALPHA_MAX = 0.99;             // R2
constexpr double T_STOP = 1.0e-4;              // R2
constexpr float ALPHA_MIN_F = 1.0f / 255.0f, ALPHA_MAX_F = 0.99f, T_STOP_F = 1.0e-4f;   // the same, as the fp32 decisions see them
// Relative margins of "borderline" decisions (R29).  The wide pair bounds which Gaussians an fp32
// implementation MAY mark as rendered; the tight pair marks the pixels where an fp32 implementation
// (alpha accurate to ~1e-6, T to ~1e-5 relative) may legitimately take the other branch.
constexpr double MARGIN_ALPHA = 1.0e-4;
constexpr double MARGIN_T = 1.0e-2;
constexpr double PIX_MARGIN_ALPHA = 5.0e-6;
constexpr double Q_EPS = 2.4e-7;           // 4 ulp of fp32: rounding of the stored parameters + of the evaluation
constexpr double PIX_MARGIN_T = 1.0e-3;

struct Cam {
  float V[16];
  float fx, fy, cx, cy;
  int W = 0, H = 0;
  float znear, zfar;
  bool set = false;
};

double now_ms() {
  using namespace std::chrono;
  return duration<double, std::milli>(steady_clock::now().time_since_epoch()).count();
}

uint32_t f2u(float f) { uint32_t u; std::memcpy(&u, &f, 4); return u; }

// ---------------------------------------------------------------- SH basis (R5)
// Real spherical harmonics, Condon-Shortley phase folded as in the constants below, order m=-l..l.
void sh_basis(int deg, const double dir[3], double* Y) {
  const double x = dir[0], y = dir[1], z = dir[2];
  Y[0] = 0.28209479177387814;                                 // sqrt(1/(4 pi))
  if (deg < 1) return;
  const double c1 = 0.4886025119029199;                       // sqrt(3/(4 pi))
  Y[1] = -c1 * y; Y[2] = c1 * z; Y[3] = -c1 * x;
  if (deg < 2) return;
  const double xx = x * x, yy = y * y, zz = z * z, xy = x * y, yz = y * z, xz = x * z;
  Y[4] = 1.0925484305920792 * xy;                             // sqrt(15/(4 pi))
  Y[5] = -1.0925484305920792 * yz;
  Y[6] = 0.31539156525252005 * (2.0 * zz - xx - yy);          // sqrt(5/(16 pi))
  Y[7] = -1.0925484305920792 * xz;
  Y[8] = 0.5462742152960396 * (xx - yy);                      // sqrt(15/(16 pi))
  if (deg < 3) return;
  Y[9] = -0.5900435899266435 * y * (3.0 * xx - yy);           // sqrt(35/(32 pi))
  Y[10] = 2.890611442640554 * xy * z;                         // sqrt(105/(4 pi))
  Y[11] = -0.4570457994644658 * y * (4.0 * zz - xx - yy);     // sqrt(21/(32 pi))
  Y[12] = 0.3731763325901154 * z * (2.0 * zz - 3.0 * xx - 3.0 * yy);  // sqrt(7/(16 pi))
  Y[13] = -0.4570457994644658 * x * (4.0 * zz - xx - yy);
  Y[14] = 1.445305721320277 * z * (xx - yy);                  // sqrt(105/(16 pi))
  Y[15] = -0.5900435899266435 * x * (xx - 3.0 * yy);
}

// ---------------------------------------------------------------- box minimum of the conic form
// PAPER.md:L119 "filter out the newly visible Gaussians with trivial contribution to their
// intersected tiles ... alpha ... 1/255" (R18): max alpha over the tile's pixel-centre box
// >= 1/255  <=>  min over the box of q(dx,dy) = A dx^2 + 2 B dx dy + C dy^2  <=  tau.
float box_qmin(float u, float v, float A, float B, float C, float x0, float x1, float y0, float y1) {
  if (u >= x0 && u <= x1 && v >= y0 && v <= y1) return 0.0f;
  float best = std::numeric_limits<float>::infinity();
  const float xl = x0 - u, xh = x1 - u, yl = y0 - v, yh = y1 - v;
  const float B2 = 2.0f * B;
  const float ex[2] = {xl, xh};
  for (int k = 0; k < 2; ++k) {           // edges x = x0, x = x1 : dy free in [yl, yh]
    const float dx = ex[k];
    float t = -(B * dx) / C;
    t = std::fmin(std::fmax(t, yl), yh);
    const float q = ((A * dx) * dx + (B2 * dx) * t) + (C * t) * t;
    best = std::fmin(best, q);
  }
  const float ey[2] = {yl, yh};
  for (int k = 0; k < 2; ++k) {           // edges y = y0, y = y1 : dx free in [xl, xh]
    const float dy = ey[k];
    float t = -(B * dy) / A;
    t = std::fmin(std::fmax(t, xl), xh);
    const float q = ((A * t) * t + (B2 * t) * dy) + (C * dy) * dy;
    best = std::fmin(best, q);
  }
  return best;
}

// rigid relative pose M = W_b * W_a^{-1} in double, rounded to 12 floats (row-major 3x4).
// PAPER.md:L88 Eq.3: K W_{t+i} W_t^{-1} D K^{-1} [x,y,1]^T.  W^{-1} = [R^T | -R^T t] (rigid).
void relative_pose(const float* Wa, const float* Wb, float* M) {
  double Ra[9], ta[3], Rb[9], tb[3];
  for (int i = 0; i < 3; ++i) {
    for (int j = 0; j < 3; ++j) { Ra[i * 3 + j] = Wa[i * 4 + j]; Rb[i * 3 + j] = Wb[i * 4 + j]; }
    ta[i] = Wa[i * 4 + 3]; tb[i] = Wb[i * 4 + 3];
  }
  double MR[9];
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j)   // MR = Rb * Ra^T
      MR[i * 3 + j] = (Rb[i * 3 + 0] * Ra[j * 3 + 0] + Rb[i * 3 + 1] * Ra[j * 3 + 1]) + Rb[i * 3 + 2] * Ra[j * 3 + 2];
  for (int i = 0; i < 3; ++i) {
    const double mt = tb[i] - ((MR[i * 3 + 0] * ta[0] + MR[i * 3 + 1] * ta[1]) + MR[i * 3 + 2] * ta[2]);
    M[i * 4 + 0] = (float)MR[i * 3 + 0]; M[i * 4 + 1] = (float)MR[i * 3 + 1]; M[i * 4 + 2] = (float)MR[i * 3 + 2];
    M[i * 4 + 3] = (float)mt;
  }
}

}  // namespace

struct ora_ctx {
  // scene
  uint32_t n = 0; int deg = 0; int K = 1;
  std::vector<float> means, opacity, sh, cov3d, tau;   // cov3d: 6 per Gaussian (xx,xy,xz,yy,yz,zz)
  Cam cam;
  ora_params prm;
  ora_sched sched{0, 0, 0, 0};
  int force_all = 0;
  // priors (O2)
  bool priors_valid = false, F_valid = false;
  std::vector<float> prior_depth, prior_sigma, prior_image;
  std::vector<uint8_t> rendered;          // G_rendered
  float F[4] = {0, 0, 0, 0};              // F_min.x, F_min.y, F_max.x, F_max.y
  float prior_view[16];
  // per-frame
  float M[12], Minv[12];
  // TGB grid of this frame (R43): ds = 1: the image grid; ds = 2: ceil(W/2) x ceil(H/2), grid pixel (i, j) sits at the
  // image position (2i + 0.5, 2j + 0.5), i.e. a pinhole camera with fx/2, fy/2, (cx - 0.5)/2, (cy - 0.5)/2
  int ds = 1, Wt = 0, Ht = 0;
  float tfx = 0, tfy = 0, tcx = 0, tcy = 0;
  std::vector<float> warp_depth, warp_sigma, fill_depth, corr_xy;
  std::vector<uint8_t> matched;
  std::vector<ora_record> rec;
  std::vector<uint64_t> keys; std::vector<uint32_t> vals; std::vector<uint32_t> ranges;
  std::vector<uint8_t> tile_mask;         // bit0 oc, bit1 um, bit2 selected
  std::vector<float> image, depth, sigma; // current frame
  std::vector<uint8_t> rendered_now, rendered_sure, rendered_maybe, borderline;
  ora_stats st{};
  int TX = 0, TY = 0;
};

namespace {

bool finite_all(const float* p, size_t n) {
  for (size_t i = 0; i < n; ++i) if (!std::isfinite(p[i])) return false;
  return true;
}

// ---------------------------------------------------------------- O9 forward warp (A1)
// PAPER.md:L86-97 Eq.3.  Nearest-pixel splat (R14), min depth / max sigma kept independently (R15),
// initialised to z_far+eps / 0 (L97, R12); sigma' = sigma |M_R[row 3] . ray| (R13).
void tgb_grid(ora_ctx* c) {
  const Cam& k = c->cam;
  c->ds = c->prm.tgb_downscale == 2 ? 2 : 1;
  if (c->ds == 1) { c->Wt = k.W; c->Ht = k.H; c->tfx = k.fx; c->tfy = k.fy; c->tcx = k.cx; c->tcy = k.cy; }
  else {
    c->Wt = (k.W + 1) / 2; c->Ht = (k.H + 1) / 2;
    c->tfx = k.fx * 0.5f; c->tfy = k.fy * 0.5f; c->tcx = (k.cx - 0.5f) * 0.5f; c->tcy = (k.cy - 0.5f) * 0.5f;
  }
}

// TGB source value of grid pixel (x, y).  ds = 2 (L142 "downscale the TGB by 2", operator unspecified -> R43): nearest
// valid depth of the 2x2 block and the largest sigma of its valid pixels -- the same "closer geometry, maximum
// deviation, for high recall" rule the paper states for colliding warped pixels (L91).
void tgb_source(const ora_ctx* c, int x, int y, float* D, float* sg) {
  const int W = c->cam.W, H = c->cam.H;
  if (c->ds == 1) { *D = c->prior_depth[(size_t)y * W + x]; *sg = c->prior_sigma[(size_t)y * W + x]; return; }
  float d = ORA_DEPTH_INVALID, s = 0.0f;
  for (int yy = 2 * y; yy < std::min(H, 2 * y + 2); ++yy)
    for (int xx = 2 * x; xx < std::min(W, 2 * x + 2); ++xx) {
      const float v = c->prior_depth[(size_t)yy * W + xx];
      if (!(v < 1.0e38f)) continue;
      d = std::fmin(d, v); s = std::fmax(s, c->prior_sigma[(size_t)yy * W + xx]);
    }
  *D = d; *sg = s;
}

void forward_warp(ora_ctx* c) {
  const Cam& k = c->cam; const int W = c->Wt, H = c->Ht; const float* M = c->M;
  const float fx = c->tfx, fy = c->tfy, cx = c->tcx, cy = c->tcy;
  c->warp_depth.assign((size_t)W * H, ORA_DEPTH_INVALID);
  c->warp_sigma.assign((size_t)W * H, 0.0f);
  for (int y = 0; y < H; ++y)
    for (int x = 0; x < W; ++x) {
      float D, sg;
      tgb_source(c, x, y, &D, &sg);
      if (!(D < 1.0e38f)) continue;                       // R11: no geometry -> not warped
      const float rx = ((float)x - cx) / fx, ry = ((float)y - cy) / fy;
      const float Px = D * rx, Py = D * ry, Pz = D;
      const float X = ((M[0] * Px + M[1] * Py) + M[2] * Pz) + M[3];
      const float Y = ((M[4] * Px + M[5] * Py) + M[6] * Pz) + M[7];
      const float Z = ((M[8] * Px + M[9] * Py) + M[10] * Pz) + M[11];
      if (!(Z > k.znear)) continue;
      const float u = (fx * X) / Z + cx, v = (fy * Y) / Z + cy;
      const float fu = std::floor(u + 0.5f), fv = std::floor(v + 0.5f);
      if (!(fu >= 0.0f && fu < (float)W && fv >= 0.0f && fv < (float)H)) continue;
      const size_t q = (size_t)(int)fv * W + (int)fu;
      const float s = sg * std::fabs((M[8] * rx + M[9] * ry) + M[10]);
      c->warp_depth[q] = std::fmin(c->warp_depth[q], Z);
      c->warp_sigma[q] = std::fmax(c->warp_sigma[q], s);
    }
}

// ---------------------------------------------------------------- O10 depth fill + correspondence (A2)
// PAPER.md:L121.  R19: 8 neighbours, single pass from the unrepaired buffer, border never filled.
// R20: matched <=> D' valid, back-projected z > z_near, nearest pixel of (x,y) inside the image.  R22: in-image pixels.
void fill_and_correspond(ora_ctx* c) {
  const int W = c->Wt, H = c->Ht; const float* M = c->Minv;
  struct { float fx, fy, cx, cy, znear; } k = {c->tfx, c->tfy, c->tcx, c->tcy, c->cam.znear};
  c->fill_depth = c->warp_depth;
  for (int y = 1; y < H - 1; ++y)
    for (int x = 1; x < W - 1; ++x) {
      if (c->warp_depth[(size_t)y * W + x] < 1.0e38f) continue;
      bool all = true; float sum = 0.0f; bool first = true;
      for (int dy = -1; dy <= 1 && all; ++dy)
        for (int dx = -1; dx <= 1; ++dx) {
          if (dx == 0 && dy == 0) continue;
          const float nb = c->warp_depth[(size_t)(y + dy) * W + (x + dx)];
          if (!(nb < 1.0e38f)) { all = false; break; }
          sum = first ? nb : sum + nb; first = false;
        }
      if (all) c->fill_depth[(size_t)y * W + x] = sum * 0.125f;
    }
  c->corr_xy.assign((size_t)W * H * 2, -1.0f);
  c->matched.assign((size_t)W * H, 0);
  for (int y = 0; y < H; ++y)
    for (int x = 0; x < W; ++x) {
      const float D = c->fill_depth[(size_t)y * W + x];
      if (!(D < 1.0e38f)) continue;
      const float rx = ((float)x - k.cx) / k.fx, ry = ((float)y - k.cy) / k.fy;
      const float Px = D * rx, Py = D * ry, Pz = D;
      const float X = ((M[0] * Px + M[1] * Py) + M[2] * Pz) + M[3];
      const float Y = ((M[4] * Px + M[5] * Py) + M[6] * Pz) + M[7];
      const float Z = ((M[8] * Px + M[9] * Py) + M[10] * Pz) + M[11];
      if (!(Z > k.znear)) continue;
      const float xs = (k.fx * X) / Z + k.cx, ys = (k.fy * Y) / Z + k.cy;
      c->corr_xy[((size_t)y * W + x) * 2 + 0] = xs;
      c->corr_xy[((size_t)y * W + x) * 2 + 1] = ys;
      const float fu = std::floor(xs + 0.5f), fv = std::floor(ys + 0.5f);   // nearest reference pixel inside the image (R20)
      if (fu >= 0.0f && fu < (float)W && fv >= 0.0f && fv < (float)H) c->matched[(size_t)y * W + x] = 1;
    }
}

// ---------------------------------------------------------------- O3 preprocess (A3)
// PAPER.md:L61 (near cull, projection, tile intersection), L109-111 (AFC), L113 (TOC), L119
// (newly visible).  EWA conventions of vanilla 3DGS as behaviour (R3).
void preprocess(ora_ctx* c, int ftype) {
  const Cam& k = c->cam; const float* V = k.V; const int W = k.W, H = k.H;
  const int TX = c->TX, TY = c->TY;
  const float tanx = (0.5f * (float)W) / k.fx, tany = (0.5f * (float)H) / k.fy;
  const float limx = 1.3f * tanx, limy = 1.3f * tany;
  const bool do_afc = (ftype != ORA_FRAME_R) && c->prm.enable_afc && c->F_valid;
  const bool do_tgb = (ftype == ORA_FRAME_S);
  // camera centre = -R^T t (double), for the SH view direction
  double cc[3];
  for (int j = 0; j < 3; ++j)
    cc[j] = -(((double)V[0 * 4 + j] * V[3] + (double)V[1 * 4 + j] * V[7]) + (double)V[2 * 4 + j] * V[11]);
  c->rec.assign(c->n, ora_record{});
  ora_stats& st = c->st;
  for (uint32_t g = 0; g < c->n; ++g) {
    ora_record& r = c->rec[g];
    const float x = c->means[3 * g], y = c->means[3 * g + 1], z = c->means[3 * g + 2];
    const float tx = ((V[0] * x + V[1] * y) + V[2] * z) + V[3];
    const float ty = ((V[4] * x + V[5] * y) + V[6] * z) + V[7];
    const float tz = ((V[8] * x + V[9] * y) + V[10] * z) + V[11];
    r.d = tz; r.o = c->opacity[g]; r.tau = c->tau[g];
    if (!(tz > k.znear)) { r.flags = ORA_CULL_NEAR; ++st.n_near; continue; }        // L61, R4
    const float u = (k.fx * tx) / tz + k.cx, v = (k.fy * ty) / tz + k.cy;
    r.u = u; r.v = v;
    if (do_afc) {                                                                      // L109-111, R6, R7
      const float nx = (2.0f * u + 1.0f) / (float)W - 1.0f, ny = (2.0f * v + 1.0f) / (float)H - 1.0f;
      if (!(c->F[0] <= nx && nx <= c->F[2] && c->F[1] <= ny && ny <= c->F[3])) { r.flags = ORA_CULL_AFC; ++st.n_afc; continue; }
    }
    uint32_t fl = 0;
    if (do_tgb && !c->rendered[g]) {                                                   // L113, L119, R16, R17
      const float fu = std::floor(u + 0.5f), fv = std::floor(v + 0.5f);
      if (fu >= 0.0f && fu < (float)W && fv >= 0.0f && fv < (float)H) {
        const size_t q = (size_t)((int)fv / c->ds) * c->Wt + (size_t)((int)fu / c->ds);   // R43: the block of the nearest pixel
        const float D = c->warp_depth[q], s = c->warp_sigma[q];
        if (c->prm.enable_toc && tz > D + c->prm.lambda2 * s) { r.flags = ORA_CULL_TOC; ++st.n_toc; continue; }
        if (tz <= D - c->prm.lambda1 * s) fl |= ORA_NEWLY_VISIBLE;
      }
    }
    // EWA projection (R3)
    const float* S = &c->cov3d[6 * (size_t)g];
    const float rxz = tx / tz, ryz = ty / tz;
    const float jx = std::fmin(limx, std::fmax(-limx, rxz)) * tz;
    const float jy = std::fmin(limy, std::fmax(-limy, ryz)) * tz;
    const float j00 = k.fx / tz, j02 = -(k.fx * jx) / (tz * tz);
    const float j11 = k.fy / tz, j12 = -(k.fy * jy) / (tz * tz);
    const float T00 = j00 * V[0] + j02 * V[8], T01 = j00 * V[1] + j02 * V[9], T02 = j00 * V[2] + j02 * V[10];
    const float T10 = j11 * V[4] + j12 * V[8], T11 = j11 * V[5] + j12 * V[9], T12 = j11 * V[6] + j12 * V[10];
    const float s0 = (S[0] * T00 + S[1] * T01) + S[2] * T02;
    const float s1 = (S[1] * T00 + S[3] * T01) + S[4] * T02;
    const float s2 = (S[2] * T00 + S[4] * T01) + S[5] * T02;
    const float q0 = (S[0] * T10 + S[1] * T11) + S[2] * T12;
    const float q1 = (S[1] * T10 + S[3] * T11) + S[4] * T12;
    const float q2 = (S[2] * T10 + S[4] * T11) + S[5] * T12;
    const float a = ((T00 * s0 + T01 * s1) + T02 * s2) + 0.3f;
    const float b = (T10 * s0 + T11 * s1) + T12 * s2;
    const float cc2 = ((T10 * q0 + T11 * q1) + T12 * q2) + 0.3f;
    const float det = a * cc2 - b * b;
    if (!(det > 0.0f)) { r.flags = ORA_CULL_DEGENERATE; ++st.n_degenerate; continue; }
    r.A = cc2 / det; r.B = -b / det; r.C = a / det;
    r.ca = a; r.cb = b; r.cc = cc2;
    const float mid = 0.5f * (a + cc2);
    const float lam = mid + std::sqrt(std::fmax(0.1f, mid * mid - det));
    const float rad = std::ceil(3.0f * std::sqrt(lam));
    r.radius = rad;
    const float fx_lo = std::fmin(std::fmax(std::floor((u - rad) / 16.0f), 0.0f), (float)TX);
    const float fx_hi = std::fmin(std::fmax(std::floor((u + rad + 15.0f) / 16.0f), 0.0f), (float)TX);
    const float fy_lo = std::fmin(std::fmax(std::floor((v - rad) / 16.0f), 0.0f), (float)TY);
    const float fy_hi = std::fmin(std::fmax(std::floor((v + rad + 15.0f) / 16.0f), 0.0f), (float)TY);
    r.x_lo = (uint16_t)fx_lo; r.x_hi = (uint16_t)fx_hi; r.y_lo = (uint16_t)fy_lo; r.y_hi = (uint16_t)fy_hi;
    if (!(r.x_hi > r.x_lo && r.y_hi > r.y_lo)) { r.flags = ORA_CULL_EMPTY; ++st.n_empty; continue; }
    r.flags = fl | ORA_VISIBLE; ++st.n_visible;
    if (fl & ORA_NEWLY_VISIBLE) ++st.n_newly_visible;
    // colour: SH -> RGB (R5), value arithmetic in double
    double dir[3] = {(double)x - cc[0], (double)y - cc[1], (double)z - cc[2]};
    const double nn = std::sqrt(dir[0] * dir[0] + dir[1] * dir[1] + dir[2] * dir[2]);
    dir[0] /= nn; dir[1] /= nn; dir[2] /= nn;
    double Y[16]; sh_basis(c->deg, dir, Y);
    double col[3] = {0.5, 0.5, 0.5};
    const float* shp = &c->sh[(size_t)g * c->K * 3];
    for (int kk = 0; kk < c->K; ++kk)
      for (int ch = 0; ch < 3; ++ch) col[ch] += Y[kk] * (double)shp[kk * 3 + ch];
    r.r = (float)std::max(0.0, col[0]); r.g = (float)std::max(0.0, col[1]); r.b = (float)std::max(0.0, col[2]);
  }
}

// ---------------------------------------------------------------- O4 tile selection (A4)
// PAPER.md:L117-123.  T_sel = T^oc U T^um; on R / P frames every tile is selected.
void select_tiles(ora_ctx* c, int ftype) {
  const Cam& k = c->cam; const int W = k.W, H = k.H, TX = c->TX, TY = c->TY;
  c->tile_mask.assign((size_t)TX * TY, 0);
  const bool sr = (ftype == ORA_FRAME_S) && c->prm.enable_sr && !c->force_all;
  if (ftype == ORA_FRAME_S) {
    // T^um: any in-image pixel of the tile unmatched (L121, R22)
    for (int ty = 0; ty < TY; ++ty)
      for (int tx = 0; tx < TX; ++tx) {
        bool um = false;
        const int tg = TILE / c->ds;                       // tile edge in TGB grid pixels
        for (int y = ty * tg; y < std::min(c->Ht, ty * tg + tg) && !um; ++y)
          for (int x = tx * tg; x < std::min(c->Wt, tx * tg + tg); ++x)
            if (!c->matched[(size_t)y * c->Wt + x]) { um = true; break; }
        if (um) c->tile_mask[(size_t)ty * TX + tx] |= 2;
      }
    // T^oc: newly visible Gaussians whose max alpha over the tile's pixel box >= 1/255 (L119, R18)
    for (uint32_t g = 0; g < c->n; ++g) {
      const ora_record& r = c->rec[g];
      if ((r.flags & (ORA_VISIBLE | ORA_NEWLY_VISIBLE)) != (ORA_VISIBLE | ORA_NEWLY_VISIBLE)) continue;
      if (!(r.tau >= 0.0f)) continue;                       // o < 1/255: alpha never reaches 1/255
      for (int ty = r.y_lo; ty < r.y_hi; ++ty)
        for (int tx = r.x_lo; tx < r.x_hi; ++tx) {
          const float x0 = (float)(tx * TILE), x1 = (float)std::min(tx * TILE + TILE - 1, W - 1);
          const float y0 = (float)(ty * TILE), y1 = (float)std::min(ty * TILE + TILE - 1, H - 1);
          if (box_qmin(r.u, r.v, r.A, r.B, r.C, x0, x1, y0, y1) <= r.tau) c->tile_mask[(size_t)ty * TX + tx] |= 1;
        }
    }
  }
  ora_stats& st = c->st;
  st.n_tiles = (uint32_t)(TX * TY);
  for (size_t t = 0; t < c->tile_mask.size(); ++t) {
    uint8_t& m = c->tile_mask[t];
    if (m & 1) ++st.n_sel_oc;
    if (m & 2) ++st.n_sel_um;
    if (!sr || (m & 3)) { m |= 4; ++st.n_sel; }
  }
}

// ---------------------------------------------------------------- O5-O7 pairs, sort, ranges (A5-A7)
// PAPER.md:L61 "Gaussians that intersect with multiple tiles are duplicated ... sorts its intersected
// Gaussians by depth from front to back"; L123 only the Gaussians intersecting T_selected are sorted.
// "Intersect" is not defined by the paper.  exact_tiles = 0: every tile of the 3-sigma rect (vanilla 3DGS, R3).
// exact_tiles = 1 (default, R39): additionally max alpha over the tile's pixel-centre box >= 1/255, the test the
// paper itself uses for tile contributions (L119).  A pair dropped by it is skipped at every pixel of the tile
// (alpha < 1/255, R2) and can never stop a loop, so the image, the TGB and G_rendered do not depend on it
// (up to alpha within rounding of 1/255); only the lists get shorter.
void bin_and_sort(ora_ctx* c) {
  const int TX = c->TX, W = c->cam.W, H = c->cam.H;
  std::vector<std::pair<uint64_t, uint32_t>> pairs;
  for (uint32_t g = 0; g < c->n; ++g) {
    ora_record& r = c->rec[g];
    if (!(r.flags & ORA_VISIBLE)) continue;
    uint32_t cnt = 0;
    for (int ty = r.y_lo; ty < r.y_hi; ++ty)
      for (int tx = r.x_lo; tx < r.x_hi; ++tx) {
        const uint32_t t = (uint32_t)(ty * TX + tx);
        if (!(c->tile_mask[t] & 4)) continue;
        if (c->prm.exact_tiles) {   // R39: "intersect" = some point of the tile's pixel box has alpha >= 1/255
          const float x0 = (float)(tx * TILE), x1 = (float)std::min(tx * TILE + TILE - 1, W - 1);
          const float y0 = (float)(ty * TILE), y1 = (float)std::min(ty * TILE + TILE - 1, H - 1);
          if (!(r.tau >= 0.0f && box_qmin(r.u, r.v, r.A, r.B, r.C, x0, x1, y0, y1) <= r.tau)) continue;
        }
        pairs.emplace_back(((uint64_t)t << 32) | f2u(r.d), g);
        ++cnt;
      }
    r.tiles_touched = cnt;
  }
  std::stable_sort(pairs.begin(), pairs.end(),
                   [](const auto& a, const auto& b) { return a.first < b.first; });   // R28: ties by ascending g
  const size_t P = pairs.size();
  c->keys.resize(P); c->vals.resize(P);
  for (size_t i = 0; i < P; ++i) { c->keys[i] = pairs[i].first; c->vals[i] = pairs[i].second; }
  c->ranges.assign((size_t)c->TX * c->TY * 2, 0);
  for (size_t i = 0; i < P; ++i) {
    const uint32_t t = (uint32_t)(c->keys[i] >> 32);
    if (i == 0 || t != (uint32_t)(c->keys[i - 1] >> 32)) c->ranges[2 * t] = (uint32_t)i;
    if (i + 1 == P || t != (uint32_t)(c->keys[i + 1] >> 32)) c->ranges[2 * t + 1] = (uint32_t)(i + 1);
  }
  c->st.n_pairs = P;
}

// ---------------------------------------------------------------- O8 blend (A8) + O11 stitch (A9)
// alpha-blending PAPER.md:L61 (constants R2); Eq.1, Eq.2 L82 with w_i = alpha_i T_i (R1);
// G_rendered L103; Eq.4 L125 stitch with bilinear TAB (L101, R21) and repaired depth (L128, R31).
void blend_and_stitch(ora_ctx* c, int ftype) {
  const Cam& k = c->cam; const int W = k.W, H = k.H, TX = c->TX, TY = c->TY;
  c->image.assign((size_t)W * H * 3, 0.0f);
  c->depth.assign((size_t)W * H, ORA_DEPTH_INVALID);
  c->sigma.assign((size_t)W * H, 0.0f);
  c->borderline.assign((size_t)W * H, 0);
  c->rendered_now.assign(c->n, 0); c->rendered_sure.assign(c->n, 0); c->rendered_maybe.assign(c->n, 0);
  uint64_t L = 0;
  for (int ty = 0; ty < TY; ++ty)
    for (int tx = 0; tx < TX; ++tx) {
      const uint32_t t = (uint32_t)(ty * TX + tx);
      const bool sel = (c->tile_mask[t] & 4) != 0;
      for (int py = ty * TILE; py < std::min(H, ty * TILE + TILE); ++py)
        for (int px = tx * TILE; px < std::min(W, tx * TILE + TILE); ++px) {
          const size_t pix = (size_t)py * W + px;
          if (!sel) {   // Eq.4 second case: warped TAB
            double xs, ys;
            const size_t tq = (size_t)(py / c->ds) * c->Wt + (size_t)(px / c->ds);
            if (c->ds == 1) { xs = c->corr_xy[pix * 2]; ys = c->corr_xy[pix * 2 + 1]; }
            else {   // R43: the pixel's own ray with the repaired depth of its TGB block, backward Eq.3 (L121, L101)
              const float D = c->fill_depth[tq]; const float* Mi = c->Minv;
              const float rx = ((float)px - k.cx) / k.fx, ry = ((float)py - k.cy) / k.fy;
              const float Px = D * rx, Py = D * ry, Pz = D;
              const float X = ((Mi[0] * Px + Mi[1] * Py) + Mi[2] * Pz) + Mi[3];
              const float Y = ((Mi[4] * Px + Mi[5] * Py) + Mi[6] * Pz) + Mi[7];
              const float Z = ((Mi[8] * Px + Mi[9] * Py) + Mi[10] * Pz) + Mi[11];
              xs = (k.fx * X) / Z + k.cx; ys = (k.fy * Y) / Z + k.cy;
            }
            const double x0 = std::floor(xs), y0 = std::floor(ys);
            const double wx = xs - x0, wy = ys - y0;
            const int ix0 = std::min(std::max((int)x0, 0), W - 1), ix1 = std::min(std::max((int)x0 + 1, 0), W - 1);
            const int iy0 = std::min(std::max((int)y0, 0), H - 1), iy1 = std::min(std::max((int)y0 + 1, 0), H - 1);
            for (int ch = 0; ch < 3; ++ch) {
              const double v00 = c->prior_image[((size_t)iy0 * W + ix0) * 3 + ch], v10 = c->prior_image[((size_t)iy0 * W + ix1) * 3 + ch];
              const double v01 = c->prior_image[((size_t)iy1 * W + ix0) * 3 + ch], v11 = c->prior_image[((size_t)iy1 * W + ix1) * 3 + ch];
              c->image[pix * 3 + ch] = (float)((v00 * (1 - wx) + v10 * wx) * (1 - wy) + (v01 * (1 - wx) + v11 * wx) * wy);
            }
            c->depth[pix] = c->fill_depth[tq];
            c->sigma[pix] = c->warp_sigma[tq];
            continue;
          }
          double T = 1.0, C[3] = {0, 0, 0}, Sw = 0, Sd = 0, Sdd = 0;
          // The skip / stop tests DECIDE integers (membership in G_rendered), so they are taken in fp32
          // (R33): alpha_f = min(0.99f, float(o e^q)), T_f <- T_f (1 - alpha_f).  With the 3DGS constants the
          // case of two alpha-clamped Gaussians lands on T = 0.01^2 ~ 1e-4, i.e. ON the stop threshold, and
          // only a fixed precision makes that decision reproducible.  Values (colour, Eq.1-2) stay in double.
          // `stopped`: the real loop has terminated; what follows is a virtual continuation that only
          // marks which Gaussians an implementation with slightly different rounding MAY still blend.
          float Tf = 1.0f;
          double Terr = 0.0;
          bool stopped = false, sure_alive = true;
          double Tv = 1.0;
          for (uint32_t i = c->ranges[2 * t]; i < c->ranges[2 * t + 1]; ++i) {
            const uint32_t g = c->vals[i];
            const ora_record& r = c->rec[g];
            if (!stopped) ++L;
            const double dx = (double)r.u - px, dy = (double)r.v - py;
            // q = -1/2 delta^T Sigma'^-1 delta, Sigma' = [[ca, cb], [cb, cc]] inverted in double (the fp32 conic A, B, C is
            // only used for the tile-selection DECISION: evaluating the form with its rounded entries loses up to
            // 1e-7 x (sum of the magnitudes of the three terms), which matters for screen-filling anisotropic splats)
            const double ca = r.ca, cb = r.cb, cc = r.cc;
            const double q = -0.5 * (cc * dx * dx - 2.0 * cb * dx * dy + ca * dy * dy) / (ca * cc - cb * cb);
            if (q > 0.0) continue;                                   // R2 (cannot happen for a positive definite Sigma')
            // Conditioning of q with respect to fp32 storage of ANY parametrisation of Sigma'^-1 (the needle-like
            // splats of Gaussians next to the camera: centre a thousand pixels away, ridge one pixel wide):
            // with t = dx - (cb/cc) dy,  q = -1/2 (cc/det t^2 + dy^2/cc)  and  dq ~ eps (2 |A t| (|dx| + |k dy|) + |q|).
            const double kk = -cb / cc, tt = dx + kk * dy, AA = cc / (ca * cc - cb * cb);
            const double q_margin = Q_EPS * (2.0 * std::fabs(AA * tt) * (std::fabs(dx) + std::fabs(kk * dy)) + 2.0 * std::fabs(q));
            const double pm_alpha = PIX_MARGIN_ALPHA + q_margin, m_alpha = MARGIN_ALPHA + 4.0 * q_margin;
            const double a_raw = (double)r.o * std::exp(q);
            const double alpha = std::min(ALPHA_MAX, a_raw);         // L61, clamp R2 (value)
            const float alpha_f = std::fmin(ALPHA_MAX_F, (float)a_raw);   // (decision)
            if (stopped) {
              if (alpha < ALPHA_MIN * (1.0 - m_alpha)) continue;
              const double Tn = Tv * (1.0 - alpha);
              if (Tn < T_STOP * (1.0 - MARGIN_T)) break;
              c->rendered_maybe[g] = 1; Tv = Tn;
              continue;
            }
            if (alpha_f < ALPHA_MIN_F) {                             // skip alpha < 1/255 (R2)
              if (alpha >= ALPHA_MIN * (1.0 - m_alpha)) c->rendered_maybe[g] = 1;
              if (alpha >= ALPHA_MIN * (1.0 - pm_alpha)) c->borderline[pix] = 1;
              continue;
            }
            const float Tn_f = Tf * (1.0f - alpha_f);
            const double Tn = (double)Tn_f;
            if (Tn_f < T_STOP_F) {                                   // stop; this record is not blended (R2)
              if (Tn < T_STOP * (1.0 - MARGIN_T)) break;
              if (Tn >= T_STOP * (1.0 - std::max(PIX_MARGIN_T, 2.0 * (Terr + pm_alpha * alpha / (1.0 - alpha)))) && alpha_f < ALPHA_MAX_F) c->borderline[pix] = 1;
              c->rendered_maybe[g] = 1; stopped = true; Tv = Tn;
              continue;
            }
            const bool a_border = alpha < ALPHA_MIN * (1.0 + m_alpha);
            if (alpha < ALPHA_MIN * (1.0 + pm_alpha)) c->borderline[pix] = 1;
            if (alpha_f < ALPHA_MAX_F) Terr += pm_alpha * alpha / (1.0 - alpha);   // relative error bound of an fp32 T
            if (Tn < T_STOP * (1.0 + std::max(PIX_MARGIN_T, 2.0 * Terr)) && alpha_f < ALPHA_MAX_F) c->borderline[pix] = 1;
            if (Tn < T_STOP * (1.0 + MARGIN_T)) sure_alive = false;
            const double w = alpha * T;                              // w_i = alpha_i T_i (R1)
            C[0] += w * r.r; C[1] += w * r.g; C[2] += w * r.b;
            Sw += w; Sd += w * (double)r.d; Sdd += w * (double)r.d * (double)r.d;   // Eq.1-2 sums
            c->rendered_now[g] = 1; c->rendered_maybe[g] = 1;        // L103
            if (sure_alive && !a_border) c->rendered_sure[g] = 1;
            T *= 1.0 - alpha; Tf = Tn_f;
          }
          for (int ch = 0; ch < 3; ++ch) c->image[pix * 3 + ch] = (float)(C[ch] + T * c->prm.bg[ch]);   // R27
          if (Sw > 0.0) {
            const double D = Sd / Sw;
            c->depth[pix] = (float)D;
            c->sigma[pix] = (float)std::sqrt(std::max(0.0, Sdd / Sw - D * D));
          }
        }
    }
  c->st.n_interactions = L;
  uint32_t nr = 0; for (uint32_t g = 0; g < c->n; ++g) nr += c->rendered_now[g];
  c->st.n_rendered = nr;
  (void)ftype;
}

// R42, prior_policy = CHAINED (north_star: "the new frame ... becomes the next frame's TGB/TAB"): after an S frame
// its stitched image, depth and sigma (Eq.4, R31) replace TAB and TGB, W_t becomes this frame's pose, and
// G_rendered (L103) grows by the Gaussians blended in the selected tiles -- the un-rendered tiles show the same
// surfaces as before, so their contributors stay members.  F (L109) stays the reference frame's.
void commit_chained(ora_ctx* c) {
  c->prior_image = c->image; c->prior_depth = c->depth; c->prior_sigma = c->sigma;
  for (uint32_t g = 0; g < c->n; ++g) c->rendered[g] = c->rendered[g] | c->rendered_now[g];
  std::memcpy(c->prior_view, c->cam.V, sizeof(c->prior_view));
}

// after an R / P frame the outputs become the priors (O2, A10); R also stores F (L109, R8)
void commit_priors(ora_ctx* c, int ftype) {
  c->prior_image = c->image; c->prior_depth = c->depth; c->prior_sigma = c->sigma;
  c->rendered = c->rendered_now;
  std::memcpy(c->prior_view, c->cam.V, sizeof(c->prior_view));
  c->priors_valid = true;
  if (ftype == ORA_FRAME_R) {
    const float inf = std::numeric_limits<float>::infinity();
    float F[4] = {inf, inf, -inf, -inf};
    const int W = c->cam.W, H = c->cam.H;
    for (uint32_t g = 0; g < c->n; ++g)
      if (c->rendered_now[g]) {
        const ora_record& r = c->rec[g];
        const float nx = (2.0f * r.u + 1.0f) / (float)W - 1.0f, ny = (2.0f * r.v + 1.0f) / (float)H - 1.0f;
        F[0] = std::fmin(F[0], nx); F[1] = std::fmin(F[1], ny); F[2] = std::fmax(F[2], nx); F[3] = std::fmax(F[3], ny);
      }
    std::memcpy(c->F, F, sizeof(F)); c->F_valid = true;
  }
}

}  // namespace

extern "C" {

void ora_default_params(ora_params* p) {
  p->lambda1 = 3.0f; p->lambda2 = 0.0f; p->lambda_tdc = 50; p->lambda_sr = 5; p->eta = 0.40f;
  p->bg[0] = p->bg[1] = p->bg[2] = 0.0f; p->enable_afc = p->enable_toc = p->enable_sr = 1; p->exact_tiles = 1;
  p->prior_policy = 0; p->tgb_downscale = 1;
}

ora_ctx* ora_create(void) { ora_ctx* c = new ora_ctx(); ora_default_params(&c->prm); return c; }
void ora_destroy(ora_ctx* c) { delete c; }

int ora_load_gaussians(ora_ctx* c, uint32_t n, int deg, const float* means, const float* scales,
                       const float* quats, const float* opacity, const float* sh) {
  if (!c || deg < 0 || deg > 3 || (n && (!means || !scales || !quats || !opacity || !sh))) return ORA_E_INVALID_ARG;
  const int K = (deg + 1) * (deg + 1);
  if (!finite_all(means, 3 * (size_t)n) || !finite_all(scales, 3 * (size_t)n) || !finite_all(quats, 4 * (size_t)n) ||
      !finite_all(opacity, n) || !finite_all(sh, (size_t)n * K * 3)) return ORA_E_INVALID_ARG;
  c->n = n; c->deg = deg; c->K = K;
  c->means.assign(means, means + 3 * (size_t)n);
  c->opacity.assign(opacity, opacity + n);
  c->sh.assign(sh, sh + (size_t)n * K * 3);
  c->cov3d.resize(6 * (size_t)n); c->tau.resize(n);
  for (uint32_t g = 0; g < n; ++g) {
    // Sigma = R S S^T R^T ("covariance matrix"), fp32 fixed order, quaternion (w,x,y,z) normalised
    float w = quats[4 * g], x = quats[4 * g + 1], y = quats[4 * g + 2], z = quats[4 * g + 3];
    const float nrm = std::sqrt(((w * w + x * x) + y * y) + z * z);
    w /= nrm; x /= nrm; y /= nrm; z /= nrm;
    const float R[9] = {1.0f - 2.0f * (y * y + z * z), 2.0f * (x * y - w * z), 2.0f * (x * z + w * y),
                        2.0f * (x * y + w * z), 1.0f - 2.0f * (x * x + z * z), 2.0f * (y * z - w * x),
                        2.0f * (x * z - w * y), 2.0f * (y * z + w * x), 1.0f - 2.0f * (x * x + y * y)};
    float Mx[9];
    for (int i = 0; i < 3; ++i) for (int kx = 0; kx < 3; ++kx) Mx[i * 3 + kx] = R[i * 3 + kx] * scales[3 * g + kx];
    auto S = [&](int i, int j) { return (Mx[i * 3] * Mx[j * 3] + Mx[i * 3 + 1] * Mx[j * 3 + 1]) + Mx[i * 3 + 2] * Mx[j * 3 + 2]; };
    float* o = &c->cov3d[6 * (size_t)g];
    o[0] = S(0, 0); o[1] = S(0, 1); o[2] = S(0, 2); o[3] = S(1, 1); o[4] = S(1, 2); o[5] = S(2, 2);
    // tau = 2 ln(255 o): alpha = o exp(-q/2) >= 1/255  <=>  q <= tau  (double log, rounded once)
    c->tau[g] = (float)(2.0 * std::log(255.0 * (double)opacity[g]));
  }
  c->priors_valid = false; c->F_valid = false; c->sched = ora_sched{0, 0, 0, 0};
  return ORA_OK;
}

int ora_set_camera(ora_ctx* c, const float view[16], float fx, float fy, float cx, float cy, int W, int H,
                   float znear, float zfar) {
  if (!c || !view || W <= 0 || H <= 0 || !(fx > 0) || !(fy > 0) || !(znear > 0) || !finite_all(view, 16)) return ORA_E_INVALID_ARG;
  const float intr[6] = {fx, fy, cx, cy, znear, zfar};
  if (!finite_all(intr, 6)) return ORA_E_INVALID_ARG;
  Cam& k = c->cam;
  if (k.set && (k.W != W || k.H != H || k.fx != fx || k.fy != fy || k.cx != cx || k.cy != cy)) { c->priors_valid = false; c->F_valid = false; c->sched.valid = 0; }
  std::memcpy(k.V, view, sizeof(k.V)); k.fx = fx; k.fy = fy; k.cx = cx; k.cy = cy; k.W = W; k.H = H; k.znear = znear; k.zfar = zfar; k.set = true;
  c->TX = (W + TILE - 1) / TILE; c->TY = (H + TILE - 1) / TILE;
  return ORA_OK;
}

int ora_set_params(ora_ctx* c, const ora_params* p) {
  if (!c || !p || p->lambda_tdc < 1 || p->lambda_sr < 1) return ORA_E_INVALID_ARG;
  c->prm = *p; return ORA_OK;
}

int ora_reset_priors(ora_ctx* c) { c->priors_valid = false; c->F_valid = false; c->sched = ora_sched{0, 0, 0, 0}; return ORA_OK; }
int ora_force_all_tiles(ora_ctx* c, int on) { c->force_all = on; return ORA_OK; }

int ora_schedule_next(ora_sched* s, int lambda_tdc, int lambda_sr) {
  // PAPER.md:L65-67, L107, L142 (R9): R every lambda_TDC frames, P every lambda_SR frames or when forced (L128)
  if (!s->valid || s->since_R >= lambda_tdc) return ORA_FRAME_R;
  if (s->since_ref >= lambda_sr || s->force_P) return ORA_FRAME_P;
  return ORA_FRAME_S;
}

void ora_schedule_feedback(ora_sched* s, int ftype, uint32_t n_sel, uint32_t n_tiles, float eta) {
  if (ftype == ORA_FRAME_R) { s->since_R = 0; s->since_ref = 0; s->valid = 1; s->force_P = 0; }
  else if (ftype == ORA_FRAME_P) { s->since_ref = 0; s->force_P = 0; }
  else s->force_P = ((float)n_sel > eta * (float)n_tiles) ? 1 : 0;      // L128 "exceeds eta(%)" (R23: strict)
  ++s->since_R; ++s->since_ref;
}

int ora_render(ora_ctx* c, int mode) {
  if (!c) return ORA_E_INVALID_ARG;
  if (!c->n) return ORA_E_NO_SCENE;
  if (!c->cam.set) return ORA_E_NO_CAMERA;
  int ftype;
  if (mode == ORA_AUTO) ftype = ora_schedule_next(&c->sched, c->prm.lambda_tdc, c->prm.lambda_sr);
  else if (mode == ORA_FULL) ftype = ORA_FRAME_R;
  else if (mode == ORA_PSEUDO_REF) ftype = ORA_FRAME_P;
  else if (mode == ORA_TEMPORAL) ftype = ORA_FRAME_S;
  else return ORA_E_INVALID_ARG;
  if (ftype != ORA_FRAME_R && !c->priors_valid) return ORA_E_NO_PRIORS;
  c->st = ora_stats{}; c->st.frame_type = ftype; c->st.n_total = c->n;
  const double t0 = now_ms();
  if (ftype == ORA_FRAME_S) {
    relative_pose(c->prior_view, c->cam.V, c->M);       // reference -> current (forward, Eq.3)
    relative_pose(c->cam.V, c->prior_view, c->Minv);    // current -> reference (backward, L121)
    tgb_grid(c);
    forward_warp(c);
    fill_and_correspond(c);
  }
  const double t1 = now_ms();
  preprocess(c, ftype);
  select_tiles(c, ftype);
  const double t2 = now_ms();
  bin_and_sort(c);
  const double t3 = now_ms();
  blend_and_stitch(c, ftype);
  if (ftype != ORA_FRAME_S) commit_priors(c, ftype);
  else if (c->prm.prior_policy == 1) commit_chained(c);
  const double t4 = now_ms();
  c->st.ms_temporal = t1 - t0; c->st.ms_preprocess = t2 - t1; c->st.ms_sort = t3 - t2; c->st.ms_blend = t4 - t3; c->st.ms_total = t4 - t0;
  // R41: the eta rule is part of selective rendering (section III-E); with SR switched off no tile is
  // "selected" by the method, so an S frame never forces a pseudo-reference frame.
  ora_schedule_feedback(&c->sched, ftype, c->prm.enable_sr ? c->st.n_sel : 0u, c->st.n_tiles, c->prm.eta);
  return ftype;
}

int ora_read_image(ora_ctx* c, float* rgb) {
  if (!c || !rgb || c->image.empty()) return ORA_E_INVALID_ARG;
  std::memcpy(rgb, c->image.data(), c->image.size() * 4); return ORA_OK;
}
int ora_read_depth(ora_ctx* c, float* depth, float* sigma) {
  if (!c || !depth || c->depth.empty()) return ORA_E_INVALID_ARG;
  std::memcpy(depth, c->depth.data(), c->depth.size() * 4);
  if (sigma) std::memcpy(sigma, c->sigma.data(), c->sigma.size() * 4);
  return ORA_OK;
}
int ora_read_tile_mask(ora_ctx* c, uint8_t* sel) {
  if (!c || !sel || c->tile_mask.empty()) return ORA_E_INVALID_ARG;
  for (size_t i = 0; i < c->tile_mask.size(); ++i) sel[i] = c->tile_mask[i];
  return ORA_OK;
}
int ora_get_stats(ora_ctx* c, ora_stats* s) { if (!c || !s) return ORA_E_INVALID_ARG; *s = c->st; return ORA_OK; }

#define ORA_GET(nm, vec)                                                                 \
  if (name == nm) {                                                                      \
    const size_t have = (vec).size() * sizeof((vec)[0]);                                 \
    if (dst) std::memcpy(dst, (vec).data(), std::min(have, bytes));                      \
    return (long long)have;                                                              \
  }

long long ora_get(ora_ctx* c, const char* nm, void* dst, size_t bytes) {
  if (!c || !nm) return ORA_E_INVALID_ARG;
  const std::string name(nm);
  ORA_GET("records", c->rec) ORA_GET("keys", c->keys) ORA_GET("vals", c->vals) ORA_GET("ranges", c->ranges)
  ORA_GET("warp_depth", c->warp_depth) ORA_GET("warp_sigma", c->warp_sigma) ORA_GET("fill_depth", c->fill_depth)
  ORA_GET("corr_xy", c->corr_xy) ORA_GET("matched", c->matched) ORA_GET("rendered", c->rendered) ORA_GET("rendered_now", c->rendered_now)
  ORA_GET("rendered_sure", c->rendered_sure) ORA_GET("rendered_maybe", c->rendered_maybe) ORA_GET("borderline", c->borderline)
  ORA_GET("prior_depth", c->prior_depth) ORA_GET("prior_sigma", c->prior_sigma) ORA_GET("prior_image", c->prior_image)
  ORA_GET("cov3d", c->cov3d) ORA_GET("tau", c->tau)
  auto raw = [&](const void* p, size_t have) { if (dst) std::memcpy(dst, p, std::min(have, bytes)); return (long long)have; };
  if (name == "F") return raw(c->F, sizeof(c->F));
  if (name == "M") return raw(c->M, sizeof(c->M));
  if (name == "Minv") return raw(c->Minv, sizeof(c->Minv));
  if (name == "prior_view") return raw(c->prior_view, sizeof(c->prior_view));
  return ORA_E_INVALID_ARG;
}

int ora_put(ora_ctx* c, const char* nm, const void* src, size_t bytes) {
  if (!c || !nm || !src || !c->cam.set) return ORA_E_INVALID_ARG;
  const std::string name(nm);
  const size_t px = (size_t)c->cam.W * c->cam.H;
  auto putf = [&](std::vector<float>& v, size_t cnt) { if (bytes != cnt * 4) return (int)ORA_E_INVALID_ARG; v.resize(cnt); std::memcpy(v.data(), src, bytes); return (int)ORA_OK; };
  if (name == "prior_depth") return putf(c->prior_depth, px);
  if (name == "prior_sigma") return putf(c->prior_sigma, px);
  if (name == "prior_image") return putf(c->prior_image, px * 3);
  if (name == "rendered") { if (bytes != c->n) return ORA_E_INVALID_ARG; c->rendered.assign((const uint8_t*)src, (const uint8_t*)src + bytes); return ORA_OK; }
  if (name == "F") { if (bytes != 16) return ORA_E_INVALID_ARG; std::memcpy(c->F, src, 16); c->F_valid = true; return ORA_OK; }
  if (name == "prior_view") {
    if (bytes != 64) return ORA_E_INVALID_ARG;
    std::memcpy(c->prior_view, src, 64);
    if (c->rendered.size() != c->n) c->rendered.assign(c->n, 0);
    c->priors_valid = c->prior_depth.size() == px && c->prior_sigma.size() == px && c->prior_image.size() == px * 3;
    if (c->priors_valid) c->sched.valid = 1;
    return c->priors_valid ? ORA_OK : ORA_E_INVALID_ARG;
  }
  return ORA_E_INVALID_ARG;
}

int ora_stage(ora_ctx* c, const char* stage) {
  if (!c || !stage || !c->priors_valid) return ORA_E_NO_PRIORS;
  const std::string s(stage);
  if (s == "warp") {
    relative_pose(c->prior_view, c->cam.V, c->M);
    relative_pose(c->cam.V, c->prior_view, c->Minv);
    tgb_grid(c);
    forward_warp(c); return ORA_OK;
  }
  if (s == "fill") { fill_and_correspond(c); return ORA_OK; }
  return ORA_E_INVALID_ARG;
}

void ora_sh_basis(int degree, const double dir[3], double* Y) { sh_basis(degree, dir, Y); }
float ora_box_qmin(float u, float v, float A, float B, float C, float x0, float x1, float y0, float y1) {
  return box_qmin(u, v, A, B, C, x0, x1, y0, y1);
}

}  // extern "C"
