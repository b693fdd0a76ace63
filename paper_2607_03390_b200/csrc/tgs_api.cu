// tgs_api.cu -- C-ABI of libtgs.so (include/tgs.h): context, host-side frame scheduler A0, buffer
// management, the per-frame launch sequence A1-A10 and the read-back / debug calls.
// No CPU fallback: every step of the path is a kernel launch; the host only computes the relative pose
// (12 floats) and the frame type.
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <exception>
#include <string>
#include <vector>

#include "tgs_internal.cuh"

#define CK(call)                                                                                   \
  do {                                                                                             \
    cudaError_t e_ = (call);                                                                       \
    if (e_ != cudaSuccess) {                                                                       \
      snprintf(c->err, sizeof(c->err), "%s:%d %s: %s", __FILE__, __LINE__, #call, cudaGetErrorString(e_)); \
      return TGS_E_CUDA;                                                                           \
    }                                                                                              \
  } while (0)

unsigned long long g_tgs_launches = 0;

struct Sched { int since_R = 0, since_ref = 0, force_P = 0; };

struct tgs_ctx {
  int device = 0;
  int num_sms = 148;
  cudaStream_t stream = nullptr;
  char err[512] = {0};
  // scene
  uint32_t n = 0; int deg = 0, K = 1;
  // camera
  bool cam_set = false;
  float view[16]; float fx, fy, cx, cy, znear, zfar; int W = 0, H = 0, TX = 0, TY = 0;
  tgs_params prm;
  // priors
  bool priors_valid = false, F_valid = false;
  float prior_view[16];
  int prior_idx = 0;           // image/depth/sigma[prior_idx] hold TAB / TGB
  int cur_idx = 0;             // buffers of the last rendered frame
  int sorted_idx = 0;          // keys/vals[sorted_idx] hold the sorted pairs of the last frame
  bool have_frame = false;
  bool put_depth = false, put_sigma = false, put_image = false;
  Sched sched;
  int force_all = 0;
  // capacities
  uint32_t max_pairs = 0; uint32_t sort_tiles_cap = 0; uint32_t dsort_tiles_cap = 0; uint32_t bin_chunks_cap = 0; int sort_passes_cap = 0; size_t px_cap = 0; int tiles_cap = 0;
  uint32_t epoch = 0;          // frame number, tag of the look-back descriptors
  uint64_t* keys64 = nullptr;  // test-only scratch of tgs_debug_get("keys")
  uint2* ranges_dec = nullptr; // test-only scratch of tgs_debug_get("ranges")
  float4* dbg_rec = nullptr;   // test-only scratch of tgs_debug_get("rec_uvdo" / "rec_conic")
  uint64_t device_bytes = 0;
  DevBuffers b;
  std::vector<void*> allocs_scene, allocs_frame, allocs_pairs;
  struct Guard { unsigned char* base; size_t bytes, body; };
  std::vector<Guard> guards;           // red zones (test-only)
  bool redzones = false;
  // stats
  Counters* h_counters = nullptr;      // pinned: the block of the last rendered frame (= h_cnt2[parity])
  Counters* h_cnt2[2] = {nullptr, nullptr};   // pinned, by frame parity: frame N - 2's statistics are complete and unchanged when frame N is set up
  uint32_t* h_sel = nullptr;           // pinned: n_sel of the last S frame (for the eta rule)
  cudaEvent_t ev_sel = nullptr, ev_done = nullptr;
  // the device counters are double-buffered by frame parity: their (latency-bound) copy to the host runs on the third
  // stream while the next frame, which uses the other block, has already started
  Counters* counters2[2] = {nullptr, nullptr};
  cudaEvent_t ev_cnt[2] = {nullptr, nullptr}, ev_post = nullptr, ev_post2 = nullptr;
  bool post2_pending = false;
  uint32_t* F_base = nullptr;          // F_key of the last R frame = F_base + 4 * F_idx; an R frame builds the other one
  int F_idx = 0;
  bool cnt_pending[2] = {false, false};
  cudaStream_t copy = nullptr;          // read-back stream of tgs_read_image_async
  cudaEvent_t ev_copy[3] = {nullptr, nullptr, nullptr};   // last asynchronous read of image[i] has finished
  bool copy_pending[3] = {false, false, false};
  cudaStream_t side = nullptr;          // second stream: work that is off the critical path of a frame (A2, A4)
  cudaStream_t side2 = nullptr;         // third stream: SH colours beside the depth sort
  cudaEvent_t ev_fork = nullptr, ev_join = nullptr, ev_fork2 = nullptr, ev_join2 = nullptr, ev_fork3 = nullptr;
  bool sel_pending = false;
  // pair-buffer overflow of the previous frame: k_bin stores the flag into pinned memory (zero-copy) and ev_bin marks the
  // end of that kernel; the next tgs_render waits for it (mid-frame: tile sort and blend are still running) before it
  // decides the frame type, so that priors committed by an overflowed frame are never used
  uint32_t* h_ovf = nullptr;            // pinned, [2] by frame parity
  cudaEvent_t ev_bin = nullptr;
  bool bin_pending = false; int bin_slot = 0;
  uint32_t nv_hint = 0;                 // visible Gaussians of a recent frame (selects the depth-sort instance)
  uint32_t nv_hint_cls[2] = {0, 0};     // the same per frame class (R / P, S): the one-launch depth sort is for lists of one tile per SM
  int last_ftype = -1; uint32_t last_n_tiles = 0;
  bool timing = false;
  bool count_interactions = false;
  // stage timing: an event before every launch group, tagged with the stage (0..7) the time up to the next event goes to
  static constexpr int MAX_EV = 48;
  cudaEvent_t ev_stage[MAX_EV];
  int ev_tag[MAX_EV]; int n_ev = 0;
  int last_n_slabs = 1;
  int dsort_mode = -1;                  // -1 automatic (short visible lists), 0 onesweep launches, 1 one-launch depth sort
  int blend_half_mode = -1;             // -1 automatic (small splats: few tests per visible Gaussian), 0 off, 1 on
  bool half_hint = false;
  // automatic choice of the number of slabs (depth_slabs = 0), per frame class (0: R / P, 1: S): pairs per test measured on
  // recent one-piece and two-piece frames; slabs are used where they drop more than half of the pairs
  struct SlabCtl {
    float p1 = -1.0f, p2 = -1.0f; int since_probe = 0; uint32_t tests = 0, tests_probe = 0; bool asked1 = false, asked2 = false, two = false;
    uint32_t split = 256, split_floor = 64; int hold = 0;      // first piece in 1/1024 of the test space (automatic mode), see tgs_render
    bool empty2 = false; int probe_k = 0;                      // the second piece of the latest two-piece frame was (nearly) empty; probes cycle through 256 / 384 / 512
  } slab_ctl[2];
  uint32_t cur_split = 0;               // automatic split of the frame being enqueued (0: not automatic)
  uint32_t hist_split[2] = {0, 0};      // split of the frame that last used each counter block (0: not the automatic one)
  int hist_cls[2] = {0, 0}, hist_slabs[2] = {1, 1};   // class and number of slabs of the frame that last used each counter block
  FrameConst fc;
};

namespace {

// Every device buffer of a context comes from here.  With red zones on (tgs_debug_run_stage("redzones_on") before the
// scene is loaded; test-only) each buffer is framed by two 256-byte guards filled with a pattern, and
// tgs_debug_run_stage("check_redzones") verifies that no kernel has written outside its buffers -- the stand-in for
// compute-sanitizer's memcheck, which is closed on this pool (profiles/r2_sanitizers.md).
constexpr size_t REDZONE = 256;
constexpr unsigned char REDZONE_BYTE = 0xA5;
template <typename T>
int dev_alloc(tgs_ctx* c, T** p, size_t count, std::vector<void*>& list, bool zero = false) {
  *p = nullptr;
  if (!count) count = 1;
  const size_t bytes = count * sizeof(T), pad = c->redzones ? REDZONE : 0;
  const size_t body = (bytes + 255) / 256 * 256;                        // the rear guard starts at the next 256-byte boundary
  unsigned char* base = nullptr;
  CK(cudaMalloc((void**)&base, pad ? body + 2 * pad : bytes));
  if (pad) {
    CK(cudaMemsetAsync(base, REDZONE_BYTE, pad, c->stream));
    CK(cudaMemsetAsync(base + pad + bytes, REDZONE_BYTE, body - bytes + pad, c->stream));
    c->guards.push_back({base, bytes, body});
  }
  *p = reinterpret_cast<T*>(base + pad);
  if (zero) CK(cudaMemsetAsync(*p, 0, bytes, c->stream));   // look-back descriptors: epoch 0 = never valid
  list.push_back(base);
  c->device_bytes += bytes;
  return TGS_OK;
}

void free_list(tgs_ctx* c, std::vector<void*>& list) {
  for (void* p : list) {
    cudaFree(p);
    for (size_t i = 0; i < c->guards.size(); ++i) if (c->guards[i].base == p) { c->guards.erase(c->guards.begin() + (long)i); break; }
  }
  list.clear();
}

// red zones intact?  0 = yes; otherwise the number of damaged guards (the first one is described in c->err)
int check_redzones(tgs_ctx* c) {
  cudaDeviceSynchronize();
  int bad = 0;
  std::vector<unsigned char> h;
  for (const auto& g : c->guards) {
    const size_t rear = g.body - g.bytes + REDZONE;
    h.resize(REDZONE + rear);
    if (cudaMemcpy(h.data(), g.base, REDZONE, cudaMemcpyDeviceToHost) != cudaSuccess ||
        cudaMemcpy(h.data() + REDZONE, g.base + REDZONE + g.bytes, rear, cudaMemcpyDeviceToHost) != cudaSuccess) return -1;
    for (size_t i = 0; i < h.size(); ++i)
      if (h[i] != REDZONE_BYTE) {
        if (!bad) snprintf(c->err, sizeof(c->err), "red zone of a %zu-byte buffer damaged %s it (offset %zu)", g.bytes, i < REDZONE ? "before" : "behind",
                           i < REDZONE ? REDZONE - i : i - REDZONE);
        ++bad;
        break;
      }
  }
  return bad;
}

bool finite_all(const float* p, size_t n) {
  for (size_t i = 0; i < n; ++i) if (!std::isfinite(p[i])) return false;
  return true;
}

// rigid relative pose M = W_b W_a^{-1}, double arithmetic, rounded once to float (Eq.3)
void relative_pose(const float* Wa, const float* Wb, float* M) {
  double Ra[9], ta[3], Rb[9], tb[3];
  for (int i = 0; i < 3; ++i) {
    for (int j = 0; j < 3; ++j) { Ra[i * 3 + j] = Wa[i * 4 + j]; Rb[i * 3 + j] = Wb[i * 4 + j]; }
    ta[i] = Wa[i * 4 + 3]; tb[i] = Wb[i * 4 + 3];
  }
  for (int i = 0; i < 3; ++i) {
    double row[3];
    for (int j = 0; j < 3; ++j) row[j] = (Rb[i * 3] * Ra[j * 3] + Rb[i * 3 + 1] * Ra[j * 3 + 1]) + Rb[i * 3 + 2] * Ra[j * 3 + 2];
    const double mt = tb[i] - ((row[0] * ta[0] + row[1] * ta[1]) + row[2] * ta[2]);
    M[i * 4] = (float)row[0]; M[i * 4 + 1] = (float)row[1]; M[i * 4 + 2] = (float)row[2]; M[i * 4 + 3] = (float)mt;
  }
}

int alloc_frame_buffers(tgs_ctx* c) {
  const size_t px = (size_t)c->W * c->H;
  const int T = c->TX * c->TY;
  if (px <= c->px_cap && T <= c->tiles_cap) return TGS_OK;
  cudaStreamSynchronize(c->stream);
  free_list(c, c->allocs_frame);
  c->ranges_dec = nullptr;
  DevBuffers& b = c->b;
  for (int i = 0; i < 3; ++i) {
    if (int r = dev_alloc(c, &b.image[i], px * 3, c->allocs_frame)) return r;
    if (int r = dev_alloc(c, &b.depth[i], px, c->allocs_frame)) return r;
    if (int r = dev_alloc(c, &b.sigma[i], px, c->allocs_frame)) return r;
  }
  if (int r = dev_alloc(c, &b.warp_tgb, px, c->allocs_frame)) return r;
  if (int r = dev_alloc(c, &b.fill_depth, px, c->allocs_frame)) return r;
  if (int r = dev_alloc(c, &b.tile_flags, (size_t)T, c->allocs_frame)) return r;
  if (int r = dev_alloc(c, &b.tile_mask, (size_t)T, c->allocs_frame)) return r;
  if (int r = dev_alloc(c, &b.sel_bits, (size_t)(T + 31) / 32 + 1, c->allocs_frame)) return r;
  if (int r = dev_alloc(c, &b.live_bits, (size_t)(T + 31) / 32 + 1, c->allocs_frame)) return r;
  b.live_sat = nullptr; b.pix_state = nullptr;      // slab buffers: allocated by the first frame that runs in several pieces
  if (int r = dev_alloc(c, &b.tile_order, (size_t)T, c->allocs_frame)) return r;
  if (int r = dev_alloc(c, &b.ranges, (size_t)T, c->allocs_frame)) return r;
  c->px_cap = px; c->tiles_cap = T;
  return TGS_OK;
}

int alloc_pair_buffers(tgs_ctx* c, uint32_t max_pairs, int passes) {
  if (max_pairs <= c->max_pairs && passes <= c->sort_passes_cap) return TGS_OK;
  if (max_pairs < c->max_pairs) max_pairs = c->max_pairs;
  if (passes < c->sort_passes_cap) passes = c->sort_passes_cap;
  c->max_pairs = 0;
  cudaStreamSynchronize(c->stream);
  free_list(c, c->allocs_pairs);
  c->keys64 = nullptr;
  DevBuffers& b = c->b;
  for (int i = 0; i < 2; ++i) {
    if (int r = dev_alloc(c, &b.keys[i], (size_t)max_pairs, c->allocs_pairs)) return r;
    if (int r = dev_alloc(c, &b.vals[i], (size_t)max_pairs, c->allocs_pairs)) return r;
  }
  const uint32_t tiles = (max_pairs + sort_tile_items() - 1) / sort_tile_items() + 1;
  if (int r = dev_alloc(c, &b.sort_desc, (size_t)passes * tiles * 256, c->allocs_pairs, true)) return r;
  c->sort_tiles_cap = tiles; c->sort_passes_cap = passes;
  // flat (Gaussian, tile) test space of k_bin: up to 4 tests per pair of capacity (and below 2^32)
  unsigned long long max_tests = (unsigned long long)max_pairs * 4ull;
  if (max_tests > 0xfff00000ull) max_tests = 0xfff00000ull;
  c->bin_chunks_cap = (uint32_t)(max_tests / bin_chunk_items()) + 2;
  if (int r = dev_alloc(c, &b.chunk_first, (size_t)c->bin_chunks_cap, c->allocs_pairs)) return r;
  if (int r = dev_alloc(c, &b.bin_desc, (size_t)c->bin_chunks_cap, c->allocs_pairs, true)) return r;
  c->max_pairs = max_pairs;
  return TGS_OK;
}

int tile_key_bits(int n_tiles) {
  int bits = 1;
  while ((1ll << bits) < n_tiles) ++bits;
  return bits;
}

uint32_t auto_max_pairs(const tgs_ctx* c) {
  // heuristic capacity: 24 pairs per Gaussian, at least 4 M, at most 2^30 - 1 (look-back value field)
  unsigned long long want = (unsigned long long)c->n * 24ull;
  if (want < (4ull << 20)) want = 4ull << 20;
  if (want > (1ull << 30) - 1) want = (1ull << 30) - 1;
  return (uint32_t)want;
}

void invalidate_priors(tgs_ctx* c) {
  c->priors_valid = false; c->F_valid = false; c->sched = Sched();
  c->put_depth = c->put_sigma = c->put_image = false;
}

int copy_out(tgs_ctx* c, void* dst, const void* src, size_t bytes, int mem) {
  if (mem == TGS_DEVICE) { CK(cudaMemcpyAsync(dst, src, bytes, cudaMemcpyDeviceToDevice, c->stream)); return TGS_OK; }
  CK(cudaMemcpyAsync(dst, src, bytes, cudaMemcpyDeviceToHost, c->stream));
  CK(cudaStreamSynchronize(c->stream));
  return TGS_OK;
}

}  // namespace

extern "C" {

const char* tgs_strerror(int code) {
  switch (code) {
    case TGS_OK: return "ok";
    case TGS_E_INVALID_ARG: return "invalid argument";
    case TGS_E_NO_SCENE: return "no Gaussians loaded";
    case TGS_E_NO_CAMERA: return "no camera set";
    case TGS_E_NO_PRIORS: return "no valid temporal priors (render a reference frame first)";
    case TGS_E_CAPACITY: return "pair buffer capacity exceeded";
    case TGS_E_CUDA: return "CUDA error";
    default: return "unknown error";
  }
}

const char* tgs_last_error(tgs_ctx* c) { return c ? c->err : "null context"; }

void tgs_default_params(tgs_params* p) {
  if (!p) return;
  p->lambda1 = 3.0f; p->lambda2 = 0.0f; p->lambda_tdc = 50; p->lambda_sr = 5; p->eta = 0.40f;
  p->bg[0] = p->bg[1] = p->bg[2] = 0.0f;
  p->enable_afc = p->enable_toc = p->enable_sr = 1;
  p->max_pairs = 0;
  p->exact_tiles = 1;
  p->prior_policy = TGS_PRIORS_ANCHORED;
  p->tgb_downscale = 1;
  p->depth_slabs = 0;
  p->slab_split[0] = p->slab_split[1] = p->slab_split[2] = 0;
}

static void destroy_ctx(tgs_ctx* c) {   // tolerates a partially constructed context (tgs_create's failure paths)
  if (!c) return;
  cudaSetDevice(c->device);
  cudaStreamSynchronize(c->stream);
  for (cudaStream_t* st : {&c->side, &c->side2, &c->copy}) if (*st) { cudaStreamSynchronize(*st); cudaStreamDestroy(*st); *st = nullptr; }
  free_list(c, c->allocs_scene); free_list(c, c->allocs_frame); free_list(c, c->allocs_pairs);
  for (auto& p : c->counters2) if (p) cudaFree(p);
  if (c->F_base) cudaFree(c->F_base);
  if (c->b.sort_hist) cudaFree(c->b.sort_hist);
  for (auto& p : c->h_cnt2) if (p) cudaFreeHost(p);
  if (c->h_sel) cudaFreeHost(c->h_sel);
  if (c->h_ovf) cudaFreeHost(c->h_ovf);
  for (auto& e : c->ev_cnt) if (e) cudaEventDestroy(e);
  for (auto& e : c->ev_copy) if (e) cudaEventDestroy(e);
  for (auto& e : c->ev_stage) if (e) cudaEventDestroy(e);
  for (cudaEvent_t* e : {&c->ev_post, &c->ev_post2, &c->ev_sel, &c->ev_done, &c->ev_bin, &c->ev_fork, &c->ev_join, &c->ev_fork2, &c->ev_join2, &c->ev_fork3})
    if (*e) cudaEventDestroy(*e);
  delete c;
}

static int create_impl(tgs_ctx** out, int device, void* stream) {
  int count = 0;
  if (cudaGetDeviceCount(&count) != cudaSuccess || device < 0 || device >= count) return TGS_E_CUDA;
  tgs_ctx* c = new tgs_ctx();
  c->device = device; c->stream = (cudaStream_t)stream;
  for (auto& e : c->ev_stage) e = nullptr;
  tgs_default_params(&c->prm);
  bool ok = cudaSetDevice(device) == cudaSuccess;
  cudaDeviceProp prop;
  ok = ok && cudaGetDeviceProperties(&prop, device) == cudaSuccess;
  if (ok) c->num_sms = prop.multiProcessorCount;
  for (auto& p : c->h_cnt2) ok = ok && cudaMallocHost((void**)&p, sizeof(Counters)) == cudaSuccess;
  ok = ok && cudaMallocHost((void**)&c->h_sel, 2 * sizeof(uint32_t)) == cudaSuccess;
  ok = ok && cudaMallocHost((void**)&c->h_ovf, 2 * sizeof(uint32_t)) == cudaSuccess;
  if (ok) { for (auto& p : c->h_cnt2) memset(p, 0, sizeof(Counters)); c->h_counters = c->h_cnt2[0]; c->h_ovf[0] = c->h_ovf[1] = 0; c->h_sel[0] = c->h_sel[1] = 0; }
  for (auto& p : c->counters2) ok = ok && cudaMalloc((void**)&p, sizeof(Counters)) == cudaSuccess;
  ok = ok && cudaMalloc((void**)&c->F_base, 8 * sizeof(uint32_t)) == cudaSuccess;   // two F's, by frame parity
  ok = ok && cudaMalloc((void**)&c->b.sort_hist, (1 + TGS_MAX_SLABS) * 4 * 256 * sizeof(uint32_t)) == cudaSuccess;
  for (auto& e : c->ev_cnt) ok = ok && cudaEventCreateWithFlags(&e, cudaEventDisableTiming) == cudaSuccess;
  for (auto& e : c->ev_copy) ok = ok && cudaEventCreateWithFlags(&e, cudaEventDisableTiming) == cudaSuccess;
  for (cudaEvent_t* e : {&c->ev_post, &c->ev_post2, &c->ev_sel, &c->ev_done, &c->ev_bin, &c->ev_fork, &c->ev_join, &c->ev_fork2, &c->ev_join2, &c->ev_fork3})
    ok = ok && cudaEventCreateWithFlags(e, cudaEventDisableTiming) == cudaSuccess;
  for (cudaStream_t* st : {&c->side, &c->side2, &c->copy}) ok = ok && cudaStreamCreateWithFlags(st, cudaStreamNonBlocking) == cudaSuccess;
  for (auto& e : c->ev_stage) ok = ok && cudaEventCreate(&e) == cudaSuccess;
  if (!ok) { cudaGetLastError(); destroy_ctx(c); return TGS_E_CUDA; }
  c->b.counters = c->counters2[0];
  c->b.F_key = c->F_base;
  sort_prepare_device();
  *out = c;
  return TGS_OK;
}

// No exception crosses the C-ABI (tgs.h): the host-side containers (std::vector, std::string) may throw std::bad_alloc.
#define TGS_NOEXCEPT_BODY(ctx, expr)                                                                        \
  try { return (expr); }                                                                                     \
  catch (const std::exception& e_) { if (ctx) snprintf((ctx)->err, sizeof((ctx)->err), "host exception: %s", e_.what()); return TGS_E_INVALID_ARG; } \
  catch (...) { return TGS_E_INVALID_ARG; }

int tgs_create(tgs_ctx** out, int device, void* stream) {
  if (!out) return TGS_E_INVALID_ARG;
  *out = nullptr;
  TGS_NOEXCEPT_BODY((tgs_ctx*)nullptr, create_impl(out, device, stream))
}

void tgs_destroy(tgs_ctx* c) { destroy_ctx(c); }

static int load_gaussians_impl(tgs_ctx* c, uint32_t n, int deg, const float* means, const float* scales, const float* quats,
                       const float* opacity, const float* sh, int mem) {
  if (!c) return TGS_E_INVALID_ARG;
  if (deg < 0 || deg > 3 || n == 0 || !means || !scales || !quats || !opacity || !sh || (mem != TGS_HOST && mem != TGS_DEVICE)) return TGS_E_INVALID_ARG;
  const int K = (deg + 1) * (deg + 1);
  CK(cudaSetDevice(c->device));
  if (mem == TGS_HOST && (!finite_all(means, 3 * (size_t)n) || !finite_all(scales, 3 * (size_t)n) || !finite_all(quats, 4 * (size_t)n) ||
                          !finite_all(opacity, n) || !finite_all(sh, (size_t)n * K * 3))) return TGS_E_INVALID_ARG;
  CK(cudaStreamSynchronize(c->stream));
  free_list(c, c->allocs_scene);
  c->dbg_rec = nullptr;
  DevBuffers& b = c->b;
  c->n = 0;
#define A(ptr, cnt) if (int r = dev_alloc(c, &ptr, (size_t)(cnt), c->allocs_scene)) return r;
#define AZ(ptr, cnt) if (int r = dev_alloc(c, &ptr, (size_t)(cnt), c->allocs_scene, true)) return r;
  A(b.cull4, n) A(b.g2, 2 * (size_t)n) A(b.sh, (size_t)n * K * 3)
  A(b.rec_bin, 2 * (size_t)n) A(b.rec_flags, (size_t)n + 4) A(b.rec_rgb, n) A(b.rec_b0, 2 * (size_t)n)
  b.rec_b1 = b.rec_b0 + 1;
  A(b.tiles_touched, (size_t)n + 4) A(b.area_prefix, (size_t)n + 4) A(b.rendered, (size_t)n + 4) A(b.rendered_next, (size_t)n + 4)
  A(b.pre_cnt, (size_t)n / preprocess_chunk_items() + 3) AZ(b.scan_desc, (size_t)n / scan_tile_items() + 3)
  A(b.ckeys[0], n) A(b.ckeys[1], (size_t)n + preprocess_chunk_items()) A(b.cvals[0], n) A(b.cvals[1], (size_t)n + preprocess_chunk_items()) A(b.nv_queue, n) A(b.bin_params, 3 * (size_t)n) A(b.vis_list, n)
  c->dsort_tiles_cap = (n + sort_tile_items() - 1) / sort_tile_items() + 1;
  AZ(b.dsort_desc, (size_t)4 * c->dsort_tiles_cap * 256)
  AZ(b.dsort_H, depth_sort_fused_words(c->dsort_tiles_cap))
  b.dsort_tiles_cap = c->dsort_tiles_cap;
#undef A
#undef AZ
  const float *d_means = means, *d_scales = scales, *d_quats = quats, *d_opacity = opacity, *d_sh = sh;
  std::vector<void*> tmp;
  if (mem == TGS_HOST) {
    auto up = [&](const float* h, size_t cnt, const float** d) -> int {
      float* p = nullptr;
      CK(cudaMalloc((void**)&p, cnt * sizeof(float)));
      tmp.push_back(p);
      CK(cudaMemcpyAsync(p, h, cnt * sizeof(float), cudaMemcpyHostToDevice, c->stream));
      *d = p;
      return TGS_OK;
    };
    int r = up(means, 3 * (size_t)n, &d_means);
    if (!r) r = up(scales, 3 * (size_t)n, &d_scales);
    if (!r) r = up(quats, 4 * (size_t)n, &d_quats);
    if (!r) r = up(opacity, n, &d_opacity);
    if (!r) r = up(sh, (size_t)n * K * 3, &d_sh);
    if (r) { for (void* p : tmp) cudaFree(p); return r; }
  }
  launch_repack(c->stream, n, K, d_means, d_scales, d_quats, d_opacity, d_sh, b);
  cudaError_t e = cudaStreamSynchronize(c->stream);
  for (void* p : tmp) cudaFree(p);
  if (e == cudaSuccess) e = cudaGetLastError();
  if (e != cudaSuccess) { snprintf(c->err, sizeof(c->err), "load: %s", cudaGetErrorString(e)); return TGS_E_CUDA; }
  c->n = n; c->deg = deg; c->K = K;
  c->nv_hint = n / 4; c->nv_hint_cls[0] = c->nv_hint_cls[1] = n / 4;
  c->slab_ctl[0] = tgs_ctx::SlabCtl(); c->slab_ctl[1] = tgs_ctx::SlabCtl();
  invalidate_priors(c);
  c->have_frame = false;
  return TGS_OK;
}

int tgs_set_camera(tgs_ctx* c, const float view[16], float fx, float fy, float cx, float cy, int W, int H, float znear, float zfar) {
  if (!c || !view || W <= 0 || H <= 0 || W > 65535 * 16 || H > 65535 * 16 || !(fx > 0) || !(fy > 0) || !(znear > 0)) return TGS_E_INVALID_ARG;
  const float intr[6] = {fx, fy, cx, cy, znear, zfar};
  if (!finite_all(view, 16) || !finite_all(intr, 6)) return TGS_E_INVALID_ARG;
  if (c->cam_set && (c->W != W || c->H != H || c->fx != fx || c->fy != fy || c->cx != cx || c->cy != cy)) { invalidate_priors(c); c->have_frame = false; }
  memcpy(c->view, view, sizeof(c->view));
  c->fx = fx; c->fy = fy; c->cx = cx; c->cy = cy; c->W = W; c->H = H; c->znear = znear; c->zfar = zfar;
  c->TX = (W + TGS_TILE - 1) / TGS_TILE; c->TY = (H + TGS_TILE - 1) / TGS_TILE;
  c->cam_set = true;
  return TGS_OK;
}

int tgs_set_params(tgs_ctx* c, const tgs_params* p) {
  if (!c || !p || p->lambda_tdc < 1 || p->lambda_sr < 1 || !std::isfinite(p->lambda1) || !std::isfinite(p->lambda2) ||
      !std::isfinite(p->eta) || !finite_all(p->bg, 3) || (p->prior_policy != TGS_PRIORS_ANCHORED && p->prior_policy != TGS_PRIORS_CHAINED) ||
      (p->tgb_downscale != 1 && p->tgb_downscale != 2) || p->depth_slabs < 0 || p->depth_slabs > TGS_MAX_SLABS) return TGS_E_INVALID_ARG;
  for (int i = 0; i < 3; ++i) if (p->slab_split[i] > 1023u) return TGS_E_INVALID_ARG;
  c->prm = *p;
  return TGS_OK;
}

// accessors for tgs_ply.cu (the context is defined in this file only)
int tgs_ply_report(tgs_ctx* c, const char* msg) { snprintf(c->err, sizeof(c->err), "%s", msg); return 0; }
cudaStream_t tgs_ply_stream(tgs_ctx* c) { return c->stream; }
int tgs_ply_device(tgs_ctx* c) { return c->device; }

int tgs_reset_priors(tgs_ctx* c) {
  if (!c) return TGS_E_INVALID_ARG;
  invalidate_priors(c);
  return TGS_OK;
}

static int render_impl(tgs_ctx* c, int mode) {
  if (!c) return TGS_E_INVALID_ARG;
  if (!c->n) return TGS_E_NO_SCENE;
  if (!c->cam_set) return TGS_E_NO_CAMERA;
  CK(cudaSetDevice(c->device));
  // ---- what the previous frame left for the host mid-frame: the overflow flag of its pair binning ...
  if (c->bin_pending) {
    // k_scan_area / the first k_bin of the previous frame have finished (its sorts and blends may still run).  0: the tests fit
    // the capacity, so no slab can overflow; otherwise the answer is only known when the frame has ended.
    CK(cudaEventSynchronize(c->ev_bin));
    c->bin_pending = false;
    bool overflowed = false;
    if (c->h_ovf[c->bin_slot]) { CK(cudaEventSynchronize(c->ev_done)); overflowed = c->h_counters->overflow != 0; }
    if (overflowed) {
      // That frame is background only (TGS_E_CAPACITY from tgs_get_stats) and whatever it committed -- TAB, TGB, G_rendered,
      // an F of (+inf, -inf) that would make AFC cull everything -- must never be used: drop the priors, so the next AUTO
      // frame is a reference frame, and grow the automatic capacity before it.
      c->h_ovf[c->bin_slot] = 0;
      invalidate_priors(c);
      c->sel_pending = false;
      if (!c->prm.max_pairs) {
        unsigned long long want = (unsigned long long)c->max_pairs * 2ull;
        if (want > (1ull << 30) - 1) want = (1ull << 30) - 1;
        if (int r = alloc_pair_buffers(c, (uint32_t)want, c->sort_passes_cap)) return r;
      }
    }
  }
  // ---- A0: frame type (R9, R23)
  if (c->sel_pending) {   // eta rule needs the selected-tile count of the previous S frame
    CK(cudaEventSynchronize(c->ev_sel));
    c->sched.force_P = (c->prm.enable_sr && (float)c->h_sel[0] > c->prm.eta * (float)c->last_n_tiles) ? 1 : 0;   // L128; R41: only with SR on
    c->sel_pending = false;
  }
  int ftype;
  if (mode == TGS_AUTO) {
    if (!c->priors_valid || c->sched.since_R >= c->prm.lambda_tdc) ftype = TGS_FRAME_R;
    else if (c->sched.since_ref >= c->prm.lambda_sr || c->sched.force_P) ftype = TGS_FRAME_P;
    else ftype = TGS_FRAME_S;
  } else if (mode == TGS_FULL) ftype = TGS_FRAME_R;
  else if (mode == TGS_PSEUDO_REF) ftype = TGS_FRAME_P;
  else if (mode == TGS_TEMPORAL) ftype = TGS_FRAME_S;
  else return TGS_E_INVALID_ARG;
  if (ftype != TGS_FRAME_R && !c->priors_valid) return TGS_E_NO_PRIORS;

  if (int r = alloc_frame_buffers(c)) return r;
  const int tile_bits = tile_key_bits(c->TX * c->TY), tile_passes = (tile_bits + 7) / 8;
  if (int r = alloc_pair_buffers(c, c->prm.max_pairs ? c->prm.max_pairs : auto_max_pairs(c), tile_passes)) return r;
  // What is known about the scene comes from the statistics of frame N - 2 (same parity: its counter block is the one this
  // frame reuses, so its export is waited for anyway; by now it has long finished).  Deterministic, unlike "whatever has
  // arrived": the choices below (depth-sort instance, number of slabs, capacity) do not depend on host timing.
  if (++c->epoch >= (1u << 28)) {   // tag wrap-around: forget every descriptor (once per 2^28 frames)
    CK(cudaMemsetAsync(c->b.scan_desc, 0, ((size_t)c->n / scan_tile_items() + 3) * 8, c->stream));
    CK(cudaMemsetAsync(c->b.dsort_desc, 0, (size_t)4 * c->dsort_tiles_cap * 256 * 8, c->stream));
    CK(cudaMemsetAsync(c->b.sort_desc, 0, (size_t)c->sort_passes_cap * c->sort_tiles_cap * 256 * 8, c->stream));
    CK(cudaMemsetAsync(c->b.bin_desc, 0, (size_t)c->bin_chunks_cap * 8, c->stream));
    c->epoch = 1;
  }
  const int ci = (int)(c->epoch & 1u);
  if (c->cnt_pending[ci]) {
    CK(cudaEventSynchronize(c->ev_cnt[ci])); c->cnt_pending[ci] = false;
    const Counters& h2 = *c->h_cnt2[ci];
    c->nv_hint = h2.n_visible; c->nv_hint_cls[c->hist_cls[ci]] = h2.n_visible;
    c->half_hint = h2.n_visible > 0 && h2.n_tests < 8ull * h2.n_visible;     // small splats: most records reach one half of a tile only
    if (!h2.overflow && h2.n_tests) {
      tgs_ctx::SlabCtl& sc = c->slab_ctl[c->hist_cls[ci]];
      sc.tests = h2.n_tests;
      const float ratio = (float)h2.n_pairs / (float)h2.n_tests;
      if (c->hist_slabs[ci] == 1) sc.p1 = ratio;
      else if (c->hist_slabs[ci] == 2) {
        sc.p2 = ratio;
        // Where the first piece ends (automatic mode only).  The fastest split is the smallest one that leaves the second
        // piece next to nothing (config 3, per class and 40-frame segment: 128 ... 512 of 1024, always the smallest with
        // pairs(2nd) / pairs(1st) ~ 0); below it the second piece has to enumerate the rest of the test space for the tiles
        // that are still alive, and the frame time rises steeply.  So: shrink by 1/8 per frame of the class while the
        // second piece stays empty, step back up by 1/4 as soon as it does not, and then leave the split alone for 24 frames
        // of the class and never go below what just failed.  Only statistics of a frame rendered with the CURRENT split count.
        if (c->hist_split[ci] != 0 && c->hist_split[ci] == sc.split) {
          const float r = (float)h2.n_pairs_slab[1] / (float)(h2.n_pairs_slab[0] ? h2.n_pairs_slab[0] : 1u);
          sc.empty2 = r < 0.03f && sc.split <= 576u;
          // (growing only helps where it makes tiles finish: stacks of thin sheets keep half of their tiles alive whatever
          // the split -- config 5 -- and are left at the default)
          const bool tiles_finish = (unsigned long long)h2.n_finished[0] * 10ull >= (unsigned long long)h2.n_sel * 6ull;
          if (r > 0.03f && tiles_finish) {
            sc.split_floor = sc.split + sc.split / 16 < 768u ? sc.split + sc.split / 16 : 768u;
            sc.split = sc.split + sc.split / 4 < 768u ? sc.split + sc.split / 4 : 768u;
            sc.hold = 24;
          } else if (r < 0.005f && sc.hold == 0) {
            const uint32_t next = sc.split - sc.split / 8;
            sc.split = next > sc.split_floor ? next : sc.split_floor;
          }
        }
      }
    }
    // grow the automatic capacity when a frame came close to it (the slabs' lists are never longer than the tests)
    if (!c->prm.max_pairs && (h2.n_pairs > c->max_pairs / 2 || h2.n_tests > c->max_pairs)) {
      unsigned long long want = (unsigned long long)c->max_pairs * 2ull;
      if (want > (1ull << 30) - 1) want = (1ull << 30) - 1;
      if (int r = alloc_pair_buffers(c, (uint32_t)want, tile_passes)) return r;
    }
  }

  FrameConst& fc = c->fc;
  CamConst& k = fc.cam;
  for (int i = 0; i < 12; ++i) k.V[i] = c->view[i];
  k.fx = c->fx; k.fy = c->fy; k.cx = c->cx; k.cy = c->cy; k.Wf = (float)c->W; k.Hf = (float)c->H;
  const float tanx = (0.5f * (float)c->W) / c->fx, tany = (0.5f * (float)c->H) / c->fy;
  k.limx = 1.3f * tanx; k.limy = 1.3f * tany;
  k.znear = c->znear;
  for (int j = 0; j < 3; ++j)
    k.campos[j] = (float)-(((double)c->view[0 * 4 + j] * c->view[3] + (double)c->view[1 * 4 + j] * c->view[7]) + (double)c->view[2 * 4 + j] * c->view[11]);
  k.W = c->W; k.H = c->H; k.TX = c->TX; k.TY = c->TY;
  if (ftype == TGS_FRAME_S) { relative_pose(c->prior_view, c->view, fc.M); relative_pose(c->view, c->prior_view, fc.Minv); }
  else { memset(fc.M, 0, sizeof(fc.M)); memset(fc.Minv, 0, sizeof(fc.Minv)); }
  TgbGrid& tg = fc.tg;
  tg.ds = c->prm.tgb_downscale == 2 ? 2 : 1;
  if (tg.ds == 1) { tg.W = c->W; tg.H = c->H; tg.fx = c->fx; tg.fy = c->fy; tg.cx = c->cx; tg.cy = c->cy; }
  else {
    tg.W = (c->W + 1) / 2; tg.H = (c->H + 1) / 2;
    tg.fx = c->fx * 0.5f; tg.fy = c->fy * 0.5f; tg.cx = (c->cx - 0.5f) * 0.5f; tg.cy = (c->cy - 0.5f) * 0.5f;
  }
  tg.Wf = (float)tg.W; tg.Hf = (float)tg.H;
  fc.lambda1 = c->prm.lambda1; fc.lambda2 = c->prm.lambda2;
  for (int j = 0; j < 3; ++j) fc.bg[j] = c->prm.bg[j];
  fc.n = c->n; fc.max_pairs = c->max_pairs; fc.sh_degree = c->deg; fc.ftype = ftype;
  fc.do_afc = (ftype != TGS_FRAME_R) && c->prm.enable_afc && c->F_valid;
  fc.do_tgb = (ftype == TGS_FRAME_S);
  fc.do_toc = fc.do_tgb && c->prm.enable_toc;
  fc.all_tiles = !(ftype == TGS_FRAME_S && c->prm.enable_sr && !c->force_all);
  fc.exact_tiles = c->prm.exact_tiles ? 1 : 0;
  fc.n_tiles = c->TX * c->TY;
  fc.epoch = c->epoch;
  // the depth sort as one launch (k_sort.cu) where the visible list of this frame class has been short enough for one tile per
  // resident CTA; longer lists keep the onesweep launches (more CTAs per SM, look-back instead of grid barriers)
  fc.dsort_fused = c->dsort_mode >= 0 ? c->dsort_mode
                   : (c->nv_hint_cls[ftype == TGS_FRAME_S ? 1 : 0] <= (uint32_t)c->num_sms * depth_sort_fused_ctas_per_sm() * depth_sort_fused_tile_items() ? 1 : 0);
  fc.blend_half = c->blend_half_mode < 0 ? (c->half_hint ? 1 : 0) : c->blend_half_mode;
  // front-to-back slabs: explicit, or automatic from the size of a recent frame's test space -- small frames
  // are launch bound and stay in one piece
  {
    int ns = c->prm.depth_slabs;
    if (ns == 0) {
      // Two pieces pay where most tiles finish inside the first one: then the second piece bins and sorts next to nothing.
      // Where the tiles stay alive (thin surfaces, clouds with gaps) the second piece only adds launches and the parking
      // of the pixel states.  Measured, not guessed: p1, p2 = pairs per test of the latest one-piece and two-piece frames of
      // this class (R / P, S); two pieces where p2 < 0.4 p1 (config 3, per 20-frame segment of the trajectory: two pieces are
      // the faster choice up to a ratio of 0.35 and the slower one from 0.46 on); small frames are launch bound and stay in one piece.
      //  * With two pieces p2 is fresh every frame and p1 is not needed again: it is a property of the tile test, not of the
      //    occlusion (0.57-0.63 over the whole trajectory), so no one-piece frame is rendered just to re-measure it.
      //  * With one piece p2 goes stale; two pieces are probed again (one frame) every 32 frames of the class -- every 8
      //    while the other class runs two pieces far below its threshold --, or as soon as the test space has grown by a
      //    quarter since the last probe.
      const int cls = ftype == TGS_FRAME_S ? 1 : 0;
      tgs_ctx::SlabCtl& sc = c->slab_ctl[cls];
      const tgs_ctx::SlabCtl& other = c->slab_ctl[1 - cls];
      if (!sc.asked1) { ns = 1; sc.asked1 = true; }                               // a one-piece sample ...
      else if (sc.tests < 2000000u) { ns = 1; sc.two = false; }                   // (small, or nothing known yet)
      else if (!sc.asked2) { ns = 2; sc.asked2 = true; sc.tests_probe = sc.tests; sc.since_probe = 0; }   // ... then ONE two-piece probe ...
      else if (sc.p1 < 0.0f || sc.p2 < 0.0f) ns = 1;                              // ... and one piece until both have been counted
      else {
        // two pieces where they drop 60 % of the pairs, or where a first piece of at most 9/16 of the tests leaves the second one empty
        sc.two = sc.p2 < 0.4f * sc.p1 || sc.empty2;
        ns = sc.two ? 2 : 1;
        ++sc.since_probe;
        if (!sc.two) {
          const bool hinted = other.two && other.p2 < 0.3f * other.p1;
          const bool grown = (unsigned long long)sc.tests * 4ull > (unsigned long long)sc.tests_probe * 5ull;
          if (sc.since_probe >= 32 || (sc.since_probe >= 8 && hinted) || (sc.since_probe >= 4 && grown)) {
            ns = 2; sc.since_probe = 0; sc.tests_probe = sc.tests;
          }
        }
      }
    }
    static const uint32_t def_split[TGS_MAX_SLABS + 1][3] = {{0, 0, 0}, {0, 0, 0}, {256, 0, 0}, {160, 448, 0}, {96, 256, 512}};
    fc.n_slabs = ns;
    fc.slab_bound[0] = 0;
    uint32_t auto_split = 0;
    if (c->prm.depth_slabs == 0 && ns == 2 && !c->prm.slab_split[0]) {
      tgs_ctx::SlabCtl& sc = c->slab_ctl[ftype == TGS_FRAME_S ? 1 : 0];
      if (!sc.two) {                                                           // a probe from one-piece mode: a quarter, three eighths, half of the tests in turn
        static const uint32_t probe_split[3] = {256, 384, 512};
        sc.split = probe_split[sc.probe_k++ % 3]; sc.split_floor = 64; sc.hold = 0;
      }
      else if (sc.hold > 0) { if (--sc.hold == 0) sc.split_floor = 64; }   // (a floor that only decays was tried: the best split of config 3 falls from 256 to 128 within 80 frames, and the floor kept it from following)
      auto_split = sc.split;
    }
    c->cur_split = auto_split;
    for (int i = 1; i < ns; ++i) {
      uint32_t v = c->prm.slab_split[i - 1] ? c->prm.slab_split[i - 1] : def_split[ns][i - 1];
      if (auto_split) v = auto_split;
      if (v < fc.slab_bound[i - 1]) v = fc.slab_bound[i - 1];
      fc.slab_bound[i] = v;
    }
    for (int i = ns; i <= TGS_MAX_SLABS; ++i) fc.slab_bound[i] = 1024;
    if (ns > 1 && !c->b.pix_state) {
      if (int r = dev_alloc(c, &c->b.live_sat, (size_t)(c->TX + 1) * (c->TY + 1), c->allocs_frame)) return r;
      if (int r = dev_alloc(c, &c->b.pix_state, (size_t)(c->TX * c->TY) * 7 * TGS_TILE * TGS_TILE, c->allocs_frame)) return r;
    }
  }
  c->b.counters = c->counters2[ci];          // ci = parity of this frame's epoch (computed above)
  c->h_counters = c->h_cnt2[ci];
  c->b.F_key = c->F_base + 4 * (ftype == TGS_FRAME_R ? ci : c->F_idx);   // R: reset + built here (k_frustum, third stream); P / S: read

  DevBuffers& b = c->b;
  cudaStream_t s = c->stream;
  const bool builds_priors = ftype != TGS_FRAME_S;
  // R42 (prior_policy = CHAINED): an S frame's stitched outputs become the priors too; its G_rendered marks are OR-ed
  // into the current set in place (k_preprocess has read the set before the blend writes it: stream order)
  const bool chains = ftype == TGS_FRAME_S && c->prm.prior_policy == TGS_PRIORS_CHAINED;
  // never the priors (they are being read), and not the previous frame's buffers either when there is a third choice:
  // an asynchronous read-back of that image may still be running (tgs_read_image_async)
  int out_idx = (c->prior_idx + 1) % 3;
  if (out_idx == c->cur_idx) out_idx = (out_idx + 1) % 3 == c->prior_idx ? out_idx : (out_idx + 1) % 3;
  const float* prior_image = c->priors_valid ? b.image[c->prior_idx] : nullptr;
  uint8_t* rendered_next = builds_priors ? b.rendered_next : nullptr;
  uint8_t* rendered_marks = chains ? b.rendered : rendered_next;
  c->n_ev = 0;
  auto mark = [&](int stage) { if (c->timing && c->n_ev < tgs_ctx::MAX_EV) { cudaEventRecord(c->ev_stage[c->n_ev], s); c->ev_tag[c->n_ev++] = stage; } };
  mark(0);                                                                     // 0: init, A1 warp, A2 fill + correspondence
  launch_frame_init(s, fc, b, ftype == TGS_FRAME_R, rendered_next);
  if (ftype == TGS_FRAME_S) launch_warp(s, fc, b, b.depth[c->prior_idx], b.sigma[c->prior_idx]);          // A1
  // A2 (depth fill, correspondence, T^um) is only needed by the tile selection: it runs beside the preprocess.
  // With stage timing on, everything stays on one stream so that the stage events bracket what they name.
  const bool fork = !c->timing;
  if (ftype == TGS_FRAME_S) {
    if (fork) { CK(cudaEventRecord(c->ev_fork2, s)); CK(cudaStreamWaitEvent(c->side, c->ev_fork2, 0)); }
    launch_fill_corr(fork ? c->side : s, fc, b);                                                           // A2
  }
  mark(1);                                                                     // 1: A3 preprocess, A4 selection
  if (c->post2_pending) { CK(cudaStreamWaitEvent(s, c->ev_post2, 0)); c->post2_pending = false; }          // k_frustum of the previous frame
  launch_preprocess(s, fc, b, c->num_sms);                                                                 // A3 (+ small-rect T^oc) + visible list
  if (ftype == TGS_FRAME_S) {
    // A4 (T^oc of larger rects, T_sel) is only needed by the pair binning: it runs beside the depth sort
    cudaStream_t s4 = fork ? c->side : s;
    if (fork) { CK(cudaEventRecord(c->ev_fork, s)); CK(cudaStreamWaitEvent(c->side, c->ev_fork, 0)); }
    launch_mark_oc(s4, fc, b, c->num_sms);                                                                 // A4: T^oc of larger rects
    launch_select(s4, fc, b, c->h_sel);                                                                    // A4: T_sel (R / P: all tiles, k_frame_init); n_sel -> host
    CK(cudaEventRecord(c->ev_sel, s4));
    c->sel_pending = true;
  }
  // SH colours of every visible Gaussian on a third stream beside the depth sort (few CTAs, most SMs idle).  Behind k_bin
  // a colour kernel only queues up behind the tile sort, whose CTAs fill the register file (measured: no overlap).
  const bool early_colour = fork;
  if (early_colour) {
    CK(cudaEventRecord(c->ev_fork3, s)); CK(cudaStreamWaitEvent(c->side2, c->ev_fork3, 0));
    launch_colour_all(c->side2, fc, b, c->num_sms);
    CK(cudaEventRecord(c->ev_join, c->side2));
  }
  mark(2);                                                                     // 2: A6 level 1
  c->h_ovf[ci] = 0;
  int dsorted = 0;                                                                                         // visible Gaussians by depth
  if (fc.dsort_fused)
    launch_depth_sort_fused(s, fc, b, bin_max_tests(c->bin_chunks_cap), c->h_ovf + ci, c->num_sms, c->nv_hint_cls[ftype == TGS_FRAME_S ? 1 : 0]);
  else
    dsorted = launch_sort(s, b.ckeys, b.cvals, &b.counters->n_visible, 32, b.sort_hist, b.dsort_desc, c->dsort_tiles_cap,
                          &b.counters->ticket_sort[0], &b.counters->error, fc.epoch, c->num_sms, c->nv_hint < 1000000u);
  if (ftype == TGS_FRAME_S && fork) CK(cudaStreamWaitEvent(s, c->ev_sel, 0));                              // join A2 + A4
  // ---- A5-A9, slab by slab (one slab: the plain pipeline)
  int sorted = 0;
  for (int k = 0; k < fc.n_slabs; ++k) {
    mark(3);                                                                   // 3: A5 pairs
    launch_bin(s, fc, b, dsorted, c->bin_chunks_cap, c->num_sms, c->h_ovf + ci, k);                        // tests -> pairs, counts
    if (k == 0) {
      CK(cudaEventRecord(c->ev_bin, s));
      c->bin_pending = true; c->bin_slot = ci;
      mark(4);                                                                 // 4: A5 colours (production: third stream, beside the depth sort)
      if (!early_colour) launch_colour_all(s, fc, b, c->num_sms);                                         // stage timing: the production kernel, in line
    }
    mark(5);                                                                   // 5: A6 level 2 + A7
    sorted = launch_sort(s, b.keys, b.vals, &b.counters->n_pairs_slab[k], tile_bits, b.sort_hist + (1 + k) * 4 * 256,
                         b.sort_desc, c->sort_tiles_cap, &b.counters->ticket_tsort[k][0], &b.counters->error, fc.epoch * 4u + (uint32_t)k, c->num_sms, false,
                         b.ranges);                                                                        // pairs by tile + A7 in the last pass
    mark(6);                                                                   // 6: A8 + A9
    if (k == 0) {
      if (fork) CK(cudaStreamWaitEvent(s, c->ev_join, 0));
      if (c->copy_pending[out_idx]) { CK(cudaStreamWaitEvent(s, c->ev_copy[out_idx], 0)); c->copy_pending[out_idx] = false; }   // an asynchronous read of this buffer
    }
    launch_blend(s, fc, b, sorted, out_idx, prior_image, rendered_marks, c->num_sms, c->count_interactions, k);
  }
  mark(7);                                                                     // 7: post
  if (builds_priors && !fork) launch_frustum(s, fc, b, b.cvals[dsorted], rendered_next, ftype == TGS_FRAME_R);      // F_min/F_max (L109)
  if (fork) {
    // post-processing on the third stream, beside the start of the next frame: F / |G_rendered| over the visible list
    // (the next frame waits for ev_post2 before it overwrites that list or reads F) and the counters' copy to the host
    CK(cudaEventRecord(c->ev_post, s)); CK(cudaStreamWaitEvent(c->side2, c->ev_post, 0));
    if (builds_priors) {
      launch_frustum(c->side2, fc, b, b.cvals[dsorted], rendered_next, ftype == TGS_FRAME_R);
      CK(cudaEventRecord(c->ev_post2, c->side2));
      c->post2_pending = true;
    }
    launch_export_counters(c->side2, b, c->h_counters);
    CK(cudaEventRecord(c->ev_done, c->side2));
    CK(cudaEventRecord(c->ev_cnt[ci], c->side2));
    c->cnt_pending[ci] = true;
  } else {
    launch_export_counters(s, b, c->h_counters);
    mark(8);                                                                   // end
    CK(cudaEventRecord(c->ev_done, s));
    CK(cudaEventRecord(c->ev_cnt[ci], s));
    c->cnt_pending[ci] = true;
  }
  CK(cudaGetLastError());
  // ---- A10: prior commit (pointer swap) and scheduler counters
  c->cur_idx = out_idx; c->sorted_idx = sorted;
  if (builds_priors) {
    c->prior_idx = out_idx;
    std::swap(b.rendered, b.rendered_next);
    memcpy(c->prior_view, c->view, sizeof(c->prior_view));
    c->priors_valid = true;
    if (ftype == TGS_FRAME_R) { c->F_valid = true; c->F_idx = ci; }
  }
  if (chains) { c->prior_idx = out_idx; memcpy(c->prior_view, c->view, sizeof(c->prior_view)); }
  if (ftype == TGS_FRAME_R) { c->sched.since_R = 0; c->sched.since_ref = 0; c->sched.force_P = 0; }
  else if (ftype == TGS_FRAME_P) { c->sched.since_ref = 0; c->sched.force_P = 0; }
  ++c->sched.since_R; ++c->sched.since_ref;
  c->last_ftype = ftype; c->last_n_tiles = (uint32_t)fc.n_tiles; c->last_n_slabs = fc.n_slabs;
  c->hist_cls[ci] = ftype == TGS_FRAME_S ? 1 : 0; c->hist_slabs[ci] = fc.n_slabs; c->hist_split[ci] = c->cur_split;
  c->have_frame = true;
  return TGS_OK;
}

int tgs_read_image(tgs_ctx* c, float* rgb, int mem) {
  if (!c || !rgb || !c->have_frame) return TGS_E_INVALID_ARG;
  return copy_out(c, rgb, c->b.image[c->cur_idx], (size_t)c->W * c->H * 3 * sizeof(float), mem);
}

int tgs_read_image_async(tgs_ctx* c, float* rgb_host) {
  if (!c || !rgb_host || !c->have_frame) return TGS_E_INVALID_ARG;
  CK(cudaSetDevice(c->device));
  CK(cudaStreamWaitEvent(c->copy, c->ev_done, 0));                     // the frame is complete
  CK(cudaMemcpyAsync(rgb_host, c->b.image[c->cur_idx], (size_t)c->W * c->H * 3 * sizeof(float), cudaMemcpyDeviceToHost, c->copy));
  CK(cudaEventRecord(c->ev_copy[c->cur_idx], c->copy));
  c->copy_pending[c->cur_idx] = true;
  return TGS_OK;
}

int tgs_wait_reads(tgs_ctx* c) {
  if (!c) return TGS_E_INVALID_ARG;
  CK(cudaSetDevice(c->device));
  CK(cudaStreamSynchronize(c->copy));
  c->copy_pending[0] = c->copy_pending[1] = c->copy_pending[2] = false;
  return TGS_OK;
}

int tgs_read_depth(tgs_ctx* c, float* depth, float* sigma, int mem) {
  if (!c || !depth || !c->have_frame) return TGS_E_INVALID_ARG;
  if (sigma) { if (int r = copy_out(c, sigma, c->b.sigma[c->cur_idx], (size_t)c->W * c->H * sizeof(float), mem)) return r; }
  return copy_out(c, depth, c->b.depth[c->cur_idx], (size_t)c->W * c->H * sizeof(float), mem);
}

int tgs_read_tile_mask(tgs_ctx* c, uint8_t* sel, int mem) {
  if (!c || !sel || !c->have_frame) return TGS_E_INVALID_ARG;
  return copy_out(c, sel, c->b.tile_mask, (size_t)c->TX * c->TY, mem);
}

int tgs_get_stats(tgs_ctx* c, tgs_stats* out) {
  if (!c || !out || !c->have_frame) return TGS_E_INVALID_ARG;
  CK(cudaEventSynchronize(c->ev_done));
  const Counters& h = *c->h_counters;
  memset(out, 0, sizeof(*out));
  out->frame_type = c->last_ftype;
  out->n_total = c->n; out->n_near = h.n_near; out->n_afc = h.n_afc; out->n_toc = h.n_toc; out->n_degenerate = h.n_degenerate;
  out->n_empty = h.n_empty; out->n_visible = h.n_visible; out->n_newly_visible = h.n_newly_visible;
  out->n_pairs = h.n_pairs; out->n_tiles = c->last_n_tiles; out->n_sel_oc = h.n_sel_oc; out->n_sel_um = h.n_sel_um; out->n_sel = h.n_sel;
  out->n_rendered = h.n_rendered; out->overflow = h.overflow; out->n_interactions = h.n_interactions; out->n_blended = h.n_blended; out->n_pixel_slots = h.n_slots;
  out->device_bytes = c->device_bytes;
  out->n_tests = h.n_tests; out->n_tests_evaluated = h.n_tests_eval; out->n_pairs_consumed = h.n_consumed; out->n_half_tile_visits = h.n_wrec; out->n_half_tile_visits_dead = h.n_wrec_dead; out->launches_total = g_tgs_launches;
  out->n_slabs = (uint32_t)c->last_n_slabs;
  for (int i = 0; i < TGS_MAX_SLABS; ++i) { out->n_pairs_slab[i] = h.n_pairs_slab[i]; out->n_finished_slab[i] = h.n_finished[i]; }
  if (c->timing) {
    for (int i = 0; i + 1 < c->n_ev; ++i) {
      float ms = 0.0f;
      cudaEventElapsedTime(&ms, c->ev_stage[i], c->ev_stage[i + 1]);
      if (c->ev_tag[i] >= 0 && c->ev_tag[i] < 8) out->ms_stage[c->ev_tag[i]] += ms;
    }
    if (c->n_ev >= 2) cudaEventElapsedTime(&out->ms_total, c->ev_stage[0], c->ev_stage[c->n_ev - 1]);
  }
  if (h.error) { snprintf(c->err, sizeof(c->err), "device watchdog: a look-back (code 1: prefix scan, 2: radix sort) or the grid barrier of the one-launch depth sort (3) stalled (code %u)", h.error); return TGS_E_CUDA; }
  if (h.overflow) return TGS_E_CAPACITY;
  return TGS_OK;
}


// ------------------------------------------------------------------ test-only access to intermediates
static uint32_t f2key_host(float f) { uint32_t b; memcpy(&b, &f, 4); return (b & 0x80000000u) ? ~b : (b | 0x80000000u); }
static float key2f_host(uint32_t k) { const uint32_t b = (k & 0x80000000u) ? (k & 0x7fffffffu) : ~k; float f; memcpy(&f, &b, 4); return f; }

static long long debug_get_impl(tgs_ctx* c, const char* nm, void* dst, size_t bytes, int mem) {
  if (!c || !nm || (mem != TGS_HOST && mem != TGS_DEVICE)) return TGS_E_INVALID_ARG;
  CK(cudaSetDevice(c->device));
  const std::string name(nm);
  if (c->post2_pending) CK(cudaStreamWaitEvent(c->stream, c->ev_post2, 0));   // k_frustum of the last frame (third stream)
  const DevBuffers& b = c->b;
  const size_t N = c->n, px = (size_t)c->W * c->H, T = (size_t)c->TX * c->TY;
  const size_t tpx = c->fc.tg.W > 0 ? (size_t)c->fc.tg.W * c->fc.tg.H : px;   // TGB grid of the last frame (R43)
  const void* src = nullptr; size_t have = 0;
  if (name == "keys" || name == "vals") {
    if (!c->have_frame) return TGS_E_INVALID_ARG;
    CK(cudaEventSynchronize(c->ev_done));
    const size_t P = c->h_counters->n_pairs_slab[c->last_n_slabs - 1];          // the list of the last slab (one slab: the whole list)
    if (name == "keys") {
      if (!c->keys64 && P) { if (int r = dev_alloc(c, &c->keys64, (size_t)c->max_pairs, c->allocs_pairs)) return r; }
      launch_keys64(c->stream, c->b, c->sorted_idx, (uint32_t)P, c->keys64);
      src = c->keys64; have = P * 8;
      if (!P) return 0;
    } else { src = b.vals[c->sorted_idx]; have = P * 4; if (!P) return 0; }
  } else if (name == "F") {
    uint32_t keys[4]; float F[4];
    CK(cudaMemcpyAsync(keys, b.F_key, sizeof(keys), cudaMemcpyDeviceToHost, c->stream));
    CK(cudaStreamSynchronize(c->stream));
    for (int i = 0; i < 4; ++i) F[i] = key2f_host(keys[i]);
    if (dst && bytes) {
      if (mem == TGS_HOST) memcpy(dst, F, bytes < 16 ? bytes : 16);
      else { CK(cudaMemcpy(dst, F, bytes < 16 ? bytes : 16, cudaMemcpyHostToDevice)); }
    }
    return 16;
  }
  else if (name == "rec_uvdo" || name == "rec_conic" || name == "rec_rect") {      // not stored as such: put together from rec_bin, the blend record and the scene
    if (!c->dbg_rec && N) { if (int r = dev_alloc(c, &c->dbg_rec, N, c->allocs_scene)) return r; }
    launch_debug_record(c->stream, c->fc, b, (uint32_t)N, name == "rec_uvdo" ? 0 : name == "rec_conic" ? 1 : 2, c->dbg_rec);
    src = c->dbg_rec; have = N * (name == "rec_rect" ? 8 : 16);
  }
  else if (name == "rec_flags") {                            // stored as bytes, reported as words
    if (!c->dbg_rec && N) { if (int r = dev_alloc(c, &c->dbg_rec, N, c->allocs_scene)) return r; }
    launch_debug_flags(c->stream, b, (uint32_t)N, reinterpret_cast<uint32_t*>(c->dbg_rec));
    src = c->dbg_rec; have = N * 4;
  }
  else if (name == "rec_rgb") { src = b.rec_rgb; have = N * 16; }
  else if (name == "tiles_touched") {
    if (!c->have_frame) return TGS_E_INVALID_ARG;
    CK(cudaEventSynchronize(c->ev_done));
    if (c->h_counters->overflow) return TGS_E_CAPACITY;
    launch_count_pairs(c->stream, c->b, c->sorted_idx, (uint32_t)c->h_counters->n_pairs_slab[c->last_n_slabs - 1], (uint32_t)N);
    src = b.tiles_touched; have = N * 4;
  }
  else if (name == "ranges") {
    if (!c->ranges_dec) { if (int r = dev_alloc(c, &c->ranges_dec, T, c->allocs_frame)) return r; }
    launch_ranges_decode(c->stream, b, (int)T, c->ranges_dec);
    src = c->ranges_dec; have = T * 8;
  }
  else if (name == "tile_order") { src = b.tile_order; have = T * 4; }
  else if (name == "warp_depth" || name == "warp_sigma") {   // de-interleave {D^min, sigma^max}: a strided copy
    have = tpx * 4;
    if (dst && bytes) {
      const size_t cnt = (bytes < have ? bytes : have) / 4;
      const float* base = reinterpret_cast<const float*>(b.warp_tgb) + (name == "warp_sigma" ? 1 : 0);
      CK(cudaMemcpy2DAsync(dst, 4, base, 8, 4, cnt, mem == TGS_DEVICE ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, c->stream));
      if (mem == TGS_HOST) CK(cudaStreamSynchronize(c->stream));
    }
    return (long long)have;
  }
  else if (name == "fill_depth") { src = b.fill_depth; have = tpx * 4; }
  else if (name == "rendered") { src = b.rendered; have = N; }
  else if (name == "prior_depth") { src = b.depth[c->prior_idx]; have = px * 4; }
  else if (name == "prior_sigma") { src = b.sigma[c->prior_idx]; have = px * 4; }
  else if (name == "prior_image") { src = b.image[c->prior_idx]; have = px * 12; }
  else if (name == "g2") { src = b.g2; have = N * 32; }
  else return TGS_E_INVALID_ARG;
  if (!src) return TGS_E_INVALID_ARG;
  if (dst && bytes && have) { if (int r = copy_out(c, dst, src, bytes < have ? bytes : have, mem)) return r; }
  return (long long)have;
}

static int debug_put_impl(tgs_ctx* c, const char* nm, const void* src, size_t bytes, int mem) {
  if (!c || !nm || !src || (mem != TGS_HOST && mem != TGS_DEVICE) || !c->cam_set || !c->n) return TGS_E_INVALID_ARG;
  CK(cudaSetDevice(c->device));
  if (int r = alloc_frame_buffers(c)) return r;
  const std::string name(nm);
  DevBuffers& b = c->b;
  const size_t N = c->n, px = (size_t)c->W * c->H;
  const cudaMemcpyKind kind = mem == TGS_HOST ? cudaMemcpyHostToDevice : cudaMemcpyDeviceToDevice;
  auto put = [&](void* dstp, size_t want) -> int {
    if (bytes != want) return TGS_E_INVALID_ARG;
    CK(cudaMemcpyAsync(dstp, src, bytes, kind, c->stream));
    CK(cudaStreamSynchronize(c->stream));
    return TGS_OK;
  };
  if (name == "prior_depth") { int r = put(b.depth[c->prior_idx], px * 4); if (!r) c->put_depth = true; return r; }
  if (name == "prior_sigma") { int r = put(b.sigma[c->prior_idx], px * 4); if (!r) c->put_sigma = true; return r; }
  if (name == "prior_image") { int r = put(b.image[c->prior_idx], px * 12); if (!r) c->put_image = true; return r; }
  if (name == "rendered") return put(b.rendered, N);
  if (name == "F") {
    if (bytes != 16) return TGS_E_INVALID_ARG;
    float F[4]; uint32_t keys[4];
    if (mem == TGS_HOST) memcpy(F, src, 16); else { CK(cudaMemcpy(F, src, 16, cudaMemcpyDeviceToHost)); }
    for (int i = 0; i < 4; ++i) keys[i] = f2key_host(F[i]);
    CK(cudaMemcpyAsync(b.F_key, keys, 16, cudaMemcpyHostToDevice, c->stream));
    CK(cudaStreamSynchronize(c->stream));
    c->F_valid = true;
    return TGS_OK;
  }
  if (name == "prior_view") {
    if (bytes != 64) return TGS_E_INVALID_ARG;
    if (mem == TGS_HOST) memcpy(c->prior_view, src, 64); else { CK(cudaMemcpy(c->prior_view, src, 64, cudaMemcpyDeviceToHost)); }
    if (!c->priors_valid) {
      if (!(c->put_depth && c->put_sigma && c->put_image)) return TGS_E_NO_PRIORS;
      c->priors_valid = true;
    }
    return TGS_OK;
  }
  return TGS_E_INVALID_ARG;
}

static int debug_run_stage_impl(tgs_ctx* c, const char* st) {
  if (!c || !st) return TGS_E_INVALID_ARG;
  const std::string s(st);
  if (s == "timing_on") { c->timing = true; return TGS_OK; }
  if (s == "timing_off") { c->timing = false; return TGS_OK; }
  if (s == "count_interactions_on") { c->count_interactions = true; return TGS_OK; }
  if (s == "count_interactions_off") { c->count_interactions = false; return TGS_OK; }
  if (s == "force_all_tiles_on") { c->force_all = 1; return TGS_OK; }
  if (s == "force_all_tiles_off") { c->force_all = 0; return TGS_OK; }
  if (s == "depth_sort_fused_on") { c->dsort_mode = 1; return TGS_OK; }
  if (s == "depth_sort_fused_off") { c->dsort_mode = 0; return TGS_OK; }
  if (s == "depth_sort_fused_auto") { c->dsort_mode = -1; return TGS_OK; }
  if (s == "blend_half_on") { c->blend_half_mode = 1; return TGS_OK; }
  if (s == "blend_half_off") { c->blend_half_mode = 0; return TGS_OK; }
  if (s == "blend_half_auto") { c->blend_half_mode = -1; return TGS_OK; }
  if (s == "redzones_on") {            // takes effect for the buffers allocated from now on: call it before tgs_load_gaussians
    if (c->n || c->px_cap) return TGS_E_INVALID_ARG;
    c->redzones = true; return TGS_OK;
  }
  if (s == "check_redzones") {
    const int bad = check_redzones(c);
    return bad == 0 ? TGS_OK : TGS_E_CUDA;
  }
  return TGS_E_INVALID_ARG;
}

int tgs_load_gaussians(tgs_ctx* c, uint32_t n, int deg, const float* means, const float* scales, const float* quats,
                       const float* opacity, const float* sh, int mem) {
  TGS_NOEXCEPT_BODY(c, load_gaussians_impl(c, n, deg, means, scales, quats, opacity, sh, mem))
}
int tgs_render(tgs_ctx* c, int mode) { TGS_NOEXCEPT_BODY(c, render_impl(c, mode)) }
long long tgs_debug_get(tgs_ctx* c, const char* nm, void* dst, size_t bytes, int mem) { TGS_NOEXCEPT_BODY(c, debug_get_impl(c, nm, dst, bytes, mem)) }
int tgs_debug_put(tgs_ctx* c, const char* nm, const void* src, size_t bytes, int mem) { TGS_NOEXCEPT_BODY(c, debug_put_impl(c, nm, src, bytes, mem)) }
int tgs_debug_run_stage(tgs_ctx* c, const char* st) { TGS_NOEXCEPT_BODY(c, debug_run_stage_impl(c, st)) }

}  // extern "C"
