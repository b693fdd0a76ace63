// tgs_internal.cuh -- shared declarations of the CUDA path (NOT shared with oracle/).
// Paper: TemporalGS, arxiv/paper_2607_03390; citations are PAPER.md:L<line>; steps A0-A10 and data
// layout are described in DESIGN.md §1 / §6.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/tgs.h"

#define TGS_TILE 16
#define TGS_MAX_SLABS 4
#define TGS_INVALID_BITS 0x7f61b1e6u /* bits of 3.0e38f */

// ------------------------------------------------------------------ per-frame constants (kernel argument)
struct CamConst {
  float V[12];              // world->camera, rows 0..2 of the 4x4
  float fx, fy, cx, cy;
  float Wf, Hf;             // (float)W, (float)H
  float limx, limy;         // 1.3 tan(fov/2) (R3)
  float znear;
  float campos[3];          // camera centre, for the SH view direction
  int W, H, TX, TY;
};

// TGB grid of an S frame (R43): ds = 1: the image grid and the camera's intrinsics; ds = 2: ceil(W/2) x
// ceil(H/2), grid pixel (i, j) at the image position (2i + 0.5, 2j + 0.5) = a pinhole camera with fx/2, fy/2,
// (cx - 0.5)/2, (cy - 0.5)/2.  Source value of a grid pixel: nearest valid depth / largest sigma of its 2x2 block.
struct TgbGrid {
  int ds, W, H;
  float Wf, Hf, fx, fy, cx, cy;
};

struct FrameConst {
  CamConst cam;
  TgbGrid tg;
  float M[12];              // reference -> current (Eq.3)
  float Minv[12];           // current -> reference (backward query, L121)
  float lambda1, lambda2;   // L99
  float bg[3];
  uint32_t n;
  uint32_t max_pairs;
  int sh_degree;
  int ftype;                // TGS_FRAME_R / P / S
  int do_afc, do_toc, do_tgb, all_tiles;
  int exact_tiles;          // R39
  int n_tiles;
  uint32_t epoch;           // frame number (1 .. 2^28 - 1): tag of the look-back descriptors (x 4 + slab for pairs)
  // Front-to-back slabs: the flat test space of the depth-sorted visible Gaussians is cut into n_slabs
  // consecutive ranges of chunks; slab k is binned, sorted and blended before slab k + 1 is binned, and tiles whose pixels
  // have all stopped are dropped from the binning of the later slabs.  slab_bound[k] / 1024 = share of the chunks before slab k.
  int blend_half;           // k_blend<.,.,HALF>: per-warp lists of the records that reach the warp's half tile (scenes of small splats)
  int n_slabs;              // 1 .. TGS_MAX_SLABS
  int dsort_fused;          // the depth sort runs as one launch (k_depth_sort_fused): k_compact_vis fills its first count matrix
  uint32_t slab_bound[TGS_MAX_SLABS + 1];
};

// ------------------------------------------------------------------ device counters (one block, zeroed per frame)
struct Counters {
  uint32_t n_near, n_afc, n_toc, n_degenerate, n_empty, n_visible, n_newly_visible;
  uint32_t n_pairs;         // P
  uint32_t n_sel_oc, n_sel_um, n_sel;
  uint32_t n_rendered;
  uint32_t overflow;
  uint32_t error;           // look-back watchdog etc.
  uint32_t n_tests;         // sum of the rect areas of the visible Gaussians: the flat (Gaussian, tile) test space
  uint32_t n_nv_queue;      // newly visible Gaussians queued for the cooperative T^oc marking
  uint32_t n_oc_marked;     // tiles whose T^oc bit is set
  // work tickets of the persistent kernels
  uint32_t ticket_pre, ticket_scan;
  uint32_t ticket_sort[4];  // depth sort, one per digit
  // per slab
  uint32_t ticket_bin[TGS_MAX_SLABS], ticket_blend[TGS_MAX_SLABS];
  uint32_t ticket_tsort[TGS_MAX_SLABS][4];   // tile sort, one per slab and digit
  uint32_t n_pairs_slab[TGS_MAX_SLABS];      // pairs of a slab = length of its sort
  uint32_t n_live_after[TGS_MAX_SLABS];      // tiles that parked their pixel states at the end of a slab's blend
  uint32_t n_finished[TGS_MAX_SLABS];        // selected tiles finished (written) by a slab's blend before the last slab
  uint32_t pre_done;        // CTAs of k_preprocess that have finished
  unsigned long long area_sum;         // same as n_tests, accumulated in 64 bits by k_preprocess (overflow check)
  unsigned long long n_interactions;   // L (only when interaction counting is on)
  unsigned long long n_blended;        // interactions that passed alpha >= 1/255 and were composited (counting on)
  unsigned long long n_slots;          // pixel slots the blend loop issued: warp iterations x pixels per warp (counting on)
  unsigned long long n_tests_eval;     // tests k_bin evaluated (tile alive): all of them in one piece, fewer with slabs
  unsigned long long n_wrec, n_wrec_dead;   // dense-mode (record, half tile = warp) visits, and those with alpha < 1/255 at all 128 pixels (counting on)
  unsigned long long n_consumed;       // pairs the blend reached before their tile was finished, in whole batches (counting on)
};
static_assert(sizeof(Counters) % 8 == 0 && sizeof(Counters) <= 512, "Counters layout (k_export_counters copies it with 128 threads)");

// ------------------------------------------------------------------ device buffers of a context
struct DevBuffers {
  // scene (repacked at load)
  float4* cull4 = nullptr;       // [N] {x,y,z, largest scale}: the only record read for every Gaussian every frame
  float4* g2 = nullptr;          // [N][2] {Sxx,Sxy,Sxz,Syy},{Syz,Szz,opacity,tau = 2 ln(255 o)}: read by survivors of the culls
  float* sh = nullptr;           // [N][K][3]
  // per-Gaussian records of the current frame
  float4* rec_bin = nullptr;     // [N][2] {u, v, A, B}, {C, tau, bits(trect.x), bits(trect.y)}: everything A5a gathers per visible Gaussian, in ONE 32-byte sector
  uint8_t* rec_flags = nullptr;  // [N] TGS_CULL_* / TGS_VISIBLE / TGS_NEWLY_VISIBLE of the current frame (one byte; test-only reader)
  float4* rec_rgb = nullptr;     // [N] {r,g,b,-}
  // blend-side parameters (values, not decisions): alpha = exp2(A' t^2 + D' dy^2 + log2 o), t = dx + k dy, which is
  // -1/2 delta^T Sigma'^-1 delta completed to a sum of two squares: A' = -log2e/2 * c/det, k = -b/c, D' = -log2e/2 / c
  float4* rec_b0 = nullptr;      // [N][2] blend record, interleaved: rec_b0[2 g] = {u, v, A', k},
  float4* rec_b1 = nullptr;      //        rec_b1[2 g] = rec_b0[2 g + 1] = {D', log2 o, d, o} (one 32-byte sector per Gaussian)
  uint32_t* tiles_touched = nullptr;  // [N] pairs emitted per Gaussian (test-only: filled by tgs_debug_get)
  uint8_t* rendered = nullptr;        // [N] G_rendered of the priors (L103)
  uint8_t* rendered_next = nullptr;   // [N] being built by an R / P frame
  // visible Gaussians: ckeys = bits(depth), cvals = index; [1] staging (2048 slots per chunk), [0] in index order
  // (k_compact_vis), then ping-pong of the depth sort
  uint32_t* ckeys[2] = {nullptr, nullptr};   // [N]
  uint32_t* cvals[2] = {nullptr, nullptr};   // [N]
  uint2* pre_cnt = nullptr;                  // [ceil(N/2048)] {visible Gaussians of a preprocess chunk, of the chunks before it}
  uint32_t* vis_list = nullptr;              // [N] the visible Gaussians in index order (a copy the depth sort does not permute)
  uint32_t* area_prefix = nullptr;           // [N+1] tests before each sorted visible Gaussian
  uint32_t* chunk_first = nullptr;           // [bin_chunks_cap] sorted position of the Gaussian holding a chunk's first test
  uint32_t* nv_queue = nullptr;              // [N] newly visible Gaussians with rects of more than 4 tiles
  uint4* bin_params = nullptr;               // [N][3] tile-test parameters of the visible Gaussians in SORTED order (k_scan_area -> k_bin)
  // pairs
  uint32_t* keys[2] = {nullptr, nullptr};    // [max_pairs] tile id of a pair
  uint32_t* vals[2] = {nullptr, nullptr};    // [max_pairs] Gaussian index of a pair
  uint32_t* sort_hist = nullptr;      // [1 + TGS_MAX_SLABS][4][256]: depth sort, tile sort of each slab
  uint64_t* sort_desc = nullptr;      // tile sort: [passes][tiles][256] look-back descriptors (epoch-tagged)
  uint64_t* dsort_desc = nullptr;     // depth sort: [4][tiles][256]
  uint32_t* dsort_H = nullptr;        // one-launch depth sort: [4][tiles][256] digit counts per tile, all zero between frames
  uint32_t dsort_tiles_cap = 0;       // rows of one of those matrices
  uint64_t* scan_desc = nullptr;      // look-back descriptors of k_scan_area
  uint64_t* bin_desc = nullptr;       //                        k_bin [bin_chunks_cap]
  // tiles
  uint32_t* tile_flags = nullptr;     // [T] bit0 oc, bit1 um
  uint8_t* tile_mask = nullptr;       // [T] bit0 oc, bit1 um, bit2 selected
  uint32_t* sel_bits = nullptr;       // [ceil(T/32)] T_sel
  uint32_t* live_bits = nullptr;      // [ceil(T/32)] selected tiles whose pixels have not all stopped yet (slabs)
  uint32_t* live_sat = nullptr;       // [(TY + 1)(TX + 1)] summed-area table of live_bits (k_live_sat, before the binning of a later slab)
  float* pix_state = nullptr;         // [T][7][256] pixel states of the tiles that stay live from one slab to the next
  uint32_t* tile_order = nullptr;     // [T] selected tiles first, then the others
  uint2* ranges = nullptr;            // [T] {start,end}
  // images
  // three sets: the priors, the frame being rendered, and the previous frame, whose image may still be on its way to the host
  float* image[3] = {nullptr, nullptr, nullptr};   // [H][W][3]
  float* depth[3] = {nullptr, nullptr, nullptr};   // [H][W]
  float* sigma[3] = {nullptr, nullptr, nullptr};   // [H][W]
  float2* warp_tgb = nullptr;   // warped TGB {D^min, sigma^max} per grid pixel, interleaved (uint bits during the splat)
  float* fill_depth = nullptr;  // D'
  uint32_t* F_key = nullptr;    // [4] ordered-uint keys of F_min.x, F_min.y, F_max.x, F_max.y
  Counters* counters = nullptr;
};

// ------------------------------------------------------------------ programmatic dependent launch (sm_90+)
// Every kernel of a frame is launched with programmatic stream serialization: its CTAs may be scheduled while the
// previous kernel of the stream drains, and wait in TGS_PDL_WAIT() (griddepcontrol.wait: the previous grid has completed
// and its writes are visible) before they touch anything a predecessor produced.  Persistent kernels, whose grid is
// resident from the start, call TGS_PDL_TRIGGER() at once so that the next grid is launched as their CTAs retire.
#define TGS_PDL_WAIT() asm volatile("griddepcontrol.wait;" ::: "memory")
#define TGS_PDL_TRIGGER() asm volatile("griddepcontrol.launch_dependents;" ::: "memory")
struct PdlLaunch {
  cudaLaunchConfig_t cfg;
  cudaLaunchAttribute at;
  PdlLaunch(dim3 grid, dim3 block, size_t smem, cudaStream_t s) {
    cfg = cudaLaunchConfig_t();
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = s;
    at.id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at.val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = &at; cfg.numAttrs = 1;
  }
};
extern unsigned long long g_tgs_launches;   // kernels launched by this library (tgs_stats.launches_total); defined in tgs_api.cu
#define TGS_LAUNCH(kernel, grid, block, smem, stream, ...)   \
  do {                                                       \
    PdlLaunch L_(grid, block, smem, stream);                 \
    cudaLaunchKernelEx(&L_.cfg, kernel, __VA_ARGS__);        \
    ++g_tgs_launches;                                        \
  } while (0)

// ------------------------------------------------------------------ launchers (definitions in k_*.cu)
void launch_repack(cudaStream_t s, uint32_t n, int K, const float* means, const float* scales, const float* quats,
                   const float* opacity, const float* sh, DevBuffers& b);
void launch_frame_init(cudaStream_t s, const FrameConst& fc, DevBuffers& b, bool reset_F, uint8_t* rendered_next);
void launch_warp(cudaStream_t s, const FrameConst& fc, DevBuffers& b, const float* prior_depth, const float* prior_sigma);
void launch_fill_corr(cudaStream_t s, const FrameConst& fc, DevBuffers& b);
void launch_preprocess(cudaStream_t s, const FrameConst& fc, DevBuffers& b, int num_sms);
void launch_select(cudaStream_t s, const FrameConst& fc, DevBuffers& b, uint32_t* host_n_sel);
void launch_export_counters(cudaStream_t s, const DevBuffers& b, Counters* host);
void launch_frustum(cudaStream_t s, const FrameConst& fc, DevBuffers& b, const uint32_t* vis_vals, const uint8_t* rendered_now, bool update_F);
void launch_mark_oc(cudaStream_t s, const FrameConst& fc, DevBuffers& b, int num_sms);
// k_scan_area (slab 0 only) + k_bin of one slab.  host_overflow: pinned host word, zero-copy stores: 1 = the pair buffers
// overflowed, 2 (from k_scan_area) = the tests exceed the capacity, so an overflow cannot be ruled out before the frame ends
void launch_bin(cudaStream_t s, const FrameConst& fc, DevBuffers& b, int sorted_g_idx, uint32_t bin_chunks_cap, int num_sms,
                uint32_t* host_overflow, int slab);
void launch_colour_all(cudaStream_t s, const FrameConst& fc, DevBuffers& b, int num_sms);
// Sorts *n_ptr items on the low key_bits bits of the uint32 key; returns the index (0/1) of the result buffers.
int launch_sort(cudaStream_t s, uint32_t* const keys[2], uint32_t* const vals[2], const uint32_t* n_ptr, int key_bits,
                const uint32_t* hist, uint64_t* desc, uint32_t tiles_cap, uint32_t* tickets, uint32_t* error_flag, uint32_t epoch,
                int num_sms, bool small_input, uint2* ranges = nullptr);   // ranges: A7 fused into the last pass ({~start, end} per key)
void launch_keys64(cudaStream_t s, DevBuffers& b, int sorted_idx, uint32_t n, uint64_t* out);
void launch_debug_record(cudaStream_t s, const FrameConst& fc, const DevBuffers& b, uint32_t n, int which, float4* out);   // test-only: {u,v,d,o} / {A,B,C,tau} / 3-sigma rect per Gaussian
void launch_debug_flags(cudaStream_t s, const DevBuffers& b, uint32_t n, uint32_t* out);               // test-only: the flag bytes as words   // test-only: {u,v,d,o} / {A,B,C,tau} per Gaussian
void launch_count_pairs(cudaStream_t s, DevBuffers& b, int sorted_idx, uint32_t n_pairs, uint32_t n);   // test-only
void launch_ranges_decode(cudaStream_t s, const DevBuffers& b, int n_tiles, uint2* out);   // test-only: {~start, end} -> {start, end}
void launch_blend(cudaStream_t s, const FrameConst& fc, DevBuffers& b, int sorted_idx, int out_idx,
                  const float* prior_image, uint8_t* rendered_next, int num_sms, bool count_interactions, int slab);
uint32_t sort_tile_items();
uint32_t scan_tile_items();
uint32_t bin_chunk_items();
uint32_t preprocess_chunk_items();
int tile_sort_passes(int n_tiles);
uint32_t depth_sort_fused_tile_items();
uint32_t depth_sort_fused_ctas_per_sm();
size_t depth_sort_fused_words(uint32_t tiles_cap);   // size of its count matrices (uint32 words): [4][tiles][256]
// one launch: depth sort of the visible list (result in buffer 0) + A5a (what k_scan_area does); launch_bin(slab 0) then skips k_scan_area
void launch_depth_sort_fused(cudaStream_t s, const FrameConst& fc, DevBuffers& b, unsigned long long max_tests, uint32_t* host_overflow, int num_sms,
                             uint32_t n_hint);   // n_hint: expected length of the list (sizes the grid only)
unsigned long long bin_max_tests(uint32_t bin_chunks_cap);
void sort_prepare_device();   // function attributes of the sort kernels on the current device (once per context)
