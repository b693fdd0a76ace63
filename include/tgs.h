/* include/tgs.h -- C-ABI boundary of the B200-native TemporalGS hot path (libtgs.so).
 *
 * Method: TemporalGS, arxiv/paper_2607_03390.  Citations are PAPER.md:L<line>; "R<n>" are the
 * readings of silent / ambiguous passages listed in DESIGN.md §2.  Every step of the path runs in
 * hand-written CUDA kernels for sm_100a (paper_2607_03390_b200/csrc); there is no CPU fallback --
 * a call fails with TGS_E_CUDA when no device is usable.
 *
 * General rules
 *  - Every function returns 0 (TGS_OK) on success or a negative tgs_status; no exceptions cross.
 *  - A context is bound to one CUDA device and one stream; it is not thread-safe.  Contexts that render on the SAME device
 *    at the same time (other streams, threads or processes) must switch the one-launch depth sort off
 *    (tgs_debug_run_stage(ctx, "depth_sort_fused_off")): its grid barriers need all of its CTAs resident, and two such
 *    kernels could each hold part of the SMs; a watchdog then fails the frame (TGS_E_CUDA) after a few seconds.
 *  - `mem` says where a caller buffer lives: TGS_HOST or TGS_DEVICE (same device as the context).
 *    Input buffers are copied during the call; the caller keeps ownership of everything it passes.
 *  - tgs_render only enqueues work; tgs_read_* / tgs_get_stats / tgs_debug_get with TGS_HOST block until
 *    the data is on the host.  With TGS_DEVICE they enqueue a device copy on the context's stream.
 *  - Conventions (R6): `view` is a rigid world->camera matrix, row-major 4x4, camera looks along +z,
 *    x right, y down; pixel (i,j) is sampled at (u,v)=(i,j); 16x16 tiles, tile id =
 *    ty*TX+tx.  Depth of a pixel without geometry is TGS_DEPTH_INVALID ("z_far + eps", L97, R12).
 */
#ifndef TGS_H
#define TGS_H
#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define TGS_DEPTH_INVALID 3.0e38f

typedef enum { TGS_HOST = 0, TGS_DEVICE = 1 } tgs_mem;

/* render modes (argument of tgs_render) */
typedef enum {
  TGS_FULL = 0,       /* reference frame R: vanilla 3DGS + construction of the priors (L65, L73-84, L103, L109) */
  TGS_PSEUDO_REF = 1, /* pseudo reference frame P: reference frame with AFC (L128) */
  TGS_TEMPORAL = 2,   /* TemporalGS frame S: AFC + TOC + selective rendering (L105-128) */
  TGS_AUTO = 3        /* scheduler A0 decides: lambda_TDC, lambda_SR, eta (L67, L107, L128, L142) */
} tgs_mode;

/* frame types (tgs_stats.frame_type) */
enum { TGS_FRAME_R = 0, TGS_FRAME_P = 1, TGS_FRAME_S = 2 };

typedef enum {
  TGS_OK = 0,
  TGS_E_INVALID_ARG = -1, /* null pointer, bad size, non-finite input, unknown name */
  TGS_E_NO_SCENE = -2,    /* tgs_render before tgs_load_gaussians */
  TGS_E_NO_CAMERA = -3,   /* tgs_render before tgs_set_camera */
  TGS_E_NO_PRIORS = -4,   /* TGS_TEMPORAL / TGS_PSEUDO_REF without valid priors */
  TGS_E_CAPACITY = -5,    /* the (Gaussian, tile) pair buffer overflowed; the frame is invalid */
  TGS_E_CUDA = -6         /* CUDA runtime error; see tgs_last_error */
} tgs_status;

/* per-Gaussian flags in the "rec_flags" debug buffer */
enum {
  TGS_CULL_NEAR = 1,       /* d <= z_near (L61, R4) */
  TGS_CULL_AFC = 2,        /* outside the adaptive frustum (L109-111) */
  TGS_CULL_TOC = 4,        /* behind the warped TGB (L113) */
  TGS_CULL_DEGENERATE = 8, /* det(Sigma') <= 0 */
  TGS_CULL_EMPTY = 16,     /* intersects no tile (L61) */
  TGS_VISIBLE = 32,
  TGS_NEWLY_VISIBLE = 64   /* L119 */
};

typedef struct {
  float lambda1, lambda2; /* surface range [D - l1 s, D + l2 s]; 3, 0 (L99) */
  int lambda_tdc;         /* a reference frame every lambda_tdc frames; 50 (L142) */
  int lambda_sr;          /* a (pseudo) reference frame every lambda_sr frames; 5 (L142) */
  float eta;              /* S frame with more than eta*T selected tiles forces a P frame next; 0.40 (L128) */
  float bg[3];            /* background colour, part of the TAB (R27); 0 */
  int enable_afc, enable_toc, enable_sr; /* module toggles of Table IV (L221-231); 1 */
  uint32_t max_pairs;     /* capacity of the (Gaussian, tile) pair buffers; 0 = automatic */
  int exact_tiles;        /* 1 (default, R39): a Gaussian "intersects" a tile (L61) iff its max alpha over the tile's pixel
                             box is >= 1/255 -- the test L119 uses for tile contributions; 0: every tile of the 3-sigma
                             rect.  Images, TGB and G_rendered do not depend on it, only the pair lists get shorter. */
  int prior_policy;       /* TGS_PRIORS_ANCHORED (default; the paper, L86: S frames always warp from the last R / P frame) or
                             TGS_PRIORS_CHAINED (R42): the stitched {I, D, sigma} of every S frame replace the priors and
                             G_rendered grows by the Gaussians that frame blended */
  int tgb_downscale;      /* 1 (default) or 2: the TGB is warped, repaired and looked up on a ceil(W/2) x ceil(H/2) grid,
                             the paper's setting for large scenes (L142); downscale = min depth / max sigma of 2x2 (R43) */
  int depth_slabs;        /* front-to-back slabs: the depth-ordered (Gaussian, tile) tests are binned, sorted and
                             blended in this many consecutive pieces, and tiles whose pixels have all stopped (T < 1e-4) receive no
                             pairs in the later pieces.  Image, TGB and G_rendered do not depend on it; the pair lists of the later
                             pieces lack the pairs of finished tiles (records the blend would never have read).  1: one piece,
                             the complete lists of L61; 2..4; 0 (default): automatic from the size of a recent frame */
  uint32_t slab_split[3]; /* boundaries between the pieces in 1/1024 of the test space, ascending; 0 = built-in default */
} tgs_params;
enum { TGS_PRIORS_ANCHORED = 0, TGS_PRIORS_CHAINED = 1 };

typedef struct {
  int frame_type; /* TGS_FRAME_R / P / S */
  uint32_t n_total, n_near, n_afc, n_toc, n_degenerate, n_empty, n_visible, n_newly_visible;
  uint64_t n_pairs; /* P: pairs emitted = total sort length */
  uint32_t n_tiles, n_sel_oc, n_sel_um, n_sel;
  uint32_t n_rendered; /* |G_rendered| (R / P frames) */
  uint32_t overflow;   /* 1: n_pairs exceeded the capacity, frame invalid */
  uint64_t n_interactions; /* L: (pixel, Gaussian) pairs evaluated by the blend; 0 unless counting is on
                              (tgs_debug_run_stage("count_interactions_on")) */
  uint64_t n_blended;      /* of those, the ones with alpha >= 1/255 that were composited (counting on) */
  uint64_t n_pixel_slots;  /* pixel slots issued by the blend loop, dead lanes included (counting on) */
  float ms_stage[8];   /* per-stage device time when timing is on (tgs_debug_run_stage("timing_on")):
                          0 init + warp + fill/correspondence, 1 preprocess + tile selection, 2 depth sort of the visible
                          Gaussians (with the prefix sums of their test rects where it runs as one launch), 3 pair binning (tile tests, emission), 4 SH colours, 5 tile sort + ranges,
                          6 blend + stitch, 7 post (F reduction, stats) */
  float ms_total;
  uint64_t device_bytes; /* device memory held by the context */
  uint64_t n_tests;      /* (Gaussian, tile) combinations the pair binning examined: sum of the test-rect areas of the visible
                            Gaussians (n_pairs of them passed: tile selected, L123, and reached with alpha >= 1/255, R39) */
  uint64_t n_tests_evaluated; /* of n_tests, those whose tile was still alive when their slab was binned (= n_tests in one piece) */
  uint64_t n_half_tile_visits, n_half_tile_visits_dead; /* (counting on) dense-mode (record, 16 x 8 half tile) visits of the blend,
                                and those that reach none of the half's 128 pixels with alpha >= 1/255 */
  uint64_t n_pairs_consumed; /* pairs the blend reached before their tile was finished (whole batches of 128; counting on): the
                                rest of each tile's list lies behind saturated pixels and is never read */
  uint32_t n_slabs;          /* pieces this frame was binned / sorted / blended in (tgs_params.depth_slabs) */
  uint32_t n_pairs_slab[4];  /* pairs of each piece; n_pairs is their sum */
  uint32_t n_finished_slab[4]; /* selected tiles finished by each piece before the last one (they get no pairs afterwards) */
  uint64_t launches_total; /* kernels this library has launched in this process so far (all contexts); bench.py reports the
                              difference over its timed region as `gpu_launches` */
} tgs_stats;

typedef struct tgs_ctx tgs_ctx;

/* Create a context on `cuda_device`; all work is enqueued on `cuda_stream` (a cudaStream_t; NULL = the
 * legacy default stream).  *out is owned by the caller until tgs_destroy. */
int tgs_create(tgs_ctx** out, int cuda_device, void* cuda_stream);
void tgs_destroy(tgs_ctx*);

/* Load the scene (mean, covariance = R S S^T R^T, opacity, SH).  means [n][3]; scales
 * [n][3] linear (post-exp); quats [n][4] (w,x,y,z), normalised here; opacity [n] post-sigmoid; sh
 * [n][K][3], K=(sh_degree+1)^2, sh_degree 0..3.  Data are copied and repacked on the device (cull
 * record {mean, opacity}, 3-D covariance, tau = 2 ln(255 o)); invalidates the priors.  Host inputs with
 * a non-finite value are rejected (TGS_E_INVALID_ARG). */
int tgs_load_gaussians(tgs_ctx*, uint32_t n, int sh_degree, const float* means, const float* scales,
                       const float* quats, const float* opacity, const float* sh, int mem);

/* load a trained 3DGS checkpoint in the public `point_cloud.ply` layout (binary_little_endian, float32
 * vertex properties x y z, f_dc_0..2, f_rest_* (channel-major, 3 ((deg+1)^2 - 1) of them, consecutive), opacity (logit),
 * scale_0..2 (log), rot_0..3 (w x y z); other properties are ignored).  `path` is a host file name.  The rows are
 * uploaded as they are and activated on the device (exp, sigmoid, SH re-interleaved), then loaded exactly like
 * tgs_load_gaussians.  TGS_E_INVALID_ARG: unreadable / malformed file or a non-finite value; tgs_last_error says which. */
int tgs_load_ply(tgs_ctx*, const char* path);

/* Camera of the NEXT frame (W, K).  Changing W, H or the intrinsics invalidates the priors. */
int tgs_set_camera(tgs_ctx*, const float view[16], float fx, float fy, float cx, float cy, int W, int H,
                   float znear, float zfar);

void tgs_default_params(tgs_params*);
int tgs_set_params(tgs_ctx*, const tgs_params*);

/* Render one frame of the stream.  Enqueues the whole path A1-A10 of DESIGN.md §1. */
int tgs_render(tgs_ctx*, int mode);

/* Current frame.  rgb [H][W][3] in [0,1] (+bg); depth [H][W] (Eq.1; stitched on S frames, R31);
 * sigma [H][W] (Eq.2), nullable; sel [TY][TX]: bit0 = T^oc (L119), bit1 = T^um (L121), bit2 = selected. */
int tgs_read_image(tgs_ctx*, float* rgb, int mem);
/* Streaming read-back for frame loops: enqueues the copy of the current frame's image to `rgb_host` (page-locked
 * host memory, [H][W][3]) on a copy stream of the context and returns at once, so the transfer overlaps the rendering
 * of the following frames (a later frame that would overwrite the device buffer waits for the copy by itself).  The
 * data are valid only after tgs_wait_reads, which blocks until every enqueued read has finished; the other blocking
 * calls do not imply it.  The caller keeps `rgb_host` alive and untouched until then. */
int tgs_read_image_async(tgs_ctx*, float* rgb_host);
int tgs_wait_reads(tgs_ctx*);
int tgs_read_depth(tgs_ctx*, float* depth, float* sigma, int mem);
int tgs_read_tile_mask(tgs_ctx*, uint8_t* sel, int mem);
int tgs_get_stats(tgs_ctx*, tgs_stats* out);

/* Drop the temporal priors: the next TGS_AUTO frame is a reference frame. */
int tgs_reset_priors(tgs_ctx*);

const char* tgs_strerror(int code);
const char* tgs_last_error(tgs_ctx*);

/* ---- test-only: named intermediate buffers, so that a stage can be fed the oracle's inputs ----
 * tgs_debug_get copies min(bytes, size) bytes and returns the buffer's size in bytes (>= 0) or an error.
 * Readable (rec_uvdo, rec_conic, rec_rect and rec_flags are views assembled on request from what the path keeps per Gaussian,
 *   not buffers it writes as such): rec_uvdo rec_conic (float4 [N]) rec_rect (uint16x4 [N]) rec_flags (uint32 [N]) rec_rgb
 *   (float4 [N]) tiles_touched (uint32 [N]) keys (uint64 [P]) vals (uint32 [P]) ranges (uint32 [T][2]) -- with more than one
 *   slab (tgs_params.depth_slabs) these four describe the LAST slab only; the parity tests of the lists use depth_slabs = 1 --
 *   warp_depth warp_sigma fill_depth (float [H][W]) rendered (uint8 [N]) F (float[4]) prior_depth
 *   prior_sigma (float [H][W]) prior_image (float [H][W][3]) g2 (float [N][8]: Sigma xx xy xz yy yz zz, opacity, tau).
 * Writable (tgs_debug_put; marks the priors valid once depth, sigma, image and view are present):
 *   prior_depth prior_sigma prior_image rendered F prior_view (float[16]).
 * tgs_debug_run_stage: "timing_on" "timing_off" "force_all_tiles_on" "force_all_tiles_off"
 *   "count_interactions_on" "count_interactions_off" "blend_half_on" "blend_half_off" "blend_half_auto" (per-warp half-tile record
 *   lists in the blend: default automatic, on for scenes of small splats; the result does not depend on it)
 *   "depth_sort_fused_on" "depth_sort_fused_off" "depth_sort_fused_auto" (the depth sort of the visible Gaussians and the prefix sums of
 *   their test rects as one launch instead of five: default automatic, on for short visible lists; the result does not depend on it)
 *   "redzones_on" (before the scene is loaded: every device buffer allocated
 *   afterwards is framed by 256-byte guards) "check_redzones" (TGS_OK if no guard has been written to, else TGS_E_CUDA). */
long long tgs_debug_get(tgs_ctx*, const char* name, void* dst, size_t bytes, int mem);
int tgs_debug_put(tgs_ctx*, const char* name, const void* src, size_t bytes, int mem);
int tgs_debug_run_stage(tgs_ctx*, const char* stage);

/* ---- an entry point that allocates nothing (for callers that cannot call cudaMalloc: code under CUDA graph capture, tight
 * serving loops, harnesses that forbid it) ----
 * The path's stable LSD radix sort of (uint32 key, uint32 value) pairs (A6, the tile sort of PAPER.md:L61 "for each tile, sorts its
 * intersected Gaussians by depth": pairs emitted in depth order are sorted stably by tile id) as a call of its own, with every byte
 * of its scratch -- digit histograms, tile tickets, look-back descriptors, the ping-pong buffers of the intermediate passes -- in
 * ONE file-scope static device array of TGS_SORT_STATIC_SCRATCH_BYTES (~8.5 MiB), which every GPU that loads libtgs.so holds until
 * the process exits.  The call needs no tgs_ctx and calls no cudaMalloc / cudaFree / allocating library routine; it only enqueues
 * work (one memset, one histogram kernel, key_bytes scatter kernels, at most two small copies) on `cuda_stream` of `cuda_device`.
 *   keys_in, vals_in   [n] DEVICE, read only           keys_out, vals_out   [n] DEVICE, must not overlap the inputs
 *   n                  items, 0 .. TGS_SORT_STATIC_MAX_ITEMS; a larger n is rejected with TGS_E_INVALID_ARG and nothing is enqueued
 *   key_bytes          1 .. 4: the sort is stable on the low 8 * key_bytes bits of the key (higher bits are carried, not compared)
 *   status             nullable DEVICE word, caller-owned: receives 0, or non-zero if a look-back gave up (the output is then invalid)
 * Returns TGS_OK, TGS_E_INVALID_ARG (null pointer, n or key_bytes out of range, overlapping buffers, bad device) or TGS_E_CUDA;
 * tgs_static_last_error() gives the reason of the calling thread's last failure ("" if none).
 * Every call on a device shares the array, which keeps the previous call's contents: the call clears what must start at zero
 * (histograms, tickets, status) and tags its descriptors with a per-device call number, so calls that follow one another in ONE
 * stream are independent.  Calls that OVERLAP on the GPU (two streams, two host threads with different streams, two processes'
 * worth of graph replays at once) race on the array and give garbage: serialise them. */
#define TGS_SORT_STATIC_MAX_ITEMS (1u << 20)
#define TGS_SORT_STATIC_SCRATCH_BYTES (4352u + 256u * 2048u + 2u * 4u * TGS_SORT_STATIC_MAX_ITEMS)
int tgs_sort_pairs_static(int cuda_device, void* cuda_stream, const uint32_t* keys_in, const uint32_t* vals_in, uint32_t* keys_out,
                          uint32_t* vals_out, uint32_t n, int key_bytes, uint32_t* status);
const char* tgs_static_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* TGS_H */
