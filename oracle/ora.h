/* oracle/ora.h -- C interface of the TemporalGS CPU oracle.
 *
 * TEST INFRASTRUCTURE ONLY.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may load this library.  It shares no code with the CUDA path
 * (paper_2607_03390_b200/csrc, include/tgs.h); the constants below are restated, not included.
 *
 * Citations are PAPER.md:L<line> (+ section / equation); "R<n>" are the readings of silent or
 * ambiguous passages listed in DESIGN.md §2.
 */
#ifndef ORA_H
#define ORA_H
#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define ORA_DEPTH_INVALID 3.0e38f /* z_far + eps sentinel, PAPER.md:L97 (R12) */

/* render modes */
enum { ORA_FULL = 0, ORA_PSEUDO_REF = 1, ORA_TEMPORAL = 2, ORA_AUTO = 3 };
/* frame types returned by ora_render / stats.frame_type: R, P, S */
enum { ORA_FRAME_R = 0, ORA_FRAME_P = 1, ORA_FRAME_S = 2 };
/* error codes */
enum { ORA_OK = 0, ORA_E_INVALID_ARG = -1, ORA_E_NO_SCENE = -2, ORA_E_NO_CAMERA = -3, ORA_E_NO_PRIORS = -4 };

/* per-Gaussian flags of a record */
enum {
  ORA_CULL_NEAR = 1,       /* d <= z_near, PAPER.md:L61 (R4) */
  ORA_CULL_AFC = 2,        /* outside [F_min, F_max] */
  ORA_CULL_TOC = 4,        /* behind the warped TGB */
  ORA_CULL_DEGENERATE = 8, /* det(Sigma') <= 0 */
  ORA_CULL_EMPTY = 16,     /* touches no tile */
  ORA_VISIBLE = 32,        /* survived every cull */
  ORA_NEWLY_VISIBLE = 64
};

typedef struct {
  float lambda1, lambda2; /* 3, 0  */
  int lambda_tdc;         /* 50 */
  int lambda_sr;          /* 5 */
  float eta;              /* 0.40 */
  float bg[3];            /* background colour (R27) */
  int enable_afc, enable_toc, enable_sr; /* Table IV toggles */
  int exact_tiles;        /* 1: a Gaussian "intersects" a tile iff max alpha over the tile's pixel box >= 1/255
                             (R39, same box test as L119); 0: every tile of the 3-sigma rect (vanilla 3DGS) */
  int prior_policy;       /* 0 ANCHORED (paper, L86: priors always come from the last R / P frame); 1 CHAINED (R42): the
                             stitched outputs of every S frame replace the priors, G_rendered grows by what it blended */
  int tgb_downscale;      /* 1 (default) or 2: TGB warped, repaired and looked up on a (W/2) x (H/2) grid (L142, R43) */
} ora_params;

typedef struct {        /* 80 bytes */
  float u, v, d, o;     /* 2-D mean (pixels), depth, opacity */
  float A, B, C, tau;   /* conic (inverse of Sigma') as fp32 decision values; tau = 2 ln(255 o) */
  float ca, cb, cc, pad0; /* Sigma' = [[ca, cb], [cb, cc]] (with the 0.3 dilation), fp32 */
  float r, g, b;        /* colour (value arithmetic, computed in double) */
  float radius;         /* ceil(3 sqrt(lambda_max)) */
  uint16_t x_lo, x_hi, y_lo, y_hi; /* tile rect, hi exclusive */
  uint32_t flags;
  uint32_t tiles_touched; /* number of SELECTED tiles in the rect (= pairs emitted) */
} ora_record;

typedef struct {
  int frame_type;
  uint32_t n_total, n_near, n_afc, n_toc, n_degenerate, n_empty, n_visible, n_newly_visible;
  uint64_t n_pairs;
  uint32_t n_tiles, n_sel_oc, n_sel_um, n_sel;
  uint32_t n_rendered;
  uint64_t n_interactions; /* L: pixel-Gaussian pairs iterated before termination */
  double ms_preprocess, ms_sort, ms_blend, ms_temporal, ms_total;
} ora_stats;

typedef struct ora_ctx ora_ctx;

ora_ctx* ora_create(void);
void ora_destroy(ora_ctx*);
int ora_load_gaussians(ora_ctx*, uint32_t n, int sh_degree, const float* means, const float* scales,
                       const float* quats, const float* opacity, const float* sh);
int ora_set_camera(ora_ctx*, const float view[16], float fx, float fy, float cx, float cy, int W, int H,
                   float znear, float zfar);
int ora_set_params(ora_ctx*, const ora_params*);
void ora_default_params(ora_params*);
int ora_render(ora_ctx*, int mode); /* >= 0: frame type; < 0: error */
int ora_read_image(ora_ctx*, float* rgb /*[H][W][3]*/);
int ora_read_depth(ora_ctx*, float* depth /*[H][W]*/, float* sigma /*nullable*/);
int ora_read_tile_mask(ora_ctx*, uint8_t* sel /*[TY][TX], bit0 = oc, bit1 = um*/);
int ora_get_stats(ora_ctx*, ora_stats*);
int ora_reset_priors(ora_ctx*);
/* force all tiles selected on the next S frames (pin P9) */
int ora_force_all_tiles(ora_ctx*, int on);

/* named intermediates; returns the number of bytes the buffer holds (copying min(bytes, that)),
 * or a negative error.  Names: records keys vals ranges warp_depth warp_sigma fill_depth corr_xy
 * matched rendered rendered_sure rendered_maybe borderline F prior_depth prior_sigma prior_image
 * prior_view M Minv cov3d */
long long ora_get(ora_ctx*, const char* name, void* dst, size_t bytes);
/* overwrite a prior buffer (prior_depth prior_sigma prior_image rendered F prior_view); marks priors valid */
int ora_put(ora_ctx*, const char* name, const void* src, size_t bytes);
/* run single stages on the current state (pins P7, P8): "warp", "fill" */
int ora_stage(ora_ctx*, const char* stage);

/* ---- pure functions, exported for the pins ---- */
/* real SH basis Y_0..Y_{K-1} at unit direction dir (R5) */
void ora_sh_basis(int degree, const double dir[3], double* Y);
/* min over the pixel-centre box [x0,x1]x[y0,y1] of A dx^2 + 2B dx dy + C dy^2, (dx,dy) = p - (u,v);
 * fp32, fixed operation order (R18) */
float ora_box_qmin(float u, float v, float A, float B, float C, float x0, float x1, float y0, float y1);
/* scheduler (R9, R23): state = {since_R, since_ref, force_P, valid};
 * returns the frame type and advances the counters; call ora_schedule_feedback after an S frame. */
typedef struct { int since_R, since_ref, force_P, valid; } ora_sched;
int ora_schedule_next(ora_sched*, int lambda_tdc, int lambda_sr);
void ora_schedule_feedback(ora_sched*, int frame_type, uint32_t n_sel, uint32_t n_tiles, float eta);

#ifdef __cplusplus
}
#endif
#endif
