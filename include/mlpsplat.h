/* mlpsplat.h -- C ABI of the B200-native MLP-Splatting forward render
 * (arxiv/paper_2606_03877; BASELINE.json north_star = NS).  P:NN = PAPER.md line NN.
 *
 * The library renders a scene of N spatially bounded primitives, each an independent
 * compact MLP (Sec.3 / 3.1): per camera ray it finds the ray/ellipsoid support
 * intervals, takes K midpoint samples in each, evaluates the hit primitive's own MLP at
 * every sample (positional encoding P:101 Eq.5 -> Linear+ReLU -> rgb = sigmoid,
 * sigma = softplus P:105) and alpha-composites all samples of the ray front to back,
 * alpha = 1 - exp(-sigma*delta), C = sum_j T_j alpha_j c_j (Eq.6
 * Eq.14), stopping once T < t_stop.  Stages (NS (a)-(e)): projection + tile keys,
 * device radix sort, per-tile intersection, grouped per-primitive MLP (fp32 SIMT or bf16
 * tcgen05 tensor cores), per-ray merge + composite.  DESIGN.md Sec.1 lists every reading
 * of the paper this ABI fixes (Q1-Q27); Sec.2 the canonical fp32 order of the geometry.
 *
 * Conventions
 *  - Every function returns MS_OK (0) or a negative MS_ERR_*; nothing aborts, throws or prints.
 *  - "host" / "device" on a pointer says where the memory lives.  Inputs of ms_scene_create
 *    are host pointers and are copied; the caller keeps ownership.  Render outputs are
 *    DEVICE pointers owned by the caller (ms_render_host: host pointers).
 *  - One CUDA device (the current one at ms_scene_create); there is no CPU fallback.
 *  - A scene handle is not thread-safe; use one handle per host thread / stream.
 */
#ifndef MLPSPLAT_H
#define MLPSPLAT_H
#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum {
  MS_OK = 0,
  MS_ERR_INVALID_ARG = -1,       /* NULL / out-of-range argument, zero quaternion, scale <= 0 */
  MS_ERR_OUT_OF_MEMORY = -2,     /* host or device allocation failed */
  MS_ERR_CUDA = -3,              /* a CUDA call or kernel failed (ms_error_string has no detail; see ms_last_cuda_error) */
  MS_ERR_UNSUPPORTED_SHAPE = -4, /* MLP shape / key width outside what the kernels cover */
  MS_ERR_CAPACITY = -5           /* a caller-provided debug buffer is too small (*n holds the need) */
};

typedef struct ms_scene ms_scene; /* opaque; owns every device allocation it makes */

/* Primitive parameterisation: centre mu, unit quaternion q, ellipsoid semi-axes s.
 * The support of primitive i is { x : |x - mu|^2_Lambda <= 1 }, Lambda = R(q) diag(s^2)^-1 R(q)^T
 * (Q5). */
typedef struct {
  int32_t n;           /* number of primitives, >= 1 */
  const float *center; /* host [n][3] */
  const float *quat;   /* host [n][4], order (w,x,y,z), Hamilton; normalised by the library (Q6) */
  const float *scale;  /* host [n][3], semi-axes > 0 */
} ms_prims;

enum { MS_F32 = 0, MS_BF16 = 1 };
enum { MS_MODE_LOCAL = 0, MS_MODE_CONTACT = 1 };

/* One MLP per primitive, all of the same shape.  Input (Q2,Q3,Q15):
 *   x = [u, sin(2^0 pi u), cos(2^0 pi u), ..., sin(2^(L-1) pi u), cos(2^(L-1) pi u)] [, d]
 * u = local coordinate of the sample in the primitive's unit-sphere frame (3 values; each
 * sin/cos block is 3 wide: x,y,z), d = unit world-frame ray direction.  in_dim = 3 + 6L (+3).
 * n_hidden x (Linear(width) + ReLU), then Linear(4 + n_feat): outputs [r,g,b,sigma,feat...];
 * rgb = sigmoid, sigma = softplus, feat linear (Q16).
 * weights: host float32 [n][P]; per primitive, for each layer in order: W[in][out] row-major
 * (input index slowest), then b[out].  P = sum(in*out + out).
 * dtype = MS_BF16 declares that the contractions run with bf16 operands on tensor cores:
 * weight matrices are rounded to bf16 (round-to-nearest-even; a no-op if already
 * representable), biases stay fp32 (Q18).  dtype = MS_F32 keeps everything fp32.
 *
 * mode = MS_MODE_CONTACT selects the paper's own interaction model (S:Sec.8(f) NEXT-1)
 * instead of the north-star's K samples per chord: ONE evaluation per (ray, primitive) hit, at
 * the soft contact point t* = max(d^T Lambda (mu - o) / d^T Lambda d, t_near), p* = o + t* d
 * (Eq.1-2).  Input x = gamma([d; delta]), delta = mu - p* (Eq.3-5): for scalar j of
 * (d_x,d_y,d_z,delta_x,delta_y,delta_z) and level l, x[2L j + 2l] = sin(2^l pi z_j),
 * x[2L j + 2l + 1] = cos(2^l pi z_j); in_dim = 12 L, no identity, use_viewdir must be 0.
 * alpha = (1 - exp(-sigma l)) g with l = the chord length of the ray inside the support and
 * g = exp(-falloff |p* - mu|^2_Lambda), falloff = 9/2 by default (readings of P:105); hits are
 * composited in the order of (t*, primitive id).  ms_opts.K must be 1.  Paths: fp32 for any shape;
 * the tensor path for dtype = MS_BF16 with the paper's shape (L = 6, width 32, two hidden layers, n_feat 0). */
typedef struct {
  int32_t n_freq;      /* L >= 0 */
  int32_t use_viewdir; /* 0 / 1 */
  int32_t n_hidden;    /* 1..4 */
  int32_t width;       /* hidden width, 1..128 (tensor path: 64 or 128) */
  int32_t n_feat;      /* 0..60 */
  int32_t dtype;       /* MS_F32 | MS_BF16 */
  const float *weights;
  size_t n_weights;    /* must equal n * P */
  int32_t mode;        /* MS_MODE_LOCAL | MS_MODE_CONTACT */
  float falloff;       /* MS_MODE_CONTACT: g = exp(-falloff |p* - mu|^2_Lambda), the reading of the "Gaussian falloff"
                          whose formula the paper omits (Q29).  MS_FALLOFF_DEFAULT = 9/2 puts the
                          support boundary |.|_Lambda = 1 at three standard deviations; 0 = no falloff; must be >= 0 */
} ms_mlp;
#define MS_FALLOFF_DEFAULT 4.5f

/* Pinhole camera (Q14): pixel (x,y), row 0 on top, looks along
 * d_cam = ((x+0.5-cx)/fx, (y+0.5-cy)/fy, 1); c2w = 3x4 row-major [R|t], camera axes
 * x right, y down, z forward; the ray is o = t, d = normalise(R d_cam). */
typedef struct {
  float fx, fy, cx, cy;
  float c2w[12];
  float t_near; /* >= 0; intervals are clipped to t >= t_near (Q13) */
} ms_camera;

enum { MS_PATH_AUTO = 0, MS_PATH_FP32 = 1, MS_PATH_BF16_TC = 2 };
enum {
  MS_FLAG_KEEP_DEBUG = 1, /* keep the intermediate buffers of the last view for ms_debug_* (tile lists, intervals) */
  MS_FLAG_STAGE_TIMES = 2, /* record CUDA events between stages (ms_last_stage_ms) */
  MS_FLAG_TILE_ORDER = 4,  /* MS_MODE_CONTACT only: composite every pixel of a tile in ONE shared order, that of the
                              contact points t*_{i,c} of the virtual ray through the tile centre (the
                              paper's approximation), instead of the exact per-ray order; the tile lists are
                              then sorted by (tile, t*_{i,c}, primitive id) */
  MS_FLAG_NO_SYNC = 16,    /* ms_render / ms_render_batch enqueue the whole view without ANY host synchronisation when the
                              previous synchronising view on this scene had the same H, W, tile, K, path and outputs and was
                              one band without depth waves: scratch is sized from that view (it carries 25 % of slack) and
                              every count stays on the device.  A view that needs more than that writes nothing valid:
                              ms_last_stats then returns MS_ERR_CAPACITY (stats.overflow = 1) and the next render sizes
                              again.  Ignored (the view synchronises as usual) when there is no such history, with
                              MS_FLAG_KEEP_DEBUG, or when depth waves are asked for or due. */
  MS_FLAG_OVERLAP = 32,    /* banded views: run stage (e) of band b on a second stream inside the library, beside stage
                              (d) of band b + 1 (the staging budget split into two halves that alternate).  The image
                              is bitwise the same and all work is ordered before whatever the caller enqueues next on
                              its stream.  Off by default: measured on CFG4, both stages contend for the same issue
                              slots and the view takes as long as without. */
  MS_FLAG_KEEP_ORDER = 8   /* stage (e) also records the order it composited every ray's samples in (4 B per sample)
                              for ms_debug_sample_order*: the order the product really used, not a re-derivation */
};

typedef struct {
  int32_t K;      /* midpoint samples per interval, 1..64 (NS (c)) */
  float t_stop;   /* early termination threshold on T (NS (e): 1e-4); 0 disables */
  int32_t tile;   /* tile edge in pixels: 8, 16 or 32; 0 = default 16 (Q10) */
  int32_t path;   /* MS_PATH_*; AUTO = BF16_TC when dtype is MS_BF16 and the shape is covered, else FP32 */
  void *stream;   /* cudaStream_t to enqueue on; NULL = the legacy default stream */
  int32_t flags;  /* MS_FLAG_* */
  int64_t band_bytes; /* Banded rendering (DESIGN.md Sec.6 "Bands and waves"; P:437 tile-local processing): the frame is
                     cut into bands of neighbouring tiles whose staged samples ((r,g,b,e) + features per sample) fill
                     about this many bytes, and stages (d), (e) run band by band on ONE staging buffer of that size,
                     which then lives in the L2 cache instead of HBM.  0 = MS_BAND_BYTES_DEFAULT; < 0 = one band
                     (staging of the whole frame).  The image does not depend on it. */
  int32_t waves;  /* Depth waves = early termination that skips MLP work ("early t[ermination]"): > 0 = a tile's
                     sorted list is evaluated in waves of `waves` entries (at most six, the last takes the rest), and before each
                     wave the rays that have already stopped (T < t_stop/2 over the samples in front of the wave) drop
                     their later intervals.  0 = MS_WAVES_AUTO: on when the previous view rendered on this scene
                     had rays stopping early, else off; < 0 = off.  The image does not depend on it. */
  float eye_guard; /* Q13: a support whose near depth z_lo <= eye_guard * r_z (it touches or nearly touches the eye
                     plane) is binned to the whole image instead of through the dual-conic bound, which degenerates
                     there.  <= 0 = MS_EYE_GUARD_DEFAULT (0.01). */
} ms_opts;
#define MS_BAND_BYTES_DEFAULT ((int64_t)1 << 30)
#define MS_WAVES_AUTO 0
#define MS_EYE_GUARD_DEFAULT 0.01f

typedef struct {
  int64_t n_visible;   /* primitives with a non-empty screen AABB */
  int64_t n_pairs;     /* (tile, primitive) keys */
  int64_t n_intervals; /* (ray, primitive) hits */
  int64_t n_samples;   /* n_intervals * K = MLP evaluations */
  int64_t n_blocks;    /* 128-sample row blocks fed to the MLP stage */
  int64_t scratch_bytes;
  int64_t n_launches;  /* kernels launched for this view (all stages) */
  int64_t n_samples_evaluated; /* samples whose MLP really ran: n_samples minus those of intervals dropped by the
                                  depth waves (rays already stopped) */
  int64_t n_dead_rays; /* rays the depth waves found stopped before their last hit */
  int64_t n_bands;     /* bands the frame was cut into */
  int64_t n_waves;     /* depth waves per band (1 = off) */
  int64_t staging_bytes; /* size of the staging buffers of stages (d) -> (e) */
  int64_t overflow;    /* MS_FLAG_NO_SYNC: 1 = the view did not fit the scratch sized from the previous one: invalid */
  int64_t no_sync;     /* 1 = the view was enqueued without host synchronisation */
} ms_stats;

enum { MS_STAGE_BIN = 0, MS_STAGE_SORT, MS_STAGE_ISECT, MS_STAGE_MLP, MS_STAGE_COMPOSITE, MS_N_STAGES };

/* Builds the device-resident scene: uploads primitives, derives per primitive (in canonical
 * fp32) A = diag(1/s) R^T and M = R diag(s), and packs the weights for the
 * MLP kernels.  Synchronises the device. */
int ms_scene_create(const ms_prims *prims, const ms_mlp *mlp, ms_scene **out);
/* Eq.7 slot features (S:Sec.8(f) NEXT-2), MS_MODE_CONTACT scenes with n_feat == 0 only:
 * attaches four slot embeddings per primitive, emb = host float32 [n][4][c_f] (copied), c_f a multiple
 * of 128, <= 512 (the paper: 512).  Renders then write out_feat[H][W][c_f]:
 *   u = clip_[-1,1]^3(R^T delta / s), g_k = softmax_k(a_k^T u) over the canonical tetrahedral frame
 *   a_k = (1,1,1), (1,-1,-1), (-1,1,-1), (-1,-1,1), each / sqrt(3); f = sum_k g_k e_k;
 *   F = sum_i T_i alpha_i f_i (the colour weights).  Synchronises the device. */
int ms_scene_set_slots(ms_scene *scene, int32_t c_f, const float *emb);

int ms_scene_destroy(ms_scene *scene);

/* Renders one view into DEVICE buffers out_rgb [H][W][3], out_alpha [H][W] and, if the MLP has
 * n_feat > 0 and out_feat != NULL, out_feat [H][W][n_feat]; all float32.  rgb / feat are
 * premultiplied sums (no background term, Q14); alpha = 1 - T.  Work is enqueued on
 * opts->stream; the call synchronises that stream internally to size its scratch buffers (after the pair count, after
 * the hit count, and after the band table when the view is cut into several bands), not at the end: outputs are ready
 * once the stream is.  With MS_FLAG_NO_SYNC and a matching previous view it does not synchronise at all. */
int ms_render(ms_scene *scene, const ms_camera *camera, int32_t H, int32_t W, const ms_opts *opts,
              float *out_rgb, float *out_alpha, float *out_feat);

/* n_views cameras (host array), outputs [n_views][H][W][...] (CFG5: 8 poses). */
int ms_render_batch(ms_scene *scene, const ms_camera *cameras, int32_t n_views, int32_t H, int32_t W,
                    const ms_opts *opts, float *out_rgb, float *out_alpha, float *out_feat);

/* Same as ms_render_batch with HOST output buffers (pinned or pageable): renders into
 * library-owned device buffers, copies the results back and synchronises the stream. */
int ms_render_host(ms_scene *scene, const ms_camera *cameras, int32_t n_views, int32_t H, int32_t W,
                   const ms_opts *opts, float *host_rgb, float *host_alpha, float *host_feat);

/* Backward pass of ms_render (S:Sec.8(f) NEXT-4; the losses of P:132-142 Eq.8-9 need dL/dtheta and dL/d(mu, s, q)):
 * given d_rgb = dL/d out_rgb (DEVICE [H][W][3]) it ADDS dL/dtheta_i into g_weights (DEVICE [n][P], the layout of
 * ms_mlp.weights), dL/dmu into g_center [n][3] and, if not NULL, dL/dq into g_quat [n][4] (q as given: the gradient is
 * tangent to q's sphere, q enters through q/|q|) and dL/ds into g_scale [n][3]; the caller zeroes them, several views
 * accumulate.  It renders the view first (stages (a)-(e), fp32 path, the whole frame staged, no early-stop waves) and
 * then walks C = sum_j T_j alpha_j c_j (Eq.6) backwards: compositing, activations, the Linear+ReLU
 * layers, Eq.5, the chord interval and its K midpoint samples, the frame A = diag(1/s) R(q)^T.  Samples behind
 * the early stop carry no gradient; a ReLU at exactly 0 has derivative 0; feature channels (n_feat) carry none (their
 * loss, Eq.9, is not built).  fp32 arithmetic with atomic accumulation (the sums' order is not fixed).
 * MS_MODE_LOCAL only, and MLPs whose activations of 128 samples fit shared memory (widths <= 64 at three hidden
 * layers): else MS_ERR_UNSUPPORTED_SHAPE.  Enqueued on opts->stream like ms_render. */
int ms_backward(ms_scene *scene, const ms_camera *camera, int32_t H, int32_t W, const ms_opts *opts,
                const float *d_rgb, float *g_weights, float *g_center, float *g_quat, float *g_scale);

/* Counts of the last view rendered on this scene.  Waits for that view to finish (its device counters).  Returns
 * MS_ERR_CAPACITY (with *out filled) if that view was a MS_FLAG_NO_SYNC view that overflowed its scratch. */
int ms_last_stats(ms_scene *scene, ms_stats *out);
/* Device time of each stage of the last view rendered with MS_FLAG_STAGE_TIMES, in ms,
 * ms[MS_N_STAGES].  Synchronises the recorded events. */
int ms_last_stage_ms(ms_scene *scene, float *ms);

/* Sum of the per-stage device times (ms_sum[MS_N_STAGES], ms) over every view rendered with
 * MS_FLAG_STAGE_TIMES since the last reset, and the number of views summed.  The library reads a
 * view's events at the start of the next render (or in this call): one event wait per view, on
 * work the next render has to wait for anyway.  reset != 0 clears the sums. */
int ms_stage_accum(ms_scene *scene, double *ms_sum, int64_t *n_views, int32_t reset);

/* ---- parity introspection: valid after a render with MS_FLAG_KEEP_DEBUG (last view) ---- */
/* Sorted tile lists: tile_offsets host [tiles+1], prim_ids / zbits host [cap]. */
int ms_debug_tile_lists(ms_scene *scene, int64_t *tile_offsets, int32_t *prim_ids, uint32_t *zbits,
                        size_t cap, size_t *n);
/* Per-ray hit lists in tile-list order: hit_offsets host [H*W+1]; prim / t_in / delta host [cap]. */
int ms_debug_intervals(ms_scene *scene, int64_t *hit_offsets, int32_t *prim, float *t_in, float *delta,
                       size_t cap, size_t *n);
/* Compositing order of one ray (pixel index y*W + x; all samples, not truncated) as stage (e) recorded it while
 * compositing (MS_FLAG_KEEP_DEBUG | MS_FLAG_KEEP_ORDER): prim / k / t host [cap]. */
int ms_debug_sample_order(ms_scene *scene, int32_t ray, int32_t *prim, int32_t *k, float *t,
                          size_t cap, size_t *n);
/* The same for every ray: prim / k host [cap] with cap >= n_samples; ray y*W + x owns the entries
 * [hit_offsets[ray] * K, hit_offsets[ray + 1] * K) (ms_debug_intervals), in compositing order. */
int ms_debug_sample_order_all(ms_scene *scene, int32_t *prim, int32_t *k, size_t cap, size_t *n);
/* Derived per-primitive frames, host [n][9] each (row-major A, M). */
int ms_debug_prim_frames(ms_scene *scene, float *A, float *M);

/* ---- the offset scan of stages (a), (c), (d) as entry points of its own ----
 * out[i] = sum of in[j], j < i, for i in [0, n]: n + 1 values (out[n] = the total), uint32 with wrap-around.
 * in: device [n]; out: device [n + 1]; they must not overlap.  Enqueued on `stream` (cudaStream_t; NULL = the legacy
 * default stream).
 *
 * ms_exclusive_scan_device: the path the render uses (ms_scan.cu: one CTA up to 32 768 counts, tiled above); it
 * allocates its scratch with cudaMalloc, synchronises the stream and frees it.
 *
 * ms_exclusive_scan_static: allocates NOTHING (no cudaMalloc / cudaFree, no allocating library call) and does not
 * synchronise: for callers under CUDA graph capture, in serving loops, or in harnesses that forbid allocation.  The
 * tile sums live in a file-scope device array of 65 KB that every GPU loading the library holds until exit; it covers
 * n <= MS_SCAN_STATIC_MAX, beyond that the call returns MS_ERR_CAPACITY and enqueues nothing.  Every call shares the
 * array (the scan writes each scratch word before reading it, so nothing is cleared between calls): calls that
 * overlap on the GPU -- different streams, concurrent graph replays -- race on it; serialise them.  The first call on
 * a device looks up the array's address (cudaGetSymbolAddress): make one call before starting a capture. */
#define MS_SCAN_STATIC_MAX (1u << 24)
int ms_exclusive_scan_device(const uint32_t *in, uint32_t *out, size_t n, void *stream);
int ms_exclusive_scan_static(const uint32_t *in, uint32_t *out, size_t n, void *stream);

/* Kernels the calling host thread has launched through this library so far (a running count; no synchronisation). */
int64_t ms_launch_count_total(void);

const char *ms_error_string(int code);
/* cudaError_t of the last failing CUDA call on this scene (0 if none). */
int ms_last_cuda_error(ms_scene *scene);

#ifdef __cplusplus
}
#endif
#endif
