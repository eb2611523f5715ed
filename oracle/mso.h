/* mso.h -- CPU ORACLE for the MLP-Splatting forward render (arxiv/paper_2606_03877).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may load it.  It shares no
 * source, header, table or helper with the CUDA path (paper_2606_03877_b200/csrc/,
 * include/mlpsplat.h); it was written from PAPER.md and BASELINE.json's north_star
 * (NS) before any kernel existed.
 *
 * What it computes (citations: P:NN = /root/reference/PAPER.md line NN):
 *   scene      N primitives (mu, s, unit quaternion q, own MLP)            P:74-76 (Sec.3.1)
 *   support    ellipsoid { x : |x-mu|^2_Lambda <= 1 },
 *              Lambda = R diag(s^2)^-1 R^T                                  P:84, NS, Q5
 *   interval   ray/ellipsoid chord [t_in, t_out], K midpoint samples       NS (c), Q1,Q7
 *   MLP input  u = S^-1 R^T (p - mu); [u, sin(2^l pi u), cos(2^l pi u)]_l
 *              [, world-frame unit d]                                       P:101 Eq.5, Q2,Q3,Q15
 *   MLP        (Linear+ReLU) x n_hidden, Linear; rgb = sigmoid,
 *              sigma = softplus, extra channels linear                      P:105, Eq.18-19
 *   composite  alpha = 1-exp(-sigma*delta), T_j = prod_{l<j}(1-alpha_l),
 *              C = sum_j T_j alpha_j c_j, front to back over all samples of
 *              the ray sorted by (t, primitive id, k); stop after the sample
 *              that brings T below t_stop                                   P:113-115 Eq.6, Eq.14
 *   binning    conservative screen-tile lists of projected supports,
 *              sorted by (tile, entry depth, primitive id)                  P:119, NS (a),(b)
 *
 * Contact-point mode (mso_mlp.mode = MSO_MODE_CONTACT; the paper's own variant, S:Sec.8(f) NEXT-1):
 *   one evaluation per hit (K must be 1) at the soft contact point
 *   t* = max(d^T Lambda (mu-o) / d^T Lambda d, t_near), p* = o + t* d        P:80-86 Eq.1-2
 *   residual delta = mu - p*, MLP input gamma([d; delta]): per scalar z_j
 *   (d_x,d_y,d_z,delta_x,delta_y,delta_z), per level l: sin(2^l pi z_j), cos(2^l pi z_j)
 *   -> 12 L dims, no identity                                                P:89-103 Eq.3-5
 *   alpha = (1 - exp(-sigma l)) g, l = chord length of the ray in the support (reading of the
 *   undefined "effective integration length"), g = exp(-falloff |p*-mu|^2_Lambda), falloff = 9/2
 *   by default (reading of the "Gaussian falloff" whose formula the paper omits: the support
 *   boundary |.|_Lambda = 1 then sits at three standard deviations); samples ordered by (t*, primitive id).
 *   Both readings are listed in DESIGN.md Sec.11.
 *   Slot features (mso_scene_set_slots; S:Sec.8(f) NEXT-2; Eq.7): u = clip_[-1,1]^3(R^T delta / s),
 *   g_k = softmax_k(a_k^T u) over the canonical tetrahedral frame a_k = (1,1,1), (1,-1,-1), (-1,1,-1),
 *   (-1,-1,1), each / sqrt(3); f = sum_k g_k e_k in R^{C_f}; F = sum_i T_i alpha_i f_i (same weights as colour).
 *
 * Precision: every geometric decision (projection, tile range, intersection,
 * sample t, sample order, local coordinate u) is evaluated in IEEE fp32,
 * round-to-nearest, NO fused multiply-add, in the operation order written in
 * mso.c -- because NS demands bit-exact tile
 * lists, interval counts and sample order.  The MLP and the compositing sum run
 * in fp64 from the given float32 weight values.
 *
 * Parity pins: tests/test_oracle_pins.py (closed forms, invariants, brute force,
 * torch fp64 MLP).  Unpinned: nothing on the render path; dataset-level quality
 * metrics (PSNR/mIoU) are out of scope ("parity unpinned").
 */
#ifndef MSO_H
#define MSO_H
#include <stdint.h>
#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct mso_scene mso_scene;

typedef struct {
  int32_t n;             /* primitives */
  const float *center;   /* [n][3] */
  const float *quat;     /* [n][4] (w,x,y,z), normalised here */
  const float *scale;    /* [n][3] ellipsoid semi-axes > 0 */
} mso_prims;

typedef struct {
  int32_t n_freq;        /* L of Eq.5 */
  int32_t use_viewdir;   /* append raw world-frame unit d after the encoding  */
  int32_t n_hidden;      /* hidden Linear+ReLU layers                                  */
  int32_t width;         /* hidden width                                               */
  int32_t n_feat;        /* linear channels after [r,g,b,sigma] */
  const float *weights;  /* [n][params]: per layer W[in][out] row-major, then b[out]   */
  int32_t mode;          /* MSO_MODE_LOCAL (0) | MSO_MODE_CONTACT (1)                  */
  float falloff;         /* contact mode: g = exp(-falloff |p*-mu|^2_Lambda), >= 0; the reading of P:105's
                            "Gaussian falloff" (Q29): MSO_FALLOFF_DEFAULT = 9/2               */
} mso_mlp;
#define MSO_FALLOFF_DEFAULT 4.5f
#define MSO_EYE_GUARD_DEFAULT 0.01f

enum { MSO_MODE_LOCAL = 0, MSO_MODE_CONTACT = 1 };
enum { MSO_ORDER_EXACT = 0, MSO_ORDER_TILE = 1 };

typedef struct {
  float fx, fy, cx, cy;
  float c2w[12];         /* 3x4 row-major; camera x right, y down, z forward */
  float t_near;
} mso_camera;

typedef struct {
  int32_t K;             /* midpoint samples per interval (NS (c)) */
  float   t_stop;        /* early termination: stop once T < t_stop (NS (e): 1e-4) */
  int32_t tile;          /* tile edge in pixels for binned mode; 0 = brute force (no binning) */
  int32_t n_threads;     /* OpenMP threads; <= 0 = all cores */
} mso_opts;

typedef struct {
  int64_t n_pixels;
  int64_t n_intervals;         /* (ray, primitive) hits */
  int64_t n_samples;           /* n_intervals * K */
  int64_t n_mlp_evals;         /* samples actually evaluated (fewer if rays terminated early) */
  int64_t n_terminated;        /* rays stopped by T < t_stop */
  int64_t n_pairs;             /* (tile, primitive) keys; 0 in brute mode */
  double  min_T;               /* smallest final transmittance over the rendered pixels */
} mso_stats;

enum { MSO_OK = 0, MSO_ERR_ARG = -1, MSO_ERR_MEM = -2, MSO_ERR_CAP = -3 };

int  mso_scene_create(const mso_prims *, const mso_mlp *, mso_scene **out);
/* contact mode: MSO_ORDER_TILE composites every pixel of a tile in ONE shared order, that of the contact
 * points t*_{i,c} of the virtual ray through the tile centre (ties by primitive id) -- the paper's
 * approximation (about 2x faster, -0.35 dB there).  Binned mode only; the tile lists are then sorted by
 * (tile, t*_{i,c}, primitive id).  Default MSO_ORDER_EXACT: per-ray order by (t*, primitive id). */
int  mso_scene_set_order(mso_scene *, int32_t order);
/* Q13: a support with z_lo <= eye_guard * r_z (touching or nearly touching the eye plane) is binned to the whole
 * image; default MSO_EYE_GUARD_DEFAULT = 0.01.  Must be > 0. */
int  mso_scene_set_eye_guard(mso_scene *, float eye_guard);
/* contact mode, n_feat == 0: attach slot embeddings emb[n][4][c_f] (copied); mso_render then writes feat[n_pix][c_f] */
int  mso_scene_set_slots(mso_scene *, int32_t c_f, const float *emb);
/* gates g[4] of primitive prim for the residual delta = mu - p* (world frame) */
int  mso_slot_gates(const mso_scene *, int32_t prim, const float *delta, double *g);
void mso_scene_destroy(mso_scene *);

/* Renders pixels pix[0..n_pix) (linear index y*W+x), or all H*W pixels in raster
 * order when pix == NULL.  Outputs are fp64: rgb[n][3], alpha[n], feat[n][n_feat]
 * (feat may be NULL).  stats may be NULL. */
int mso_render(const mso_scene *, const mso_camera *, int H, int W, const mso_opts *,
               const int32_t *pix, int64_t n_pix,
               double *out_rgb, double *out_alpha, double *out_feat, mso_stats *stats);

/* ---- parity artefacts (NS: "tile lists, interval counts and sample ordering bit-exact") ---- */

/* Sorted (tile, z_entry bits, primitive) keys.  tile_offsets[tiles+1]; prim_ids/zbits[cap].
 * Returns MSO_ERR_CAP (with *n set) if cap is too small; call with cap = 0 to size. */
int mso_tile_lists(const mso_scene *, const mso_camera *, int H, int W, int tile,
                   int64_t *tile_offsets, int32_t *prim_ids, uint32_t *zbits,
                   size_t cap, size_t *n);

/* Per-pixel hit counts for the whole image (binned if opts->tile > 0). hit_count[H*W]. */
int mso_hit_counts(const mso_scene *, const mso_camera *, int H, int W, const mso_opts *,
                   int32_t *hit_count);

/* Intervals of one pixel, sorted by primitive id: prim, t_in, delta = (t_out - t_in)/K. */
int mso_ray_intervals(const mso_scene *, const mso_camera *, int H, int W, const mso_opts *,
                      int32_t pixel, int32_t *prim, float *t_in, float *delta,
                      size_t cap, size_t *n);

/* Intervals of every pixel (each ray's list sorted by primitive id): offsets[H*W+1].
 * Call with cap = 0 to size (*n), then again. */
int mso_intervals_all(const mso_scene *, const mso_camera *, int H, int W, const mso_opts *,
                      int64_t *offsets, int32_t *prim, float *t_in, float *delta,
                      size_t cap, size_t *n);

/* All samples of one pixel in compositing order (not truncated by early termination). */
int mso_ray_samples(const mso_scene *, const mso_camera *, int H, int W, const mso_opts *,
                    int32_t pixel, int32_t *prim, int32_t *k, float *t,
                    size_t cap, size_t *n);

/* (primitive, k) of every sample of every pixel in compositing order (not truncated); pixel q owns the entries
 * [K offsets[q], K offsets[q+1]) of mso_intervals_all's offsets.  cap = 0 to size (*n). */
int mso_samples_all(const mso_scene *, const mso_camera *, int H, int W, const mso_opts *,
                    int32_t *prim, int32_t *k, size_t cap, size_t *n);

/* ---- pieces exposed so tests can pin them one by one ---- */

/* world->unit-sphere frame A = diag(1/s) R^T and its inverse-ish M = R diag(s), both [n][9]. */
int mso_prim_frames(const mso_scene *, float *A, float *M);
/* ray of pixel (x, y): origin o[3], unit direction d[3]. */
int mso_ray(const mso_camera *, int x, int y, float *o, float *d);
/* screen-space AABB of one primitive: rect = {px0, px1, py0, py1} inclusive; *visible = 0 if culled. */
int mso_project(const mso_scene *, const mso_camera *, int H, int W, int32_t prim,
                int32_t *visible, int32_t *rect, float *z_entry);
/* MLP of one primitive at local coordinate u (and world direction d): raw[out_dim] and
 * act[out_dim] = (sigmoid rgb, softplus sigma, linear features). */
int mso_mlp_eval(const mso_scene *, int32_t prim, const float *u, const float *d,
                 double *raw, double *act);
/* contact mode only: x[in_dim], raw[out_dim], act[out_dim], |p*-mu|^2_Lambda of primitive prim at o + t d */
int mso_contact_eval(const mso_scene *, int32_t prim, const float *o, const float *d, float t,
                     double *x, double *raw, double *act, double *r2);
/* encoded input vector x[in_dim] for (u, d). */
int mso_encode(const mso_scene *, const float *u, const float *d, double *x);

/* ---- backward pass (mso_grad.c; S:Sec.8(f) NEXT-4) ----
 * fp64 forward + backward of the render of pixels pix[0..n_pix) (all of them, in raster order, if pix == NULL) for
 * a scene given as fp64 arrays (center[n][3], quat[n][4], scale[n][3], weights[n][params]; mlp->weights is ignored),
 * north-star mode only.  loss = sum over pixels and channels of |C - target| (the L1 term of Eq.8) when
 * target != NULL; dL/dC = sign(C - target), or g_in[n_pix][3] if given.  Any of the outputs may be NULL: rgb_out
 * [n_pix][3], g_weights[n][params], g_center[n][3], g_quat[n][4], g_scale[n][3].  All gradient outputs NULL =
 * forward only (the finite-difference leg of the pins). */
int mso_loss_grad_f64(int32_t n, const double *center, const double *quat, const double *scale,
                      const double *weights, const mso_mlp *mlp, const mso_camera *cam, int H, int W, int K,
                      double t_stop, const int32_t *pix, int64_t n_pix, const double *target, const double *g_in,
                      double *loss, double *rgb_out, double *g_weights, double *g_center, double *g_quat,
                      double *g_scale);

#ifdef __cplusplus
}
#endif
#endif
