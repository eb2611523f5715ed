/* mso.c -- CPU ORACLE for the MLP-Splatting forward render.  TEST INFRASTRUCTURE ONLY;
 * see mso.h for scope, citations and the precision contract.
 *
 * Build: gcc -O2 -std=c11 -ffp-contract=off -fno-fast-math -fopenmp -shared -fPIC mso.c -lm
 * (-ffp-contract=off: no fused multiply-add may be formed; every fp32 operation below
 *  rounds once, in the order written -- DESIGN.md "Canonical fp32 order".)
 *
 * Plain and slow on purpose: no blocking, no SIMD intrinsics, no shared tables.  The
 * per-ray work is the algorithm of SURVEY.md Sec.8(c) in its order: candidates ->
 * intersection -> samples -> sort -> MLP -> composite.
 */
#include "mso.h"
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define MSO_PI 3.14159265358979323846

/* ------------------------------------------------------------------------------------------
 * Scene
 * ---------------------------------------------------------------------------------------- */
struct mso_scene {
  int32_t n;
  int32_t n_freq, use_viewdir, n_hidden, width, n_feat, mode;
  int32_t c_f;           /* Eq.7 slot embeddings: width (0 = none) */
  int32_t order;         /* MSO_ORDER_EXACT | MSO_ORDER_TILE (contact mode, binned only) */
  float falloff;         /* contact mode: g = exp(-falloff r2)  (reading Q29; MSO_FALLOFF_DEFAULT = 9/2) */
  float eye_guard;       /* Q13: z_lo <= eye_guard * r_z -> whole image (MSO_EYE_GUARD_DEFAULT = 0.01) */
  float *slots;          /* [n][4][c_f] */
  int32_t in_dim, out_dim, n_layers, params;
  float *center;  /* [n][3] */
  float *A;       /* [n][9] world -> unit-sphere frame: diag(1/s) R^T    (Lambda = A^T A) */
  float *M;       /* [n][9] unit-sphere -> world:        R diag(s)                              */
  float *weights; /* [n][params] copy */
};

/* canonical 3-term dot product: (a0*b0 + a1*b1) + a2*b2, fp32, no FMA */
static inline float dot3(float a0, float a1, float a2, float b0, float b1, float b2) {
  float p0 = a0 * b0;
  float p1 = a1 * b1;
  float p2 = a2 * b2;
  float s = p0 + p1;
  return s + p2;
}

/* P:74 unit quaternion -> rotation matrix (Hamilton convention, (w,x,y,z)); row-major R[9]. */
static int quat_to_rot(const float *q, float *R) {
  float w = q[0], x = q[1], y = q[2], z = q[3];
  float n2 = ((w * w + x * x) + y * y) + z * z;
  if (!(n2 > 0.0f) || !isfinite(n2)) return MSO_ERR_ARG;
  float nrm = sqrtf(n2);
  w = w / nrm; x = x / nrm; y = y / nrm; z = z / nrm;
  float xx = x * x, yy = y * y, zz = z * z;
  float xy = x * y, xz = x * z, yz = y * z;
  float wx = w * x, wy = w * y, wz = w * z;
  R[0] = 1.0f - 2.0f * (yy + zz); R[1] = 2.0f * (xy - wz);        R[2] = 2.0f * (xz + wy);
  R[3] = 2.0f * (xy + wz);        R[4] = 1.0f - 2.0f * (xx + zz); R[5] = 2.0f * (yz - wx);
  R[6] = 2.0f * (xz - wy);        R[7] = 2.0f * (yz + wx);        R[8] = 1.0f - 2.0f * (xx + yy);
  return MSO_OK;
}

int mso_scene_create(const mso_prims *p, const mso_mlp *m, mso_scene **out) {
  if (!p || !m || !out || p->n <= 0 || !p->center || !p->quat || !p->scale || !m->weights)
    return MSO_ERR_ARG;
  if (m->n_freq < 0 || m->n_hidden < 1 || m->width < 1 || m->n_feat < 0) return MSO_ERR_ARG;
  if (m->mode != MSO_MODE_LOCAL && m->mode != MSO_MODE_CONTACT) return MSO_ERR_ARG;
  if (m->mode == MSO_MODE_CONTACT && (m->n_freq < 1 || m->use_viewdir)) return MSO_ERR_ARG;
  if (m->mode == MSO_MODE_CONTACT && !(m->falloff >= 0.0f)) return MSO_ERR_ARG;
  mso_scene *s = (mso_scene *)calloc(1, sizeof(*s));
  if (!s) return MSO_ERR_MEM;
  s->n = p->n;
  s->falloff = m->falloff;
  s->eye_guard = MSO_EYE_GUARD_DEFAULT;
  s->n_freq = m->n_freq; s->use_viewdir = m->use_viewdir ? 1 : 0;
  s->n_hidden = m->n_hidden; s->width = m->width; s->n_feat = m->n_feat;
  s->mode = m->mode;
  s->in_dim = m->mode == MSO_MODE_CONTACT ? 12 * m->n_freq : 3 + 6 * m->n_freq + (s->use_viewdir ? 3 : 0);
  s->out_dim = 4 + m->n_feat;
  s->n_layers = m->n_hidden + 1;
  int params = 0, in = s->in_dim;
  for (int l = 0; l < s->n_layers; ++l) {
    int o = (l == s->n_layers - 1) ? s->out_dim : s->width;
    params += in * o + o;
    in = o;
  }
  s->params = params;
  size_t n = (size_t)p->n;
  s->center = (float *)malloc(n * 3 * sizeof(float));
  s->A = (float *)malloc(n * 9 * sizeof(float));
  s->M = (float *)malloc(n * 9 * sizeof(float));
  s->weights = (float *)malloc(n * (size_t)params * sizeof(float));
  if (!s->center || !s->A || !s->M || !s->weights) { mso_scene_destroy(s); return MSO_ERR_MEM; }
  memcpy(s->center, p->center, n * 3 * sizeof(float));
  memcpy(s->weights, m->weights, n * (size_t)params * sizeof(float));
  for (size_t i = 0; i < n; ++i) {
    float R[9];
    const float *sc = p->scale + 3 * i;
    if (!(sc[0] > 0.0f) || !(sc[1] > 0.0f) || !(sc[2] > 0.0f) ||
        quat_to_rot(p->quat + 4 * i, R) != MSO_OK) {
      mso_scene_destroy(s);
      return MSO_ERR_ARG;
    }
    for (int r = 0; r < 3; ++r)
      for (int c = 0; c < 3; ++c) {
        s->A[9 * i + 3 * r + c] = R[3 * c + r] / sc[r];   /* A = diag(1/s) R^T */
        s->M[9 * i + 3 * r + c] = R[3 * r + c] * sc[c];   /* M = R diag(s)     */
      }
  }
  *out = s;
  return MSO_OK;
}

int mso_scene_set_eye_guard(mso_scene *s, float eye_guard) {
  if (!s || !(eye_guard > 0.0f)) return MSO_ERR_ARG;
  s->eye_guard = eye_guard;
  return MSO_OK;
}

int mso_scene_set_order(mso_scene *s, int32_t order) {
  if (!s || (order != MSO_ORDER_EXACT && order != MSO_ORDER_TILE)) return MSO_ERR_ARG;
  if (order == MSO_ORDER_TILE && s->mode != MSO_MODE_CONTACT) return MSO_ERR_ARG;
  s->order = order;
  return MSO_OK;
}

int mso_scene_set_slots(mso_scene *s, int32_t c_f, const float *emb) {
  if (!s || c_f < 1 || !emb || s->mode != MSO_MODE_CONTACT || s->n_feat != 0) return MSO_ERR_ARG;
  float *p = (float *)malloc((size_t)s->n * 4 * (size_t)c_f * sizeof(float));
  if (!p) return MSO_ERR_MEM;
  memcpy(p, emb, (size_t)s->n * 4 * (size_t)c_f * sizeof(float));
  free(s->slots);
  s->slots = p; s->c_f = c_f;
  return MSO_OK;
}

/* Eq.7: u = clip(R^T delta / s) = clip(A delta), g = softmax_k(a_k^T u) over the tetrahedral frame */
static void slot_gates(const mso_scene *s, int i, const float *delta, double *g) {
  static const double TET[4][3] = {{1, 1, 1}, {1, -1, -1}, {-1, 1, -1}, {-1, -1, 1}};
  const float *A = s->A + 9 * i;
  double u[3], z[4], m = -1e300, sum = 0.0;
  for (int r = 0; r < 3; ++r) {
    double v = (double)A[3 * r] * delta[0] + (double)A[3 * r + 1] * delta[1] + (double)A[3 * r + 2] * delta[2];
    u[r] = v < -1.0 ? -1.0 : (v > 1.0 ? 1.0 : v);
  }
  for (int k = 0; k < 4; ++k) {
    z[k] = (TET[k][0] * u[0] + TET[k][1] * u[1] + TET[k][2] * u[2]) / sqrt(3.0);
    if (z[k] > m) m = z[k];
  }
  for (int k = 0; k < 4; ++k) { g[k] = exp(z[k] - m); sum += g[k]; }
  for (int k = 0; k < 4; ++k) g[k] /= sum;
}

int mso_slot_gates(const mso_scene *s, int32_t prim, const float *delta, double *g) {
  if (!s || prim < 0 || prim >= s->n || !delta || !g) return MSO_ERR_ARG;
  slot_gates(s, prim, delta, g);
  return MSO_OK;
}

void mso_scene_destroy(mso_scene *s) {
  if (!s) return;
  free(s->center); free(s->A); free(s->M); free(s->weights); free(s->slots);
  free(s);
}

int mso_prim_frames(const mso_scene *s, float *A, float *M) {
  if (!s) return MSO_ERR_ARG;
  if (A) memcpy(A, s->A, (size_t)s->n * 9 * sizeof(float));
  if (M) memcpy(M, s->M, (size_t)s->n * 9 * sizeof(float));
  return MSO_OK;
}

/* ------------------------------------------------------------------------------------------
 * Camera ray (Q14: pixel centres at +0.5, row 0 on top, OpenCV frame)
 * ---------------------------------------------------------------------------------------- */
/* ray through the image point (px, py) in pixel units; pixel (x, y) has its centre at (x + 0.5, y + 0.5) */
static void point_ray(const mso_camera *c, float px, float py, float *o, float *d) {
  float dcx = (px - c->cx) / c->fx;
  float dcy = (py - c->cy) / c->fy;
  const float *m = c->c2w;   /* rows: [r00 r01 r02 tx] ... */
  float wx = (m[0] * dcx + m[1] * dcy) + m[2];
  float wy = (m[4] * dcx + m[5] * dcy) + m[6];
  float wz = (m[8] * dcx + m[9] * dcy) + m[10];
  float n2 = (wx * wx + wy * wy) + wz * wz;
  float nrm = sqrtf(n2);
  d[0] = wx / nrm; d[1] = wy / nrm; d[2] = wz / nrm;
  o[0] = m[3]; o[1] = m[7]; o[2] = m[11];
}

static void camera_ray(const mso_camera *c, int x, int y, float *o, float *d) {
  point_ray(c, (float)x + 0.5f, (float)y + 0.5f, o, d);
}

int mso_ray(const mso_camera *c, int x, int y, float *o, float *d) {
  if (!c || !o || !d) return MSO_ERR_ARG;
  camera_ray(c, x, y, o, d);
  return MSO_OK;
}

/* ------------------------------------------------------------------------------------------
 * Projection: conservative screen-space AABB of an ellipsoid ("conservative overlap
 * tests based on their projected support regions"; "AABB-tile-frustum intersection").
 *
 * Camera space: c = R_c^T (mu - o), M_c = R_c^T M; the support is { c + M_c w : |w| <= 1 }.
 * z extent: c_z -/+ |row_z(M_c)|.  A plane x = tau z through the eye is tangent to the
 * ellipsoid iff  zz tau^2 - 2 xz tau + xx = 0  with  zz = |r_z|^2 - c_z^2, xz = r_x.r_z - c_x c_z,
 * xx = |r_x|^2 - c_x^2  (r_x, r_z rows of M_c); its roots bound x/z over the support.
 * ---------------------------------------------------------------------------------------- */
typedef struct { int visible; int px0, px1, py0, py1; float z_entry; } proj_t;

static void axis_bounds(float rxx, float rxy, float rxz, float cxv,
                        float rzx, float rzy, float rzz, float czv, float zz,
                        float focal, float centre, float *lo, float *hi) {
  float xz = dot3(rxx, rxy, rxz, rzx, rzy, rzz) - cxv * czv;
  float xx = dot3(rxx, rxy, rxz, rxx, rxy, rxz) - cxv * cxv;
  float m = xz / zz;
  float q = m * m - xx / zz;
  float h = sqrtf(q > 0.0f ? q : 0.0f);
  *lo = focal * (m - h) + centre;
  *hi = focal * (m + h) + centre;
}

static int clamp_lo(float v, int n) {          /* max(0, floor(v)) without int overflow */
  float f = floorf(v);
  if (!(f > 0.0f)) return 0;                   /* also catches NaN */
  if (f > (float)n) return n;                  /* beyond the image: caller sees empty range */
  return (int)f;
}
static int clamp_hi(float v, int n) {          /* min(n-1, ceil(v)) */
  float f = ceilf(v);
  if (!(f < (float)(n - 1))) return n - 1;     /* also catches NaN */
  if (f < 0.0f) return -1;
  return (int)f;
}

static proj_t project(const mso_scene *s, const mso_camera *cam, int H, int W, int i) {
  proj_t r; memset(&r, 0, sizeof(r));
  const float *m = cam->c2w;
  const float *mu = s->center + 3 * i;
  const float *M = s->M + 9 * i;
  float v0 = mu[0] - m[3], v1 = mu[1] - m[7], v2 = mu[2] - m[11];
  /* columns of the c2w rotation are the camera axes: c_j = column_j . v */
  float cxv = dot3(m[0], m[4], m[8], v0, v1, v2);
  float cyv = dot3(m[1], m[5], m[9], v0, v1, v2);
  float czv = dot3(m[2], m[6], m[10], v0, v1, v2);
  float Mc[9];
  for (int a = 0; a < 3; ++a)          /* camera axis a */
    for (int j = 0; j < 3; ++j)
      Mc[3 * a + j] = dot3(m[a], m[4 + a], m[8 + a], M[j], M[3 + j], M[6 + j]);
  float rz = sqrtf(dot3(Mc[6], Mc[7], Mc[8], Mc[6], Mc[7], Mc[8]));
  float z_lo = czv - rz;
  float z_hi = czv + rz;
  if (!(z_hi > 0.0f)) return r;                       /* entirely behind the eye plane */
  r.z_entry = z_lo > 0.0f ? z_lo : 0.0f;
  if (z_lo <= s->eye_guard * rz) {
    /* Touches / nears the eye plane (Q13): the tangent-plane bound degenerates.  Bound the camera-space box of the
     * support instead, clipped at a depth z_n in front of which every point of the support projects off the image:
     * the support lies in c -/+ (r_x, r_y, r_z) (r_a = |row_a(M_c)|), so its points are at least
     * d_box = |max(|c| - r, 0)| from the eye; one with 0 < z < z_n has (x^2 + y^2)/z^2 > d_box^2/z_n^2 - 1, beyond the
     * farthest image corner rho_max once z_n < d_box / sqrt(1 + rho_max^2) (half of that is taken).  The part with
     * z >= z_c = max(z_lo, z_n) projects inside [x_l, x_h] / [z_c, z_hi].  Eye inside the box: whole image. */
    float rx = sqrtf(dot3(Mc[0], Mc[1], Mc[2], Mc[0], Mc[1], Mc[2]));
    float ry = sqrtf(dot3(Mc[3], Mc[4], Mc[5], Mc[3], Mc[4], Mc[5]));
    float ex = fabsf(cxv) - rx, ey = fabsf(cyv) - ry, ez = fabsf(czv) - rz;
    ex = ex > 0.0f ? ex : 0.0f; ey = ey > 0.0f ? ey : 0.0f; ez = ez > 0.0f ? ez : 0.0f;
    float d2 = (ex * ex + ey * ey) + ez * ez;
    r.visible = 1; r.px0 = 0; r.px1 = W - 1; r.py0 = 0; r.py1 = H - 1;
    if (!(d2 > 0.0f)) return r;
    float wx = (float)W - cam->cx, wy = (float)H - cam->cy;
    float tx = (cam->cx > wx ? cam->cx : wx) / cam->fx, ty = (cam->cy > wy ? cam->cy : wy) / cam->fy;
    float zn = (0.5f * sqrtf(d2)) / sqrtf(1.0f + (tx * tx + ty * ty));
    float zc = z_lo > zn ? z_lo : zn;
    zc = zc < z_hi ? zc : z_hi;
    float xl = cxv - rx, xh = cxv + rx, yl = cyv - ry, yh = cyv + ry;
    float x_lo = cam->fx * (xl < 0.0f ? xl / zc : xl / z_hi) + cam->cx;
    float x_hi = cam->fx * (xh > 0.0f ? xh / zc : xh / z_hi) + cam->cx;
    float y_lo = cam->fy * (yl < 0.0f ? yl / zc : yl / z_hi) + cam->cy;
    float y_hi = cam->fy * (yh > 0.0f ? yh / zc : yh / z_hi) + cam->cy;
    r.px0 = clamp_lo(x_lo - 0.5f, W);
    r.px1 = clamp_hi(x_hi - 0.5f, W);
    r.py0 = clamp_lo(y_lo - 0.5f, H);
    r.py1 = clamp_hi(y_hi - 0.5f, H);
    r.visible = (r.px0 <= r.px1) && (r.py0 <= r.py1);
    return r;
  }
  float zz = dot3(Mc[6], Mc[7], Mc[8], Mc[6], Mc[7], Mc[8]) - czv * czv;   /* < 0 here */
  float x_lo, x_hi, y_lo, y_hi;
  axis_bounds(Mc[0], Mc[1], Mc[2], cxv, Mc[6], Mc[7], Mc[8], czv, zz, cam->fx, cam->cx, &x_lo, &x_hi);
  axis_bounds(Mc[3], Mc[4], Mc[5], cyv, Mc[6], Mc[7], Mc[8], czv, zz, cam->fy, cam->cy, &y_lo, &y_hi);
  /* pixel x is covered if x + 0.5 in [x_lo, x_hi]; one pixel of slack absorbs fp32 rounding */
  r.px0 = clamp_lo(x_lo - 0.5f, W);
  r.px1 = clamp_hi(x_hi - 0.5f, W);
  r.py0 = clamp_lo(y_lo - 0.5f, H);
  r.py1 = clamp_hi(y_hi - 0.5f, H);
  r.visible = (r.px0 <= r.px1) && (r.py0 <= r.py1);
  return r;
}

int mso_project(const mso_scene *s, const mso_camera *cam, int H, int W, int32_t prim,
                int32_t *visible, int32_t *rect, float *z_entry) {
  if (!s || !cam || prim < 0 || prim >= s->n) return MSO_ERR_ARG;
  proj_t r = project(s, cam, H, W, prim);
  if (visible) *visible = r.visible;
  if (rect) { rect[0] = r.px0; rect[1] = r.px1; rect[2] = r.py0; rect[3] = r.py1; }
  if (z_entry) *z_entry = r.z_entry;
  return MSO_OK;
}

/* ------------------------------------------------------------------------------------------
 * Tile lists: keys (tile, z_entry bits, primitive) sorted ascending  (NS (a),(b))
 * ---------------------------------------------------------------------------------------- */
typedef struct { uint32_t tile; uint32_t zbits; int32_t prim; } tkey_t;

static int tkey_cmp(const void *a, const void *b) {
  const tkey_t *x = (const tkey_t *)a, *y = (const tkey_t *)b;
  if (x->tile != y->tile) return x->tile < y->tile ? -1 : 1;
  if (x->zbits != y->zbits) return x->zbits < y->zbits ? -1 : 1;
  if (x->prim != y->prim) return x->prim < y->prim ? -1 : 1;
  return 0;
}

typedef struct { int tiles_x, tiles_y; int64_t *offsets; tkey_t *keys; size_t n; } tlists_t;

static void tlists_free(tlists_t *t) { free(t->offsets); free(t->keys); memset(t, 0, sizeof(*t)); }

/* "a representative virtual ray passing through the tile center" orders the tile's primitives
 * for every pixel of the tile: t*_{i,c} of Eq.2 for the ray through the centre point of tile (a, b). */
static float tile_center_tstar(const mso_scene *s, const mso_camera *cam, int i, int a, int b, int tile) {
  float o[3], d[3];
  point_ray(cam, (float)(a * tile) + 0.5f * (float)tile, (float)(b * tile) + 0.5f * (float)tile, o, d);
  const float *A = s->A + 9 * i;
  const float *mu = s->center + 3 * i;
  float v0 = o[0] - mu[0], v1 = o[1] - mu[1], v2 = o[2] - mu[2];
  float o0 = dot3(A[0], A[1], A[2], v0, v1, v2);
  float o1 = dot3(A[3], A[4], A[5], v0, v1, v2);
  float o2 = dot3(A[6], A[7], A[8], v0, v1, v2);
  float d0 = dot3(A[0], A[1], A[2], d[0], d[1], d[2]);
  float d1 = dot3(A[3], A[4], A[5], d[0], d[1], d[2]);
  float d2 = dot3(A[6], A[7], A[8], d[0], d[1], d[2]);
  float aa = dot3(d0, d1, d2, d0, d1, d2);
  float bb = dot3(o0, o1, o2, d0, d1, d2);
  float ts = (-bb) / aa;
  return ts > 0.0f ? ts : 0.0f;
}

static int tlists_build(const mso_scene *s, const mso_camera *cam, int H, int W, int tile, tlists_t *out) {
  memset(out, 0, sizeof(*out));
  int tx = (W + tile - 1) / tile, ty = (H + tile - 1) / tile;
  out->tiles_x = tx; out->tiles_y = ty;
  size_t cap = 1024, n = 0;
  tkey_t *keys = (tkey_t *)malloc(cap * sizeof(tkey_t));
  if (!keys) return MSO_ERR_MEM;
  for (int i = 0; i < s->n; ++i) {
    proj_t r = project(s, cam, H, W, i);
    if (!r.visible) continue;
    uint32_t zb; memcpy(&zb, &r.z_entry, 4);
    for (int b = r.py0 / tile; b <= r.py1 / tile; ++b)
      for (int a = r.px0 / tile; a <= r.px1 / tile; ++a) {
        if (n == cap) {
          cap *= 2;
          tkey_t *k2 = (tkey_t *)realloc(keys, cap * sizeof(tkey_t));
          if (!k2) { free(keys); return MSO_ERR_MEM; }
          keys = k2;
        }
        if (s->order == MSO_ORDER_TILE) { float tc = tile_center_tstar(s, cam, i, a, b, tile); memcpy(&zb, &tc, 4); }
        keys[n].tile = (uint32_t)(b * tx + a); keys[n].zbits = zb; keys[n].prim = i; ++n;
      }
  }
  qsort(keys, n, sizeof(tkey_t), tkey_cmp);
  int64_t *off = (int64_t *)calloc((size_t)tx * ty + 1, sizeof(int64_t));
  if (!off) { free(keys); return MSO_ERR_MEM; }
  for (size_t j = 0; j < n; ++j) off[keys[j].tile + 1]++;
  for (int t = 0; t < tx * ty; ++t) off[t + 1] += off[t];
  out->offsets = off; out->keys = keys; out->n = n;
  return MSO_OK;
}

int mso_tile_lists(const mso_scene *s, const mso_camera *cam, int H, int W, int tile,
                   int64_t *tile_offsets, int32_t *prim_ids, uint32_t *zbits, size_t cap, size_t *n) {
  if (!s || !cam || tile <= 0 || H <= 0 || W <= 0) return MSO_ERR_ARG;
  tlists_t t;
  int rc = tlists_build(s, cam, H, W, tile, &t);
  if (rc != MSO_OK) return rc;
  if (n) *n = t.n;
  if (cap < t.n) { tlists_free(&t); return MSO_ERR_CAP; }
  if (tile_offsets) memcpy(tile_offsets, t.offsets, ((size_t)t.tiles_x * t.tiles_y + 1) * sizeof(int64_t));
  for (size_t j = 0; j < t.n; ++j) {
    if (prim_ids) prim_ids[j] = t.keys[j].prim;
    if (zbits) zbits[j] = t.keys[j].zbits;
  }
  tlists_free(&t);
  return MSO_OK;
}

/* ------------------------------------------------------------------------------------------
 * Ray / ellipsoid intersection (NS (c); Q13).  In the unit-sphere frame the
 * support is |o' + t d'| <= 1 with o' = A (o - mu), d' = A d.
 * ---------------------------------------------------------------------------------------- */
typedef struct { int32_t prim; float t_in, delta; } hit_t;

static int intersect(const mso_scene *s, int i, const float *o, const float *d,
                     float t_near, int K, hit_t *h) {
  const float *A = s->A + 9 * i;
  const float *mu = s->center + 3 * i;
  float v0 = o[0] - mu[0], v1 = o[1] - mu[1], v2 = o[2] - mu[2];
  float o0 = dot3(A[0], A[1], A[2], v0, v1, v2);
  float o1 = dot3(A[3], A[4], A[5], v0, v1, v2);
  float o2 = dot3(A[6], A[7], A[8], v0, v1, v2);
  float d0 = dot3(A[0], A[1], A[2], d[0], d[1], d[2]);
  float d1 = dot3(A[3], A[4], A[5], d[0], d[1], d[2]);
  float d2 = dot3(A[6], A[7], A[8], d[0], d[1], d[2]);
  float a = dot3(d0, d1, d2, d0, d1, d2);
  float b = dot3(o0, o1, o2, d0, d1, d2);
  float c = dot3(o0, o1, o2, o0, o1, o2) - 1.0f;
  float bb = b * b;
  float ac = a * c;
  float disc = bb - ac;
  if (!(disc > 0.0f)) return 0;                 /* tangent or miss */
  float sq = sqrtf(disc);
  float t0 = (-b - sq) / a;
  float t1 = (-b + sq) / a;
  if (!(t1 > t_near)) return 0;                 /* support entirely before t_near */
  float t_in = t0 > t_near ? t0 : t_near;       /* eye inside the support: start at t_near */
  float delta = (t1 - t_in) / (float)K;
  if (!(delta > 0.0f)) return 0;
  h->prim = i; h->t_in = t_in; h->delta = delta;
  if (s->mode == MSO_MODE_CONTACT) {
    /* Eq.2: t* = max(0, d^T Lambda (mu - o) / d^T Lambda d) = max(-b/a, .); the hit keeps
     * (t*, chord length): K = 1, so delta above IS the chord length t1 - max(t0, t_near). */
    float ts = (-b) / a;
    h->t_in = ts > t_near ? ts : t_near;
  }
  return 1;
}

static inline float sample_t(float t_in, float delta, int k) {   /* MSO_MODE_LOCAL; contact mode: the sample IS t_in = t* */
  float kf = (float)k + 0.5f;
  float off = kf * delta;
  return t_in + off;
}

/* local coordinate of the sample point: p = o + t d; u = A (p - mu)   (Q2) */
static inline void sample_u(const mso_scene *s, int i, const float *o, const float *d, float t, float *u) {
  const float *A = s->A + 9 * i;
  const float *mu = s->center + 3 * i;
  float p0 = o[0] + t * d[0], p1 = o[1] + t * d[1], p2 = o[2] + t * d[2];
  float w0 = p0 - mu[0], w1 = p1 - mu[1], w2 = p2 - mu[2];
  u[0] = dot3(A[0], A[1], A[2], w0, w1, w2);
  u[1] = dot3(A[3], A[4], A[5], w0, w1, w2);
  u[2] = dot3(A[6], A[7], A[8], w0, w1, w2);
}

/* ------------------------------------------------------------------------------------------
 * MLP (fp64): positional encoding Eq.5 with the identity prepended (Q3),
 * Linear+ReLU hidden layers, output activations P:105.
 * ---------------------------------------------------------------------------------------- */
static void encode(const mso_scene *s, const float *u, const float *d, double *x) {
  int j = 0;
  for (int a = 0; a < 3; ++a) x[j++] = (double)u[a];
  for (int l = 0; l < s->n_freq; ++l) {
    double f = ldexp(MSO_PI, l);                       /* 2^l * pi */
    for (int a = 0; a < 3; ++a) x[j++] = sin(f * (double)u[a]);
    for (int a = 0; a < 3; ++a) x[j++] = cos(f * (double)u[a]);
  }
  if (s->use_viewdir) for (int a = 0; a < 3; ++a) x[j++] = (double)d[a];
}

/* Contact-point input (Eq.3-5): p* = o + t* d, delta = mu - p*, z = [d; delta];
 * gamma(z): per scalar z_j, per level l: sin(2^l pi z_j), cos(2^l pi z_j).  Also returns
 * r2 = |p* - mu|^2_Lambda = |A (p* - mu)|^2 for the falloff.  p* and A (p* - mu) in
 * canonical fp32 (the same sample_u as the local mode), the rest fp64. */
static void encode_contact(const mso_scene *s, int i, const float *o, const float *d, float t, double *x, double *r2,
                           float *delta_out) {
  const float *mu = s->center + 3 * i;
  float p0 = o[0] + t * d[0], p1 = o[1] + t * d[1], p2 = o[2] + t * d[2];
  float z[6] = {d[0], d[1], d[2], mu[0] - p0, mu[1] - p1, mu[2] - p2};
  if (delta_out) { delta_out[0] = z[3]; delta_out[1] = z[4]; delta_out[2] = z[5]; }
  int j = 0;
  for (int c = 0; c < 6; ++c)
    for (int l = 0; l < s->n_freq; ++l) {
      double f = ldexp(MSO_PI, l);
      x[j++] = sin(f * (double)z[c]);
      x[j++] = cos(f * (double)z[c]);
    }
  float u[3];
  sample_u(s, i, o, d, t, u);
  *r2 = (double)u[0] * u[0] + (double)u[1] * u[1] + (double)u[2] * u[2];
}

#define MSO_MAXW 1024

static void mlp_forward(const mso_scene *s, int prim, const double *x, double *raw) {
  double h0[MSO_MAXW], h1[MSO_MAXW];
  const float *w = s->weights + (size_t)prim * s->params;
  const double *in = x;
  double *cur = h0, *nxt = h1;
  int n_in = s->in_dim;
  for (int l = 0; l < s->n_layers; ++l) {
    int last = (l == s->n_layers - 1);
    int n_out = last ? s->out_dim : s->width;
    double *dst = last ? raw : cur;
    const float *W = w, *b = w + (size_t)n_in * n_out;
    for (int o = 0; o < n_out; ++o) dst[o] = (double)b[o];
    for (int i = 0; i < n_in; ++i) {
      double hi = in[i];
      const float *Wi = W + (size_t)i * n_out;
      for (int o = 0; o < n_out; ++o) dst[o] += hi * (double)Wi[o];
    }
    if (!last) {
      for (int o = 0; o < n_out; ++o) dst[o] = dst[o] > 0.0 ? dst[o] : 0.0;   /* ReLU */
      in = dst;
      double *t = cur; cur = nxt; nxt = t;
    }
    w = b + n_out;
    n_in = n_out;
  }
}

static void activate(const mso_scene *s, const double *raw, double *act) {
  for (int c = 0; c < 3; ++c) act[c] = 1.0 / (1.0 + exp(-raw[c]));              /* sigmoid  */
  double r = raw[3];
  act[3] = (r > 0.0 ? r : 0.0) + log1p(exp(-fabs(r)));                            /* softplus */
  for (int c = 4; c < s->out_dim; ++c) act[c] = raw[c];                           /* linear   */
}

int mso_encode(const mso_scene *s, const float *u, const float *d, double *x) {
  if (!s || !u || !x || (s->use_viewdir && !d) || s->mode != MSO_MODE_LOCAL) return MSO_ERR_ARG;
  encode(s, u, d, x);
  return MSO_OK;
}

int mso_mlp_eval(const mso_scene *s, int32_t prim, const float *u, const float *d, double *raw, double *act) {
  if (!s || prim < 0 || prim >= s->n || !u || (s->use_viewdir && !d) || s->mode != MSO_MODE_LOCAL) return MSO_ERR_ARG;
  if (s->in_dim > MSO_MAXW || s->width > MSO_MAXW || s->out_dim > MSO_MAXW) return MSO_ERR_ARG;
  double x[MSO_MAXW], r[MSO_MAXW], a[MSO_MAXW];
  encode(s, u, d, x);
  mlp_forward(s, prim, x, r);
  activate(s, r, a);
  if (raw) memcpy(raw, r, (size_t)s->out_dim * sizeof(double));
  if (act) memcpy(act, a, (size_t)s->out_dim * sizeof(double));
  return MSO_OK;
}

/* ------------------------------------------------------------------------------------------
 * Per-ray pipeline
 * ---------------------------------------------------------------------------------------- */
typedef struct { float t; int32_t prim; int32_t k; int32_t hit; } samp_t;

static int samp_cmp(const void *a, const void *b) {          /* (t, prim id, k) ascending (Q12) */
  const samp_t *x = (const samp_t *)a, *y = (const samp_t *)b;
  if (x->t != y->t) return x->t < y->t ? -1 : 1;
  if (x->prim != y->prim) return x->prim < y->prim ? -1 : 1;
  if (x->k != y->k) return x->k < y->k ? -1 : 1;
  return 0;
}

static int hit_cmp_prim(const void *a, const void *b) {
  const hit_t *x = (const hit_t *)a, *y = (const hit_t *)b;
  return x->prim < y->prim ? -1 : (x->prim > y->prim ? 1 : 0);
}

typedef struct { hit_t *hits; size_t hcap; samp_t *samps; size_t scap; } raybuf_t;

static void raybuf_free(raybuf_t *b) { free(b->hits); free(b->samps); memset(b, 0, sizeof(*b)); }

/* candidates -> hits.  Binned: the tile's list in key order; brute: every primitive. */
static long gather_hits(const mso_scene *s, const mso_camera *cam, const tlists_t *tl, int tile,
                        int W, int pixel, int K, float *o, float *d, raybuf_t *rb) {
  int x = pixel % W, y = pixel / W;
  camera_ray(cam, x, y, o, d);
  size_t nh = 0;
  size_t ncand; const tkey_t *cand = NULL;
  if (tl) {
    int t = (y / tile) * tl->tiles_x + (x / tile);
    cand = tl->keys + tl->offsets[t];
    ncand = (size_t)(tl->offsets[t + 1] - tl->offsets[t]);
  } else {
    ncand = (size_t)s->n;
  }
  for (size_t c = 0; c < ncand; ++c) {
    int i = cand ? cand[c].prim : (int)c;
    hit_t h;
    if (!intersect(s, i, o, d, cam->t_near, K, &h)) continue;
    if (nh == rb->hcap) {
      size_t nc = rb->hcap ? rb->hcap * 2 : 32;
      hit_t *h2 = (hit_t *)realloc(rb->hits, nc * sizeof(hit_t));
      if (!h2) return -1;
      rb->hits = h2; rb->hcap = nc;
    }
    rb->hits[nh++] = h;
  }
  return (long)nh;
}

static long build_samples(const mso_scene *s, long nh, int K, raybuf_t *rb) {
  size_t ns = (size_t)nh * (size_t)K;
  if (ns > rb->scap) {
    samp_t *s2 = (samp_t *)realloc(rb->samps, ns * sizeof(samp_t));
    if (!s2) return -1;
    rb->samps = s2; rb->scap = ns;
  }
  size_t j = 0;
  for (long h = 0; h < nh; ++h)
    for (int k = 0; k < K; ++k) {
      rb->samps[j].t = s->mode == MSO_MODE_CONTACT ? rb->hits[h].t_in   /* the contact point t* itself */
                                                   : sample_t(rb->hits[h].t_in, rb->hits[h].delta, k);
      rb->samps[j].prim = rb->hits[h].prim; rb->samps[j].k = k; rb->samps[j].hit = (int32_t)h;
      ++j;
    }
  if (s->order != MSO_ORDER_TILE) qsort(rb->samps, ns, sizeof(samp_t), samp_cmp);   /* tile order: the tile list's order as it is */
  return (long)ns;
}

/* contact mode: input vector, raw outputs, activations and |p*-mu|^2_Lambda at o + t d (for the pins) */
int mso_contact_eval(const mso_scene *s, int32_t prim, const float *o, const float *d, float t,
                     double *x_out, double *raw, double *act, double *r2_out) {
  if (!s || prim < 0 || prim >= s->n || !o || !d || s->mode != MSO_MODE_CONTACT) return MSO_ERR_ARG;
  if (s->in_dim > MSO_MAXW || s->width > MSO_MAXW || s->out_dim > MSO_MAXW) return MSO_ERR_ARG;
  double x[MSO_MAXW], r[MSO_MAXW], a[MSO_MAXW], r2;
  encode_contact(s, prim, o, d, t, x, &r2, NULL);
  mlp_forward(s, prim, x, r);
  activate(s, r, a);
  if (x_out) memcpy(x_out, x, (size_t)s->in_dim * sizeof(double));
  if (raw) memcpy(raw, r, (size_t)s->out_dim * sizeof(double));
  if (act) memcpy(act, a, (size_t)s->out_dim * sizeof(double));
  if (r2_out) *r2_out = r2;
  return MSO_OK;
}

int mso_render(const mso_scene *s, const mso_camera *cam, int H, int W, const mso_opts *opt,
               const int32_t *pix, int64_t n_pix, double *out_rgb, double *out_alpha,
               double *out_feat, mso_stats *stats) {
  if (!s || !cam || !opt || H <= 0 || W <= 0 || opt->K <= 0 || opt->tile < 0 || !out_rgb || !out_alpha)
    return MSO_ERR_ARG;
  if (s->mode == MSO_MODE_CONTACT && opt->K != 1) return MSO_ERR_ARG;
  if (s->order == MSO_ORDER_TILE && opt->tile <= 0) return MSO_ERR_ARG;   /* the shared order is a property of the tiling */
  if (s->in_dim > MSO_MAXW || s->width > MSO_MAXW || s->out_dim > MSO_MAXW) return MSO_ERR_ARG;
  if (!pix) n_pix = (int64_t)H * W;
  tlists_t tl; memset(&tl, 0, sizeof(tl));
  if (opt->tile > 0) {
    int rc = tlists_build(s, cam, H, W, opt->tile, &tl);
    if (rc != MSO_OK) return rc;
  }
  const tlists_t *tlp = opt->tile > 0 ? &tl : NULL;
  const int K = opt->K;
  const double t_stop = (double)opt->t_stop;
  const int nf = s->c_f ? s->c_f : s->n_feat;
  int64_t tot_hits = 0, tot_evals = 0, tot_term = 0;
  double min_T = 1.0;
  int failed = 0;
#ifdef _OPENMP
  int nt = opt->n_threads > 0 ? opt->n_threads : omp_get_max_threads();
#pragma omp parallel num_threads(nt) reduction(+ : tot_hits, tot_evals, tot_term) reduction(min : min_T)
#endif
  {
    raybuf_t rb; memset(&rb, 0, sizeof(rb));
    double x[MSO_MAXW], raw[MSO_MAXW], act[MSO_MAXW];
#ifdef _OPENMP
#pragma omp for schedule(dynamic, 64)
#endif
    for (int64_t q = 0; q < n_pix; ++q) {
      int pixel = pix ? pix[q] : (int)q;
      float o[3], d[3];
      long nh = gather_hits(s, cam, tlp, opt->tile, W, pixel, K, o, d, &rb);
      long ns = nh >= 0 ? build_samples(s, nh, K, &rb) : -1;
      if (ns < 0) {
#ifdef _OPENMP
#pragma omp atomic write
#endif
        failed = 1;
        continue;
      }
      tot_hits += nh;
      /* Eq.14: front-to-back, T_j = prod_{l<j} (1 - alpha_l) */
      double T = 1.0, C[3] = {0.0, 0.0, 0.0};
      double *F = out_feat ? out_feat + (size_t)q * nf : NULL;
      if (F) for (int c = 0; c < nf; ++c) F[c] = 0.0;
      for (long j = 0; j < ns; ++j) {
        const samp_t *sp = &rb.samps[j];
        double e;                                                     /* 1 - alpha */
        float dlt[3] = {0.f, 0.f, 0.f};
        if (s->mode == MSO_MODE_CONTACT) {
          double r2;
          encode_contact(s, sp->prim, o, d, sp->t, x, &r2, dlt);
          mlp_forward(s, sp->prim, x, raw);
          activate(s, raw, act);
          /* alpha = (1 - exp(-sigma l)) g,  g = exp(-falloff r2), falloff = 9/2 by default (readings: mso.h header) */
          e = 1.0 - (1.0 - exp(-act[3] * (double)rb.hits[sp->hit].delta)) * exp(-(double)s->falloff * r2);
        } else {
          float u[3];
          sample_u(s, sp->prim, o, d, sp->t, u);
          encode(s, u, d, x);
          mlp_forward(s, sp->prim, x, raw);
          activate(s, raw, act);
          e = exp(-act[3] * (double)rb.hits[sp->hit].delta);
        }
        ++tot_evals;
        double w = T * (1.0 - e);
        C[0] += w * act[0]; C[1] += w * act[1]; C[2] += w * act[2];
        if (F && s->c_f) {                                            /* Eq.7: f_i = sum_k g_ik e_ik, F += T alpha f_i */
          double g[4];
          slot_gates(s, sp->prim, dlt, g);
          const float *e0 = s->slots + (size_t)sp->prim * 4 * (size_t)nf;
          for (int c = 0; c < nf; ++c) {
            double f = 0.0;
            for (int k = 0; k < 4; ++k) f += g[k] * (double)e0[(size_t)k * nf + c];
            F[c] += w * f;
          }
        } else if (F) {
          for (int c = 0; c < nf; ++c) F[c] += w * act[4 + c];
        }
        T = T * e;
        if (T < t_stop) { ++tot_term; break; }                       /* P:437; NS (e) */
      }
      out_rgb[3 * q + 0] = C[0]; out_rgb[3 * q + 1] = C[1]; out_rgb[3 * q + 2] = C[2];
      out_alpha[q] = 1.0 - T;
      if (T < min_T) min_T = T;
    }
    raybuf_free(&rb);
  }
  if (stats) {
    stats->n_pixels = n_pix; stats->n_intervals = tot_hits; stats->n_samples = tot_hits * K;
    stats->n_mlp_evals = tot_evals; stats->n_terminated = tot_term;
    stats->n_pairs = (int64_t)tl.n; stats->min_T = min_T;
  }
  tlists_free(&tl);
  return failed ? MSO_ERR_MEM : MSO_OK;
}

int mso_hit_counts(const mso_scene *s, const mso_camera *cam, int H, int W, const mso_opts *opt,
                   int32_t *hit_count) {
  if (!s || !cam || !opt || !hit_count || opt->K <= 0) return MSO_ERR_ARG;
  tlists_t tl; memset(&tl, 0, sizeof(tl));
  if (opt->tile > 0) { int rc = tlists_build(s, cam, H, W, opt->tile, &tl); if (rc) return rc; }
  const tlists_t *tlp = opt->tile > 0 ? &tl : NULL;
  int failed = 0;
#ifdef _OPENMP
  int nt = opt->n_threads > 0 ? opt->n_threads : omp_get_max_threads();
#pragma omp parallel num_threads(nt)
#endif
  {
    raybuf_t rb; memset(&rb, 0, sizeof(rb));
#ifdef _OPENMP
#pragma omp for schedule(dynamic, 256)
#endif
    for (int64_t q = 0; q < (int64_t)H * W; ++q) {
      float o[3], d[3];
      long nh = gather_hits(s, cam, tlp, opt->tile, W, (int)q, opt->K, o, d, &rb);
      if (nh < 0) {
#ifdef _OPENMP
#pragma omp atomic write
#endif
        failed = 1;
        nh = 0;
      }
      hit_count[q] = (int32_t)nh;
    }
    raybuf_free(&rb);
  }
  tlists_free(&tl);
  return failed ? MSO_ERR_MEM : MSO_OK;
}

static int one_ray(const mso_scene *s, const mso_camera *cam, int H, int W, const mso_opts *opt,
                   int32_t pixel, raybuf_t *rb, long *nh, long *ns) {
  if (!s || !cam || !opt || opt->K <= 0 || pixel < 0 || pixel >= H * W) return MSO_ERR_ARG;
  tlists_t tl; memset(&tl, 0, sizeof(tl));
  if (opt->tile > 0) { int rc = tlists_build(s, cam, H, W, opt->tile, &tl); if (rc) return rc; }
  float o[3], d[3];
  *nh = gather_hits(s, cam, opt->tile > 0 ? &tl : NULL, opt->tile, W, pixel, opt->K, o, d, rb);
  tlists_free(&tl);
  if (*nh < 0) return MSO_ERR_MEM;
  if (ns) { *ns = build_samples(s, *nh, opt->K, rb); if (*ns < 0) return MSO_ERR_MEM; }
  return MSO_OK;
}

int mso_ray_intervals(const mso_scene *s, const mso_camera *cam, int H, int W, const mso_opts *opt,
                      int32_t pixel, int32_t *prim, float *t_in, float *delta, size_t cap, size_t *n) {
  raybuf_t rb; memset(&rb, 0, sizeof(rb));
  long nh = 0;
  int rc = one_ray(s, cam, H, W, opt, pixel, &rb, &nh, NULL);
  if (rc) { raybuf_free(&rb); return rc; }
  if (n) *n = (size_t)nh;
  if ((size_t)nh > cap) { raybuf_free(&rb); return MSO_ERR_CAP; }
  qsort(rb.hits, (size_t)nh, sizeof(hit_t), hit_cmp_prim);
  for (long j = 0; j < nh; ++j) {
    if (prim) prim[j] = rb.hits[j].prim;
    if (t_in) t_in[j] = rb.hits[j].t_in;
    if (delta) delta[j] = rb.hits[j].delta;
  }
  raybuf_free(&rb);
  return MSO_OK;
}

int mso_ray_samples(const mso_scene *s, const mso_camera *cam, int H, int W, const mso_opts *opt,
                    int32_t pixel, int32_t *prim, int32_t *k, float *t, size_t cap, size_t *n) {
  raybuf_t rb; memset(&rb, 0, sizeof(rb));
  long nh = 0, ns = 0;
  int rc = one_ray(s, cam, H, W, opt, pixel, &rb, &nh, &ns);
  if (rc) { raybuf_free(&rb); return rc; }
  if (n) *n = (size_t)ns;
  if ((size_t)ns > cap) { raybuf_free(&rb); return MSO_ERR_CAP; }
  for (long j = 0; j < ns; ++j) {
    if (prim) prim[j] = rb.samps[j].prim;
    if (k) k[j] = rb.samps[j].k;
    if (t) t[j] = rb.samps[j].t;
  }
  raybuf_free(&rb);
  return MSO_OK;
}

/* (primitive, k) of every sample of every pixel in compositing order; pixel q owns [K offsets[q], K offsets[q+1])
 * of mso_intervals_all's offsets.  The same gather_hits + build_samples the renderer runs. */
int mso_samples_all(const mso_scene *s, const mso_camera *cam, int H, int W, const mso_opts *opt,
                    int32_t *prim, int32_t *k, size_t cap, size_t *n) {
  if (!s || !cam || !opt || opt->K <= 0) return MSO_ERR_ARG;
  tlists_t tl; memset(&tl, 0, sizeof(tl));
  if (opt->tile > 0) { int rc = tlists_build(s, cam, H, W, opt->tile, &tl); if (rc) return rc; }
  const tlists_t *tlp = opt->tile > 0 ? &tl : NULL;
  raybuf_t rb; memset(&rb, 0, sizeof(rb));
  size_t tot = 0;
  int rc = MSO_OK;
  for (int64_t q = 0; q < (int64_t)H * W; ++q) {
    float o[3], d[3];
    long nh = gather_hits(s, cam, tlp, opt->tile, W, (int)q, opt->K, o, d, &rb);
    if (nh < 0) { rc = MSO_ERR_MEM; break; }
    long ns = build_samples(s, nh, opt->K, &rb);
    if (ns < 0) { rc = MSO_ERR_MEM; break; }
    for (long j = 0; j < ns; ++j, ++tot) {
      if (tot < cap) {
        if (prim) prim[tot] = rb.samps[j].prim;
        if (k) k[tot] = rb.samps[j].k;
      }
    }
  }
  if (n) *n = tot;
  raybuf_free(&rb);
  tlists_free(&tl);
  if (rc == MSO_OK && tot > cap) rc = MSO_ERR_CAP;
  return rc;
}

/* Intervals of every pixel (each ray's list sorted by primitive id): offsets[H*W+1]. */
int mso_intervals_all(const mso_scene *s, const mso_camera *cam, int H, int W, const mso_opts *opt,
                      int64_t *offsets, int32_t *prim, float *t_in, float *delta, size_t cap, size_t *n) {
  if (!s || !cam || !opt || !offsets || opt->K <= 0) return MSO_ERR_ARG;
  tlists_t tl; memset(&tl, 0, sizeof(tl));
  if (opt->tile > 0) { int rc = tlists_build(s, cam, H, W, opt->tile, &tl); if (rc) return rc; }
  const tlists_t *tlp = opt->tile > 0 ? &tl : NULL;
  raybuf_t rb; memset(&rb, 0, sizeof(rb));
  size_t tot = 0;
  int rc = MSO_OK;
  for (int64_t q = 0; q < (int64_t)H * W; ++q) {
    float o[3], d[3];
    offsets[q] = (int64_t)tot;
    long nh = gather_hits(s, cam, tlp, opt->tile, W, (int)q, opt->K, o, d, &rb);
    if (nh < 0) { rc = MSO_ERR_MEM; break; }
    qsort(rb.hits, (size_t)nh, sizeof(hit_t), hit_cmp_prim);
    for (long j = 0; j < nh; ++j, ++tot) {
      if (tot < cap) {
        if (prim) prim[tot] = rb.hits[j].prim;
        if (t_in) t_in[tot] = rb.hits[j].t_in;
        if (delta) delta[tot] = rb.hits[j].delta;
      }
    }
  }
  offsets[(int64_t)H * W] = (int64_t)tot;
  if (n) *n = tot;
  raybuf_free(&rb);
  tlists_free(&tl);
  if (rc == MSO_OK && tot > cap) rc = MSO_ERR_CAP;
  return rc;
}
