/* mso_grad.c -- CPU ORACLE of the BACKWARD pass of the MLP-Splatting render (S:Sec.8(f) NEXT-4).
 *
 * TEST INFRASTRUCTURE, NOT THE PRODUCT (same rules as mso.c / mso.h).  Written from the paper before any
 * backward kernel exists: the losses of P:132-134 (Eq.8; here its L1 term, lambda = 0 -- the SSIM term needs whole
 * images and is out of scope) need dL/dtheta_i and dL/d(mu_i, s_i, q_i) of
 *     C = sum_j T_j alpha_j c_j,  T_j = prod_{l<j} (1 - alpha_l),  alpha_j = 1 - exp(-sigma_j delta)      P:113-115 Eq.6,
 *                                                                                                          P:513-516 Eq.14
 * through the per-primitive MLP (c = sigmoid, sigma = softplus), the encoding (Eq.5 with identity,
 * DESIGN.md Q3), the local coordinate u = S^-1 R^T (p - mu) and the chord interval [t_in, t_out] with its
 * K midpoint samples (north_star (c); Q1, Q7).  North-star (K-sample) mode only.
 *
 * Everything here is fp64 -- geometry included -- so that the function is smooth where it should be and central
 * finite differences pin the gradients (tests/test_oracle_grad_pins.py); the same tests check that this fp64
 * forward is the render of mso.c (canonical fp32 geometry) to rounding.  Candidates: every primitive against every
 * ray (brute force; the binning of mso.c is conservative, pin P6, so the sets agree).
 *
 * The forward is the algorithm of mso.c step by step; the backward is the chain rule written out:
 *   g = dL/dC (sign(C - target) for the L1 loss, or given)
 *   dL/dc_j = T_j alpha_j g;   dL/de_j = -T_j (c_j.g) + (sum_{m>j} T_m alpha_m (c_m.g)) / e_j,   e_j = exp(-sigma_j delta)
 *   dL/dsigma_j = -delta e_j dL/de_j;   dL/ddelta += -sigma_j e_j dL/de_j
 *   MLP backward -> dL/dtheta, dL/dx;   Eq.5: dL/du = dx_id + sum_l 2^l pi (cos dx_sin - sin dx_cos)
 *   u = o' + t d' (o' = A (o - mu), d' = A d):   dL/do' += du, dL/dd' += t du, dL/dt = du.d'
 *   t_k = t_in + (k + 1/2) delta,  delta = (t1 - t_in)/K,  t_in = max(t0, t_near)
 *   t0,1 = (-b -+ s)/a,  s = sqrt(b^2 - a c),  a = d'.d', b = o'.d', c = o'.o' - 1
 *   A = diag(1/s) R(q/|q|)^T -> dL/ds, dL/dq;  dL/dmu = -A^T dL/do'
 * Samples behind the early stop (T < t_stop after a sample, Q9) carry no weight and no gradient.
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>

#include "mso.h"

#define PI 3.14159265358979323846

typedef struct {
  int prim, k, hit;
  double t;
} gs_samp;

typedef struct {
  int prim;
  double A[9], op[3], dp[3];     /* A, o' = A (o - mu), d' = A d */
  double a, b, c, s, t0, t1, t_in, delta;
  int clamped;                   /* t_in == t_near */
  double g_op[3], g_dp[3], g_tin, g_delta;   /* accumulated gradients */
} gs_hit;

static int samp_cmp(const void *pa, const void *pb) {
  const gs_samp *a = (const gs_samp *)pa, *b = (const gs_samp *)pb;
  if (a->t < b->t) return -1;
  if (a->t > b->t) return 1;
  if (a->prim != b->prim) return a->prim < b->prim ? -1 : 1;
  return a->k < b->k ? -1 : (a->k > b->k ? 1 : 0);
}

static void quat_rot(const double *q, double *R, double *qn, double *nrm) {
  double n = sqrt(q[0] * q[0] + q[1] * q[1] + q[2] * q[2] + q[3] * q[3]);
  double w = q[0] / n, x = q[1] / n, y = q[2] / n, z = q[3] / n;
  qn[0] = w; qn[1] = x; qn[2] = y; qn[3] = z; *nrm = n;
  R[0] = 1 - 2 * (y * y + z * z); R[1] = 2 * (x * y - w * z); R[2] = 2 * (x * z + w * y);
  R[3] = 2 * (x * y + w * z); R[4] = 1 - 2 * (x * x + z * z); R[5] = 2 * (y * z - w * x);
  R[6] = 2 * (x * z - w * y); R[7] = 2 * (y * z + w * x); R[8] = 1 - 2 * (x * x + y * y);
}

int mso_loss_grad_f64(int32_t n, const double *center, const double *quat, const double *scale,
                      const double *weights, const mso_mlp *mlp, const mso_camera *cam, int H, int W, int K,
                      double t_stop, const int32_t *pix, int64_t n_pix, const double *target, const double *g_in,
                      double *loss, double *rgb_out, double *g_weights, double *g_center, double *g_quat,
                      double *g_scale) {
  if (n <= 0 || !center || !quat || !scale || !weights || !mlp || !cam || K <= 0 || n_pix < 0) return MSO_ERR_ARG;
  if (mlp->mode != MSO_MODE_LOCAL) return MSO_ERR_ARG;
  const int L = mlp->n_freq, vd = mlp->use_viewdir ? 1 : 0, nh = mlp->n_hidden, Wd = mlp->width;
  const int in_dim = 3 + 6 * L + 3 * vd, out_dim = 4 + mlp->n_feat, n_layers = nh + 1;
  int params = 0, li = in_dim, max_w = in_dim > out_dim ? in_dim : out_dim;
  if (Wd > max_w) max_w = Wd;
  for (int l = 0; l < n_layers; ++l) { int o = l == nh ? out_dim : Wd; params += li * o + o; li = o; }
  const int want_grad = g_weights || g_center || g_quat || g_scale;
  if (g_weights) memset(g_weights, 0, sizeof(double) * (size_t)n * params);
  if (g_center) memset(g_center, 0, sizeof(double) * (size_t)n * 3);
  if (g_quat) memset(g_quat, 0, sizeof(double) * (size_t)n * 4);
  if (g_scale) memset(g_scale, 0, sizeof(double) * (size_t)n * 3);

  double *Aall = (double *)malloc(sizeof(double) * (size_t)n * 9);
  double *Rall = (double *)malloc(sizeof(double) * (size_t)n * 9);
  double *gA = (double *)calloc((size_t)n * 9, sizeof(double));
  gs_hit *hits = (gs_hit *)malloc(sizeof(gs_hit) * (size_t)n);
  gs_samp *samps = (gs_samp *)malloc(sizeof(gs_samp) * (size_t)n * K);
  /* per sample: activations of every layer (for the backward), e, c, raw */
  const size_t act_stride = (size_t)(n_layers + 1) * max_w;
  double *acts = (double *)malloc(sizeof(double) * (size_t)n * K * act_stride);
  double *se = (double *)malloc(sizeof(double) * (size_t)n * K * 8);   /* e, T, c[3], sigma, raw3, - */
  double *gx = (double *)malloc(sizeof(double) * 2 * (size_t)max_w);
  if (!Aall || !Rall || !gA || !hits || !samps || !acts || !se || !gx) {
    free(Aall); free(Rall); free(gA); free(hits); free(samps); free(acts); free(se); free(gx);
    return MSO_ERR_MEM;
  }
  for (int i = 0; i < n; ++i) {
    double qn[4], nr;
    quat_rot(quat + 4 * i, Rall + 9 * i, qn, &nr);
    for (int r = 0; r < 3; ++r)
      for (int c = 0; c < 3; ++c) Aall[9 * i + 3 * r + c] = Rall[9 * i + 3 * c + r] / scale[3 * i + r];
  }
  const double fx = cam->fx, fy = cam->fy, cx = cam->cx, cy = cam->cy, t_near = cam->t_near;
  const float *m = cam->c2w;
  const double o[3] = {m[3], m[7], m[11]};
  double total = 0.0;

  for (int64_t pi = 0; pi < n_pix; ++pi) {
    const int q = pix ? pix[pi] : (int)pi;
    const int px = q % W, py = q / W;
    (void)H;
    const double dcx = (px + 0.5 - cx) / fx, dcy = (py + 0.5 - cy) / fy;
    double d[3] = {m[0] * dcx + m[1] * dcy + m[2], m[4] * dcx + m[5] * dcy + m[6], m[8] * dcx + m[9] * dcy + m[10]};
    const double dn = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
    d[0] /= dn; d[1] /= dn; d[2] /= dn;
    /* ---- intervals ---- */
    int nhit = 0;
    for (int i = 0; i < n; ++i) {
      gs_hit h; memset(&h, 0, sizeof(h));
      h.prim = i;
      memcpy(h.A, Aall + 9 * i, sizeof(h.A));
      const double v[3] = {o[0] - center[3 * i], o[1] - center[3 * i + 1], o[2] - center[3 * i + 2]};
      for (int r = 0; r < 3; ++r) {
        h.op[r] = h.A[3 * r] * v[0] + h.A[3 * r + 1] * v[1] + h.A[3 * r + 2] * v[2];
        h.dp[r] = h.A[3 * r] * d[0] + h.A[3 * r + 1] * d[1] + h.A[3 * r + 2] * d[2];
      }
      h.a = h.dp[0] * h.dp[0] + h.dp[1] * h.dp[1] + h.dp[2] * h.dp[2];
      h.b = h.op[0] * h.dp[0] + h.op[1] * h.dp[1] + h.op[2] * h.dp[2];
      h.c = h.op[0] * h.op[0] + h.op[1] * h.op[1] + h.op[2] * h.op[2] - 1.0;
      const double disc = h.b * h.b - h.a * h.c;
      if (!(disc > 0.0)) continue;
      h.s = sqrt(disc);
      h.t0 = (-h.b - h.s) / h.a; h.t1 = (-h.b + h.s) / h.a;
      if (!(h.t1 > t_near)) continue;
      h.clamped = !(h.t0 > t_near);
      h.t_in = h.clamped ? t_near : h.t0;
      h.delta = (h.t1 - h.t_in) / K;
      if (!(h.delta > 0.0)) continue;
      hits[nhit++] = h;
    }
    int ns = 0;
    for (int hi = 0; hi < nhit; ++hi)
      for (int k = 0; k < K; ++k) {
        samps[ns].prim = hits[hi].prim; samps[ns].k = k; samps[ns].hit = hi;
        samps[ns].t = hits[hi].t_in + (k + 0.5) * hits[hi].delta;
        ++ns;
      }
    qsort(samps, (size_t)ns, sizeof(gs_samp), samp_cmp);
    /* ---- forward: MLP per sample, compositing with the early stop ---- */
    double T = 1.0, C[3] = {0, 0, 0};
    int n_used = 0;
    for (int j = 0; j < ns; ++j) {
      const gs_samp *sp = &samps[j];
      const gs_hit *h = &hits[sp->hit];
      double *x = acts + (size_t)j * act_stride;
      double u[3];
      for (int r = 0; r < 3; ++r) u[r] = h->op[r] + sp->t * h->dp[r];
      int ni = 0;
      x[ni++] = u[0]; x[ni++] = u[1]; x[ni++] = u[2];
      for (int l = 0; l < L; ++l) {
        const double f = ldexp(PI, l);
        for (int r = 0; r < 3; ++r) x[ni + r] = sin(f * u[r]);
        for (int r = 0; r < 3; ++r) x[ni + 3 + r] = cos(f * u[r]);
        ni += 6;
      }
      if (vd) { x[ni++] = d[0]; x[ni++] = d[1]; x[ni++] = d[2]; }
      const double *w = weights + (size_t)sp->prim * params;
      int nin = in_dim;
      for (int l = 0; l < n_layers; ++l) {
        const int no = l == nh ? out_dim : Wd;
        const double *bias = w + (size_t)nin * no;
        double *src = acts + (size_t)j * act_stride + (size_t)l * max_w, *dst = src + max_w;
        for (int oo = 0; oo < no; ++oo) {
          double acc = bias[oo];
          for (int i = 0; i < nin; ++i) acc += src[i] * w[(size_t)i * no + oo];
          dst[oo] = (l == nh) ? acc : (acc > 0.0 ? acc : 0.0);
        }
        w = bias + no; nin = no;
      }
      const double *raw = acts + (size_t)j * act_stride + (size_t)n_layers * max_w;
      double *s8 = se + (size_t)j * 8;
      for (int c = 0; c < 3; ++c) s8[2 + c] = 1.0 / (1.0 + exp(-raw[c]));
      const double sigma = (raw[3] > 0 ? raw[3] : 0.0) + log1p(exp(-fabs(raw[3])));
      s8[5] = sigma; s8[6] = raw[3];
      const double e = exp(-sigma * h->delta);
      s8[0] = e; s8[1] = T;
      const double wgt = T * (1.0 - e);
      for (int c = 0; c < 3; ++c) C[c] += wgt * s8[2 + c];
      T *= e;
      n_used = j + 1;
      if (T < t_stop) break;                       /* Q9: the stopping sample still contributes */
    }
    if (rgb_out) { rgb_out[3 * pi] = C[0]; rgb_out[3 * pi + 1] = C[1]; rgb_out[3 * pi + 2] = C[2]; }
    double g[3] = {0, 0, 0};
    for (int c = 0; c < 3; ++c) {
      if (target) {
        const double df = C[c] - target[3 * pi + c];
        total += fabs(df);
        g[c] = df > 0 ? 1.0 : (df < 0 ? -1.0 : 0.0);
      }
      if (g_in) g[c] = g_in[3 * pi + c];           /* a given dL/dC overrides the L1 sign */
    }
    if (!want_grad) continue;
    /* ---- backward ---- */
    double suffix = 0.0;
    for (int j = n_used - 1; j >= 0; --j) {
      const gs_samp *sp = &samps[j];
      gs_hit *h = &hits[sp->hit];
      const double *s8 = se + (size_t)j * 8;
      const double e = s8[0], Tj = s8[1], sigma = s8[5], raw3 = s8[6];
      const double cg = s8[2] * g[0] + s8[3] * g[1] + s8[4] * g[2];
      const double g_e = -Tj * cg + suffix / e;
      suffix += Tj * (1.0 - e) * cg;
      double *graw = gx;                       /* dL/draw[out_dim] */
      for (int c = 0; c < out_dim; ++c) graw[c] = 0.0;
      for (int c = 0; c < 3; ++c) graw[c] = Tj * (1.0 - e) * g[c] * s8[2 + c] * (1.0 - s8[2 + c]);
      const double g_sigma = -h->delta * e * g_e;
      graw[3] = g_sigma / (1.0 + exp(-raw3));  /* softplus' = sigmoid */
      h->g_delta += -sigma * e * g_e;
      /* MLP backward */
      double *gcur = gx, *gnext = gx + max_w;
      int off_w[8], ins[8], outs[8];
      {
        int off = 0, nin = in_dim;
        for (int l = 0; l < n_layers; ++l) {
          const int no = l == nh ? out_dim : Wd;
          off_w[l] = off; ins[l] = nin; outs[l] = no;
          off += nin * no + no; nin = no;
        }
      }
      const double *wp = weights + (size_t)sp->prim * params;
      double *gw = g_weights ? g_weights + (size_t)sp->prim * params : NULL;
      for (int l = n_layers - 1; l >= 0; --l) {
        const int nin = ins[l], no = outs[l];
        const double *src = acts + (size_t)j * act_stride + (size_t)l * max_w;     /* layer input */
        const double *out = src + max_w;                                           /* layer output */
        if (l != nh)
          for (int oo = 0; oo < no; ++oo) if (!(out[oo] > 0.0)) gcur[oo] = 0.0;   /* ReLU */
        const double *w = wp + off_w[l];
        for (int i = 0; i < nin; ++i) {
          double acc = 0.0;
          for (int oo = 0; oo < no; ++oo) {
            acc += w[(size_t)i * no + oo] * gcur[oo];
            if (gw) gw[off_w[l] + (size_t)i * no + oo] += src[i] * gcur[oo];
          }
          gnext[i] = acc;
        }
        if (gw) for (int oo = 0; oo < no; ++oo) gw[off_w[l] + (size_t)nin * no + oo] += gcur[oo];
        double *tmp = gcur; gcur = gnext; gnext = tmp;
      }
      /* gcur = dL/dx[in_dim] -> dL/du (Eq.5) */
      const double *x = acts + (size_t)j * act_stride;
      double gu[3] = {gcur[0], gcur[1], gcur[2]};
      for (int l = 0; l < L; ++l) {
        const double f = ldexp(PI, l);
        for (int r = 0; r < 3; ++r) {
          const double sn = x[3 + 6 * l + r], cs = x[3 + 6 * l + 3 + r];
          gu[r] += f * (cs * gcur[3 + 6 * l + r] - sn * gcur[3 + 6 * l + 3 + r]);
        }
      }
      double gt = 0.0;
      for (int r = 0; r < 3; ++r) {
        h->g_op[r] += gu[r];
        h->g_dp[r] += sp->t * gu[r];
        gt += gu[r] * h->dp[r];
      }
      h->g_tin += gt;
      h->g_delta += (sp->k + 0.5) * gt;
    }
    /* ---- per hit: interval -> (o', d') -> (A, mu) ---- */
    for (int hi = 0; hi < nhit; ++hi) {
      gs_hit *h = &hits[hi];
      const double G1 = h->g_delta / K;
      double G0 = h->g_tin - h->g_delta / K;
      if (h->clamped) G0 = 0.0;
      const double ia = 1.0 / h->a;
      const double gb = -(G0 + G1) * ia + (G1 - G0) * ia * h->b / h->s;
      const double ga = -(G0 * h->t0 + G1 * h->t1) * ia - (G1 - G0) * ia * h->c / (2.0 * h->s);
      const double gc = -(G1 - G0) / (2.0 * h->s);
      double gop[3], gdp[3];
      for (int r = 0; r < 3; ++r) {
        gop[r] = h->g_op[r] + h->dp[r] * gb + 2.0 * h->op[r] * gc;
        gdp[r] = h->g_dp[r] + 2.0 * h->dp[r] * ga + h->op[r] * gb;
      }
      const int i = h->prim;
      const double v[3] = {o[0] - center[3 * i], o[1] - center[3 * i + 1], o[2] - center[3 * i + 2]};
      for (int r = 0; r < 3; ++r)
        for (int c = 0; c < 3; ++c) gA[9 * i + 3 * r + c] += gop[r] * v[c] + gdp[r] * d[c];
      if (g_center)
        for (int c = 0; c < 3; ++c)
          g_center[3 * i + c] -= h->A[c] * gop[0] + h->A[3 + c] * gop[1] + h->A[6 + c] * gop[2];
    }
  }
  /* ---- A = diag(1/s) R^T -> scale, quaternion ---- */
  if (g_scale || g_quat)
    for (int i = 0; i < n; ++i) {
      double G[9];                                  /* dL/dR */
      for (int r = 0; r < 3; ++r)
        for (int c = 0; c < 3; ++c) {
          const double ga = gA[9 * i + 3 * r + c];
          if (g_scale) g_scale[3 * i + r] -= ga * Aall[9 * i + 3 * r + c] / scale[3 * i + r];
          G[3 * c + r] = ga / scale[3 * i + r];     /* A[r][c] = R[c][r] / s[r] */
        }
      if (g_quat) {
        double R[9], qn[4], nr;
        quat_rot(quat + 4 * i, R, qn, &nr);
        const double w = qn[0], x = qn[1], y = qn[2], z = qn[3];
        double gq[4];
        gq[0] = 2 * (-z * G[1] + y * G[2] + z * G[3] - x * G[5] - y * G[6] + x * G[7]);
        gq[1] = 2 * (y * G[1] + z * G[2] + y * G[3] - 2 * x * G[4] - w * G[5] + z * G[6] + w * G[7] - 2 * x * G[8]);
        gq[2] = 2 * (-2 * y * G[0] + x * G[1] + w * G[2] + x * G[3] + z * G[5] - w * G[6] + z * G[7] - 2 * y * G[8]);
        gq[3] = 2 * (-2 * z * G[0] - w * G[1] + x * G[2] + w * G[3] - 2 * z * G[4] + y * G[5] + x * G[6] + y * G[7]);
        const double dot = gq[0] * qn[0] + gq[1] * qn[1] + gq[2] * qn[2] + gq[3] * qn[3];
        for (int c = 0; c < 4; ++c) g_quat[4 * i + c] = (gq[c] - dot * qn[c]) / nr;   /* through q / |q| */
      }
    }
  if (loss) *loss = total;
  free(Aall); free(Rall); free(gA); free(hits); free(samps); free(acts); free(se); free(gx);
  return MSO_OK;
}
