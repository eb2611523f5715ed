// ms_backward.cu -- backward pass of the render, fp32 SIMT (S:Sec.8(f) NEXT-4; the losses of P:132-134 Eq.8 need
// dL/dtheta_i and dL/d(mu_i, s_i, q_i)).  North-star (K-sample) mode.  After the forward stages (a)-(d) and the
// compositing backward of ms_composite.cu (which leaves (dL/dc, dL/de) per sample):
//   mlp_bwd_kernel       one CTA per 128-sample row block of one primitive, one thread per sample: recomputes the
//                        sample's activations into shared memory, backpropagates through sigmoid / softplus,
//                        the Linear+ReLU layers and Eq.5; the weight gradients of the block are the
//                        contractions X_l^T G_l over its 128 samples (threads over (in, out) pairs), added to
//                        g_weights with one atomic per weight and block; dL/du goes on to the interval:
//                        u = o' + t d'  ->  dL/do' += du, dL/dd' += t du, dL/dt_in += du.d', dL/ddelta += (k+1/2) du.d'
//   interval_bwd_kernel  one thread per (ray, primitive) interval: through delta = (t1 - t_in)/K, t_in = max(t0, t_near),
//                        t0,1 = (-b -+ s)/a, s = sqrt(b^2 - a c), a = d'.d', b = o'.d', c = o'.o' - 1 to (o', d'), then
//                        o' = A (o - mu), d' = A d: dL/dA += ..., dL/dmu -= A^T dL/do'
//   prim_bwd_kernel      one thread per primitive: A = diag(1/s) R(q/|q|)^T  ->  dL/ds, dL/dq
// Written from the chain rule itself; it shares no code with the test oracle, which states the same chain in fp64.
#include "ms_internal.cuh"

namespace {

constexpr int BT = MS_ROWS;   // threads per CTA = samples per row block

// odd leading dimension: a thread walking its own row and a warp walking one column are both conflict-free
__host__ __device__ inline int ld_of(int n) { return n | 1; }

struct BwdLayout {
  int ld0, ldw, ldg;          // leading dimensions of X0 (encoded input), H_l (hidden), G (gradients)
  size_t off_h[5];            // float offsets of X0 (index 0) and H_1..H_nh
  size_t off_g0, off_g1;      // the two gradient buffers
  size_t floats;
};
__host__ __device__ inline BwdLayout bwd_layout(const MsMlpShape &sh) {
  BwdLayout L;
  L.ld0 = ld_of(sh.in_dim); L.ldw = ld_of(sh.width);
  const int gmax = sh.width > sh.in_dim ? sh.width : sh.in_dim;
  L.ldg = ld_of(gmax);
  size_t o = 0;
  L.off_h[0] = o; o += (size_t)BT * L.ld0;
  for (int l = 1; l <= sh.n_hidden; ++l) { L.off_h[l] = o; o += (size_t)BT * L.ldw; }
  L.off_g0 = o; o += (size_t)BT * L.ldg;
  L.off_g1 = o; o += (size_t)BT * L.ldg;
  L.floats = o;
  return L;
}

__device__ __forceinline__ int find_seg(const uint32_t *__restrict__ bo, int n, uint32_t base, uint32_t b) {
  int lo = 0, hi = n;
  while (hi - lo > 1) {
    int mid = (lo + hi) >> 1;
    if (bo[mid] - base <= b) lo = mid; else hi = mid;
  }
  return lo;
}

__global__ void __launch_bounds__(BT) mlp_bwd_kernel(MsMlpBwdArgs a) {
  extern __shared__ __align__(16) float sm[];
  __shared__ int s_seg;
  const MsMlpShape &sh = a.shape;
  const BwdLayout L = bwd_layout(sh);
  const int tid = threadIdx.x;
  const uint2 r = *a.segs.range;
  const uint32_t *bo = a.segs.blk_off + r.x;
  const uint32_t base = bo[0], n_blocks = bo[r.y - r.x] - base;
  const int nh = sh.n_hidden, NL = nh + 1;
  for (uint32_t blk = blockIdx.x; blk < n_blocks; blk += gridDim.x) {
    __syncthreads();
    if (tid == 0) s_seg = find_seg(bo, (int)(r.y - r.x), base, blk);
    __syncthreads();
    const uint32_t g = r.x + (uint32_t)s_seg;
    const int prim = a.segs.prim ? (int)a.segs.prim[g] : (int)g;
    const uint32_t first = a.segs.iv0[g], count = a.segs.cnt ? a.segs.cnt[g] : a.segs.iv0[g + 1] - first;
    const uint64_t srow = (uint64_t)(blk - (bo[s_seg] - base)) * BT + tid;
    const uint32_t j = (uint32_t)(srow / (uint32_t)a.K);
    const int k = (int)(srow % (uint32_t)a.K);
    const bool live = j < count;
    const float *wp = a.weights_f32 + (size_t)prim * sh.params;
    const float *Ap = a.A + 9 * (size_t)prim, *mu = a.center + 3 * (size_t)prim;
    MsInterval iv;
    iv.t_in = 0.f; iv.delta = 0.f; iv.slot = 0; iv.dx = 0.f; iv.dy = 0.f; iv.dz = 1.f; iv.ray = 0; iv.prim = prim;
    if (live) iv = a.intervals[first + j];
    const float d[3] = {iv.dx, iv.dy, iv.dz};
    const float t = ms_sample_t(iv.t_in, iv.delta, k);
    float u[3];
    ms_sample_u(Ap, mu, a.cam.o, d, t, u);
    // ---- forward, activations into shared memory (a dead row carries zeros) ----
    float *X0 = sm + L.off_h[0] + (size_t)tid * L.ld0;
    {
      int ni = 0;
      X0[ni++] = u[0]; X0[ni++] = u[1]; X0[ni++] = u[2];
      float scale = 1.0f;
      for (int l = 0; l < sh.n_freq; ++l) {
        float sv[3], cv[3];
#pragma unroll
        for (int c = 0; c < 3; ++c) sincospif(scale * u[c], &sv[c], &cv[c]);
        X0[ni++] = sv[0]; X0[ni++] = sv[1]; X0[ni++] = sv[2];
        X0[ni++] = cv[0]; X0[ni++] = cv[1]; X0[ni++] = cv[2];
        scale *= 2.0f;
      }
      if (sh.use_viewdir) { X0[ni++] = d[0]; X0[ni++] = d[1]; X0[ni++] = d[2]; }
    }
    int off_w[5], n_in_l[5];
    {
      int off = 0, nin = sh.in_dim;
      for (int l = 0; l < NL; ++l) {
        const int no = l == nh ? sh.out_dim : sh.width;
        off_w[l] = off; n_in_l[l] = nin;
        off += nin * no + no; nin = no;
      }
    }
    for (int l = 0; l < nh; ++l) {
      const float *src = sm + L.off_h[l] + (size_t)tid * (l == 0 ? L.ld0 : L.ldw);
      float *dst = sm + L.off_h[l + 1] + (size_t)tid * L.ldw;
      const float *w = wp + off_w[l];
      const int nin = n_in_l[l], no = sh.width;
      const float *bias = w + nin * no;
      for (int o = 0; o < no; ++o) {
        float acc = __ldg(bias + o);
        for (int i = 0; i < nin; ++i) acc = fmaf(src[i], __ldg(w + i * no + o), acc);
        dst[o] = acc > 0.0f ? acc : 0.0f;
      }
    }
    float raw[4];
    {
      const float *src = sm + L.off_h[nh] + (size_t)tid * L.ldw;
      const float *w = wp + off_w[nh];
      const int nin = sh.width, no = sh.out_dim;
#pragma unroll
      for (int o = 0; o < 4; ++o) {
        float acc = __ldg(w + nin * no + o);
        for (int i = 0; i < nin; ++i) acc = fmaf(src[i], __ldg(w + i * no + o), acc);
        raw[o] = acc;
      }
    }
    // ---- gradient of the head's four outputs ----
    float *G = sm + L.off_g0, *Gn = sm + L.off_g1;
    float g_delta = 0.0f;
    {
      float gr[4] = {0.f, 0.f, 0.f, 0.f};
      if (live) {
        const size_t idx = (size_t)(uint32_t)iv.slot * (size_t)a.K + (size_t)k;
        const float4 gs = a.gstage[idx];
        const float e = a.staging[idx].w;
        const float c0 = 1.0f / (1.0f + expf(-raw[0])), c1 = 1.0f / (1.0f + expf(-raw[1])), c2 = 1.0f / (1.0f + expf(-raw[2]));
        gr[0] = gs.x * c0 * (1.0f - c0); gr[1] = gs.y * c1 * (1.0f - c1); gr[2] = gs.z * c2 * (1.0f - c2);
        const float sigma = fmaxf(raw[3], 0.0f) + log1pf(expf(-fabsf(raw[3])));
        gr[3] = -iv.delta * e * gs.w / (1.0f + expf(-raw[3]));     // softplus' = sigmoid
        g_delta = -sigma * e * gs.w;
      }
      float *gp = G + (size_t)tid * L.ldg;
#pragma unroll
      for (int o = 0; o < 4; ++o) gp[o] = gr[o];
    }
    // ---- layers, last to first: weight gradients of the block, then the gradient of the layer's input ----
    for (int l = nh; l >= 0; --l) {
      __syncthreads();                                   // G of every sample is written
      const int nin = n_in_l[l];
      const int no_ld = l == nh ? sh.out_dim : sh.width;   // stride of W's rows
      const int no = l == nh ? 4 : sh.width;               // outputs that carry a gradient
      const float *Xl = sm + L.off_h[l];
      const int ldx = l == 0 ? L.ld0 : L.ldw;
      float *gw = a.g_weights + (size_t)prim * sh.params + off_w[l];
      for (int idx = tid; idx < nin * no; idx += BT) {
        const int i = idx / no, o = idx - i * no;
        float acc = 0.0f;
        for (int s = 0; s < BT; ++s) acc = fmaf(Xl[(size_t)s * ldx + i], G[(size_t)s * L.ldg + o], acc);
        if (acc != 0.0f) atomicAdd(gw + i * no_ld + o, acc);
      }
      for (int o = tid; o < no; o += BT) {
        float acc = 0.0f;
        for (int s = 0; s < BT; ++s) acc += G[(size_t)s * L.ldg + o];
        if (acc != 0.0f) atomicAdd(gw + nin * no_ld + o, acc);
      }
      // gradient of this thread's layer input (ReLU of the previous layer folded in)
      const float *w = wp + off_w[l];
      const float *gp = G + (size_t)tid * L.ldg;
      const float *xin = Xl + (size_t)tid * ldx;
      float *gn = Gn + (size_t)tid * L.ldg;
      for (int i = 0; i < nin; ++i) {
        float acc = 0.0f;
        for (int o = 0; o < no; ++o) acc = fmaf(__ldg(w + i * no_ld + o), gp[o], acc);
        gn[i] = (l > 0 && !(xin[i] > 0.0f)) ? 0.0f : acc;
      }
      float *tmp = G; G = Gn; Gn = tmp;
    }
    // ---- Eq.5: dL/du, then the interval ----
    if (live) {
      const float *gx = G + (size_t)tid * L.ldg;
      float gu[3] = {gx[0], gx[1], gx[2]};
      float scale = 3.14159265358979323846f;
      for (int l = 0; l < sh.n_freq; ++l) {
#pragma unroll
        for (int c = 0; c < 3; ++c) {
          const float sn = X0[3 + 6 * l + c], cs = X0[3 + 6 * l + 3 + c];
          gu[c] += scale * (cs * gx[3 + 6 * l + c] - sn * gx[3 + 6 * l + 3 + c]);
        }
        scale *= 2.0f;
      }
      float dp[3];
#pragma unroll
      for (int rr = 0; rr < 3; ++rr) dp[rr] = Ap[3 * rr] * d[0] + Ap[3 * rr + 1] * d[1] + Ap[3 * rr + 2] * d[2];
      const float gt = gu[0] * dp[0] + gu[1] * dp[1] + gu[2] * dp[2];
      float *ig = a.ivgrad + (size_t)(first + j) * 8;
      atomicAdd(ig + 0, gu[0]); atomicAdd(ig + 1, gu[1]); atomicAdd(ig + 2, gu[2]);
      atomicAdd(ig + 3, t * gu[0]); atomicAdd(ig + 4, t * gu[1]); atomicAdd(ig + 5, t * gu[2]);
      atomicAdd(ig + 6, gt);
      atomicAdd(ig + 7, ((float)k + 0.5f) * gt + g_delta);
    }
  }
}

// The same computation for hidden widths 8 / 16 / 32 / 64 (a multiple of 4: weight rows are 16-byte aligned): the
// layer outputs and gradients of a thread's sample live in registers while a weight row streams through float4
// loads (one row feeds WD FMAs), and the weight gradients are register tiles of 4 inputs x (WD / 32 or 1) outputs per
// lane, so a shared-memory load feeds several FMAs.  Arithmetic order of the sums differs from the generic kernel
// (and from the oracle) only in the order fp32 atomics arrive.
template <int WD>
__global__ void __launch_bounds__(BT) mlp_bwd_fast_kernel(MsMlpBwdArgs a) {
  extern __shared__ __align__(16) float sm[];
  __shared__ int s_seg;
  const MsMlpShape &sh = a.shape;
  const BwdLayout L = bwd_layout(sh);
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const uint2 r = *a.segs.range;
  const uint32_t *bo = a.segs.blk_off + r.x;
  const uint32_t base = bo[0], n_blocks = bo[r.y - r.x] - base;
  const int nh = sh.n_hidden, NL = nh + 1;
  int off_w[5], n_in_l[5];
  {
    int off = 0, nin = sh.in_dim;
    for (int l = 0; l < NL; ++l) {
      const int no = l == nh ? sh.out_dim : WD;
      off_w[l] = off; n_in_l[l] = nin;
      off += nin * no + no; nin = no;
    }
  }
  for (uint32_t blk = blockIdx.x; blk < n_blocks; blk += gridDim.x) {
    __syncthreads();
    if (tid == 0) s_seg = find_seg(bo, (int)(r.y - r.x), base, blk);
    __syncthreads();
    const uint32_t g = r.x + (uint32_t)s_seg;
    const int prim = a.segs.prim ? (int)a.segs.prim[g] : (int)g;
    const uint32_t first = a.segs.iv0[g], count = a.segs.cnt ? a.segs.cnt[g] : a.segs.iv0[g + 1] - first;
    const uint64_t srow = (uint64_t)(blk - (bo[s_seg] - base)) * BT + tid;
    const uint32_t j = (uint32_t)(srow / (uint32_t)a.K);
    const int k = (int)(srow % (uint32_t)a.K);
    const bool live = j < count;
    const float *wp = a.weights_f32 + (size_t)prim * sh.params;
    const float *Ap = a.A + 9 * (size_t)prim, *mu = a.center + 3 * (size_t)prim;
    MsInterval iv;
    iv.t_in = 0.f; iv.delta = 0.f; iv.slot = 0; iv.dx = 0.f; iv.dy = 0.f; iv.dz = 1.f; iv.ray = 0; iv.prim = prim;
    if (live) iv = a.intervals[first + j];
    const float d[3] = {iv.dx, iv.dy, iv.dz};
    const float t = ms_sample_t(iv.t_in, iv.delta, k);
    float u[3];
    ms_sample_u(Ap, mu, a.cam.o, d, t, u);
    float *X0 = sm + L.off_h[0] + (size_t)tid * L.ld0;
    {
      int ni = 0;
      X0[ni++] = u[0]; X0[ni++] = u[1]; X0[ni++] = u[2];
      float scale = 1.0f;
      for (int l = 0; l < sh.n_freq; ++l) {
        float sv[3], cv[3];
#pragma unroll
        for (int c = 0; c < 3; ++c) sincospif(scale * u[c], &sv[c], &cv[c]);
        X0[ni++] = sv[0]; X0[ni++] = sv[1]; X0[ni++] = sv[2];
        X0[ni++] = cv[0]; X0[ni++] = cv[1]; X0[ni++] = cv[2];
        scale *= 2.0f;
      }
      if (sh.use_viewdir) { X0[ni++] = d[0]; X0[ni++] = d[1]; X0[ni++] = d[2]; }
    }
    // ---- forward ----
    float acc[WD];
    for (int l = 0; l < nh; ++l) {
      const float *src = sm + L.off_h[l] + (size_t)tid * (l == 0 ? L.ld0 : L.ldw);
      float *dst = sm + L.off_h[l + 1] + (size_t)tid * L.ldw;
      const float *w = wp + off_w[l];
      const int nin = n_in_l[l];
      {
        const float4 *b4 = reinterpret_cast<const float4 *>(w + nin * WD);
#pragma unroll
        for (int q = 0; q < WD / 4; ++q) {
          const float4 v = __ldg(b4 + q);
          acc[4 * q] = v.x; acc[4 * q + 1] = v.y; acc[4 * q + 2] = v.z; acc[4 * q + 3] = v.w;
        }
      }
      for (int i = 0; i < nin; ++i) {
        const float xi = src[i];
        const float4 *w4 = reinterpret_cast<const float4 *>(w + i * WD);
#pragma unroll
        for (int q = 0; q < WD / 4; ++q) {
          const float4 v = __ldg(w4 + q);
          acc[4 * q] = fmaf(xi, v.x, acc[4 * q]); acc[4 * q + 1] = fmaf(xi, v.y, acc[4 * q + 1]);
          acc[4 * q + 2] = fmaf(xi, v.z, acc[4 * q + 2]); acc[4 * q + 3] = fmaf(xi, v.w, acc[4 * q + 3]);
        }
      }
#pragma unroll
      for (int o = 0; o < WD; ++o) dst[o] = acc[o] > 0.0f ? acc[o] : 0.0f;
    }
    float raw[4];
    {
      const float *src = sm + L.off_h[nh] + (size_t)tid * L.ldw;
      const float *w = wp + off_w[nh];
      const int no = sh.out_dim;
#pragma unroll
      for (int o = 0; o < 4; ++o) raw[o] = __ldg(w + WD * no + o);
      for (int i = 0; i < WD; ++i) {
        const float xi = src[i];
#pragma unroll
        for (int o = 0; o < 4; ++o) raw[o] = fmaf(xi, __ldg(w + i * no + o), raw[o]);
      }
    }
    // ---- gradient of the head's four outputs ----
    float *G = sm + L.off_g0, *Gn = sm + L.off_g1;
    float g_delta = 0.0f;
    {
      float gr[4] = {0.f, 0.f, 0.f, 0.f};
      if (live) {
        const size_t idx = (size_t)(uint32_t)iv.slot * (size_t)a.K + (size_t)k;
        const float4 gs = a.gstage[idx];
        const float e = a.staging[idx].w;
        const float c0 = 1.0f / (1.0f + expf(-raw[0])), c1 = 1.0f / (1.0f + expf(-raw[1])), c2 = 1.0f / (1.0f + expf(-raw[2]));
        gr[0] = gs.x * c0 * (1.0f - c0); gr[1] = gs.y * c1 * (1.0f - c1); gr[2] = gs.z * c2 * (1.0f - c2);
        const float sigma = fmaxf(raw[3], 0.0f) + log1pf(expf(-fabsf(raw[3])));
        gr[3] = -iv.delta * e * gs.w / (1.0f + expf(-raw[3]));
        g_delta = -sigma * e * gs.w;
      }
      float *gp = G + (size_t)tid * L.ldg;
#pragma unroll
      for (int o = 0; o < 4; ++o) gp[o] = gr[o];
    }
    for (int l = nh; l >= 0; --l) {
      __syncthreads();
      const int nin = n_in_l[l];
      const int no_ld = l == nh ? sh.out_dim : WD;
      const int no = l == nh ? 4 : WD;
      const float *Xl = sm + L.off_h[l];
      const int ldx = l == 0 ? L.ld0 : L.ldw;
      float *gw = a.g_weights + (size_t)prim * sh.params + off_w[l];
      // weight gradients: warp w takes the input rows 4 (w + 4 m) .. + 3, lane the outputs lane (+ 32)
      constexpr int OC = WD > 32 ? 2 : 1;
      for (int i0 = 4 * warp; i0 < nin + 1; i0 += 16) {      // row nin = the bias (input 1)
        float t4[4][OC];
#pragma unroll
        for (int ii = 0; ii < 4; ++ii)
#pragma unroll
          for (int c = 0; c < OC; ++c) t4[ii][c] = 0.0f;
        for (int s = 0; s < BT; ++s) {
          float xv[4];
#pragma unroll
          for (int ii = 0; ii < 4; ++ii) {
            const int i = i0 + ii;
            xv[ii] = i < nin ? Xl[(size_t)s * ldx + i] : (i == nin ? 1.0f : 0.0f);
          }
#pragma unroll
          for (int c = 0; c < OC; ++c) {
            const int o = lane + 32 * c;
            const float gv = o < no ? G[(size_t)s * L.ldg + o] : 0.0f;
#pragma unroll
            for (int ii = 0; ii < 4; ++ii) t4[ii][c] = fmaf(xv[ii], gv, t4[ii][c]);
          }
        }
#pragma unroll
        for (int ii = 0; ii < 4; ++ii)
#pragma unroll
          for (int c = 0; c < OC; ++c) {
            const int i = i0 + ii, o = lane + 32 * c;
            if (i <= nin && o < no && t4[ii][c] != 0.0f) atomicAdd(gw + i * no_ld + o, t4[ii][c]);
          }
      }
      // gradient of this thread's layer input
      const float *w = wp + off_w[l];
      const float *xin = Xl + (size_t)tid * ldx;
      float *gn = Gn + (size_t)tid * L.ldg;
      if (l == nh) {
        const float *gp = G + (size_t)tid * L.ldg;
        const float g0 = gp[0], g1 = gp[1], g2 = gp[2], g3 = gp[3];
        for (int i = 0; i < nin; ++i) {
          const float v = __ldg(w + i * no_ld) * g0 + __ldg(w + i * no_ld + 1) * g1 + __ldg(w + i * no_ld + 2) * g2 +
                          __ldg(w + i * no_ld + 3) * g3;
          gn[i] = xin[i] > 0.0f ? v : 0.0f;
        }
      } else {
        const float *gp = G + (size_t)tid * L.ldg;
#pragma unroll
        for (int o = 0; o < WD; ++o) acc[o] = gp[o];
        for (int i = 0; i < nin; ++i) {
          const float4 *w4 = reinterpret_cast<const float4 *>(w + i * WD);
          float v = 0.0f;
#pragma unroll
          for (int q = 0; q < WD / 4; ++q) {
            const float4 ww = __ldg(w4 + q);
            v = fmaf(ww.x, acc[4 * q], v); v = fmaf(ww.y, acc[4 * q + 1], v);
            v = fmaf(ww.z, acc[4 * q + 2], v); v = fmaf(ww.w, acc[4 * q + 3], v);
          }
          gn[i] = (l > 0 && !(xin[i] > 0.0f)) ? 0.0f : v;
        }
      }
      float *tmp = G; G = Gn; Gn = tmp;
    }
    if (live) {
      const float *gx = G + (size_t)tid * L.ldg;
      float gu[3] = {gx[0], gx[1], gx[2]};
      float scale = 3.14159265358979323846f;
      for (int l = 0; l < sh.n_freq; ++l) {
#pragma unroll
        for (int c = 0; c < 3; ++c) {
          const float sn = X0[3 + 6 * l + c], cs = X0[3 + 6 * l + 3 + c];
          gu[c] += scale * (cs * gx[3 + 6 * l + c] - sn * gx[3 + 6 * l + 3 + c]);
        }
        scale *= 2.0f;
      }
      float dp[3];
#pragma unroll
      for (int rr = 0; rr < 3; ++rr) dp[rr] = Ap[3 * rr] * d[0] + Ap[3 * rr + 1] * d[1] + Ap[3 * rr + 2] * d[2];
      const float gt = gu[0] * dp[0] + gu[1] * dp[1] + gu[2] * dp[2];
      float *ig = a.ivgrad + (size_t)(first + j) * 8;
      atomicAdd(ig + 0, gu[0]); atomicAdd(ig + 1, gu[1]); atomicAdd(ig + 2, gu[2]);
      atomicAdd(ig + 3, t * gu[0]); atomicAdd(ig + 4, t * gu[1]); atomicAdd(ig + 5, t * gu[2]);
      atomicAdd(ig + 6, gt);
      atomicAdd(ig + 7, ((float)k + 0.5f) * gt + g_delta);
    }
  }
}

__global__ void interval_bwd_kernel(MsMlpBwdArgs a) {
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= a.n_hits) return;
  const MsInterval iv = a.intervals[i];
  const int prim = iv.prim;
  const float *A = a.A + 9 * (size_t)prim, *mu = a.center + 3 * (size_t)prim;
  const float *ig = a.ivgrad + i * 8;
  const float v[3] = {a.cam.o[0] - mu[0], a.cam.o[1] - mu[1], a.cam.o[2] - mu[2]};
  const float d[3] = {iv.dx, iv.dy, iv.dz};
  float op[3], dp[3];
#pragma unroll
  for (int r = 0; r < 3; ++r) {
    op[r] = A[3 * r] * v[0] + A[3 * r + 1] * v[1] + A[3 * r + 2] * v[2];
    dp[r] = A[3 * r] * d[0] + A[3 * r + 1] * d[1] + A[3 * r + 2] * d[2];
  }
  const float qa = dp[0] * dp[0] + dp[1] * dp[1] + dp[2] * dp[2];
  const float qb = op[0] * dp[0] + op[1] * dp[1] + op[2] * dp[2];
  const float qc = op[0] * op[0] + op[1] * op[1] + op[2] * op[2] - 1.0f;
  const float disc = qb * qb - qa * qc;
  const float s = sqrtf(disc > 1e-30f ? disc : 1e-30f);
  const float t0 = (-qb - s) / qa, t1 = (-qb + s) / qa;
  const float Kf = (float)a.K;
  const float G1 = ig[7] / Kf;
  const float G0 = t0 > a.cam.t_near ? ig[6] - ig[7] / Kf : 0.0f;     // t_in clamped at t_near does not move
  const float ia = 1.0f / qa;
  const float gb = -(G0 + G1) * ia + (G1 - G0) * ia * qb / s;
  const float ga = -(G0 * t0 + G1 * t1) * ia - (G1 - G0) * ia * qc / (2.0f * s);
  const float gc = -(G1 - G0) / (2.0f * s);
  float gop[3], gdp[3];
#pragma unroll
  for (int r = 0; r < 3; ++r) {
    gop[r] = ig[r] + dp[r] * gb + 2.0f * op[r] * gc;
    gdp[r] = ig[3 + r] + 2.0f * dp[r] * ga + op[r] * gb;
  }
  float *gA = a.gA + 9 * (size_t)prim;
#pragma unroll
  for (int r = 0; r < 3; ++r)
#pragma unroll
    for (int c = 0; c < 3; ++c) atomicAdd(gA + 3 * r + c, gop[r] * v[c] + gdp[r] * d[c]);
#pragma unroll
  for (int c = 0; c < 3; ++c)
    atomicAdd(a.g_center + 3 * (size_t)prim + c, -(A[c] * gop[0] + A[3 + c] * gop[1] + A[6 + c] * gop[2]));
}

__global__ void prim_bwd_kernel(MsMlpBwdArgs a) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= a.n_prims) return;
  const float *A = a.A + 9 * (size_t)i, *gA = a.gA + 9 * (size_t)i, *sc = a.scale + 3 * (size_t)i;
  float G[9];     // dL/dR
#pragma unroll
  for (int r = 0; r < 3; ++r) {
    float gs = 0.0f;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      gs -= gA[3 * r + c] * A[3 * r + c] / sc[r];
      G[3 * c + r] = gA[3 * r + c] / sc[r];            // A[r][c] = R[c][r] / s[r]
    }
    if (a.g_scale) a.g_scale[3 * (size_t)i + r] += gs;
  }
  if (!a.g_quat) return;
  const float *qq = a.quat + 4 * (size_t)i;
  const float nr = sqrtf(qq[0] * qq[0] + qq[1] * qq[1] + qq[2] * qq[2] + qq[3] * qq[3]);
  const float w = qq[0] / nr, x = qq[1] / nr, y = qq[2] / nr, z = qq[3] / nr;
  float gq[4];
  gq[0] = 2 * (-z * G[1] + y * G[2] + z * G[3] - x * G[5] - y * G[6] + x * G[7]);
  gq[1] = 2 * (y * G[1] + z * G[2] + y * G[3] - 2 * x * G[4] - w * G[5] + z * G[6] + w * G[7] - 2 * x * G[8]);
  gq[2] = 2 * (-2 * y * G[0] + x * G[1] + w * G[2] + x * G[3] + z * G[5] - w * G[6] + z * G[7] - 2 * y * G[8]);
  gq[3] = 2 * (-2 * z * G[0] - w * G[1] + x * G[2] + w * G[3] - 2 * z * G[4] + y * G[5] + x * G[6] + y * G[7]);
  const float dot = gq[0] * w + gq[1] * x + gq[2] * y + gq[3] * z;
  const float qn[4] = {w, x, y, z};
#pragma unroll
  for (int c = 0; c < 4; ++c) a.g_quat[4 * (size_t)i + c] += (gq[c] - dot * qn[c]) / nr;   // through q / |q|
}

}  // namespace

size_t ms_mlp_bwd_smem(const MsMlpShape &sh) {
  if (sh.mode != MS_MODE_LOCAL || sh.n_hidden > 4) return 0;
  const size_t b = bwd_layout(sh).floats * sizeof(float);
  return b <= 220 * 1024 ? b : 0;
}

cudaError_t ms_mlp_bwd(const MsMlpBwdArgs &a, cudaStream_t s) {
  const size_t smem = ms_mlp_bwd_smem(a.shape);
  if (smem == 0) return cudaErrorNotSupported;
  void (*fn)(MsMlpBwdArgs) = mlp_bwd_kernel;
  const bool aligned = a.shape.params % 4 == 0;       // float4 loads of the weight rows
  if (aligned && a.shape.width == 8) fn = mlp_bwd_fast_kernel<8>;
  else if (aligned && a.shape.width == 16) fn = mlp_bwd_fast_kernel<16>;
  else if (aligned && a.shape.width == 32) fn = mlp_bwd_fast_kernel<32>;
  else if (aligned && a.shape.width == 64) fn = mlp_bwd_fast_kernel<64>;
  cudaError_t e = cudaFuncSetAttribute((const void *)fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  static int n_sm = 0;
  if (n_sm == 0) {
    int dev = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
  }
  int occ = 1;
  if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, (const void *)fn, BT, smem) != cudaSuccess || occ < 1) {
    (void)cudaGetLastError();
    occ = 1;
  }
  fn<<<(unsigned)(n_sm * occ * 4), BT, smem, s>>>(a);
  MS_LAUNCHED();
  e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  if (a.n_hits > 0) {
    interval_bwd_kernel<<<(unsigned)((a.n_hits + 255) / 256), 256, 0, s>>>(a);
    MS_LAUNCHED();
    e = cudaGetLastError();
    if (e != cudaSuccess) return e;
  }
  prim_bwd_kernel<<<(unsigned)((a.n_prims + 127) / 128), 128, 0, s>>>(a);
  MS_LAUNCHED();
  return cudaGetLastError();
}
