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
// leading dimension = 4 (mod 8) for the 4-threads-per-sample kernel: rows are 16-byte aligned and the float4 accesses
// of the eight threads of a quarter warp (each on its own row) fall on 32 different banks
__host__ __device__ inline int ld4_of(int n) { int m = (n + 3) & ~3; return (m & 4) ? m : m + 4; }

struct BwdLayout {
  int ld0, ldw, ldg;          // leading dimensions of X0 (encoded input), H_l (hidden), G (gradients)
  size_t off_h[5];            // float offsets of X0 (index 0) and H_1..H_nh
  size_t off_g0, off_g1;      // the two gradient buffers
  size_t floats;
};
__host__ __device__ inline BwdLayout bwd_layout(const MsMlpShape &sh, bool vec4 = false, int rows = BT) {
  BwdLayout L;
  const int gmax = sh.width > sh.in_dim ? sh.width : sh.in_dim;
  if (vec4) { L.ld0 = ld4_of(sh.in_dim); L.ldw = ld4_of(sh.width); L.ldg = ld4_of(gmax); }
  else { L.ld0 = ld_of(sh.in_dim); L.ldw = ld_of(sh.width); L.ldg = ld_of(gmax); }
  size_t o = 0;
  L.off_h[0] = o; o += (size_t)rows * L.ld0;
  for (int l = 1; l <= sh.n_hidden; ++l) { L.off_h[l] = o; o += (size_t)rows * L.ldw; }
  L.off_g0 = o; o += (size_t)rows * L.ldg;
  L.off_g1 = o; o += (size_t)rows * L.ldg;
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

// The same computation for hidden widths 16 / 32 / 64 / 128 with CG threads per sample (512 threads per CTA; one CTA
// per SM is resident: the activations of BS samples fill shared memory, so the warps have to come from inside the
// block.  BS = 128 = one row block, CG = 4 up to width 64; width 128 takes the row block in two halves of BS = 64
// with CG = 8).  Thread (cg, s) owns the output columns [cg WD/CG, (cg+1) WD/CG) of sample s in the forward pass and
// every CG-th 4-row chunk of the layer input in the backward pass: accumulators stay in registers, weight rows stream through
// warp-uniform float4 loads, activations and gradients move as float4 (leading dimensions = 4 mod 8).  The weight
// gradients X_l^T G_l are register tiles of 8 inputs x (WD / 32) outputs per lane, one (tile, sample range) item per
// warp.  The sums differ from the generic kernel (and from the fp64 statement of the chain) only in the order of the
// fp32 additions.
constexpr int BT4 = 512;              // threads per CTA
constexpr int NW4 = BT4 / 32;         // warps per CTA

__device__ __forceinline__ float4 lds4(const float *p) { return *reinterpret_cast<const float4 *>(p); }
__device__ __forceinline__ void sts4(float *p, float x, float y, float z, float w) {
  *reinterpret_cast<float4 *>(p) = make_float4(x, y, z, w);
}
__device__ __forceinline__ float4 ldg4(const float *p) { return __ldg(reinterpret_cast<const float4 *>(p)); }

template <int WD, int CG>
__global__ void __launch_bounds__(BT4, 1) mlp_bwd_fast_kernel(MsMlpBwdArgs a) {
  constexpr int BS = BT4 / CG;        // samples per pass
  constexpr int PASSES = BT / BS;     // passes per 128-row block
  constexpr int WQ = WD / CG;         // output columns per thread in the forward pass
  constexpr int OC = WD > 32 ? WD / 32 : 1;
  static_assert(WQ % 4 == 0, "float4 weight segments");
  extern __shared__ __align__(16) float sm[];
  __shared__ int s_seg;
  const MsMlpShape &sh = a.shape;
  const BwdLayout L = bwd_layout(sh, true, BS);
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int srow_in = tid & (BS - 1), cg = tid / BS;      // sample row inside the block, column group
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
  for (uint32_t unit = blockIdx.x; unit < n_blocks * PASSES; unit += gridDim.x) {
    const uint32_t blk = unit / PASSES, pass = unit % PASSES;
    __syncthreads();
    if (tid == 0) s_seg = find_seg(bo, (int)(r.y - r.x), base, blk);
    __syncthreads();
    const uint32_t g = r.x + (uint32_t)s_seg;
    const int prim = a.segs.prim ? (int)a.segs.prim[g] : (int)g;
    const uint32_t first = a.segs.iv0[g], count = a.segs.cnt ? a.segs.cnt[g] : a.segs.iv0[g + 1] - first;
    const uint64_t srow = (uint64_t)(blk - (bo[s_seg] - base)) * BT + pass * BS + srow_in;
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
    float *X0 = sm + L.off_h[0] + (size_t)srow_in * L.ld0;
    {                                 // the encoded input of the sample: frequency l by column group l mod 4
      float u[3];
      ms_sample_u(Ap, mu, a.cam.o, d, t, u);
      if (cg == 0) {
        X0[0] = u[0]; X0[1] = u[1]; X0[2] = u[2];
        if (sh.use_viewdir) { float *v = X0 + 3 + 6 * sh.n_freq; v[0] = d[0]; v[1] = d[1]; v[2] = d[2]; }
      }
      for (int l = cg; l < sh.n_freq; l += CG) {
        const float scale = (float)(1 << l);
        float sv[3], cv[3];
#pragma unroll
        for (int c = 0; c < 3; ++c) sincospif(scale * u[c], &sv[c], &cv[c]);
        float *x = X0 + 3 + 6 * l;
        x[0] = sv[0]; x[1] = sv[1]; x[2] = sv[2];
        x[3] = cv[0]; x[4] = cv[1]; x[5] = cv[2];
      }
    }
    __syncthreads();
    // ---- forward: this thread's WQ columns of every hidden layer ----
    for (int l = 0; l < nh; ++l) {
      const float *src = sm + L.off_h[l] + (size_t)srow_in * (l == 0 ? L.ld0 : L.ldw);
      float *dst = sm + L.off_h[l + 1] + (size_t)srow_in * L.ldw + cg * WQ;
      const float *w = wp + off_w[l] + cg * WQ;
      const int nin = n_in_l[l];
      float acc[WQ];
#pragma unroll
      for (int q = 0; q < WQ / 4; ++q) {
        const float4 v = ldg4(w + nin * WD + 4 * q);
        acc[4 * q] = v.x; acc[4 * q + 1] = v.y; acc[4 * q + 2] = v.z; acc[4 * q + 3] = v.w;
      }
      int i = 0;
      for (; i + 4 <= nin; i += 4) {
        const float4 x4 = lds4(src + i);
        const float xs[4] = {x4.x, x4.y, x4.z, x4.w};
#pragma unroll
        for (int ii = 0; ii < 4; ++ii) {
          const float *wr = w + (i + ii) * WD;
#pragma unroll
          for (int q = 0; q < WQ / 4; ++q) {
            const float4 v = ldg4(wr + 4 * q);
            acc[4 * q] = fmaf(xs[ii], v.x, acc[4 * q]); acc[4 * q + 1] = fmaf(xs[ii], v.y, acc[4 * q + 1]);
            acc[4 * q + 2] = fmaf(xs[ii], v.z, acc[4 * q + 2]); acc[4 * q + 3] = fmaf(xs[ii], v.w, acc[4 * q + 3]);
          }
        }
      }
      for (; i < nin; ++i) {
        const float xi = src[i];
        const float *wr = w + i * WD;
#pragma unroll
        for (int q = 0; q < WQ / 4; ++q) {
          const float4 v = ldg4(wr + 4 * q);
          acc[4 * q] = fmaf(xi, v.x, acc[4 * q]); acc[4 * q + 1] = fmaf(xi, v.y, acc[4 * q + 1]);
          acc[4 * q + 2] = fmaf(xi, v.z, acc[4 * q + 2]); acc[4 * q + 3] = fmaf(xi, v.w, acc[4 * q + 3]);
        }
      }
#pragma unroll
      for (int q = 0; q < WQ / 4; ++q)
        sts4(dst + 4 * q, fmaxf(acc[4 * q], 0.0f), fmaxf(acc[4 * q + 1], 0.0f), fmaxf(acc[4 * q + 2], 0.0f),
             fmaxf(acc[4 * q + 3], 0.0f));
      __syncthreads();
    }
    // ---- head: partial sums over this thread's WQ inputs, summed by column group 0 ----
    float *G = sm + L.off_g0, *Gn = sm + L.off_g1;
    const int no_h = sh.out_dim;
    {
      const float *src = sm + L.off_h[nh] + (size_t)srow_in * L.ldw + cg * WQ;
      const float *w = wp + off_w[nh] + (size_t)(cg * WQ) * no_h;
      float pr[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
      for (int q = 0; q < WQ / 4; ++q) {
        const float4 x4 = lds4(src + 4 * q);
        const float xs[4] = {x4.x, x4.y, x4.z, x4.w};
#pragma unroll
        for (int ii = 0; ii < 4; ++ii)
#pragma unroll
          for (int o = 0; o < 4; ++o) pr[o] = fmaf(xs[ii], __ldg(w + (4 * q + ii) * no_h + o), pr[o]);
      }
      sts4(Gn + (size_t)srow_in * L.ldg + 4 * cg, pr[0], pr[1], pr[2], pr[3]);
    }
    __syncthreads();
    float g_delta = 0.0f;
    if (cg == 0) {                    // gradient of the head's four outputs (sigmoid colour, softplus density)
      float raw[4], gr[4] = {0.f, 0.f, 0.f, 0.f};
      const float *pp = Gn + (size_t)srow_in * L.ldg;
      const float *bh = wp + off_w[nh] + WD * no_h;
      float4 ps = lds4(pp);
#pragma unroll
      for (int c = 1; c < CG; ++c) {
        const float4 pc = lds4(pp + 4 * c);
        ps.x += pc.x; ps.y += pc.y; ps.z += pc.z; ps.w += pc.w;
      }
      raw[0] = __ldg(bh) + ps.x; raw[1] = __ldg(bh + 1) + ps.y; raw[2] = __ldg(bh + 2) + ps.z; raw[3] = __ldg(bh + 3) + ps.w;
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
      sts4(G + (size_t)srow_in * L.ldg, gr[0], gr[1], gr[2], gr[3]);
    }
    for (int l = nh; l >= 0; --l) {
      __syncthreads();
      const int nin = n_in_l[l];
      const float *Xl = sm + L.off_h[l];
      const int ldx = l == 0 ? L.ld0 : L.ldw;
      float *gw = a.g_weights + (size_t)prim * sh.params + off_w[l];
      if (l == nh) {
        // head weights (WD x 4): lane = input row, four outputs per lane; warps over (row group, sample range)
        constexpr int RG = (WD + 31) / 32, SSH = NW4 / RG, PER = BS / SSH;
        const int rg = warp % RG, part = warp / RG, row = rg * 32 + lane;
        const bool on = row < WD;
        float t4[4] = {0.f, 0.f, 0.f, 0.f}, tb[4] = {0.f, 0.f, 0.f, 0.f};
        const float *xr = Xl + (size_t)(part * PER) * ldx + (on ? row : 0);
        const float *gp = G + (size_t)(part * PER) * L.ldg;
        for (int s = 0; s < PER; ++s, xr += ldx, gp += L.ldg) {
          const float4 g4 = lds4(gp);
          const float x = *xr;
          t4[0] = fmaf(x, g4.x, t4[0]); t4[1] = fmaf(x, g4.y, t4[1]); t4[2] = fmaf(x, g4.z, t4[2]); t4[3] = fmaf(x, g4.w, t4[3]);
          tb[0] += g4.x; tb[1] += g4.y; tb[2] += g4.z; tb[3] += g4.w;
        }
        if (on) {
#pragma unroll
          for (int o = 0; o < 4; ++o) if (t4[o] != 0.0f) atomicAdd(gw + row * no_h + o, t4[o]);
        }
        if (rg == 0 && lane == 0) {
#pragma unroll
          for (int o = 0; o < 4; ++o) if (tb[o] != 0.0f) atomicAdd(gw + WD * no_h + o, tb[o]);
        }
      } else {
        // hidden weights (nin x WD): items = (8-row tile, sample range), lane = output column (+ 32 c)
        const int n_tiles = (nin + 7) >> 3;
        int SS = 1;
        while (2 * SS * n_tiles <= NW4 && SS < 8) SS *= 2;
        const int per = BS / SS;
        for (int item = warp; item < n_tiles * SS; item += NW4) {
          const int tile = item / SS, part = item - tile * SS, i0 = tile * 8;
          float t8[8][OC], tb[OC];
#pragma unroll
          for (int c = 0; c < OC; ++c) {
            tb[c] = 0.0f;
#pragma unroll
            for (int ii = 0; ii < 8; ++ii) t8[ii][c] = 0.0f;
          }
          const float *xr = Xl + (size_t)(part * per) * ldx + i0;
          const float *gp = G + (size_t)(part * per) * L.ldg + (WD >= 32 ? lane : (lane & (WD - 1)));
          for (int s = 0; s < per; ++s, xr += ldx, gp += L.ldg) {
            const float4 xa = lds4(xr), xb = lds4(xr + 4);
#pragma unroll
            for (int c = 0; c < OC; ++c) {
              const float gv = gp[32 * c];
              t8[0][c] = fmaf(xa.x, gv, t8[0][c]); t8[1][c] = fmaf(xa.y, gv, t8[1][c]);
              t8[2][c] = fmaf(xa.z, gv, t8[2][c]); t8[3][c] = fmaf(xa.w, gv, t8[3][c]);
              t8[4][c] = fmaf(xb.x, gv, t8[4][c]); t8[5][c] = fmaf(xb.y, gv, t8[5][c]);
              t8[6][c] = fmaf(xb.z, gv, t8[6][c]); t8[7][c] = fmaf(xb.w, gv, t8[7][c]);
              tb[c] += gv;
            }
          }
          if (WD >= 32 || lane < WD) {
#pragma unroll
            for (int c = 0; c < OC; ++c) {
              const int o = lane + 32 * c;
#pragma unroll
              for (int ii = 0; ii < 8; ++ii)
                if (i0 + ii < nin && t8[ii][c] != 0.0f) atomicAdd(gw + (i0 + ii) * WD + o, t8[ii][c]);
              if (tile == 0 && tb[c] != 0.0f) atomicAdd(gw + nin * WD + o, tb[c]);
            }
          }
        }
      }
      // gradient of the layer input: this thread's 4-row chunks (every fourth chunk)
      const float *w = wp + off_w[l];
      const float *xin = Xl + (size_t)srow_in * ldx;
      const float *gpr = G + (size_t)srow_in * L.ldg;
      float *gn = Gn + (size_t)srow_in * L.ldg;
      if (l == nh) {
        const float4 g4 = lds4(gpr);
        for (int i0 = 4 * cg; i0 < nin; i0 += 4 * CG) {
          const float4 x4 = lds4(xin + i0);
          const float xs[4] = {x4.x, x4.y, x4.z, x4.w};
          float v[4];
#pragma unroll
          for (int ii = 0; ii < 4; ++ii) {
            const float *wr = w + (i0 + ii) * no_h;
            const float vv = __ldg(wr) * g4.x + __ldg(wr + 1) * g4.y + __ldg(wr + 2) * g4.z + __ldg(wr + 3) * g4.w;
            v[ii] = xs[ii] > 0.0f ? vv : 0.0f;
          }
          sts4(gn + i0, v[0], v[1], v[2], v[3]);
        }
      } else {
        for (int i0 = 4 * cg; i0 < nin; i0 += 4 * CG) {
          const float *wr[4];
#pragma unroll
          for (int ii = 0; ii < 4; ++ii) wr[ii] = w + (size_t)min(i0 + ii, nin - 1) * WD;   // rows past nin: discarded
          float v[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll 4
          for (int o = 0; o < WD; o += 4) {
            const float4 g4 = lds4(gpr + o);
#pragma unroll
            for (int ii = 0; ii < 4; ++ii) {
              const float4 ww = ldg4(wr[ii] + o);
              v[ii] = fmaf(ww.x, g4.x, v[ii]); v[ii] = fmaf(ww.y, g4.y, v[ii]);
              v[ii] = fmaf(ww.z, g4.z, v[ii]); v[ii] = fmaf(ww.w, g4.w, v[ii]);
            }
          }
          if (l > 0) {
            const float4 x4 = lds4(xin + i0);
            v[0] = x4.x > 0.0f ? v[0] : 0.0f; v[1] = x4.y > 0.0f ? v[1] : 0.0f;
            v[2] = x4.z > 0.0f ? v[2] : 0.0f; v[3] = x4.w > 0.0f ? v[3] : 0.0f;
          }
          sts4(gn + i0, v[0], v[1], v[2], v[3]);
        }
      }
      float *tmp = G; G = Gn; Gn = tmp;
    }
    __syncthreads();
    if (live && cg == 0) {
      const float *gx = G + (size_t)srow_in * L.ldg;
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

// which kernel serves the shape: 2 = several threads per sample (widths 16 / 32 / 64 / 128, float4 weight rows),
// 1 = generic
static int bwd_kind(const MsMlpShape &sh, size_t *smem) {
  *smem = 0;
  if (sh.mode != MS_MODE_LOCAL || sh.n_hidden > 4 || sh.n_hidden < 1) return 0;
  const size_t cap = 220 * 1024;
  const bool fast_w = sh.width == 16 || sh.width == 32 || sh.width == 64 || sh.width == 128;
  if (fast_w && sh.params % 4 == 0) {
    const size_t b = bwd_layout(sh, true, sh.width == 128 ? 64 : BT).floats * sizeof(float);
    if (b <= cap) { *smem = b; return 2; }
  }
  const size_t b = bwd_layout(sh).floats * sizeof(float);
  if (b > cap) return 0;
  *smem = b;
  return 1;
}

size_t ms_mlp_bwd_smem(const MsMlpShape &sh) {
  size_t b = 0;
  bwd_kind(sh, &b);
  return b;
}

cudaError_t ms_mlp_bwd(const MsMlpBwdArgs &a, cudaStream_t s) {
  size_t smem = 0;
  const int kind = bwd_kind(a.shape, &smem);
  if (kind == 0) return cudaErrorNotSupported;
  void (*fn)(MsMlpBwdArgs) = mlp_bwd_kernel;
  int threads = BT;
  if (kind == 2) {
    threads = BT4;
    fn = a.shape.width == 16 ? mlp_bwd_fast_kernel<16, 4> : a.shape.width == 32 ? mlp_bwd_fast_kernel<32, 4>
       : a.shape.width == 64 ? mlp_bwd_fast_kernel<64, 4> : mlp_bwd_fast_kernel<128, 8>;
  }
  cudaError_t e = cudaFuncSetAttribute((const void *)fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  static int n_sm = 0;
  if (n_sm == 0) {
    int dev = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
  }
  int occ = 1;
  if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, (const void *)fn, threads, smem) != cudaSuccess || occ < 1) {
    (void)cudaGetLastError();
    occ = 1;
  }
  fn<<<(unsigned)(n_sm * occ * (kind == 2 ? 1 : 4)), threads, smem, s>>>(a);
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
