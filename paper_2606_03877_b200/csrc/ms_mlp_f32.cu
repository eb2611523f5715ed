// ms_mlp_f32.cu -- stage (d), fp32 SIMT path (NS: "rgb/alpha within 1e-5 max abs for the fp32
// path"; CFG1).  One CTA = one 128-sample row block of ONE primitive, whose fp32 weights are
// staged in shared memory once per CTA; one thread = one sample: canonical u,
// positional encoding Eq.5 with exact-argument sincospif(2^l u), Linear+ReLU layers with
// fp32 FMA accumulation, rgb = sigmoid, sigma = softplus, e = exp(-sigma*delta).
// This path is the accuracy reference on the device; the throughput path is ms_mlp_tc.cu.
#include "ms_internal.cuh"

namespace {

// segment of block b of the launch: largest s with bo[s] - base <= b
__device__ __forceinline__ int find_seg(const uint32_t *__restrict__ bo, int n, uint32_t base, uint32_t b) {
  int lo = 0, hi = n;
  while (hi - lo > 1) {
    int mid = (lo + hi) >> 1;
    if (bo[mid] - base <= b) lo = mid; else hi = mid;
  }
  return lo;
}

// The launch's segments and band (device tables, ms_band.cu); every CTA walks blocks blockIdx.x, + gridDim.x, ...
struct LaunchView {
  uint2 r;
  MsBand band;
  const uint32_t *bo;
  uint32_t base, n_blocks;
  __device__ LaunchView(const MsSegs &sg) {
    r = *sg.range;
    band = *sg.band;
    bo = sg.blk_off + r.x;
    base = bo[0];
    n_blocks = bo[r.y - r.x] - base;
  }
};

__global__ void __launch_bounds__(MS_ROWS) mlp_f32_kernel(MsMlpArgs a) {
  extern __shared__ float w_s[];
  __shared__ int s_seg;
  const MsMlpShape &sh = a.shape;
  const LaunchView lv(a.segs);
  int cur_prim = -1;
  // the CTA walks a contiguous run of the launch's blocks: the weights are reloaded only when the primitive changes
  const uint32_t blk_lo = (uint32_t)(((uint64_t)lv.n_blocks * blockIdx.x) / gridDim.x);
  const uint32_t blk_hi = (uint32_t)(((uint64_t)lv.n_blocks * (blockIdx.x + 1)) / gridDim.x);
  for (uint32_t blk = blk_lo; blk < blk_hi; ++blk) {
  __syncthreads();                       // the previous block is done with w_s and s_seg
  if (threadIdx.x == 0) {
    int sgm = blk == blk_lo ? find_seg(lv.bo, (int)(lv.r.y - lv.r.x), lv.base, blk) : s_seg;
    while (lv.bo[sgm + 1] - lv.base <= blk) ++sgm;     // segments without blocks are skipped
    s_seg = sgm;
  }
  __syncthreads();
  const uint32_t g = lv.r.x + (uint32_t)s_seg;
  const int prim = a.segs.prim ? (int)a.segs.prim[g] : (int)g;
  if (prim != cur_prim) {
    const float *wg = a.weights_f32 + (size_t)prim * sh.params;
    for (int i = threadIdx.x; i < sh.params; i += blockDim.x) w_s[i] = wg[i];
    cur_prim = prim;
  }
  __syncthreads();

  const uint32_t first = a.segs.iv0[g], count = a.segs.cnt ? a.segs.cnt[g] : a.segs.iv0[g + 1] - first;
  const uint64_t s = (uint64_t)(blk - (lv.bo[s_seg] - lv.base)) * MS_ROWS + threadIdx.x;
  const uint32_t j = (uint32_t)(s / (uint32_t)a.K);
  const int k = (int)(s % (uint32_t)a.K);
  if (j >= count) continue;
  const MsInterval iv = a.intervals[first + j];
  const float d[3] = {iv.dx, iv.dy, iv.dz};
  const bool contact = sh.mode == MS_MODE_CONTACT;
  const float t = ms_sample_tm(iv.t_in, iv.delta, k, contact);
  float u[3];
  ms_sample_u(a.A + 9 * (size_t)prim, a.center + 3 * (size_t)prim, a.cam.o, d, t, u);

  float ha[MS_MAX_WIDTH], hb[MS_MAX_WIDTH];
  int n_in = 0;
  if (contact) {
    // P:89-103 Eq.3-5: z = [d; mu - p*], x[2L j + 2l] = sin(2^l pi z_j), x[2L j + 2l + 1] = cos(2^l pi z_j)
    const float *mu = a.center + 3 * (size_t)prim;
    float z[6] = {d[0], d[1], d[2], 0.f, 0.f, 0.f};
#pragma unroll
    for (int c = 0; c < 3; ++c) z[3 + c] = __fsub_rn(mu[c], __fadd_rn(a.cam.o[c], __fmul_rn(t, d[c])));
    for (int c = 0; c < 6; ++c) {
      float scale = 1.0f;
      for (int l = 0; l < sh.n_freq; ++l) {
        sincospif(scale * z[c], &ha[n_in], &ha[n_in + 1]);  // 2^l z is exact
        n_in += 2;
        scale *= 2.0f;
      }
    }
  } else {
  ha[n_in++] = u[0]; ha[n_in++] = u[1]; ha[n_in++] = u[2];
  float scale = 1.0f;
  for (int l = 0; l < sh.n_freq; ++l) {
    float sv[3], cv[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) sincospif(scale * u[c], &sv[c], &cv[c]);  // 2^l u is exact
    ha[n_in++] = sv[0]; ha[n_in++] = sv[1]; ha[n_in++] = sv[2];
    ha[n_in++] = cv[0]; ha[n_in++] = cv[1]; ha[n_in++] = cv[2];
    scale *= 2.0f;
  }
  if (sh.use_viewdir) { ha[n_in++] = d[0]; ha[n_in++] = d[1]; ha[n_in++] = d[2]; }
  }

  float *src = ha, *dst = hb;
  const float *w = w_s;
  for (int l = 0; l < sh.n_layers; ++l) {
    const bool last = l == sh.n_layers - 1;
    const int n_out = last ? sh.out_dim : sh.width;
    const float *bias = w + n_in * n_out;
    for (int o = 0; o < n_out; ++o) {
      float acc = bias[o];
      for (int i = 0; i < n_in; ++i) acc = fmaf(src[i], w[i * n_out + o], acc);
      dst[o] = last ? acc : fmaxf(acc, 0.0f);
    }
    w = bias + n_out;
    n_in = n_out;
    float *tmp = src; src = dst; dst = tmp;
  }
  const float *raw = src;
  float4 r;
  r.x = 1.0f / (1.0f + expf(-raw[0]));
  r.y = 1.0f / (1.0f + expf(-raw[1]));
  r.z = 1.0f / (1.0f + expf(-raw[2]));
  const float sigma = fmaxf(raw[3], 0.0f) + log1pf(expf(-fabsf(raw[3])));
  r.w = expf(-sigma * iv.delta);  // e = 1 - alpha
  if (contact) {  // alpha = (1 - exp(-sigma l)) g, g = exp(-(9/2) |p* - mu|^2_Lambda)  (include/mlpsplat.h)
    const float r2 = u[0] * u[0] + u[1] * u[1] + u[2] * u[2];
    r.w = 1.0f - (1.0f - r.w) * expf(-a.falloff * r2);
  }
  const size_t out = (size_t)((uint32_t)iv.slot - lv.band.slot0) * (size_t)a.K + (size_t)k;
  a.staging[out] = r;
  if (a.staging_gate) a.staging_gate[out] = ms_slot_gates(u);
  if (a.staging_feat)
    for (int c = 0; c < sh.n_feat; ++c) reinterpret_cast<float *>(a.staging_feat)[out * sh.n_feat + c] = raw[4 + c];
  }
}


// 32-wide MLPs (CFG1 27-32-32-4; the paper's own 72-32-32-4): the same arithmetic in the same
// order as mlp_f32_kernel (acc = b; acc = fma(x_i, W[i][o], acc) for i ascending), but the 32
// accumulators and activations live in registers and the encoded input is fed one element at a time
// as it is produced, each with one broadcast row of W1 (8 x LDS.128) -- no local-memory arrays.
// Each thread carries SPT = 2 samples (rows r and r + 64 of the block) so that a weight row loaded
// from shared memory feeds 64 FMAs: with one sample per thread the kernel was bound by the
// shared-memory wavefronts of the broadcast loads (84 % of peak, profiles/r1e_summary.md).
template <int NH, int SPT>
__global__ void __launch_bounds__(MS_ROWS / SPT, 6) mlp_f32_w32_kernel(MsMlpArgs a) {
  extern __shared__ __align__(16) float w_s[];
  __shared__ int s_seg;
  const MsMlpShape &sh = a.shape;
  const LaunchView lv(a.segs);
  int cur_prim = -1;
  // the CTA walks a contiguous run of the launch's blocks: the weights are reloaded only when the primitive changes
  const uint32_t blk_lo = (uint32_t)(((uint64_t)lv.n_blocks * blockIdx.x) / gridDim.x);
  const uint32_t blk_hi = (uint32_t)(((uint64_t)lv.n_blocks * (blockIdx.x + 1)) / gridDim.x);
  for (uint32_t blk = blk_lo; blk < blk_hi; ++blk) {
  __syncthreads();                       // the previous block is done with w_s and s_seg
  if (threadIdx.x == 0) {
    int sgm = blk == blk_lo ? find_seg(lv.bo, (int)(lv.r.y - lv.r.x), lv.base, blk) : s_seg;
    while (lv.bo[sgm + 1] - lv.base <= blk) ++sgm;     // segments without blocks are skipped
    s_seg = sgm;
  }
  __syncthreads();
  const uint32_t g = lv.r.x + (uint32_t)s_seg;
  const int prim = a.segs.prim ? (int)a.segs.prim[g] : (int)g;
  if (prim != cur_prim) {
    const float4 *wg = reinterpret_cast<const float4 *>(a.weights_f32 + (size_t)prim * sh.params);   // params % 4 == 0 for these shapes
    float4 *ws4 = reinterpret_cast<float4 *>(w_s);
    for (int i = threadIdx.x; i < sh.params / 4; i += blockDim.x) ws4[i] = __ldg(wg + i);
    cur_prim = prim;
  }
  __syncthreads();

  const uint32_t first = a.segs.iv0[g], count = a.segs.cnt ? a.segs.cnt[g] : a.segs.iv0[g + 1] - first;
  const uint32_t blk_in_seg = blk - (lv.bo[s_seg] - lv.base);
  const bool contact = sh.mode == MS_MODE_CONTACT;
  const float *mu = a.center + 3 * (size_t)prim;
  bool live[SPT];
  int kk[SPT];
  MsInterval iv[SPT];
  float u[SPT][3], z[SPT][6];
#pragma unroll
  for (int q = 0; q < SPT; ++q) {
    const uint64_t s = (uint64_t)blk_in_seg * MS_ROWS + threadIdx.x + q * (MS_ROWS / SPT);
    const uint32_t j = (uint32_t)(s / (uint32_t)a.K);
    kk[q] = (int)(s % (uint32_t)a.K);
    live[q] = j < count;
    iv[q] = a.intervals[first + (live[q] ? j : 0u)];   // a dead row recomputes interval 0 and stores nothing
    const float d[3] = {iv[q].dx, iv[q].dy, iv[q].dz};
    const float t = ms_sample_tm(iv[q].t_in, iv[q].delta, kk[q], contact);
    ms_sample_u(a.A + 9 * (size_t)prim, mu, a.cam.o, d, t, u[q]);
    // P:89-103 Eq.3-5: z = [d; mu - p*]
    z[q][0] = d[0]; z[q][1] = d[1]; z[q][2] = d[2];
#pragma unroll
    for (int c = 0; c < 3; ++c) z[q][3 + c] = __fsub_rn(mu[c], __fadd_rn(a.cam.o[c], __fmul_rn(t, d[c])));
  }
  if (count == 0) continue;

  float acc[SPT][32];
  const int n_in = sh.in_dim;
  {
    const float4 *b4 = reinterpret_cast<const float4 *>(w_s + n_in * 32);
#pragma unroll
    for (int q = 0; q < 8; ++q) {
      const float4 v = b4[q];
#pragma unroll
      for (int p = 0; p < SPT; ++p) { acc[p][4 * q] = v.x; acc[p][4 * q + 1] = v.y; acc[p][4 * q + 2] = v.z; acc[p][4 * q + 3] = v.w; }
    }
  }
  int row = 0;
  auto feed = [&](const float (&x)[SPT]) {   // acc[p] += x[p] * W1[row][:]
    const float4 *wr = reinterpret_cast<const float4 *>(w_s + row * 32);
#pragma unroll
    for (int q = 0; q < 8; ++q) {
      const float4 v = wr[q];
#pragma unroll
      for (int p = 0; p < SPT; ++p) {
        acc[p][4 * q] = fmaf(x[p], v.x, acc[p][4 * q]); acc[p][4 * q + 1] = fmaf(x[p], v.y, acc[p][4 * q + 1]);
        acc[p][4 * q + 2] = fmaf(x[p], v.z, acc[p][4 * q + 2]); acc[p][4 * q + 3] = fmaf(x[p], v.w, acc[p][4 * q + 3]);
      }
    }
    ++row;
  };
  if (contact) {
    // x[2L j + 2l] = sin(2^l pi z_j), x[2L j + 2l + 1] = cos(2^l pi z_j)
#pragma unroll
    for (int c = 0; c < 6; ++c) {
      float scale = 1.0f;
      for (int l = 0; l < sh.n_freq; ++l) {
        float sv[SPT], cv[SPT];
#pragma unroll
        for (int p = 0; p < SPT; ++p) sincospif(scale * z[p][c], &sv[p], &cv[p]);  // 2^l z is exact
        feed(sv); feed(cv);
        scale *= 2.0f;
      }
    }
  } else {
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      float x[SPT];
#pragma unroll
      for (int p = 0; p < SPT; ++p) x[p] = u[p][c];
      feed(x);
    }
    float scale = 1.0f;
    for (int l = 0; l < sh.n_freq; ++l) {
      float sv[3][SPT], cv[3][SPT];
#pragma unroll
      for (int c = 0; c < 3; ++c)
#pragma unroll
        for (int p = 0; p < SPT; ++p) sincospif(scale * u[p][c], &sv[c][p], &cv[c][p]);  // 2^l u is exact
      feed(sv[0]); feed(sv[1]); feed(sv[2]);
      feed(cv[0]); feed(cv[1]); feed(cv[2]);
      scale *= 2.0f;
    }
    if (sh.use_viewdir) {
#pragma unroll
      for (int c = 0; c < 3; ++c) {
        float x[SPT];
#pragma unroll
        for (int p = 0; p < SPT; ++p) x[p] = z[p][c];
        feed(x);
      }
    }
  }
  float h[SPT][32];
#pragma unroll
  for (int p = 0; p < SPT; ++p)
#pragma unroll
    for (int o = 0; o < 32; ++o) h[p][o] = fmaxf(acc[p][o], 0.0f);
  const float *w = w_s + n_in * 32 + 32;
#pragma unroll
  for (int l = 1; l < NH; ++l) {
    const float4 *b4 = reinterpret_cast<const float4 *>(w + 32 * 32);
#pragma unroll
    for (int q = 0; q < 8; ++q) {
      const float4 v = b4[q];
#pragma unroll
      for (int p = 0; p < SPT; ++p) { acc[p][4 * q] = v.x; acc[p][4 * q + 1] = v.y; acc[p][4 * q + 2] = v.z; acc[p][4 * q + 3] = v.w; }
    }
#pragma unroll
    for (int i = 0; i < 32; ++i) {
      const float4 *wr = reinterpret_cast<const float4 *>(w + i * 32);
#pragma unroll
      for (int q = 0; q < 8; ++q) {
        const float4 v = wr[q];
#pragma unroll
        for (int p = 0; p < SPT; ++p) {
          acc[p][4 * q] = fmaf(h[p][i], v.x, acc[p][4 * q]); acc[p][4 * q + 1] = fmaf(h[p][i], v.y, acc[p][4 * q + 1]);
          acc[p][4 * q + 2] = fmaf(h[p][i], v.z, acc[p][4 * q + 2]); acc[p][4 * q + 3] = fmaf(h[p][i], v.w, acc[p][4 * q + 3]);
        }
      }
    }
#pragma unroll
    for (int p = 0; p < SPT; ++p)
#pragma unroll
      for (int o = 0; o < 32; ++o) h[p][o] = fmaxf(acc[p][o], 0.0f);
    w += 32 * 32 + 32;
  }
  // head: raw[o] = b[o] + sum_i h[i] Wh[i][o]
  const int n_out = sh.out_dim;
  const float *bh = w + 32 * n_out;
#pragma unroll
  for (int p = 0; p < SPT; ++p) {
    if (!live[p]) continue;
    float raw4[4];
#pragma unroll
    for (int o = 0; o < 4; ++o) {
      float r = bh[o];
#pragma unroll
      for (int i = 0; i < 32; ++i) r = fmaf(h[p][i], w[i * n_out + o], r);
      raw4[o] = r;
    }
    float4 r;
    r.x = 1.0f / (1.0f + expf(-raw4[0]));
    r.y = 1.0f / (1.0f + expf(-raw4[1]));
    r.z = 1.0f / (1.0f + expf(-raw4[2]));
    const float sigma = fmaxf(raw4[3], 0.0f) + log1pf(expf(-fabsf(raw4[3])));
    r.w = expf(-sigma * iv[p].delta);  // e = 1 - alpha
    if (contact) {  // alpha = (1 - exp(-sigma l)) g, g = exp(-(9/2) |p* - mu|^2_Lambda)  (include/mlpsplat.h)
      const float r2 = u[p][0] * u[p][0] + u[p][1] * u[p][1] + u[p][2] * u[p][2];
      r.w = 1.0f - (1.0f - r.w) * expf(-a.falloff * r2);
    }
    const size_t out = (size_t)((uint32_t)iv[p].slot - lv.band.slot0) * (size_t)a.K + (size_t)kk[p];
    a.staging[out] = r;
    if (a.staging_gate) a.staging_gate[out] = ms_slot_gates(u[p]);
    if (a.staging_feat)
      for (int c = 0; c < sh.n_feat; ++c) {
        float f = bh[4 + c];
#pragma unroll
        for (int i = 0; i < 32; ++i) f = fmaf(h[p][i], w[i * n_out + 4 + c], f);
        reinterpret_cast<float *>(a.staging_feat)[out * sh.n_feat + c] = f;
      }
  }
  }
}

// Wide MLPs (16 / 64 / 128 hidden units; north-star mode): the same arithmetic in the same order as mlp_f32_kernel
// (acc = b; acc = fma(x_i, W[i][o], acc) for i ascending -- bitwise the same staging), laid out for throughput.  CG
// threads share a pair of samples: thread (cg, sp) owns the output columns [cg WD/CG, (cg+1) WD/CG) of the samples sp
// and sp + 64 of the row block, activations live in shared memory (rows 16-byte aligned, leading dimension = 4 mod 8:
// the float4 reads of a quarter warp fall on 32 different banks), weight rows stream through warp-uniform float4 loads
// and each serves two samples (8 FMAs per loaded float4).
__host__ __device__ inline int ld4_of(int n) { int m = (n + 3) & ~3; return (m & 4) ? m : m + 4; }
__device__ __forceinline__ float4 lds4(const float *p) { return *reinterpret_cast<const float4 *>(p); }
__device__ __forceinline__ float4 ldg4(const float *p) { return __ldg(reinterpret_cast<const float4 *>(p)); }

template <int WD, int CG>
__global__ void __launch_bounds__(MS_ROWS * CG / 2) mlp_f32_wide_kernel(MsMlpArgs a) {
  constexpr int HS = MS_ROWS / 2;     // thread (cg, sp): rows sp and sp + HS
  constexpr int WQ = WD / CG;
  static_assert(WQ % 4 == 0, "float4 weight segments");
  extern __shared__ __align__(16) float sm[];
  __shared__ int s_seg;
  const MsMlpShape &sh = a.shape;
  const LaunchView lv(a.segs);
  const int ld0 = ld4_of(sh.in_dim), ldw = ld4_of(WD);
  float *X0 = sm, *HA = X0 + (size_t)MS_ROWS * ld0, *HB = HA + (size_t)MS_ROWS * ldw;
  const int tid = threadIdx.x, sp = tid & (HS - 1), cg = tid / HS;
  const uint32_t blk_lo = (uint32_t)(((uint64_t)lv.n_blocks * blockIdx.x) / gridDim.x);
  const uint32_t blk_hi = (uint32_t)(((uint64_t)lv.n_blocks * (blockIdx.x + 1)) / gridDim.x);
  for (uint32_t blk = blk_lo; blk < blk_hi; ++blk) {
    __syncthreads();
    if (tid == 0) {
      int sgm = blk == blk_lo ? find_seg(lv.bo, (int)(lv.r.y - lv.r.x), lv.base, blk) : s_seg;
      while (lv.bo[sgm + 1] - lv.base <= blk) ++sgm;
      s_seg = sgm;
    }
    __syncthreads();
    const uint32_t g = lv.r.x + (uint32_t)s_seg;
    const int prim = a.segs.prim ? (int)a.segs.prim[g] : (int)g;
    const float *wp = a.weights_f32 + (size_t)prim * sh.params;
    const uint32_t first = a.segs.iv0[g], count = a.segs.cnt ? a.segs.cnt[g] : a.segs.iv0[g + 1] - first;
    const uint64_t s0 = (uint64_t)(blk - (lv.bo[s_seg] - lv.base)) * MS_ROWS;
    bool live[2];
    int kk[2];
    float delta[2];
    uint32_t slot[2];
#pragma unroll
    for (int p = 0; p < 2; ++p) {
      const int row = sp + p * HS;
      const uint64_t s = s0 + row;
      const uint32_t j = (uint32_t)(s / (uint32_t)a.K);
      kk[p] = (int)(s % (uint32_t)a.K);
      live[p] = j < count;
      MsInterval iv;
      iv.t_in = 0.f; iv.delta = 0.f; iv.slot = 0; iv.dx = 0.f; iv.dy = 0.f; iv.dz = 1.f; iv.ray = 0; iv.prim = prim;
      if (live[p]) iv = a.intervals[first + j];
      delta[p] = iv.delta; slot[p] = (uint32_t)iv.slot;
      const float d[3] = {iv.dx, iv.dy, iv.dz};
      const float t = ms_sample_tm(iv.t_in, iv.delta, kk[p], false);
      float u[3];
      ms_sample_u(a.A + 9 * (size_t)prim, a.center + 3 * (size_t)prim, a.cam.o, d, t, u);
      float *x = X0 + (size_t)row * ld0;                  // Eq.5: frequency l by column group l mod CG
      if (cg == 0) {
        x[0] = u[0]; x[1] = u[1]; x[2] = u[2];
        if (sh.use_viewdir) { float *v = x + 3 + 6 * sh.n_freq; v[0] = d[0]; v[1] = d[1]; v[2] = d[2]; }
        if (a.staging_gate && live[p])
          a.staging_gate[(size_t)(slot[p] - lv.band.slot0) * (size_t)a.K + (size_t)kk[p]] = ms_slot_gates(u);
      }
      for (int l = cg; l < sh.n_freq; l += CG) {
        const float scale = (float)(1 << l);
        float sv[3], cv[3];
#pragma unroll
        for (int c = 0; c < 3; ++c) sincospif(scale * u[c], &sv[c], &cv[c]);  // 2^l u is exact
        float *y = x + 3 + 6 * l;
        y[0] = sv[0]; y[1] = sv[1]; y[2] = sv[2];
        y[3] = cv[0]; y[4] = cv[1]; y[5] = cv[2];
      }
    }
    __syncthreads();
    const float *src = X0;
    float *dst = HA;
    int ldx = ld0, n_in = sh.in_dim;
    const float *w = wp;
    for (int l = 0; l < sh.n_hidden; ++l) {
      const float *x0 = src + (size_t)sp * ldx, *x1 = x0 + (size_t)HS * ldx;
      const float *wc = w + cg * WQ;
      float acc[2][WQ];
#pragma unroll
      for (int q = 0; q < WQ / 4; ++q) {
        const float4 v = ldg4(wc + n_in * WD + 4 * q);
        acc[0][4 * q] = acc[1][4 * q] = v.x; acc[0][4 * q + 1] = acc[1][4 * q + 1] = v.y;
        acc[0][4 * q + 2] = acc[1][4 * q + 2] = v.z; acc[0][4 * q + 3] = acc[1][4 * q + 3] = v.w;
      }
      int i = 0;
      for (; i + 4 <= n_in; i += 4) {
        const float4 a4 = lds4(x0 + i), b4 = lds4(x1 + i);
        const float xa[4] = {a4.x, a4.y, a4.z, a4.w}, xb[4] = {b4.x, b4.y, b4.z, b4.w};
#pragma unroll
        for (int ii = 0; ii < 4; ++ii) {
          const float *wr = wc + (i + ii) * WD;
#pragma unroll
          for (int q = 0; q < WQ / 4; ++q) {
            const float4 v = ldg4(wr + 4 * q);
            acc[0][4 * q] = fmaf(xa[ii], v.x, acc[0][4 * q]); acc[0][4 * q + 1] = fmaf(xa[ii], v.y, acc[0][4 * q + 1]);
            acc[0][4 * q + 2] = fmaf(xa[ii], v.z, acc[0][4 * q + 2]); acc[0][4 * q + 3] = fmaf(xa[ii], v.w, acc[0][4 * q + 3]);
            acc[1][4 * q] = fmaf(xb[ii], v.x, acc[1][4 * q]); acc[1][4 * q + 1] = fmaf(xb[ii], v.y, acc[1][4 * q + 1]);
            acc[1][4 * q + 2] = fmaf(xb[ii], v.z, acc[1][4 * q + 2]); acc[1][4 * q + 3] = fmaf(xb[ii], v.w, acc[1][4 * q + 3]);
          }
        }
      }
      for (; i < n_in; ++i) {
        const float xa = x0[i], xb = x1[i];
        const float *wr = wc + i * WD;
#pragma unroll
        for (int q = 0; q < WQ / 4; ++q) {
          const float4 v = ldg4(wr + 4 * q);
          acc[0][4 * q] = fmaf(xa, v.x, acc[0][4 * q]); acc[0][4 * q + 1] = fmaf(xa, v.y, acc[0][4 * q + 1]);
          acc[0][4 * q + 2] = fmaf(xa, v.z, acc[0][4 * q + 2]); acc[0][4 * q + 3] = fmaf(xa, v.w, acc[0][4 * q + 3]);
          acc[1][4 * q] = fmaf(xb, v.x, acc[1][4 * q]); acc[1][4 * q + 1] = fmaf(xb, v.y, acc[1][4 * q + 1]);
          acc[1][4 * q + 2] = fmaf(xb, v.z, acc[1][4 * q + 2]); acc[1][4 * q + 3] = fmaf(xb, v.w, acc[1][4 * q + 3]);
        }
      }
#pragma unroll
      for (int p = 0; p < 2; ++p) {
        float *y = dst + (size_t)(sp + p * HS) * ldw + cg * WQ;
#pragma unroll
        for (int q = 0; q < WQ / 4; ++q)
          *reinterpret_cast<float4 *>(y + 4 * q) = make_float4(fmaxf(acc[p][4 * q], 0.0f), fmaxf(acc[p][4 * q + 1], 0.0f),
                                                               fmaxf(acc[p][4 * q + 2], 0.0f), fmaxf(acc[p][4 * q + 3], 0.0f));
      }
      __syncthreads();
      w += n_in * WD + WD;
      n_in = WD; ldx = ldw;
      src = dst; dst = dst == HA ? HB : HA;
    }
    // head: output o by column group o mod CG, raw values into the free buffer
    {
      const int n_out = sh.out_dim;
      const float *x0 = src + (size_t)sp * ldw, *x1 = x0 + (size_t)HS * ldw;
      const float *bh = w + WD * n_out;
      for (int o = cg; o < n_out; o += CG) {
        float r0 = __ldg(bh + o), r1 = r0;
#pragma unroll 4
        for (int i = 0; i < WD; i += 4) {
          const float4 a4 = lds4(x0 + i), b4 = lds4(x1 + i);
          const float w0 = __ldg(w + i * n_out + o), w1 = __ldg(w + (i + 1) * n_out + o);
          const float w2 = __ldg(w + (i + 2) * n_out + o), w3 = __ldg(w + (i + 3) * n_out + o);
          r0 = fmaf(a4.x, w0, r0); r0 = fmaf(a4.y, w1, r0); r0 = fmaf(a4.z, w2, r0); r0 = fmaf(a4.w, w3, r0);
          r1 = fmaf(b4.x, w0, r1); r1 = fmaf(b4.y, w1, r1); r1 = fmaf(b4.z, w2, r1); r1 = fmaf(b4.w, w3, r1);
        }
        dst[(size_t)sp * ldw + o] = r0;
        dst[(size_t)(sp + HS) * ldw + o] = r1;
      }
    }
    __syncthreads();
    if (cg == 0) {
#pragma unroll
      for (int p = 0; p < 2; ++p) {
        if (!live[p]) continue;
        const float *raw = dst + (size_t)(sp + p * HS) * ldw;
        float4 r;
        r.x = 1.0f / (1.0f + expf(-raw[0]));
        r.y = 1.0f / (1.0f + expf(-raw[1]));
        r.z = 1.0f / (1.0f + expf(-raw[2]));
        const float sigma = fmaxf(raw[3], 0.0f) + log1pf(expf(-fabsf(raw[3])));
        r.w = expf(-sigma * delta[p]);  // e = 1 - alpha
        const size_t out = (size_t)(slot[p] - lv.band.slot0) * (size_t)a.K + (size_t)kk[p];
        a.staging[out] = r;
        if (a.staging_feat)
          for (int c = 0; c < sh.n_feat; ++c) reinterpret_cast<float *>(a.staging_feat)[out * sh.n_feat + c] = raw[4 + c];
      }
    }
  }
}

}  // namespace

cudaError_t ms_mlp_f32(const MsMlpArgs &a, cudaStream_t s) {
  size_t smem = (size_t)a.shape.params * sizeof(float);
  void (*fn)(MsMlpArgs) = mlp_f32_kernel;
  int threads = MS_ROWS;
  const int wd = a.shape.width;
  const size_t smem_wide = (size_t)MS_ROWS * (ld4_of(a.shape.in_dim) + 2 * ld4_of(wd)) * sizeof(float);
  if (wd == 32 && a.shape.params % 4 == 0 && a.shape.n_hidden >= 1 && a.shape.n_hidden <= 3) {
    fn = a.shape.n_hidden == 1 ? mlp_f32_w32_kernel<1, 2> : (a.shape.n_hidden == 2 ? mlp_f32_w32_kernel<2, 2> : mlp_f32_w32_kernel<3, 2>);
    threads = MS_ROWS / 2;
  } else if ((wd == 16 || wd == 32 || wd == 64 || wd == 128) && a.shape.mode == MS_MODE_LOCAL && a.shape.params % 4 == 0 &&
             a.shape.out_dim <= wd && a.shape.n_hidden >= 1 && smem_wide <= 200 * 1024) {
    const int cg = wd == 128 ? 8 : 4;
    fn = wd == 16 ? mlp_f32_wide_kernel<16, 4> : wd == 32 ? mlp_f32_wide_kernel<32, 4>
       : wd == 64 ? mlp_f32_wide_kernel<64, 4> : mlp_f32_wide_kernel<128, 8>;
    threads = MS_ROWS * cg / 2;
    smem = smem_wide;
  }
  cudaError_t e = cudaFuncSetAttribute((const void *)fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  // a CTA per block while they fit a few waves of resident CTAs, else a grid-stride walk (the block count of a band
  // lives on the device)
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
  unsigned grid = (unsigned)(n_sm * occ) * 4u;       // whole rounds of resident CTAs: no ragged last round
  if (a.n_blocks_hint > 0 && a.n_blocks_hint < grid) grid = a.n_blocks_hint;
  fn<<<grid, threads, smem, s>>>(a);
  MS_LAUNCHED();
  return cudaGetLastError();
}
