// ms_mlp_f32.cu -- stage (d), fp32 SIMT path (NS: "rgb/alpha within 1e-5 max abs for the fp32
// path"; CFG1).  One CTA = one 128-sample row block of ONE primitive, whose fp32 weights are
// staged in shared memory once per CTA; one thread = one sample: canonical u,
// positional encoding Eq.5 with exact-argument sincospif(2^l u), Linear+ReLU layers with
// fp32 FMA accumulation, rgb = sigmoid, sigma = softplus, e = exp(-sigma*delta).
// This path is the accuracy reference on the device; the throughput path is ms_mlp_tc.cu.
#include "ms_internal.cuh"
#include "ms_tile_gemm.cuh"

namespace {

// sin(pi x), cos(pi x) on the special-function unit: exact reduction to [-1, 1], then MUFU.SIN / MUFU.COS, whose
// absolute error on [-pi, pi] is 2^-21.4 / 2^-21.2 (CUDA C Programming Guide, intrinsic functions)
__device__ __forceinline__ void sincospi_mufu(float x, float *s, float *c) {
  const float r = x - 2.0f * rintf(0.5f * x);
  const float a = 3.14159265358979323846f * r;
  *s = __sinf(a);
  *c = __cosf(a);
}

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
  float *const h_s = w_s + ((sh.params + 3) & ~3);     // [SPT][32][MS_ROWS / SPT]: the inputs of the hidden layers 2..
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
    // (a runtime loop: six unrolled copies of this body put the kernel beyond the 32 KB instruction cache and the
    // warps of an SM, each at a place of its own, stalled on instruction fetch -- 1.3 stall cycles per issue, ncu)
#pragma unroll 1
    for (int c = 0; c < 6; ++c) {
      float zc[SPT];
#pragma unroll
      for (int p = 0; p < SPT; ++p)
        zc[p] = c == 0 ? z[p][0] : c == 1 ? z[p][1] : c == 2 ? z[p][2] : c == 3 ? z[p][3] : c == 4 ? z[p][4] : z[p][5];
      float scale = 1.0f;
#pragma unroll 1
      for (int l = 0; l < sh.n_freq; ++l) {
        float sv[SPT], cv[SPT];
#pragma unroll
        for (int p = 0; p < SPT; ++p) sincospi_mufu(scale * zc[p], &sv[p], &cv[p]);  // 2^l z is exact; 36 pairs per hit:
        // sincospif here was 19 % of the kernel's instructions; with the SFU the image stays 2e-7 from the oracle (bar 1e-5)
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
    // the layer's inputs go through shared memory (column tid of h_s: conflict-free), so that the loop over them need
    // not be unrolled for register indexing: 2 048 FMAs of straight-line code per layer otherwise
    __syncwarp();
#pragma unroll
    for (int p = 0; p < SPT; ++p)
#pragma unroll
      for (int i = 0; i < 32; ++i) h_s[(p * 32 + i) * (MS_ROWS / SPT) + threadIdx.x] = h[p][i];
    __syncwarp();
#pragma unroll 2
    for (int i = 0; i < 32; ++i) {
      const float4 *wr = reinterpret_cast<const float4 *>(w + i * 32);
      float x[SPT];
#pragma unroll
      for (int p = 0; p < SPT; ++p) x[p] = h_s[(p * 32 + i) * (MS_ROWS / SPT) + threadIdx.x];
#pragma unroll
      for (int q = 0; q < 8; ++q) {
        const float4 v = wr[q];
#pragma unroll
        for (int p = 0; p < SPT; ++p) {
          acc[p][4 * q] = fmaf(x[p], v.x, acc[p][4 * q]); acc[p][4 * q + 1] = fmaf(x[p], v.y, acc[p][4 * q + 1]);
          acc[p][4 * q + 2] = fmaf(x[p], v.z, acc[p][4 * q + 2]); acc[p][4 * q + 3] = fmaf(x[p], v.w, acc[p][4 * q + 3]);
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

// North-star mode, hidden widths that are multiples of 4: the layers as register-tiled fp32 GEMMs over the 128 samples
// of a row block (ms_tile_gemm.cuh: feature-major activations in shared memory, 4 x 4 thread tiles, staged weight
// panels).  The same arithmetic in the same order as mlp_f32_kernel (acc = b; acc = fma(x_i, W[i][o], acc) for i
// ascending) -- bitwise the same staging.  Shared memory: X0^T, two buffers that alternate as layer outputs (the head's
// raw outputs land in the free one), the weight panel.
struct WideLayout {
  int R0, LS, LW;
  size_t off_a, off_b, off_ws, floats;
};
__host__ __device__ inline WideLayout wide_layout(const MsMlpShape &sh) {
  WideLayout L;
  L.R0 = (sh.in_dim + 3) & ~3;
  L.LS = MS_ROWS + 4;
  const int rows = sh.width > sh.out_dim ? sh.width : ((sh.out_dim + 3) & ~3);
  L.LW = rows + 4;
  size_t o = (size_t)L.R0 * L.LS;
  L.off_a = o; o += (size_t)rows * L.LS;
  L.off_b = o; o += (size_t)rows * L.LS;
  L.off_ws = o; o += (size_t)TG_KP * L.LW;
  L.floats = o;
  return L;
}

__global__ void __launch_bounds__(TG_NT) mlp_f32_tile_kernel(MsMlpArgs a) {
  constexpr int BS = MS_ROWS, NCG = TG_NT / BS;
  extern __shared__ __align__(16) float sm[];
  __shared__ int s_seg;
  const MsMlpShape &sh = a.shape;
  const LaunchView lv(a.segs);
  const WideLayout L = wide_layout(sh);
  const int LS = L.LS, LW = L.LW, WD = sh.width;
  float *const X0T = sm, *const HA = sm + L.off_a, *const HB = sm + L.off_b, *const WS = sm + L.off_ws;
  const int tid = threadIdx.x, srow_in = tid & (BS - 1), cg = tid / BS;
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
    const uint64_t s = (uint64_t)(blk - (lv.bo[s_seg] - lv.base)) * MS_ROWS + srow_in;
    const uint32_t j = (uint32_t)(s / (uint32_t)a.K);
    const int k = (int)(s % (uint32_t)a.K);
    const bool live = j < count;
    MsInterval iv;
    iv.t_in = 0.f; iv.delta = 0.f; iv.slot = 0; iv.dx = 0.f; iv.dy = 0.f; iv.dz = 1.f; iv.ray = 0; iv.prim = prim;
    if (live) iv = a.intervals[first + j];
    const size_t out = (size_t)((uint32_t)iv.slot - lv.band.slot0) * (size_t)a.K + (size_t)k;
    {                                 // Eq.5 into this sample's column of X0^T: frequency l by helper l mod NCG
      const float d[3] = {iv.dx, iv.dy, iv.dz};
      const float t = ms_sample_tm(iv.t_in, iv.delta, k, false);
      float u[3];
      ms_sample_u(a.A + 9 * (size_t)prim, a.center + 3 * (size_t)prim, a.cam.o, d, t, u);
      float *x = X0T + srow_in;
      if (cg == 0) {
        x[0] = u[0]; x[LS] = u[1]; x[2 * LS] = u[2];
        if (sh.use_viewdir) { float *v = x + (size_t)(3 + 6 * sh.n_freq) * LS; v[0] = d[0]; v[LS] = d[1]; v[2 * LS] = d[2]; }
        if (a.staging_gate && live) a.staging_gate[out] = ms_slot_gates(u);
      }
      for (int l = cg; l < sh.n_freq; l += NCG) {
        const float scale = (float)(1 << l);
        float sv[3], cv[3];
#pragma unroll
        for (int c = 0; c < 3; ++c) sincospif(scale * u[c], &sv[c], &cv[c]);  // 2^l u is exact
        float *y = x + (size_t)(3 + 6 * l) * LS;
        y[0] = sv[0]; y[LS] = sv[1]; y[2 * LS] = sv[2];
        y[3 * LS] = cv[0]; y[4 * LS] = cv[1]; y[5 * LS] = cv[2];
      }
    }
    const float *src = X0T;
    float *dst = HA;
    int n_in = sh.in_dim;
    const float *w = wp;
    for (int l = 0; l < sh.n_hidden; ++l) {
      tg_fwd<BS>(src, n_in, w, WD, WD, true, dst, WS, LS, LW);
      w += n_in * WD + WD;
      n_in = WD;
      src = dst; dst = dst == HA ? HB : HA;
    }
    const int n_out = sh.out_dim, n_out4 = n_out & ~3;
    if (n_out4) tg_fwd<BS>(src, WD, w, n_out, n_out4, false, dst, WS, LS, LW);
    if (n_out4 < n_out) {             // outputs past the last group of four: one thread per (sample, output)
      const float *x = src + srow_in;
      for (int o = n_out4 + cg; o < n_out; o += NCG) {
        float acc = __ldg(w + WD * n_out + o);
        for (int i = 0; i < WD; ++i) acc = fmaf(x[(size_t)i * LS], __ldg(w + i * n_out + o), acc);
        dst[(size_t)o * LS + srow_in] = acc;
      }
      __syncthreads();
    }
    if (cg == 0 && live) {
      const float *raw = dst + srow_in;
      float4 r;
      r.x = 1.0f / (1.0f + expf(-raw[0]));
      r.y = 1.0f / (1.0f + expf(-raw[LS]));
      r.z = 1.0f / (1.0f + expf(-raw[2 * LS]));
      const float r3 = raw[3 * LS];
      const float sigma = fmaxf(r3, 0.0f) + log1pf(expf(-fabsf(r3)));
      r.w = expf(-sigma * iv.delta);  // e = 1 - alpha
      a.staging[out] = r;
    }
    if (a.staging_feat && live)       // feature channel c by helper c mod NCG
      for (int c = cg; c < sh.n_feat; c += NCG)
        reinterpret_cast<float *>(a.staging_feat)[out * sh.n_feat + c] = dst[(size_t)(4 + c) * LS + srow_in];
  }
}

}  // namespace

cudaError_t ms_mlp_f32(const MsMlpArgs &a, cudaStream_t s) {
  size_t smem = (size_t)a.shape.params * sizeof(float);
  void (*fn)(MsMlpArgs) = mlp_f32_kernel;
  int threads = MS_ROWS;
  const int wd = a.shape.width;
  const size_t smem_tile = wide_layout(a.shape).floats * sizeof(float);
  if (wd == 32 && a.shape.params % 4 == 0 && a.shape.n_hidden >= 1 && a.shape.n_hidden <= 3) {
    fn = a.shape.n_hidden == 1 ? mlp_f32_w32_kernel<1, 2> : (a.shape.n_hidden == 2 ? mlp_f32_w32_kernel<2, 2> : mlp_f32_w32_kernel<3, 2>);
    threads = MS_ROWS / 2;
    if (a.shape.n_hidden > 1) smem = ((size_t)((a.shape.params + 3) & ~3) + (size_t)32 * MS_ROWS) * sizeof(float);
  } else if (wd % 4 == 0 && wd >= 8 && a.shape.mode == MS_MODE_LOCAL && a.shape.n_hidden >= 1 && smem_tile <= 226 * 1024) {
    fn = mlp_f32_tile_kernel;
    threads = TG_NT;
    smem = smem_tile;
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
