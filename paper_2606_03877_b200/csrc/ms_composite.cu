// ms_composite.cu -- stage (e): per-ray merge of the hit intervals' sample streams in
// (t, primitive id, k) order and front-to-back compositing (Eq.6, Eq.14):
//   w = T (1 - e); C += w rgb; F += w feat; T <- T e; stop once T < t_stop (NS (e), Q9).
// Each stream t_k = t_in + (k + 1/2) delta is already sorted in k (fp32 rounding is monotone),
// so a cursor per hit and a min-selection over the ray's hits reproduces the full sort.
// One thread per ray; cursor state lives in a global scratch array (8 B per hit) so any number
// of hits per ray is handled.  HBM-bound: reads 16 B (+ 4 n_feat B) per sample.
#include "ms_internal.cuh"
#include <math_constants.h>

namespace {

template <int NF, bool DEBUG>
__global__ void __launch_bounds__(128) composite_kernel(MsCompositeArgs a, int dbg_ray, int *dbg_prim, int *dbg_k,
                                                        float *dbg_t) {
  int ray = DEBUG ? dbg_ray : (int)(blockIdx.x * blockDim.x + threadIdx.x);
  if (ray >= a.n_rays || (DEBUG && (blockIdx.x != 0 || threadIdx.x != 0))) return;
  const uint32_t off = a.ray_off[ray];
  const int n = (int)(a.ray_off[ray + 1] - off);
  const int K = a.K;
  const int nf = NF >= 0 ? NF : a.n_feat;
  float T = 1.0f, C0 = 0.f, C1 = 0.f, C2 = 0.f;
  float F[NF > 0 ? NF : (NF < 0 ? MS_MAX_OUT : 1)];
#pragma unroll
  for (int c = 0; c < (NF > 0 ? NF : (NF < 0 ? MS_MAX_OUT : 1)); ++c) F[c] = 0.f;
  const MsHit *hits = a.hits + off;
  float2 *cur = reinterpret_cast<float2 *>(a.cur_t) + off;  // (t of the next sample, its k)
  for (int h = 0; h < n; ++h) cur[h] = make_float2(ms_sample_t(hits[h].t_in, hits[h].delta, 0), __int_as_float(0));
  const long total = (long)n * K;
  for (long it = 0; it < total; ++it) {
    int best = -1, best_prim = 0;
    float bt = CUDART_INF_F;
    for (int h = 0; h < n; ++h) {
      const float t = cur[h].x;  // +inf once the stream is exhausted
      if (t < bt) {
        bt = t; best = h; best_prim = -1;
      } else if (t == bt && best >= 0) {
        if (best_prim < 0) best_prim = hits[best].prim;
        const int p = hits[h].prim;
        if (p < best_prim) { best = h; best_prim = p; }
      }
    }
    if (best < 0) break;  // only if some t is NaN/inf; cannot happen for finite inputs
    const MsHit hb = hits[best];
    const int k = __float_as_int(cur[best].y);
    cur[best] = make_float2(k + 1 < K ? ms_sample_t(hb.t_in, hb.delta, k + 1) : CUDART_INF_F, __int_as_float(k + 1));
    if (DEBUG) {
      dbg_prim[it] = hb.prim; dbg_k[it] = k; dbg_t[it] = bt;
      continue;
    }
    const size_t s = (size_t)(off + (uint32_t)best) * (size_t)K + (size_t)k;
    const float4 v = a.staging[s];
    const float w = T * (1.0f - v.w);
    C0 = fmaf(w, v.x, C0); C1 = fmaf(w, v.y, C1); C2 = fmaf(w, v.z, C2);
    if (NF != 0 && a.staging_feat) {
      const float *f = a.staging_feat + s * (size_t)nf;
      if (NF > 0) {
#pragma unroll
        for (int c = 0; c < (NF > 0 ? NF : 1); c += 4) {
          const float4 q = *reinterpret_cast<const float4 *>(f + c);
          F[c] = fmaf(w, q.x, F[c]); F[c + 1] = fmaf(w, q.y, F[c + 1]);
          F[c + 2] = fmaf(w, q.z, F[c + 2]); F[c + 3] = fmaf(w, q.w, F[c + 3]);
        }
      } else {
        for (int c = 0; c < nf; ++c) F[c] = fmaf(w, f[c], F[c]);
      }
    }
    T *= v.w;
    if (T < a.t_stop) break;
  }
  if (DEBUG) return;
  a.out_rgb[3 * (size_t)ray + 0] = C0;
  a.out_rgb[3 * (size_t)ray + 1] = C1;
  a.out_rgb[3 * (size_t)ray + 2] = C2;
  a.out_alpha[ray] = 1.0f - T;
  if (NF != 0 && a.out_feat)
    for (int c = 0; c < nf; ++c) a.out_feat[(size_t)ray * nf + c] = F[c];
}

}  // namespace

cudaError_t ms_composite(const MsCompositeArgs &a, cudaStream_t s) {
  if (a.n_rays == 0) return cudaSuccess;
  unsigned grid = (unsigned)((a.n_rays + 127) / 128);
  const bool feat = a.n_feat > 0 && a.out_feat && a.staging_feat;
  if (!feat) composite_kernel<0, false><<<grid, 128, 0, s>>>(a, 0, nullptr, nullptr, nullptr);
  else if (a.n_feat == 32) composite_kernel<32, false><<<grid, 128, 0, s>>>(a, 0, nullptr, nullptr, nullptr);
  else composite_kernel<-1, false><<<grid, 128, 0, s>>>(a, 0, nullptr, nullptr, nullptr);
  MS_LAUNCHED();
  return cudaGetLastError();
}

cudaError_t ms_sample_order(const MsCompositeArgs &a, int ray, int *prim, int *k, float *t, cudaStream_t s) {
  composite_kernel<0, true><<<1, 32, 0, s>>>(a, ray, prim, k, t);
  MS_LAUNCHED();
  return cudaGetLastError();
}
