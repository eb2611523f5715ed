// ms_tile_gemm.cuh -- the forward GEMM of the register-tiled fp32 MLP kernels (ms_mlp_f32.cu: stage (d) on the fp32
// path; ms_backward.cu: the recomputation inside the backward kernel).  512 threads; activations FEATURE-major in shared
// memory, X^T[feature][sample] with leading dimension LS = BS + 4 (= 4 mod 32 words); a thread owns 4 outputs x 4
// samples, a warp is 8 sample tiles x 4 output tiles: one float4 of X^T and one of the staged weight panel per lane and
// contraction step, 8 resp. 4 distinct 16-byte chunks per warp.
#pragma once
#include <cuda_runtime.h>

constexpr int TG_NT = 512;            // threads per CTA
constexpr int TG_NW = TG_NT / 32;     // warps per CTA
constexpr int TG_KP = 64;             // contraction steps of one staged weight panel

__device__ __forceinline__ float4 tg_lds4(const float *p) { return *reinterpret_cast<const float4 *>(p); }
__device__ __forceinline__ void tg_sts4(float *p, float x, float y, float z, float w) {
  *reinterpret_cast<float4 *>(p) = make_float4(x, y, z, w);
}

// Z^T[o][s] = b[o] + sum_i W[i][o] X^T[i][s] for the n_out (multiple of 4) leading outputs of a layer whose weight rows
// are ldw floats apart and whose bias follows its n_in rows; sums in the order bias, i = 0, 1, ...  WS: panel of
// TG_KP x LW floats.  Every thread of the CTA calls it; it ends with a barrier (OUT is visible to all).
template <int BS>
__device__ __forceinline__ void tg_fwd(const float *XT, int n_in, const float *Wg, int ldw, int n_out, bool relu,
                                       float *OUT, float *WS, int LS, int LW) {
  constexpr int NSW = BS / 32;                 // warps side by side over the samples
  constexpr int NFW = (TG_NW / NSW) * 4;       // output tiles (of 4) the CTA covers in one pass
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int sg = (warp % NSW) * 8 + (lane & 7), ft = (warp / NSW) * 4 + (lane >> 3);
  const int n_ft = n_out >> 2;
  const float *bias = Wg + (size_t)n_in * ldw;
  for (int f0 = 0; f0 < n_ft; f0 += NFW) {
    const int f = f0 + ft;
    const bool on = f < n_ft;
    float acc[4][4];
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      const float b = on ? __ldg(bias + 4 * f + q) : 0.0f;
#pragma unroll
      for (int p = 0; p < 4; ++p) acc[q][p] = b;
    }
    for (int i0 = 0; i0 < n_in; i0 += TG_KP) {
      const int kp = min(TG_KP, n_in - i0);
      __syncthreads();                                   // the panel's previous readers are done
      for (int e = tid; e < kp * n_out; e += TG_NT) {
        const int rr = e / n_out, c = e - rr * n_out;
        WS[rr * LW + c] = __ldg(Wg + (size_t)(i0 + rr) * ldw + c);
      }
      __syncthreads();
      if (on) {
        const float *xp = XT + (size_t)i0 * LS + 4 * sg, *wq = WS + 4 * f;
#pragma unroll 4
        for (int rr = 0; rr < kp; ++rr) {
          const float4 x4 = tg_lds4(xp + (size_t)rr * LS), w4 = tg_lds4(wq + rr * LW);
          const float xs[4] = {x4.x, x4.y, x4.z, x4.w}, ws[4] = {w4.x, w4.y, w4.z, w4.w};
#pragma unroll
          for (int q = 0; q < 4; ++q)
#pragma unroll
            for (int p = 0; p < 4; ++p) acc[q][p] = fmaf(xs[p], ws[q], acc[q][p]);
        }
      }
    }
    if (on) {
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        float *y = OUT + (size_t)(4 * f + q) * LS + 4 * sg;
        if (relu) tg_sts4(y, fmaxf(acc[q][0], 0.0f), fmaxf(acc[q][1], 0.0f), fmaxf(acc[q][2], 0.0f), fmaxf(acc[q][3], 0.0f));
        else tg_sts4(y, acc[q][0], acc[q][1], acc[q][2], acc[q][3]);
      }
    }
  }
  __syncthreads();
}
