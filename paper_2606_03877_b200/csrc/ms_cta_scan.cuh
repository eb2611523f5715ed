// ms_cta_scan.cuh -- exclusive scan of uint32 counts by ONE CTA (small frames: a launch saved is 3 us saved).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

// out[i] = sum of in[j], j < i, for i in [0, n] (n + 1 values).  Every thread of the NT-thread CTA calls it; chunks of
// NT * 8 elements with a running carry.  wt: shared scratch of NT / 32 + 1 words.  in and out must not overlap; reads
// of out by other threads need a __syncthreads() after the call.  (No __restrict__: in may have been written earlier in
// the same kernel, so its loads must not take the non-coherent path.)
template <int NT>
__device__ __forceinline__ void cta_exclusive_scan_u32(const uint32_t *in, uint32_t *out, size_t n, uint32_t *wt) {
  constexpr int ITEMS = 8, NW = NT / 32;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  uint32_t carry = 0;
  for (size_t c0 = 0; c0 < n; c0 += (size_t)NT * ITEMS) {
    const size_t base = c0 + (size_t)threadIdx.x * ITEMS;
    uint32_t v[ITEMS], tsum = 0;
#pragma unroll
    for (int i = 0; i < ITEMS; ++i) {
      v[i] = base + i < n ? in[base + i] : 0u;
      tsum += v[i];
    }
    uint32_t inc = tsum;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
      const uint32_t o = __shfl_up_sync(0xffffffffu, inc, d);
      if (lane >= d) inc += o;
    }
    __syncthreads();                                     // the previous chunk's totals have been read
    if (lane == 31) wt[warp] = inc;
    __syncthreads();
    if (warp == 0) {
      uint32_t w = lane < NW ? wt[lane] : 0u;
#pragma unroll
      for (int d = 1; d < 32; d <<= 1) {
        const uint32_t o = __shfl_up_sync(0xffffffffu, w, d);
        if (lane >= d) w += o;
      }
      if (lane < NW) wt[lane] = w;                       // inclusive over the warps
    }
    __syncthreads();
    uint32_t excl = carry + inc - tsum + (warp > 0 ? wt[warp - 1] : 0u);
#pragma unroll
    for (int i = 0; i < ITEMS; ++i) {
      if (base + i < n) out[base + i] = excl;
      excl += v[i];
    }
    carry += wt[NW - 1];
  }
  if (threadIdx.x == 0) out[n] = carry;
}
