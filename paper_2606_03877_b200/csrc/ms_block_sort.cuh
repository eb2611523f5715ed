// ms_block_sort.cuh -- the one-CTA radix sort of small key sets as a device function: the body of
// radix_block_sort_kernel (ms_sort.cu) and a step of the fused small-frame kernel of stages (a) + (b) (ms_bin.cu).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

// Small key sets (<= 16 384 keys: CFG1's 52 and CFG2's 9 938 pairs): ALL passes in one CTA.  The keys live in
// registers (16 per thread, warp w owns the keys [512 w, 512 (w + 1)) in rounds of 32) and go through one shared-
// memory buffer between passes; ranking inside a pass is the scatter kernel's (match_any per round, per-warp digit
// counters), the digit offsets come from a 256-wide scan.  Replaces 2 launches per pass by one launch per sort --
// these frames are bound by launch latency, not by bandwidth.
constexpr int SB_THREADS = 1024;
constexpr int SB_WARPS = SB_THREADS / 32;
constexpr int SB_ITEMS = 16;
constexpr int SB_MAX = SB_THREADS * SB_ITEMS;

// ITEMS keys per thread (1, 4 or 16: the kernel picks the smallest that holds n -- a frame with a few hundred keys
// pays for 1 024 of them, not 16 384); only the warps that hold keys take part in the digit counts
template <int ITEMS>
__device__ __forceinline__ void block_sort_body(const uint64_t *keys, uint64_t *out, uint32_t n,
                                                int first_bit, int n_bits, uint64_t *buf, uint32_t (*wc)[256],
                                                uint32_t *dsum) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const uint32_t lt = (1u << lane) - 1u;
  const uint32_t wbase = (uint32_t)warp * 32 * ITEMS;
  const int n_aw = (int)((n + 32 * ITEMS - 1) / (32 * ITEMS));       // warps that hold keys
  uint64_t key[ITEMS];
#pragma unroll
  for (int r = 0; r < ITEMS; ++r) {
    const uint32_t i = wbase + r * 32 + lane;
    key[r] = i < n ? keys[i] : ~0ull;
  }
  for (int shift = first_bit; shift < n_bits; shift += 8) {
    for (int i = threadIdx.x; i < n_aw * 256; i += SB_THREADS) (&wc[0][0])[i] = 0;
    __syncthreads();
    uint32_t rank[ITEMS];
    if (warp < n_aw) {
#pragma unroll
      for (int r = 0; r < ITEMS; ++r) {
        const uint32_t i = wbase + r * 32 + lane;
        const bool valid = i < n;
        const uint32_t d = valid ? ((uint32_t)(key[r] >> shift) & 255u) : 256u;
        const uint32_t peers = __match_any_sync(0xffffffffu, d);
        const uint32_t prior = valid ? wc[warp][d] : 0u;
        __syncwarp();
        if (valid && (peers & lt) == 0u) wc[warp][d] = prior + __popc(peers);
        __syncwarp();
        rank[r] = prior + __popc(peers & lt);
      }
    }
    __syncthreads();
    if (threadIdx.x < 256) {       // thread t owns digit t: totals over the warps, exclusive scan over the digits
      uint32_t total = 0;
      for (int w = 0; w < n_aw; ++w) total += wc[w][threadIdx.x];
      uint32_t incl = total;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const uint32_t v = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += v;
      }
      if (lane == 31) dsum[warp] = incl;
      asm volatile("bar.sync 1, 256;");                    // the eight warps that own digits
      uint32_t run = incl - total;
      for (int w = 0; w < warp; ++w) run += dsum[w];
      for (int w = 0; w < n_aw; ++w) {                     // (digit, warp) offsets
        const uint32_t c = wc[w][threadIdx.x];
        wc[w][threadIdx.x] = run;
        run += c;
      }
    }
    __syncthreads();
    if (warp < n_aw) {
#pragma unroll
      for (int r = 0; r < ITEMS; ++r) {
        const uint32_t i = wbase + r * 32 + lane;
        if (i < n) buf[wc[warp][(uint32_t)(key[r] >> shift) & 255u] + rank[r]] = key[r];
      }
    }
    __syncthreads();
#pragma unroll
    for (int r = 0; r < ITEMS; ++r) {
      const uint32_t i = wbase + r * 32 + lane;
      key[r] = i < n ? buf[i] : ~0ull;
    }
    __syncthreads();
  }
#pragma unroll
  for (int r = 0; r < ITEMS; ++r) {
    const uint32_t i = wbase + r * 32 + lane;
    if (i < n) out[i] = key[r];
  }
}


// shared memory of the sort: SB_MAX keys + SB_WARPS x 256 digit counters (dynamic), 8 words of digit sums (static)
constexpr size_t SB_SMEM_BYTES = (size_t)SB_MAX * 8 + (size_t)SB_WARPS * 256 * 4;

// sorts keys[0, n) into out[0, n) by the bits [first_bit, n_bits); every thread of the SB_THREADS-thread CTA calls it.
// keys may have been written earlier in the same kernel by this CTA (after a __syncthreads()).
__device__ __forceinline__ void block_sort(const uint64_t *keys, uint64_t *out, uint32_t n, int first_bit, int n_bits,
                                           uint8_t *smem, uint32_t *dsum) {
  uint64_t *buf = reinterpret_cast<uint64_t *>(smem);                                    // [SB_MAX]
  uint32_t(*wc)[256] = reinterpret_cast<uint32_t(*)[256]>(smem + (size_t)SB_MAX * 8);     // [SB_WARPS][256]
  if (n <= SB_THREADS) block_sort_body<1>(keys, out, n, first_bit, n_bits, buf, wc, dsum);
  else if (n <= 4 * SB_THREADS) block_sort_body<4>(keys, out, n, first_bit, n_bits, buf, wc, dsum);
  else block_sort_body<SB_ITEMS>(keys, out, n, first_bit, n_bits, buf, wc, dsum);
}
