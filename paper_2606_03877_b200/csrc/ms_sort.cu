// ms_sort.cu -- stage (b): device LSD radix sort of the 64-bit (tile | z_entry bits | prim)
// keys (NS (b); the paper sorts per tile inside one 256-thread block).
// 8-bit digits, stable; only the bits actually used are sorted.  Each pass: per-block digit
// histogram -> exclusive scan (digit-major, block-minor) -> stable scatter.  The key set is
// <= ~0.5 M keys (L2-resident), so this stage is launch-latency-bound, not HBM-bound.
#include "ms_internal.cuh"
#include "ms_block_sort.cuh"

namespace {

constexpr int RS_THREADS = 256;
constexpr int RS_WARPS = RS_THREADS / 32;
constexpr int RS_ITEMS = 8;
constexpr int RS_TILE = RS_THREADS * RS_ITEMS;

// n_dev != NULL: the key count lives on the device (ms_render without host synchronisation); n is then its capacity
__global__ void __launch_bounds__(RS_THREADS) radix_hist_kernel(const uint64_t *__restrict__ keys, size_t n, int shift,
                                                                uint32_t *__restrict__ counts, uint32_t n_blocks,
                                                                const uint32_t *__restrict__ n_dev) {
  __shared__ uint32_t hist[256];
  if (n_dev) n = *n_dev < n ? (size_t)*n_dev : n;
  hist[threadIdx.x] = 0;
  __syncthreads();
  size_t base = (size_t)blockIdx.x * RS_TILE;
#pragma unroll
  for (int r = 0; r < RS_ITEMS; ++r) {
    size_t i = base + (size_t)r * RS_THREADS + threadIdx.x;
    if (i < n) atomicAdd(&hist[(uint32_t)(keys[i] >> shift) & 255u], 1u);
  }
  __syncthreads();
  counts[(size_t)threadIdx.x * n_blocks + blockIdx.x] = hist[threadIdx.x];
}

// Key order inside a block: warp w owns keys [w*32*ITEMS, (w+1)*32*ITEMS), visited in rounds of 32.
__global__ void __launch_bounds__(RS_THREADS) radix_scatter_kernel(const uint64_t *__restrict__ keys,
                                                                   uint64_t *__restrict__ out, size_t n, int shift,
                                                                   const uint32_t *__restrict__ offsets,
                                                                   const uint32_t *__restrict__ counts,
                                                                   uint32_t n_blocks, const uint32_t *__restrict__ n_dev) {
  __shared__ uint32_t wc[RS_WARPS][256];
  if (n_dev) n = *n_dev < n ? (size_t)*n_dev : n;
  __shared__ uint32_t wsum[RS_WARPS];
  for (int i = threadIdx.x; i < RS_WARPS * 256; i += RS_THREADS) (&wc[0][0])[i] = 0;
  __syncthreads();
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const uint32_t lt = (1u << lane) - 1u;
  size_t base = (size_t)blockIdx.x * RS_TILE + (size_t)warp * 32 * RS_ITEMS;
  uint64_t key[RS_ITEMS];
  uint32_t rank[RS_ITEMS];
#pragma unroll
  for (int r = 0; r < RS_ITEMS; ++r) {
    size_t i = base + (size_t)r * 32 + lane;
    bool valid = i < n;
    key[r] = valid ? keys[i] : 0ull;
    uint32_t d = valid ? ((uint32_t)(key[r] >> shift) & 255u) : 256u;
    uint32_t peers = __match_any_sync(0xffffffffu, d);
    uint32_t prior = valid ? wc[warp][d] : 0u;
    __syncwarp();
    if (valid && (peers & lt) == 0u) wc[warp][d] = prior + __popc(peers);
    __syncwarp();
    rank[r] = prior + __popc(peers & lt);
  }
  __syncthreads();
  {  // thread t owns digit t: exclusive prefix over warps + global offset of (digit, block)
    uint32_t run;
    if (offsets) {
      run = offsets[(size_t)threadIdx.x * n_blocks + blockIdx.x];
    } else {
      // few blocks (the usual case: <= 0.5 M keys): the (digit, block) offset straight from the count matrix --
      // digits below mine over all blocks, plus my digit in the blocks before this one -- no scan launches
      const uint32_t *row = counts + (size_t)threadIdx.x * n_blocks;
      uint32_t total = 0, before = 0;
      for (uint32_t b = 0; b < n_blocks; ++b) {
        const uint32_t c = row[b];
        before += b < blockIdx.x ? c : 0u;
        total += c;
      }
      uint32_t incl = total;   // inclusive scan of the digit totals over the 256 threads
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const uint32_t v = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += v;
      }
      if (lane == 31) wsum[warp] = incl;
      __syncthreads();
      uint32_t wbase = 0;
      for (int w = 0; w < warp; ++w) wbase += wsum[w];
      run = wbase + incl - total + before;
    }
#pragma unroll
    for (int w = 0; w < RS_WARPS; ++w) {
      uint32_t c = wc[w][threadIdx.x];
      wc[w][threadIdx.x] = run;
      run += c;
    }
  }
  __syncthreads();
#pragma unroll
  for (int r = 0; r < RS_ITEMS; ++r) {
    size_t i = base + (size_t)r * 32 + lane;
    if (i < n) {
      uint32_t d = (uint32_t)(key[r] >> shift) & 255u;
      out[wc[warp][d] + rank[r]] = key[r];
    }
  }
}

__global__ void __launch_bounds__(SB_THREADS) radix_block_sort_kernel(const uint64_t *keys, uint64_t *out,
                                                                      uint32_t n_host, const uint32_t *__restrict__ n_dev,
                                                                      int first_bit, int n_bits) {
  extern __shared__ __align__(16) uint8_t sb_smem[];
  __shared__ uint32_t dsum[8];
  const uint32_t n = n_dev ? (*n_dev < n_host ? *n_dev : n_host) : n_host;
  block_sort(keys, out, n, first_bit, n_bits, sb_smem, dsum);
}

static_assert((size_t)SB_MAX == MS_BLOCK_SORT_MAX, "ms_internal.cuh states the block sort's capacity");

}  // namespace

size_t ms_sort_scratch_elems(size_t n) {
  size_t nb = (n + RS_TILE - 1) / RS_TILE;
  if (nb == 0) nb = 1;
  size_t m = 256 * nb;
  return 2 * (m + 1) + ms_scan_scratch_elems(m) + 8;
}

cudaError_t ms_radix_sort_u64(uint64_t *a, uint64_t *b, size_t n, int first_bit, int n_bits, uint32_t *scratch,
                              uint64_t **result, cudaStream_t s, const uint32_t *n_dev) {
  *result = a;
  if ((n <= 1 && !n_dev) || n == 0 || n_bits <= 0) return cudaSuccess;
  if (n <= (size_t)SB_MAX) {       // one CTA, one launch (capacity n in the no-sync case: the count is read on the device)
    const size_t smem = SB_SMEM_BYTES;
    static bool attr_set = false;
    if (!attr_set) {
      cudaError_t e = cudaFuncSetAttribute((const void *)radix_block_sort_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
      if (e != cudaSuccess) return e;
      attr_set = true;
    }
    radix_block_sort_kernel<<<1, SB_THREADS, smem, s>>>(a, b, (uint32_t)n, n_dev, first_bit, n_bits);
    MS_LAUNCHED();
    *result = b;
    return cudaGetLastError();
  }
  size_t nb = (n + RS_TILE - 1) / RS_TILE;
  size_t m = 256 * nb;
  uint32_t *counts = scratch;
  uint32_t *offsets = scratch + m + 1;
  uint32_t *scan_scratch = scratch + 2 * (m + 1);
  uint64_t *src = a, *dst = b;
  // LSD and stable: bits below first_bit need no pass when the input is already ordered by them
  for (int shift = first_bit; shift < n_bits; shift += 8) {
    radix_hist_kernel<<<(unsigned)nb, RS_THREADS, 0, s>>>(src, n, shift, counts, (uint32_t)nb, n_dev);
  MS_LAUNCHED();
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    const bool self_scan = nb <= 256;   // the scatter kernel derives its offsets from the count matrix itself
    if (!self_scan) {
      e = ms_exclusive_scan_u32(counts, offsets, m, scan_scratch, s);
      if (e != cudaSuccess) return e;
    }
    radix_scatter_kernel<<<(unsigned)nb, RS_THREADS, 0, s>>>(src, dst, n, shift, self_scan ? nullptr : offsets, counts,
                                                             (uint32_t)nb, n_dev);
  MS_LAUNCHED();
    e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    uint64_t *t = src;
    src = dst;
    dst = t;
  }
  *result = src;
  return cudaSuccess;
}
