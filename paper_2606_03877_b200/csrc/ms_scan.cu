// ms_scan.cu -- device exclusive scan of uint32 counts (used by stages (a), (c), (d) to turn
// per-primitive / per-pair / per-ray counts into offsets).  HBM-bound, one read + one write
// per element per level; levels shrink by 2048x.
#include <mutex>
#include "ms_internal.cuh"
#include "ms_cta_scan.cuh"

namespace {

constexpr int SCAN_THREADS = 256;
constexpr int SCAN_ITEMS = 8;
constexpr int SCAN_TILE = SCAN_THREADS * SCAN_ITEMS;

// Local exclusive scan of one tile; the tile total goes to sums[blockIdx.x] (or out[n] if sums == NULL).
__global__ void __launch_bounds__(SCAN_THREADS) scan_tile_kernel(const uint32_t *__restrict__ in,
                                                                 uint32_t *__restrict__ out, size_t n,
                                                                 uint32_t *__restrict__ sums) {
  __shared__ uint32_t warp_tot[SCAN_THREADS / 32];
  size_t base = (size_t)blockIdx.x * SCAN_TILE + (size_t)threadIdx.x * SCAN_ITEMS;
  uint32_t v[SCAN_ITEMS];
  uint32_t tsum = 0;
#pragma unroll
  for (int i = 0; i < SCAN_ITEMS; ++i) {
    v[i] = (base + i < n) ? in[base + i] : 0u;
    tsum += v[i];
  }
  int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  uint32_t inc = tsum;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    uint32_t o = __shfl_up_sync(0xffffffffu, inc, d);
    if (lane >= d) inc += o;
  }
  if (lane == 31) warp_tot[warp] = inc;
  __syncthreads();
  if (warp == 0) {
    uint32_t w = lane < SCAN_THREADS / 32 ? warp_tot[lane] : 0u;
#pragma unroll
    for (int d = 1; d < SCAN_THREADS / 32; d <<= 1) {
      uint32_t o = __shfl_up_sync(0xffffffffu, w, d);
      if (lane >= d) w += o;
    }
    if (lane < SCAN_THREADS / 32) warp_tot[lane] = w;  // inclusive over warps
  }
  __syncthreads();
  uint32_t excl = inc - tsum + (warp > 0 ? warp_tot[warp - 1] : 0u);
#pragma unroll
  for (int i = 0; i < SCAN_ITEMS; ++i) {
    if (base + i < n) out[base + i] = excl;
    excl += v[i];
  }
  if (threadIdx.x == SCAN_THREADS - 1) {
    uint32_t total = warp_tot[SCAN_THREADS / 32 - 1];
    if (sums) sums[blockIdx.x] = total;
    else out[n] = total;
  }
}

__global__ void __launch_bounds__(SCAN_THREADS) scan_add_kernel(uint32_t *__restrict__ out, size_t n,
                                                                const uint32_t *__restrict__ sums_scan,
                                                                uint32_t n_tiles) {
  uint32_t add = sums_scan[blockIdx.x];
  size_t base = (size_t)blockIdx.x * SCAN_TILE + (size_t)threadIdx.x * SCAN_ITEMS;
#pragma unroll
  for (int i = 0; i < SCAN_ITEMS; ++i)
    if (base + i < n) out[base + i] += add;
  if (blockIdx.x == 0 && threadIdx.x == 0) out[n] = sums_scan[n_tiles];
}

// up to SCAN_ONE_CTA elements: one CTA, one launch (three launches of the tiled form cost more than the loop)
constexpr int SCAN_ONE_THREADS = 1024;
constexpr size_t SCAN_ONE_CTA = 4 * (size_t)SCAN_ONE_THREADS * 8;
__global__ void __launch_bounds__(SCAN_ONE_THREADS) scan_one_cta_kernel(const uint32_t *in, uint32_t *out, size_t n) {
  __shared__ uint32_t wt[SCAN_ONE_THREADS / 32 + 1];
  cta_exclusive_scan_u32<SCAN_ONE_THREADS>(in, out, n, wt);
}

}  // namespace

size_t ms_scan_scratch_elems(size_t n) {
  size_t tot = 0;
  while (n > SCAN_TILE) {
    size_t nb = (n + SCAN_TILE - 1) / SCAN_TILE;
    tot += 2 * (nb + 1);
    n = nb;
  }
  return tot + 8;
}

cudaError_t ms_exclusive_scan_u32(const uint32_t *in, uint32_t *out, size_t n, uint32_t *scratch, cudaStream_t s) {
  if (n == 0) return cudaMemsetAsync(out, 0, sizeof(uint32_t), s);
  size_t nb = (n + SCAN_TILE - 1) / SCAN_TILE;
  if (nb == 1) {
    scan_tile_kernel<<<1, SCAN_THREADS, 0, s>>>(in, out, n, nullptr);
  MS_LAUNCHED();
    return cudaGetLastError();
  }
  if (n <= SCAN_ONE_CTA) {
    scan_one_cta_kernel<<<1, SCAN_ONE_THREADS, 0, s>>>(in, out, n);
  MS_LAUNCHED();
    return cudaGetLastError();
  }
  uint32_t *sums = scratch;            // [nb]
  uint32_t *sums_scan = scratch + nb + 1;  // [nb+1]
  scan_tile_kernel<<<(unsigned)nb, SCAN_THREADS, 0, s>>>(in, out, n, sums);
  MS_LAUNCHED();
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  e = ms_exclusive_scan_u32(sums, sums_scan, nb, scratch + 2 * (nb + 1), s);
  if (e != cudaSuccess) return e;
  scan_add_kernel<<<(unsigned)nb, SCAN_THREADS, 0, s>>>(out, n, sums_scan, (uint32_t)nb);
  MS_LAUNCHED();
  return cudaGetLastError();
}

// ---- the scan as entry points of its own (include/mlpsplat.h) ---------------------------------------------------
// ms_exclusive_scan_static: for callers that cannot allocate (CUDA graph capture, serving loops, harnesses that forbid
// cudaMalloc).  The tile sums of every level live in ONE file-scope device array of a fixed size instead of a
// cudaMalloc'ed scratch buffer: every GPU that loads the library holds these 65 KB until exit, every call shares them.
// The scan writes each scratch word before it reads it (scan_tile_kernel writes sums[0..nb), the next level writes
// sums_scan[0..nb]), so nothing has to be cleared between calls -- but two calls that overlap on the GPU (different
// streams, or graphs replayed concurrently) race on the array.
constexpr size_t SCAN_STATIC_MAX_N = (size_t)MS_SCAN_STATIC_MAX;
// levels of the tiled scan for n = 2^24: 8192 tile sums, then 4: 2 (8192 + 1) + 2 (4 + 1) + 8 words, rounded up
constexpr size_t SCAN_STATIC_WORDS = 16640;
static __device__ __align__(256) uint32_t ms_scan_static_scratch[SCAN_STATIC_WORDS];

namespace {

// the tiled scan with its scratch given: always the scan_tile_kernel / scan_add_kernel pair above one tile (the
// one-CTA shortcut of ms_exclusive_scan_u32 needs no scratch and is not taken here)
cudaError_t scan_tiled(const uint32_t *in, uint32_t *out, size_t n, uint32_t *scratch, cudaStream_t s) {
  if (n == 0) return cudaMemsetAsync(out, 0, sizeof(uint32_t), s);
  const size_t nb = (n + SCAN_TILE - 1) / SCAN_TILE;
  if (nb == 1) {
    scan_tile_kernel<<<1, SCAN_THREADS, 0, s>>>(in, out, n, nullptr);
    MS_LAUNCHED();
    return cudaGetLastError();
  }
  uint32_t *sums = scratch, *sums_scan = scratch + nb + 1;
  scan_tile_kernel<<<(unsigned)nb, SCAN_THREADS, 0, s>>>(in, out, n, sums);
  MS_LAUNCHED();
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  e = scan_tiled(sums, sums_scan, nb, scratch + 2 * (nb + 1), s);
  if (e != cudaSuccess) return e;
  scan_add_kernel<<<(unsigned)nb, SCAN_THREADS, 0, s>>>(out, n, sums_scan, (uint32_t)nb);
  MS_LAUNCHED();
  return cudaGetLastError();
}

// In host code the array's name is a host-side stand-in, not a device address: the address a kernel can use comes from
// cudaGetSymbolAddress, asked once per device with that device current.
constexpr int SCAN_MAX_DEVICES = 64;
std::mutex scan_static_mutex;
uint32_t *scan_static_ptr[SCAN_MAX_DEVICES] = {};

int scan_static_scratch(uint32_t **out) {
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= SCAN_MAX_DEVICES) {
    (void)cudaGetLastError();
    return MS_ERR_CUDA;
  }
  std::lock_guard<std::mutex> lock(scan_static_mutex);
  if (!scan_static_ptr[dev]) {
    if (ms_scan_scratch_elems(SCAN_STATIC_MAX_N) > SCAN_STATIC_WORDS) return MS_ERR_CAPACITY;   // the array is sized for the maximum
    void *p = nullptr;
    if (cudaGetSymbolAddress(&p, ms_scan_static_scratch) != cudaSuccess || !p) {
      (void)cudaGetLastError();
      return MS_ERR_CUDA;
    }
    scan_static_ptr[dev] = static_cast<uint32_t *>(p);
  }
  *out = scan_static_ptr[dev];
  return MS_OK;
}

}  // namespace

extern "C" {

int ms_exclusive_scan_static(const uint32_t *in, uint32_t *out, size_t n, void *stream) {
  if (!out || (n > 0 && !in)) return MS_ERR_INVALID_ARG;
  if (n > SCAN_STATIC_MAX_N) return MS_ERR_CAPACITY;
  uint32_t *scratch = nullptr;
  const int rc = scan_static_scratch(&scratch);
  if (rc != MS_OK) return rc;
  if (scan_tiled(in, out, n, scratch, static_cast<cudaStream_t>(stream)) != cudaSuccess) {
    (void)cudaGetLastError();
    return MS_ERR_CUDA;
  }
  return MS_OK;
}

int ms_exclusive_scan_device(const uint32_t *in, uint32_t *out, size_t n, void *stream) {
  if (!out || (n > 0 && !in)) return MS_ERR_INVALID_ARG;
  if (n >= (1ull << 32)) return MS_ERR_INVALID_ARG;
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  uint32_t *scratch = nullptr;
  if (cudaMalloc(&scratch, (ms_scan_scratch_elems(n) + 16) * sizeof(uint32_t)) != cudaSuccess) {
    (void)cudaGetLastError();
    return MS_ERR_OUT_OF_MEMORY;
  }
  cudaError_t e = ms_exclusive_scan_u32(in, out, n, scratch, s);
  if (e == cudaSuccess) e = cudaStreamSynchronize(s);     // the scratch is freed below
  cudaFree(scratch);
  if (e != cudaSuccess) {
    (void)cudaGetLastError();
    return MS_ERR_CUDA;
  }
  return MS_OK;
}

}  // extern "C"
