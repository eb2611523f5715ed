// ms_bin.cu -- scene prep and stage (a): projection of each ellipsoid support to a
// conservative screen-space AABB and emission of (tile | z_entry | prim) keys
// ("conservative overlap tests based on their projected support regions";
//  P:148 "AABB-tile-frustum intersection test"; NS (a)).  All arithmetic is the canonical
// fp32 sequence of DESIGN.md Sec.2.  Bytes: N*(3+9+9)*4 in, P*8 out -- negligible.
#include "ms_internal.cuh"
#include "ms_block_sort.cuh"
#include "ms_cta_scan.cuh"

namespace {

// P:74 / P:84: q -> R (Hamilton, (w,x,y,z)); A = diag(1/s) R^T; M = R diag(s)
__global__ void prep_prims_kernel(int n, const float *__restrict__ quat, const float *__restrict__ scale,
                                  float *__restrict__ A, float *__restrict__ M, int *__restrict__ bad) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  float w = quat[4 * i], x = quat[4 * i + 1], y = quat[4 * i + 2], z = quat[4 * i + 3];
  float s0 = scale[3 * i], s1 = scale[3 * i + 1], s2 = scale[3 * i + 2];
  float n2 = __fadd_rn(__fadd_rn(__fadd_rn(__fmul_rn(w, w), __fmul_rn(x, x)), __fmul_rn(y, y)), __fmul_rn(z, z));
  if (!(n2 > 0.0f) || isinf(n2) || !(s0 > 0.0f) || !(s1 > 0.0f) || !(s2 > 0.0f)) {
    atomicExch(bad, 1);
    return;
  }
  float nrm = __fsqrt_rn(n2);
  w = __fdiv_rn(w, nrm); x = __fdiv_rn(x, nrm); y = __fdiv_rn(y, nrm); z = __fdiv_rn(z, nrm);
  float xx = __fmul_rn(x, x), yy = __fmul_rn(y, y), zz = __fmul_rn(z, z);
  float xy = __fmul_rn(x, y), xz = __fmul_rn(x, z), yz = __fmul_rn(y, z);
  float wx = __fmul_rn(w, x), wy = __fmul_rn(w, y), wz = __fmul_rn(w, z);
  float R[9];
  R[0] = __fsub_rn(1.0f, __fmul_rn(2.0f, __fadd_rn(yy, zz)));
  R[1] = __fmul_rn(2.0f, __fsub_rn(xy, wz));
  R[2] = __fmul_rn(2.0f, __fadd_rn(xz, wy));
  R[3] = __fmul_rn(2.0f, __fadd_rn(xy, wz));
  R[4] = __fsub_rn(1.0f, __fmul_rn(2.0f, __fadd_rn(xx, zz)));
  R[5] = __fmul_rn(2.0f, __fsub_rn(yz, wx));
  R[6] = __fmul_rn(2.0f, __fsub_rn(xz, wy));
  R[7] = __fmul_rn(2.0f, __fadd_rn(yz, wx));
  R[8] = __fsub_rn(1.0f, __fmul_rn(2.0f, __fadd_rn(xx, yy)));
  float s[3] = {s0, s1, s2};
#pragma unroll
  for (int r = 0; r < 3; ++r)
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      A[9 * i + 3 * r + c] = __fdiv_rn(R[3 * c + r], s[r]);
      M[9 * i + 3 * r + c] = __fmul_rn(R[3 * r + c], s[c]);
    }
}

__device__ __forceinline__ void axis_bounds(const float *rx, float cxv, const float *rz, float czv, float zz,
                                            float focal, float centre, float *lo, float *hi) {
  float xz = __fsub_rn(ms_dot3(rx[0], rx[1], rx[2], rz[0], rz[1], rz[2]), __fmul_rn(cxv, czv));
  float xx = __fsub_rn(ms_dot3(rx[0], rx[1], rx[2], rx[0], rx[1], rx[2]), __fmul_rn(cxv, cxv));
  float m = __fdiv_rn(xz, zz);
  float q = __fsub_rn(__fmul_rn(m, m), __fdiv_rn(xx, zz));
  float h = __fsqrt_rn(q > 0.0f ? q : 0.0f);
  *lo = __fadd_rn(__fmul_rn(focal, __fsub_rn(m, h)), centre);
  *hi = __fadd_rn(__fmul_rn(focal, __fadd_rn(m, h)), centre);
}

__device__ __forceinline__ int clamp_lo(float v, int n) {
  float f = floorf(v);
  if (!(f > 0.0f)) return 0;
  if (f > (float)n) return n;
  return (int)f;
}
__device__ __forceinline__ int clamp_hi(float v, int n) {
  float f = ceilf(v);
  if (!(f < (float)(n - 1))) return n - 1;
  if (f < 0.0f) return -1;
  return (int)f;
}

__device__ __forceinline__ void project_body(int i, const float *__restrict__ center, const float *__restrict__ A,
                                             const float *__restrict__ M, const MsCam &cam, int tile, float eye_guard,
                                             uint32_t *tile_count, int4 *rect, float *z_entry, float *oprime,
                                             uint32_t *counters) {
  const float *mu = center + 3 * i;
  const float *Mi = M + 9 * i;
  const float *Ai = A + 9 * i;
  // o' = A (o - mu), reused by every ray of this view (stage (c))
  {
    float v0 = __fsub_rn(cam.o[0], mu[0]), v1 = __fsub_rn(cam.o[1], mu[1]), v2 = __fsub_rn(cam.o[2], mu[2]);
    oprime[3 * i + 0] = ms_dot3(Ai[0], Ai[1], Ai[2], v0, v1, v2);
    oprime[3 * i + 1] = ms_dot3(Ai[3], Ai[4], Ai[5], v0, v1, v2);
    oprime[3 * i + 2] = ms_dot3(Ai[6], Ai[7], Ai[8], v0, v1, v2);
  }
  float v0 = __fsub_rn(mu[0], cam.o[0]), v1 = __fsub_rn(mu[1], cam.o[1]), v2 = __fsub_rn(mu[2], cam.o[2]);
  const float *r = cam.r;
  float cv[3], Mc[9];
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    cv[a] = ms_dot3(r[a], r[3 + a], r[6 + a], v0, v1, v2);
#pragma unroll
    for (int j = 0; j < 3; ++j) Mc[3 * a + j] = ms_dot3(r[a], r[3 + a], r[6 + a], Mi[j], Mi[3 + j], Mi[6 + j]);
  }
  float rz2 = ms_dot3(Mc[6], Mc[7], Mc[8], Mc[6], Mc[7], Mc[8]);
  float rz = __fsqrt_rn(rz2);
  float z_lo = __fsub_rn(cv[2], rz);
  float z_hi = __fadd_rn(cv[2], rz);
  int4 rc = make_int4(0, 0, -1, -1);
  uint32_t cnt = 0;
  float ze = 0.0f;
  if (z_hi > 0.0f) {
    ze = z_lo > 0.0f ? z_lo : 0.0f;
    int px0, px1, py0, py1;
    if (z_lo <= __fmul_rn(eye_guard, rz)) {
      // Q13: touches / nears the eye plane, where the tangent-plane bound degenerates.  The camera-space box
      // c -/+ (r_x, r_y, r_z) of the support is bounded instead, clipped at a depth z_n in front of which every point
      // of the support projects beyond the farthest image corner; eye inside the box: whole image.
      px0 = 0; px1 = cam.W - 1; py0 = 0; py1 = cam.H - 1;
      const float rx = __fsqrt_rn(ms_dot3(Mc[0], Mc[1], Mc[2], Mc[0], Mc[1], Mc[2]));
      const float ry = __fsqrt_rn(ms_dot3(Mc[3], Mc[4], Mc[5], Mc[3], Mc[4], Mc[5]));
      float ex = __fsub_rn(fabsf(cv[0]), rx), ey = __fsub_rn(fabsf(cv[1]), ry), ez = __fsub_rn(fabsf(cv[2]), rz);
      ex = ex > 0.0f ? ex : 0.0f; ey = ey > 0.0f ? ey : 0.0f; ez = ez > 0.0f ? ez : 0.0f;
      const float d2 = __fadd_rn(__fadd_rn(__fmul_rn(ex, ex), __fmul_rn(ey, ey)), __fmul_rn(ez, ez));
      if (d2 > 0.0f) {
        const float wx = __fsub_rn((float)cam.W, cam.cx), wy = __fsub_rn((float)cam.H, cam.cy);
        const float tx = __fdiv_rn(cam.cx > wx ? cam.cx : wx, cam.fx), ty = __fdiv_rn(cam.cy > wy ? cam.cy : wy, cam.fy);
        const float zn = __fdiv_rn(__fmul_rn(0.5f, __fsqrt_rn(d2)),
                                   __fsqrt_rn(__fadd_rn(1.0f, __fadd_rn(__fmul_rn(tx, tx), __fmul_rn(ty, ty)))));
        float zc = z_lo > zn ? z_lo : zn;
        zc = zc < z_hi ? zc : z_hi;
        const float xl = __fsub_rn(cv[0], rx), xh = __fadd_rn(cv[0], rx), yl = __fsub_rn(cv[1], ry), yh = __fadd_rn(cv[1], ry);
        const float x_lo = __fadd_rn(__fmul_rn(cam.fx, xl < 0.0f ? __fdiv_rn(xl, zc) : __fdiv_rn(xl, z_hi)), cam.cx);
        const float x_hi = __fadd_rn(__fmul_rn(cam.fx, xh > 0.0f ? __fdiv_rn(xh, zc) : __fdiv_rn(xh, z_hi)), cam.cx);
        const float y_lo = __fadd_rn(__fmul_rn(cam.fy, yl < 0.0f ? __fdiv_rn(yl, zc) : __fdiv_rn(yl, z_hi)), cam.cy);
        const float y_hi = __fadd_rn(__fmul_rn(cam.fy, yh > 0.0f ? __fdiv_rn(yh, zc) : __fdiv_rn(yh, z_hi)), cam.cy);
        px0 = clamp_lo(__fsub_rn(x_lo, 0.5f), cam.W);
        px1 = clamp_hi(__fsub_rn(x_hi, 0.5f), cam.W);
        py0 = clamp_lo(__fsub_rn(y_lo, 0.5f), cam.H);
        py1 = clamp_hi(__fsub_rn(y_hi, 0.5f), cam.H);
      }
    } else {
      float zz = __fsub_rn(rz2, __fmul_rn(cv[2], cv[2]));
      float xl, xh, yl, yh;
      axis_bounds(Mc, cv[0], Mc + 6, cv[2], zz, cam.fx, cam.cx, &xl, &xh);
      axis_bounds(Mc + 3, cv[1], Mc + 6, cv[2], zz, cam.fy, cam.cy, &yl, &yh);
      px0 = clamp_lo(__fsub_rn(xl, 0.5f), cam.W);
      px1 = clamp_hi(__fsub_rn(xh, 0.5f), cam.W);
      py0 = clamp_lo(__fsub_rn(yl, 0.5f), cam.H);
      py1 = clamp_hi(__fsub_rn(yh, 0.5f), cam.H);
    }
    if (px0 <= px1 && py0 <= py1) {
      rc = make_int4(px0 / tile, py0 / tile, px1 / tile, py1 / tile);
      cnt = (uint32_t)(rc.z - rc.x + 1) * (uint32_t)(rc.w - rc.y + 1);
    }
  }
  if (cnt) {   // 64-bit pair total (a wrapped 32-bit scan would undersize every buffer) and the visible count
    atomicAdd(reinterpret_cast<unsigned long long *>(counters + MS_CNT_PAIRS), (unsigned long long)cnt);
    atomicAdd(&counters[MS_CNT_VISIBLE], 1u);
  }
  tile_count[i] = cnt;
  rect[i] = rc;
  z_entry[i] = ze;
}

__global__ void project_kernel(int n, const float *__restrict__ center, const float *__restrict__ A,
                               const float *__restrict__ M, MsCam cam, int tile, float eye_guard,
                               uint32_t *__restrict__ tile_count, int4 *__restrict__ rect, float *__restrict__ z_entry,
                               float *__restrict__ oprime, uint32_t *__restrict__ counters) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) project_body(i, center, A, M, cam, tile, eye_guard, tile_count, rect, z_entry, oprime, counters);
}

// no-sync views: the pair count the later kernels read, and whether it fits the scratch sized from the previous view
__device__ __forceinline__ uint32_t pair_guard(uint32_t P, uint32_t cap, uint32_t *counters) {
  counters[MS_CNT_P_EFF] = P < cap ? P : cap;
  if (P > cap) {
    counters[MS_CNT_OVERFLOW] = 1u;
    counters[MS_CNT_STICKY_OVERFLOW] = 1u;               // survives the per-view reset: any view of a batch
  }
  return P < cap ? P : cap;
}

// one warp per primitive; emission order: tile rows, then columns (row-major inside the rect).  Plain pointers: the
// fused small-frame kernel reads what it has written itself.
__device__ __forceinline__ void emit_body(int i, int lane, const uint32_t *emit_off, const int4 *rect, const float *z_entry,
                                          int tiles_x, int prim_bits, uint64_t *keys, int tile_order, const MsCam &cam,
                                          int tile, const float *A, const float *oprime, uint32_t cap) {
  uint32_t beg = emit_off[i], cnt = emit_off[i + 1] - beg;
  if (cnt == 0) return;
  int4 rc = rect[i];
  int tw = rc.z - rc.x + 1;
  uint64_t low = ((uint64_t)__float_as_uint(z_entry[i]) << prim_bits) | (uint64_t)(uint32_t)i;
  for (uint32_t j = lane; j < cnt; j += 32) {
    int ty = rc.y + (int)(j / (uint32_t)tw), tx = rc.x + (int)(j % (uint32_t)tw);
    uint64_t t = (uint64_t)(uint32_t)(ty * tiles_x + tx);
    if (tile_order) {  // order of the contact points of the virtual ray through the tile centre
      float d[3];
      ms_point_ray(cam, __fadd_rn((float)(tx * tile), __fmul_rn(0.5f, (float)tile)),
                   __fadd_rn((float)(ty * tile), __fmul_rn(0.5f, (float)tile)), d);
      const float tc = ms_contact_t(A + 9 * (size_t)i, oprime + 3 * (size_t)i, d);
      low = ((uint64_t)__float_as_uint(tc) << prim_bits) | (uint64_t)(uint32_t)i;
    }
    if (beg + j < cap) keys[beg + j] = (t << (32 + prim_bits)) | low;     // cap: the buffer's capacity (no-sync renders)
  }
}

__global__ void emit_keys_kernel(int n, const uint32_t *__restrict__ emit_off, const int4 *__restrict__ rect,
                                 const float *__restrict__ z_entry, int tiles_x, int prim_bits,
                                 uint64_t *__restrict__ keys, int tile_order, MsCam cam, int tile,
                                 const float *__restrict__ A, const float *__restrict__ oprime, uint32_t cap,
                                 uint32_t *__restrict__ counters) {
  int i = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  int lane = threadIdx.x & 31;
  if (counters && blockIdx.x == 0 && threadIdx.x == 0) pair_guard(emit_off[n], cap, counters);
  if (i >= n) return;
  emit_body(i, lane, emit_off, rect, z_entry, tiles_x, prim_bits, keys, tile_order, cam, tile, A, oprime, cap);
}

__device__ __forceinline__ void tile_ranges_body(uint32_t i, const uint64_t *keys, uint32_t n_pairs, int n_tiles, int shift,
                                                 uint32_t *tile_start) {
  int t = (int)(keys[i] >> shift);
  int prev = i == 0 ? -1 : (int)(keys[i - 1] >> shift);
  for (int u = prev + 1; u <= t; ++u) tile_start[u] = i;
  if (i == n_pairs - 1)
    for (int u = t + 1; u <= n_tiles; ++u) tile_start[u] = n_pairs;
}

__global__ void tile_ranges_kernel(const uint64_t *__restrict__ keys, uint32_t n_pairs, int n_tiles, int shift,
                                   uint32_t *__restrict__ tile_start, const uint32_t *__restrict__ n_dev) {
  uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (n_dev) {                                   // the pair count lives on the device; n_pairs is its capacity
    n_pairs = *n_dev < n_pairs ? *n_dev : n_pairs;
    if (n_pairs == 0 && i == 0)
      for (int u = 0; u <= n_tiles; ++u) tile_start[u] = 0u;
  }
  if (i < n_pairs) tile_ranges_body(i, keys, n_pairs, n_tiles, shift, tile_start);
}

// Small frames rendered without host synchronisation (N <= MS_SMALL_PRIMS primitives, pair capacity <= SB_MAX): the
// whole of stages (a) and (b) by ONE CTA in one launch -- counters reset, projection, offset scan, pair guard, key
// emit, radix sort, tile ranges (7 stream operations otherwise; such a frame is bound by launch latency).  The same
// device functions as the separate kernels: bitwise the same keys, tile lists and counters.
struct MsBinSmallArgs {
  int n;
  const float *center, *A, *M;
  MsCam cam;
  int tile, tiles_x, n_tiles, prim_bits, tile_order, n_bits;
  float eye_guard;
  uint32_t cap;                     // pair capacity of keys_a / keys_b / the pair tables
  uint32_t *tile_count, *emit_off, *counters, *tile_start, *pair_hits_j;
  int4 *rect;
  float *z_entry, *oprime;
  uint64_t *keys_a, *keys_b;
};

__global__ void __launch_bounds__(SB_THREADS) bin_sort_small_kernel(MsBinSmallArgs a) {
  extern __shared__ __align__(16) uint8_t sb_smem[];
  __shared__ uint32_t dsum[8];
  __shared__ uint32_t wt[SB_THREADS / 32 + 1];
  __shared__ uint32_t s_P;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  if (tid < MS_CNT_N) a.counters[tid] = 0u;                // the sticky overflow flag behind them stays
  for (uint32_t e = tid; e < a.cap + 2; e += SB_THREADS) a.pair_hits_j[e] = 0u;   // slots beyond the pair count (stage (c))
  __syncthreads();
  for (int i = tid; i < a.n; i += SB_THREADS)
    project_body(i, a.center, a.A, a.M, a.cam, a.tile, a.eye_guard, a.tile_count, a.rect, a.z_entry, a.oprime, a.counters);
  __syncthreads();
  cta_exclusive_scan_u32<SB_THREADS>(a.tile_count, a.emit_off, (size_t)a.n, wt);
  __syncthreads();
  if (tid == 0) s_P = pair_guard(a.emit_off[a.n], a.cap, a.counters);
  for (int i = warp; i < a.n; i += SB_THREADS / 32)
    emit_body(i, lane, a.emit_off, a.rect, a.z_entry, a.tiles_x, a.prim_bits, a.keys_a, a.tile_order, a.cam, a.tile, a.A,
              a.oprime, a.cap);
  __syncthreads();
  const uint32_t P = s_P;
  block_sort(a.keys_a, a.keys_b, P, a.prim_bits, a.n_bits, sb_smem, dsum);
  __syncthreads();
  if (P == 0) {
    for (int u = tid; u <= a.n_tiles; u += SB_THREADS) a.tile_start[u] = 0u;
  } else {
    for (uint32_t i = tid; i < P; i += SB_THREADS) tile_ranges_body(i, a.keys_b, P, a.n_tiles, 32 + a.prim_bits, a.tile_start);
  }
}

// ms_render without host synchronisation: the pair count against the capacity the scratch was sized for
}  // namespace

cudaError_t ms_prep_prims(int n, const float *center, const float *quat, const float *scale, float *A, float *M,
                          int *bad, cudaStream_t s) {
  (void)center;
  prep_prims_kernel<<<(n + 127) / 128, 128, 0, s>>>(n, quat, scale, A, M, bad);
  MS_LAUNCHED();
  return cudaGetLastError();
}

cudaError_t ms_project(int n, const float *center, const float *A, const float *M, MsCam cam, int tile, float eye_guard,
                       uint32_t *tile_count, int4 *rect, float *z_entry, float *oprime, uint32_t *counters,
                       cudaStream_t s) {
  project_kernel<<<(n + 127) / 128, 128, 0, s>>>(n, center, A, M, cam, tile, eye_guard, tile_count, rect, z_entry, oprime,
                                                 counters);
  MS_LAUNCHED();
  return cudaGetLastError();
}

cudaError_t ms_emit_keys(int n, const uint32_t *emit_off, const int4 *rect, const float *z_entry, int tiles_x,
                         int prim_bits, uint64_t *keys, int tile_order, MsCam cam, int tile, const float *A,
                         const float *oprime, cudaStream_t s, uint32_t cap, uint32_t *counters) {
  long threads = (long)n * 32;
  emit_keys_kernel<<<(unsigned)((threads + 255) / 256), 256, 0, s>>>(n, emit_off, rect, z_entry, tiles_x, prim_bits,
                                                                    keys, tile_order, cam, tile, A, oprime, cap, counters);
  MS_LAUNCHED();
  return cudaGetLastError();
}

bool ms_bin_sort_small_fits(int n_prims, size_t pair_cap) { return n_prims <= MS_SMALL_PRIMS && pair_cap <= (size_t)SB_MAX; }

cudaError_t ms_bin_sort_small(int n, const float *center, const float *A, const float *M, MsCam cam, int tile, float eye_guard,
                              int tiles_x, int n_tiles, int prim_bits, int tile_order, int n_bits, uint32_t cap,
                              uint32_t *tile_count, uint32_t *emit_off, int4 *rect, float *z_entry, float *oprime,
                              uint32_t *counters, uint64_t *keys_a, uint64_t *keys_b, uint32_t *tile_start,
                              uint32_t *pair_hits_j, cudaStream_t s) {
  static bool attr_set = false;
  if (!attr_set) {
    cudaError_t e = cudaFuncSetAttribute((const void *)bin_sort_small_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)SB_SMEM_BYTES);
    if (e != cudaSuccess) return e;
    attr_set = true;
  }
  MsBinSmallArgs a;
  a.n = n; a.center = center; a.A = A; a.M = M; a.cam = cam; a.tile = tile; a.tiles_x = tiles_x; a.n_tiles = n_tiles;
  a.prim_bits = prim_bits; a.tile_order = tile_order; a.n_bits = n_bits; a.eye_guard = eye_guard; a.cap = cap;
  a.tile_count = tile_count; a.emit_off = emit_off; a.counters = counters; a.tile_start = tile_start;
  a.pair_hits_j = pair_hits_j; a.rect = rect; a.z_entry = z_entry; a.oprime = oprime; a.keys_a = keys_a; a.keys_b = keys_b;
  bin_sort_small_kernel<<<1, SB_THREADS, SB_SMEM_BYTES, s>>>(a);
  MS_LAUNCHED();
  return cudaGetLastError();
}

cudaError_t ms_tile_ranges(const uint64_t *keys, size_t n_pairs, int n_tiles, int prim_bits, uint32_t *tile_start,
                           cudaStream_t s, const uint32_t *n_dev) {
  if (n_pairs == 0) return cudaMemsetAsync(tile_start, 0, (size_t)(n_tiles + 1) * sizeof(uint32_t), s);
  tile_ranges_kernel<<<(unsigned)((n_pairs + 255) / 256), 256, 0, s>>>(keys, (uint32_t)n_pairs, n_tiles,
                                                                      32 + prim_bits, tile_start, n_dev);
  MS_LAUNCHED();
  return cudaGetLastError();
}
