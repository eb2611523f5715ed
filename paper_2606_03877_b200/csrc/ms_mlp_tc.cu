// ms_mlp_tc.cu -- stage (d) on the 5th-generation tensor cores (NS (d): "batches a tile's samples
// by primitive and runs them as dense contractions on tcgen05 tensor cores, with that
// primitive's weights staged into shared memory by TMA").
//
// Work unit: a row block of 128 consecutive samples of ONE primitive (one TMEM lane per sample).
// The primitive-major interval list of stage (c) makes every primitive's samples contiguous, so a
// persistent CTA (one per SM) walks a contiguous range of row blocks and re-stages weights only when
// the primitive changes (a handful of times per frame per CTA) -- one 1-D bulk async copy
// (cp.async.bulk, mbarrier complete_tx) of a host-prepacked shared-memory image.
//
// Per row block:   x = posenc(u) (bf16, smem, K-major no-swizzle core-matrix layout)
//   layer 1        D[128 x W]  = x . W1^T            tcgen05.mma SS  (A, B from shared memory)
//   epilogue       h = relu(D + b) -> bf16 -> TMEM   tcgen05.ld / cvt.rn.relu.bf16x2 / tcgen05.st
//   layers 2..NH   D = h . Wl^T                      tcgen05.mma TS  (A from tensor memory)
//   head           D[128 x NOUT] = h . Wh^T ; rgb = sigmoid, sigma = softplus, e = exp(-sigma delta)
// Accumulators never leave TMEM between layers; activations never touch shared or global memory.
//
// Warp roles (320 threads): warp 0 weight loader + TMEM owner, warp 1 MMA issuer (one lane),
// warps 2-5 and 6-9 two epilogue groups that ping-pong two row blocks so the tensor pipe works on
// one block while the other is in its CUDA-core phase.  All hand-offs are mbarriers.
#include <cuda_bf16.h>

#include <vector>

#include "ms_mlp_tc.cuh"

namespace {

constexpr int TC_THREADS = 320;
constexpr int TC_GROUP_THREADS = 128;
constexpr uint32_t TC_MIN_SMEM = 116 * 1024;  // > half of the SM's shared memory: one CTA per SM (it owns all 512 TMEM columns)

// ---------------------------------------------------------------------------------------------
// PTX wrappers (validated one by one against a CPU GEMM on B200 before this kernel was written)
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  asm volatile(
      "{\n.reg .pred p;\nMS_WAIT:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra MS_DONE;\nbra MS_WAIT;\nMS_DONE:\n}\n" ::"r"(bar),
      "r"(parity)
      : "memory");
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void *src, uint32_t bytes, uint32_t bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
               "l"(src), "r"(bytes), "r"(bar)
               : "memory");
}
// K-major, no swizzle: core matrix = 8 rows x 16 B contiguous; LBO = byte stride between the two
// K-adjacent core matrices of one MMA, SBO = byte stride between 8-row groups.
__device__ __forceinline__ uint64_t umma_desc(uint32_t addr, uint32_t lbo, uint32_t sbo) {
  return (uint64_t)((addr >> 4) & 0x3fffu) | ((uint64_t)((lbo >> 4) & 0x3fffu) << 16) |
         ((uint64_t)((sbo >> 4) & 0x3fffu) << 32) | ((uint64_t)1 << 46);
}
// kind::f16, A = B = bf16, D = fp32, both K-major, M = 128
__host__ __device__ constexpr uint32_t umma_idesc(int n) {
  return (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(n >> 3) << 17) | ((uint32_t)(128 >> 4) << 24);
}
__device__ __forceinline__ void mma_ss(uint32_t d_tmem, uint64_t a, uint64_t b, uint32_t idesc, uint32_t acc) {
  asm volatile("{\n.reg .pred p;\nsetp.ne.b32 p, %4, 0;\ntcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n}\n" ::"r"(d_tmem),
               "l"(a), "l"(b), "r"(idesc), "r"(acc)
               : "memory");
}
__device__ __forceinline__ void mma_ts(uint32_t d_tmem, uint32_t a_tmem, uint64_t b, uint32_t idesc, uint32_t acc) {
  asm volatile("{\n.reg .pred p;\nsetp.ne.b32 p, %4, 0;\ntcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p;\n}\n" ::"r"(d_tmem),
               "r"(a_tmem), "l"(b), "r"(idesc), "r"(acc)
               : "memory");
}
__device__ __forceinline__ void mma_commit(uint32_t bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }

__device__ __forceinline__ void tmem_ld32(uint32_t taddr, uint32_t *r) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
      "{%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31}, [%32];"
      : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
        "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]), "=r"(r[16]),
        "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]), "=r"(r[24]),
        "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
      : "r"(taddr));
}
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, uint32_t *r) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
      : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
        "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
      : "r"(taddr));
}
__device__ __forceinline__ void tmem_ld_wait() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tmem_st16(uint32_t taddr, const uint32_t *r) {
  asm volatile(
      "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16};" ::"r"(taddr),
      "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]), "r"(r[8]), "r"(r[9]),
      "r"(r[10]), "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15])
      : "memory");
}
__device__ __forceinline__ void tmem_st_wait() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }

// relu + round-to-nearest-even to bf16, two values per register: lo = element k, hi = element k+1
__device__ __forceinline__ uint32_t relu_pack_bf16(float lo, float hi) {
  uint32_t d;
  asm("cvt.rn.relu.bf16x2.f32 %0, %1, %2;" : "=r"(d) : "f"(hi), "f"(lo));
  return d;
}
__device__ __forceinline__ uint32_t pack_bf16(float lo, float hi) {
  uint32_t d;
  asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(d) : "f"(hi), "f"(lo));
  return d;
}

// ---------------------------------------------------------------------------------------------
// image layout (bytes), shared by the host packer and the kernel
// ---------------------------------------------------------------------------------------------
struct TcLayout {
  int k1, width, nh, nout;
  uint32_t off_w[6];   // W^T of layer l (l = 0..nh-1 hidden, nh = head)
  uint32_t off_bias;   // fp32 biases: nh x width, then nout
  uint32_t bytes;      // multiple of 128
};

__host__ __device__ inline TcLayout tc_layout(int k1, int width, int nh, int nout) {
  TcLayout L;
  L.k1 = k1; L.width = width; L.nh = nh; L.nout = nout;
  uint32_t o = 0;
  L.off_w[0] = o; o += (uint32_t)(k1 * width * 2);
  for (int l = 1; l < nh; ++l) { L.off_w[l] = o; o += (uint32_t)(width * width * 2); }
  L.off_w[nh] = o; o += (uint32_t)(nout * width * 2);
  L.off_bias = o; o += (uint32_t)((nh * width + nout) * 4);
  L.bytes = (o + 127u) & ~127u;
  return L;
}

struct TcParams {
  MsCam cam;
  int K, n_prims, in_dim, n_feat, nh, k1;
  uint32_t n_blocks;
  const float *center, *A;
  const uint32_t *prim_start, *blk_off;
  const MsInterval *intervals;
  const uint8_t *image;
  uint32_t image_bytes;
  float4 *staging;
  float *staging_feat;
};

__device__ __forceinline__ int find_prim(const uint32_t *__restrict__ blk_off, int n, uint32_t b) {
  int lo = 0, hi = n;
  while (hi - lo > 1) {
    int mid = (lo + hi) >> 1;
    if (blk_off[mid] <= b) lo = mid; else hi = mid;
  }
  return lo;
}

// Segment walk: the CTA's block range [b0, b1) cut at primitive boundaries.
struct SegWalk {
  const uint32_t *blk_off;
  uint32_t cur, b1;
  int p;
  __device__ SegWalk(const uint32_t *bo, int n, uint32_t b0, uint32_t b1_) : blk_off(bo), cur(b0), b1(b1_), p(0) {
    if (b0 < b1_) p = find_prim(bo, n, b0);
  }
  // returns false when done; else (prim, first block inside prim, number of blocks)
  __device__ bool next(int &prim, uint32_t &first, uint32_t &count) {
    while (cur < b1) {
      uint32_t pe = blk_off[p + 1];
      uint32_t end = pe < b1 ? pe : b1;
      if (end > cur) {
        prim = p; first = cur - blk_off[p]; count = end - cur;
        cur = end;
        if (cur == pe) ++p;
        return true;
      }
      ++p;
    }
    return false;
  }
};

// positional encoding of one sample into K-major bf16 chunks (16 B each), Eq.5 with identity
// first (Q3): [u, sin(2^l pi u) xyz, cos(2^l pi u) xyz]_l [, d].  sin/cos of level 0 from the SFU on
// the exact product pi*u (|u| <= 1), higher levels by the double-angle recurrence in fp32; the
// RESULT is rounded to bf16 (never the argument: S:H8).
template <int NFREQ, int VIEWDIR, int K1>
__device__ __forceinline__ void encode_row(const float *u, const float *d, uint8_t *dst_row /* + chunk*2048 */) {
  constexpr int IN = 3 + 6 * NFREQ + 3 * VIEWDIR;
  static_assert(IN <= K1, "padded input too small");
  float x[K1];
#pragma unroll
  for (int i = 0; i < K1; ++i) x[i] = 0.0f;
  x[0] = u[0]; x[1] = u[1]; x[2] = u[2];
  float s[3], c[3];
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    float arg = 3.14159265358979323846f * u[a];
    s[a] = __sinf(arg);
    c[a] = __cosf(arg);
  }
#pragma unroll
  for (int l = 0; l < NFREQ; ++l) {
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      x[3 + 6 * l + a] = s[a];
      x[3 + 6 * l + 3 + a] = c[a];
      float s2 = 2.0f * s[a] * c[a];
      float c2 = fmaf(-2.0f * s[a], s[a], 1.0f);
      s[a] = s2; c[a] = c2;
    }
  }
  if (VIEWDIR) {
    x[3 + 6 * NFREQ + 0] = d[0]; x[3 + 6 * NFREQ + 1] = d[1]; x[3 + 6 * NFREQ + 2] = d[2];
  }
#pragma unroll
  for (int ch = 0; ch < K1 / 8; ++ch) {
    uint4 v;
    v.x = pack_bf16(x[8 * ch + 0], x[8 * ch + 1]);
    v.y = pack_bf16(x[8 * ch + 2], x[8 * ch + 3]);
    v.z = pack_bf16(x[8 * ch + 4], x[8 * ch + 5]);
    v.w = pack_bf16(x[8 * ch + 6], x[8 * ch + 7]);
    *reinterpret_cast<uint4 *>(dst_row + ch * (MS_ROWS * 16)) = v;
  }
}

template <int NFREQ, int VIEWDIR, int WIDTH, int NOUT>
__global__ void __launch_bounds__(TC_THREADS, 1) mlp_tc_kernel(const TcParams p) {
  constexpr int K1 = ((3 + 6 * NFREQ + 3 * VIEWDIR) + 15) / 16 * 16;
  extern __shared__ __align__(1024) uint8_t smem[];
  // [ weight image | A1[0] | A1[1] ]
  __shared__ uint64_t bars[8];
  __shared__ uint32_t tmem_base_s;
  const TcLayout L = tc_layout(K1, WIDTH, p.nh, NOUT);
  uint8_t *s_img = smem;
  uint8_t *s_a1 = smem + L.bytes;
  constexpr uint32_t A1_BYTES = MS_ROWS * K1 * 2;
  const uint32_t bar_w_full = smem_u32(&bars[0]), bar_w_free = smem_u32(&bars[1]);
  const uint32_t bar_a_full0 = smem_u32(&bars[2]);  // [2], [3]
  const uint32_t bar_d_full0 = smem_u32(&bars[4]);  // [4], [5]

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  if (tid == 0) {
    mbar_init(bar_w_full, 1);
    mbar_init(bar_w_free, 9);  // 8 epilogue warps + the MMA warp's commit
    mbar_init(bar_a_full0, 4); mbar_init(bar_a_full0 + 8, 4);
    mbar_init(bar_d_full0, 1); mbar_init(bar_d_full0 + 8, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == 0) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&tmem_base_s)), "r"(512));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = tmem_base_s;

  const uint32_t b0 = (uint32_t)(((uint64_t)p.n_blocks * blockIdx.x) / gridDim.x);
  const uint32_t b1 = (uint32_t)(((uint64_t)p.n_blocks * (blockIdx.x + 1)) / gridDim.x);
  const int nh = p.nh;

  if (warp == 0) {
    // ===== weight loader: one bulk async copy per segment =====
    if (lane == 0) {
      SegWalk w(p.blk_off, p.n_prims, b0, b1);
      int prim; uint32_t first, count, seg = 0;
      while (w.next(prim, first, count)) {
        if (seg > 0) mbar_wait(bar_w_free, (seg - 1) & 1);
        mbar_expect_tx(bar_w_full, p.image_bytes);
        bulk_g2s(smem_u32(s_img), p.image + (size_t)prim * p.image_bytes, p.image_bytes, bar_w_full);
        ++seg;
      }
    }
  } else if (warp == 1) {
    // ===== MMA issuer =====
    if (lane == 0) {
      SegWalk w(p.blk_off, p.n_prims, b0, b1);
      int prim; uint32_t first, count, seg = 0;
      uint32_t pa[2] = {0, 0};
      const uint32_t idesc_w = umma_idesc(WIDTH), idesc_o = umma_idesc(NOUT);
      const uint32_t img = smem_u32(s_img);
      while (w.next(prim, first, count)) {
        mbar_wait(bar_w_full, seg & 1);
        const uint32_t iters = (count + 1) >> 1;
        for (uint32_t it = 0; it < iters; ++it) {
          for (int l = 0; l <= nh; ++l) {
#pragma unroll
            for (int g = 0; g < 2; ++g) {
              if (2 * it + g >= count) continue;
              mbar_wait(bar_a_full0 + 8 * g, pa[g]);
              pa[g] ^= 1;
              tc_fence_after();
              const uint32_t d_tmem = tmem + 256 * g;
              const uint32_t a_tmem = tmem + 256 * g + 128;
              if (l == 0) {
                const uint32_t a1 = smem_u32(s_a1) + g * A1_BYTES;
#pragma unroll
                for (int j = 0; j < K1 / 16; ++j) {
                  uint64_t da = umma_desc(a1 + j * 2 * (MS_ROWS * 16), MS_ROWS * 16, 128);
                  uint64_t db = umma_desc(img + L.off_w[0] + j * 2 * (WIDTH * 16), WIDTH * 16, 128);
                  mma_ss(d_tmem, da, db, idesc_w, j > 0);
                }
              } else if (l < nh) {
#pragma unroll
                for (int j = 0; j < WIDTH / 16; ++j) {
                  uint64_t db = umma_desc(img + L.off_w[l] + j * 2 * (WIDTH * 16), WIDTH * 16, 128);
                  mma_ts(d_tmem, a_tmem + j * 8, db, idesc_w, j > 0);
                }
              } else {
#pragma unroll
                for (int j = 0; j < WIDTH / 16; ++j) {
                  uint64_t db = umma_desc(img + L.off_w[nh] + j * 2 * (NOUT * 16), NOUT * 16, 128);
                  mma_ts(d_tmem, a_tmem + j * 8, db, idesc_o, j > 0);
                }
              }
              mma_commit(bar_d_full0 + 8 * g);
            }
          }
        }
        mma_commit(bar_w_free);  // arrives once every MMA of this segment has read its weights
        ++seg;
      }
    }
  } else {
    // ===== epilogue groups: g = 0 (warps 2-5), g = 1 (warps 6-9) =====
    const int g = (warp - 2) >> 2;
    const int quarter = warp & 3;                  // TMEM lanes this warp may touch: 32*quarter .. +31
    const int row = quarter * 32 + lane;           // sample row inside the block = TMEM lane
    const uint32_t lane_addr = (uint32_t)(quarter * 32) << 16;
    const uint32_t d_tmem = tmem + 256 * g + lane_addr;
    const uint32_t a_tmem = tmem + 256 * g + 128 + lane_addr;
    const uint32_t bar_a = bar_a_full0 + 8 * g, bar_d = bar_d_full0 + 8 * g;
    uint8_t *a1_row = s_a1 + g * A1_BYTES + row * 16;
    const float *bias_s = reinterpret_cast<const float *>(s_img + L.off_bias);
    uint32_t pd = 0;
    SegWalk w(p.blk_off, p.n_prims, b0, b1);
    int prim; uint32_t first, count, seg = 0;
    const uint32_t K = (uint32_t)p.K;
    while (w.next(prim, first, count)) {
      mbar_wait(bar_w_full, seg & 1);              // biases live in the weight image
      const uint32_t iv_first = p.prim_start[prim], iv_count = p.prim_start[prim + 1] - iv_first;
      float Al[9], mu[3];
#pragma unroll
      for (int q = 0; q < 9; ++q) Al[q] = __ldg(p.A + 9 * (size_t)prim + q);
#pragma unroll
      for (int q = 0; q < 3; ++q) mu[q] = __ldg(p.center + 3 * (size_t)prim + q);
      for (uint32_t i = (uint32_t)g; i < count; i += 2) {
        // ---- stage 0: sample -> u -> encoding -> smem (A operand of layer 1) ----
        const uint64_t s = (uint64_t)(first + i) * MS_ROWS + (uint32_t)row;
        const uint32_t j = (uint32_t)(s / K);
        const uint32_t k = (uint32_t)(s - (uint64_t)j * K);
        const bool valid = j < iv_count;
        float delta = 0.f;
        size_t out_idx = 0;
        {
          float u[3] = {0.f, 0.f, 0.f}, d[3] = {0.f, 0.f, 0.f};
          if (valid) {
            const float4 *ivp = reinterpret_cast<const float4 *>(p.intervals + iv_first + j);
            const float4 q0 = __ldg(ivp), q1 = __ldg(ivp + 1);
            const float t = ms_sample_t(q0.y, q0.z, (int)k);
            delta = q0.z;
            out_idx = (size_t)(uint32_t)__float_as_int(q0.w) * K + k;
            d[0] = q1.x; d[1] = q1.y; d[2] = q1.z;
            ms_sample_u(Al, mu, p.cam.o, d, t, u);
          }
          encode_row<NFREQ, VIEWDIR, K1>(u, d, a1_row);
        }
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        __syncwarp();
        if (lane == 0) mbar_arrive(bar_a);
        // ---- hidden layers: D -> +bias, relu, bf16 -> TMEM (A operand of the next layer) ----
        for (int l = 0; l < nh; ++l) {
          mbar_wait(bar_d, pd);
          pd ^= 1;
          tc_fence_after();
          const float *b = bias_s + l * WIDTH;
#pragma unroll
          for (int c0 = 0; c0 < WIDTH; c0 += 32) {
            uint32_t r[32], o[16];
            tmem_ld32(d_tmem + c0, r);
            tmem_ld_wait();
#pragma unroll
            for (int q = 0; q < 16; ++q) {
              const float2 bb = *reinterpret_cast<const float2 *>(b + c0 + 2 * q);
              o[q] = relu_pack_bf16(__uint_as_float(r[2 * q]) + bb.x, __uint_as_float(r[2 * q + 1]) + bb.y);
            }
            tmem_st16(a_tmem + c0 / 2, o);
          }
          tmem_st_wait();
          tc_fence_before();
          __syncwarp();
          if (lane == 0) mbar_arrive(bar_a);
        }
        // ---- head: raw -> rgb = sigmoid, sigma = softplus, e = exp(-sigma delta) ----
        mbar_wait(bar_d, pd);
        pd ^= 1;
        tc_fence_after();
        {
          const float *b = bias_s + nh * WIDTH;
          uint32_t r[16];
          tmem_ld16(d_tmem, r);
          tmem_ld_wait();
          if (valid) {
            const float r0 = __uint_as_float(r[0]) + b[0], r1 = __uint_as_float(r[1]) + b[1];
            const float r2 = __uint_as_float(r[2]) + b[2], r3 = __uint_as_float(r[3]) + b[3];
            float4 v;
            v.x = __fdividef(1.0f, 1.0f + __expf(-r0));
            v.y = __fdividef(1.0f, 1.0f + __expf(-r1));
            v.z = __fdividef(1.0f, 1.0f + __expf(-r2));
            const float sigma = fmaxf(r3, 0.0f) + __logf(1.0f + __expf(-fabsf(r3)));
            v.w = __expf(-sigma * delta);
            p.staging[out_idx] = v;
            if (p.staging_feat) {
              float *f = p.staging_feat + out_idx * (size_t)p.n_feat;
#pragma unroll
              for (int c = 4; c < 16; ++c)
                if (c - 4 < p.n_feat) f[c - 4] = __uint_as_float(r[c]) + b[c];
            }
          }
          if (NOUT > 16) {
#pragma unroll
            for (int c0 = 16; c0 < NOUT; c0 += 16) {
              tmem_ld16(d_tmem + c0, r);
              tmem_ld_wait();
              if (valid && p.staging_feat) {
                float *f = p.staging_feat + out_idx * (size_t)p.n_feat;
#pragma unroll
                for (int c = 0; c < 16; ++c)
                  if (c0 + c - 4 < p.n_feat) f[c0 + c - 4] = __uint_as_float(r[c]) + b[c0 + c];
              }
            }
          }
        }
        tc_fence_before();  // the next block's layer-1 MMA overwrites D: order our loads before the arrive
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(bar_w_free);
      ++seg;
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"(512));
}

// ---------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------
uint16_t bf16_bits(float f) {  // values are already bf16-representable (ms_api.cu rounds them)
  uint32_t u;
  memcpy(&u, &f, 4);
  uint32_t lsb = (u >> 16) & 1u;
  u += 0x7fffu + lsb;
  return (uint16_t)(u >> 16);
}

// W [in][out] row-major -> W^T as B operand: element (n = out, k = in) at chunk (k/8) slab
// [rows x 16 B], row n, position k%8.
void pack_wT(const float *W, int in, int out, int k_pad, int n_pad, uint8_t *dst) {
  uint16_t *d = reinterpret_cast<uint16_t *>(dst);
  for (int k = 0; k < k_pad; ++k)
    for (int n = 0; n < n_pad; ++n) {
      float v = (k < in && n < out) ? W[(size_t)k * out + n] : 0.0f;
      d[(size_t)(k / 8) * (n_pad * 8) + (size_t)n * 8 + (k % 8)] = bf16_bits(v);
    }
}

using KernelFn = void (*)(const TcParams);

template <int NFREQ, int VIEWDIR, int WIDTH, int NOUT>
KernelFn kernel_ptr() { return mlp_tc_kernel<NFREQ, VIEWDIR, WIDTH, NOUT>; }

KernelFn select_kernel(int n_freq, int viewdir, int width, int nout) {
#define MS_TC_CASE(F, V, W, O) \
  if (n_freq == F && viewdir == V && width == W && nout == O) return kernel_ptr<F, V, W, O>();
  MS_TC_CASE(4, 0, 64, 16)
  MS_TC_CASE(4, 1, 64, 16)
  MS_TC_CASE(4, 1, 64, 48)
  MS_TC_CASE(4, 0, 64, 48)
  MS_TC_CASE(6, 0, 128, 16)
  MS_TC_CASE(6, 1, 128, 16)
  MS_TC_CASE(4, 0, 128, 16)
  MS_TC_CASE(4, 1, 128, 16)
  MS_TC_CASE(6, 0, 64, 16)
  MS_TC_CASE(6, 0, 128, 48)
#undef MS_TC_CASE
  return nullptr;
}

int nout_pad(int out_dim) { return out_dim <= 16 ? 16 : (out_dim <= 48 ? 48 : 0); }

}  // namespace

int ms_tc_pack(const MsMlpShape &sh, int n_prims, const float *weights, MsTcWeights *out) {
  out->valid = false;
  const int nout = nout_pad(sh.out_dim);
  if (nout == 0 || !select_kernel(sh.n_freq, sh.use_viewdir, sh.width, nout)) return MS_OK;  // shape not covered
  const int k1 = (sh.in_dim + 15) / 16 * 16;
  const TcLayout L = tc_layout(k1, sh.width, sh.n_hidden, nout);
  std::vector<uint8_t> img;
  try {
    img.assign((size_t)n_prims * L.bytes, 0);
  } catch (...) {
    return MS_ERR_OUT_OF_MEMORY;
  }
  for (int i = 0; i < n_prims; ++i) {
    const float *w = weights + (size_t)i * sh.params;
    uint8_t *dst = img.data() + (size_t)i * L.bytes;
    float *bias = reinterpret_cast<float *>(dst + L.off_bias);
    int in = sh.in_dim;
    for (int l = 0; l <= sh.n_hidden; ++l) {
      const bool last = l == sh.n_hidden;
      const int o = last ? sh.out_dim : sh.width;
      pack_wT(w, in, o, l == 0 ? k1 : sh.width, last ? nout : sh.width, dst + L.off_w[l]);
      const float *b = w + (size_t)in * o;
      for (int q = 0; q < o; ++q) bias[l * sh.width + q] = b[q];
      w = b + o;
      in = o;
    }
  }
  if (cudaMalloc(&out->image, img.size()) != cudaSuccess) {
    (void)cudaGetLastError();
    return MS_ERR_OUT_OF_MEMORY;
  }
  if (cudaMemcpy(out->image, img.data(), img.size(), cudaMemcpyHostToDevice) != cudaSuccess) return MS_ERR_CUDA;
  out->bytes_per_prim = L.bytes;
  out->k1_pad = k1;
  out->n_out_pad = nout;
  out->valid = true;
  return MS_OK;
}

void ms_tc_free(MsTcWeights *w) {
  if (w->image) cudaFree(w->image);
  w->image = nullptr;
  w->valid = false;
}

cudaError_t ms_mlp_tc(const MsTcWeights &w, const MsMlpArgs &a, cudaStream_t s) {
  if (a.n_blocks == 0) return cudaSuccess;
  if (!w.valid) return cudaErrorNotSupported;
  KernelFn fn = select_kernel(a.shape.n_freq, a.shape.use_viewdir, a.shape.width, w.n_out_pad);
  if (!fn) return cudaErrorNotSupported;
  TcParams p;
  p.cam = a.cam; p.K = a.K; p.n_prims = a.n_prims; p.in_dim = a.shape.in_dim; p.n_feat = a.shape.n_feat;
  p.nh = a.shape.n_hidden; p.k1 = w.k1_pad; p.n_blocks = a.n_blocks;
  p.center = a.center; p.A = a.A; p.prim_start = a.prim_start; p.blk_off = a.blk_off; p.intervals = a.intervals;
  p.image = (const uint8_t *)w.image; p.image_bytes = (uint32_t)w.bytes_per_prim;
  p.staging = a.staging; p.staging_feat = a.staging_feat;
  size_t smem = w.bytes_per_prim + 2 * (size_t)MS_ROWS * w.k1_pad * 2;
  if (smem < TC_MIN_SMEM) smem = TC_MIN_SMEM;
  static int n_sm = 0;
  if (n_sm == 0) {
    int dev = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
  }
  cudaError_t e = cudaFuncSetAttribute((const void *)fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  unsigned grid = a.n_blocks < (uint32_t)n_sm ? a.n_blocks : (unsigned)n_sm;
  fn<<<grid, TC_THREADS, smem, s>>>(p);
  MS_LAUNCHED();
  return cudaGetLastError();
}
