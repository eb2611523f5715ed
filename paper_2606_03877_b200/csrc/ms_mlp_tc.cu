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
// Per row block:   x = [posenc(u), 1, 1] (bf16, smem, K-major no-swizzle core-matrix layout)
//   layer 1        D[128 x W]  = x . [W1; b1_hi; b1_lo]^T      tcgen05.mma SS  (A, B from shared memory)
//   epilogue       h = relu(D) -> bf16 -> TMEM                 tcgen05.ld / cvt.rn.relu.bf16x2 / tcgen05.st
//   layers 2..NH   D = [h, 1, 1] . [Wl; bl_hi; bl_lo]^T        tcgen05.mma TS  (A from tensor memory)
//   head           D[128 x NOUT] = [h, 1, 1] . [Wh; bh_hi; bh_lo]^T ; rgb = sigmoid, sigma = softplus,
//                  e = exp(-sigma delta)
// The bias rides in the contraction: every A operand carries two constant 1 columns and every
// weight matrix two extra K rows holding the bias split into bf16 hi + lo parts (b = hi + lo to
// 2^-17 relative; products with 1 are exact, accumulation is fp32), so the hidden epilogue is
// load / relu-pack / store only.  Accumulators never leave TMEM between layers; activations
// never touch shared or global memory.
//
// Warp roles and the pipeline are described above the kernel.
#include <cuda_bf16.h>

#include <string.h>

#include <thread>
#include <vector>

#include "ms_mlp_tc.cuh"

namespace {


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
// The MMA warp stays converged; one elected lane issues.  (Issued from a divergent `if (lane == 0)`
// block, every tcgen05.mma costs ~95 cycles: ptxas wraps it in a per-lane R2UR loop.  Converged +
// unrolled, the issue cost is ~20-30 cycles; measured on B200.)
__device__ __forceinline__ void mma_ss(uint32_t d_tmem, uint64_t a, uint64_t b, uint32_t idesc, uint32_t acc) {
  asm volatile(
      "{\n.reg .pred p, e;\nelect.sync _|e, 0xffffffff;\nsetp.ne.b32 p, %4, 0;\n"
      "@e tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n}\n" ::"r"(d_tmem),
      "l"(a), "l"(b), "r"(idesc), "r"(acc)
      : "memory");
}
__device__ __forceinline__ void mma_ts(uint32_t d_tmem, uint32_t a_tmem, uint64_t b, uint32_t idesc, uint32_t acc) {
  asm volatile(
      "{\n.reg .pred p, e;\nelect.sync _|e, 0xffffffff;\nsetp.ne.b32 p, %4, 0;\n"
      "@e tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p;\n}\n" ::"r"(d_tmem),
      "r"(a_tmem), "l"(b), "r"(idesc), "r"(acc)
      : "memory");
}
__device__ __forceinline__ void mma_commit(uint32_t bar) {
  asm volatile(
      "{\n.reg .pred e;\nelect.sync _|e, 0xffffffff;\n"
      "@e tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];\n}\n" ::"r"(bar)
      : "memory");
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
__device__ __forceinline__ void tmem_st8(uint32_t taddr, const uint32_t *r) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};" ::"r"(taddr), "r"(r[0]), "r"(r[1]),
               "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7])
               : "memory");
}
__device__ __forceinline__ void tmem_ld4(uint32_t taddr, uint32_t *r) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0,%1,%2,%3}, [%4];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3])
               : "r"(taddr));
}

// relu + round-to-nearest-even to bf16, two values per register: lo = element k, hi = element k+1
__device__ __forceinline__ uint32_t relu_pack_bf16(float lo, float hi) {
  uint32_t d;
  asm("cvt.rn.relu.bf16x2.f32 %0, %1, %2;" : "=r"(d) : "f"(hi), "f"(lo));
  return d;
}
__device__ __forceinline__ uint32_t pack_f16(float lo, float hi) {
  uint32_t d;
  asm("cvt.rn.f16x2.f32 %0, %1, %2;" : "=r"(d) : "f"(hi), "f"(lo));
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
// Layer 0:  [W1; b1_hi; b1_lo; 0...]^T,  K = k1 = pad16(in_dim + 2), N = width
// Layer l:  [Wl; bl_hi; bl_lo; 0...]^T,  K = width + 16,             N = width   (l = 1..nh-1)
// Head:     [Wh; bh_hi; bh_lo; 0...]^T,  K = width + 16,             N = nout (padded)
// Each as the UMMA B operand, K-major without swizzle: element (n, k) at 16-byte chunk (k/8) of an
// [N rows x 16 B] slab, row n, position k%8.
struct TcLayout {
  uint32_t off_w[6];   // layer l (l = 0..nh-1 hidden, nh = head)
  uint32_t bytes;      // multiple of 128
};

__host__ __device__ constexpr uint32_t tc_off_w(int k1, int width, int l) {
  return l == 0 ? 0u : (uint32_t)(k1 * width * 2 + (l - 1) * (width + 16) * width * 2);
}
__host__ __device__ constexpr uint32_t tc_image_bytes(int k1, int width, int nh, int nout) {
  return (tc_off_w(k1, width, nh) + (uint32_t)((width + 16) * nout * 2) + 127u) & ~127u;
}

inline TcLayout tc_layout(int k1, int width, int nh, int nout) {
  TcLayout L;
  for (int l = 0; l <= nh; ++l) L.off_w[l] = tc_off_w(k1, width, l);
  L.bytes = tc_image_bytes(k1, width, nh, nout);
  return L;
}

struct TcParams {
  MsCam cam;
  int K, n_feat;
  float falloff;          // CONTACT: g = exp(-falloff |p* - mu|^2_Lambda)
  const float *center, *A;
  MsSegs segs;            // segment tables, segment range and band of this launch (device)
  const MsInterval *intervals;
  const uint8_t *image;
  float4 *staging;
  void *staging_feat;     // n_feat == 32: fp16 rows of 64 B; other widths: fp32
  float4 *staging_gate;   // CONTACT + Eq.7 slot features: the four gates of every hit, or NULL
};

// Segment walk: the CTA's block range [b0, b1) of the launch cut at segment boundaries (a segment = the
// intervals of one primitive inside the launch's band and wave).  Every role walks the same segments (a pure
// function of the device tables), so no role has to tell another what comes next.
struct SegWalk {
  const MsSegs &sg;        // the kernel parameter itself: its pointers stay in the constant bank, not in registers
  uint32_t s, cur, b1;     // absolute segment index; absolute block numbers (in blk_off's numbering)
  __device__ SegWalk(const MsSegs &sg_, uint2 r, uint32_t b0, uint32_t b1_) : sg(sg_), s(r.x) {
    const uint32_t base = sg.blk_off[r.x];
    cur = base + b0; b1 = base + b1_;
    if (b0 < b1_) {
      uint32_t lo = r.x, hi = r.y;
      while (hi - lo > 1) {
        const uint32_t mid = (lo + hi) >> 1;
        if (sg.blk_off[mid] <= cur) lo = mid; else hi = mid;
      }
      s = lo;
    }
  }
  // returns false when done; else (segment, its primitive, first block inside the segment, number of blocks)
  __device__ bool next(uint32_t &seg, int &prim, uint32_t &first, uint32_t &count) {
    while (cur < b1) {
      const uint32_t pe = sg.blk_off[s + 1];
      const uint32_t end = pe < b1 ? pe : b1;
      if (end > cur) {
        seg = s;
        prim = sg.prim ? (int)sg.prim[s] : (int)s;
        first = cur - sg.blk_off[s]; count = end - cur;
        cur = end;
        if (cur == pe) ++s;
        return true;
      }
      ++s;
    }
    return false;
  }
};

// positional encoding of one sample into K-major bf16 chunks (16 B each), Eq.5 with identity
// first (Q3): [u, sin(2^l pi u) xyz, cos(2^l pi u) xyz]_l [, d], then the two bias columns (1, 1).
// sin/cos of level 0 from the SFU on the exact product pi*u (|u| <= 1), higher levels by the
// double-angle recurrence in fp32; the RESULT is rounded to bf16 (never the argument: S:H8).
template <int NFREQ, int VIEWDIR, int K1>
__device__ __forceinline__ void encode_row(const float *u, const float *d, uint8_t *dst_row /* + chunk*2048 */) {
  constexpr int IN = 3 + 6 * NFREQ + 3 * VIEWDIR;
  static_assert(IN + 2 <= K1, "padded input too small");
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
  x[IN] = 1.0f; x[IN + 1] = 1.0f;   // bias columns
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

// Contact-point input (MS_MODE_CONTACT; Eq.3-5): z = [d; mu - p*], x[2L j + 2l] = sin(2^l pi z_j),
// x[2L j + 2l + 1] = cos(2^l pi z_j), then the two bias columns.  Two scalars fill 4L values = whole
// 16-byte chunks (L even), so the row is produced and stored pair by pair (24 live values, not 80).
template <int NFREQ, int K1>
__device__ __forceinline__ void encode_contact_row(const float *z, uint8_t *dst_row /* + chunk*2048 */) {
  constexpr int IN = 12 * NFREQ, PER = 4 * NFREQ;
  static_assert(PER % 8 == 0 && IN + 2 <= K1 && K1 == IN + 8, "contact layout");
#pragma unroll
  for (int jp = 0; jp < 3; ++jp) {
    float x[PER];
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      // delta = mu - p* is in world units and unbounded (|u| <= 1 is not): reduce z to [-1, 1] first -- exact in fp32,
      // sin / cos(pi z) have period 2 -- so the SFU sees |arg| <= pi and the five doublings stay accurate
      const float zr = z[2 * jp + h] - 2.0f * rintf(0.5f * z[2 * jp + h]);
      const float arg = 3.14159265358979323846f * zr;
      float sv = __sinf(arg), cv = __cosf(arg);
#pragma unroll
      for (int l = 0; l < NFREQ; ++l) {
        x[2 * NFREQ * h + 2 * l] = sv;
        x[2 * NFREQ * h + 2 * l + 1] = cv;
        const float s2 = 2.0f * sv * cv, c2 = fmaf(-2.0f * sv, sv, 1.0f);
        sv = s2; cv = c2;
      }
    }
#pragma unroll
    for (int c = 0; c < PER / 8; ++c) {
      uint4 v;
      v.x = pack_bf16(x[8 * c + 0], x[8 * c + 1]);
      v.y = pack_bf16(x[8 * c + 2], x[8 * c + 3]);
      v.z = pack_bf16(x[8 * c + 4], x[8 * c + 5]);
      v.w = pack_bf16(x[8 * c + 6], x[8 * c + 7]);
      *reinterpret_cast<uint4 *>(dst_row + (jp * (PER / 8) + c) * (MS_ROWS * 16)) = v;
    }
  }
  *reinterpret_cast<uint4 *>(dst_row + (IN / 8) * (MS_ROWS * 16)) = make_uint4(0x3f803f80u, 0u, 0u, 0u);   // bias columns (1, 1)
}

// ---------------------------------------------------------------------------------------------
// kernel
// ---------------------------------------------------------------------------------------------
// Warp roles (one CTA per SM):
//   warp NSLOT        (128-wide MLPs only) head MMA issuer (N = NOUT MMAs of every block, in block order);
//                     also the weight loader (one bulk copy per segment) and the TMEM owner.  Narrower
//                     MLPs: the slot warps issue their heads, slot warp 0 loads (24 warps -> 80 registers)
//   warps 0..NSLOT-1  MMA issuers, one per slot: a converged warp, one elected lane issues (see mma_ss).
//                     One warp per slot because the issue path is latency-bound: ~45 cycles per
//                     tcgen05.mma (four R2UR each) and ~90 per mbarrier try_wait, 30 MMAs and 6 waits
//                     per block -- more than the 1416 tensor cycles the block needs
//   next 4 or 8 warps EN: sample -> u -> encoding -> A1 ring in shared memory (runs ahead of the tensor pipe);
//                     two groups taking alternate blocks when the MLP is 64 wide
//   next 4 warps      HD: head accumulator -> sigmoid / softplus / exp -> staging store
//   last 8 warps      HE: hidden-layer epilogue, D (fp32, TMEM) -> relu, bf16 -> A (TMEM); two warps per
//                     TMEM lane quarter, each on one half of the columns
// Every role walks the same static schedule (SegWalk; block i of a segment runs in slot i % NSLOT), so all
// hand-offs are plain mbarriers: EN -a1_full-> MMA -d_full-> HE -a_ready-> MMA ... -h_full-> HD,
// and back: MMA commit -a1_free-> EN, HD -h_free-> MMA.  NSLOT row blocks are in flight in the
// tensor pipe (slot s: D at column s*SLOT_COLS, A at +W, the two constant 1 columns at +3W/2); the
// head accumulators live in HPS small regions per slot after the slots (private to the slot's MMA
// warp, so every mbarrier has one producer and one consumer walking it in order), and a slot is
// released to its next block as soon as the block's head MMA is issued.  The tensor pipe completes in issue order.
constexpr uint32_t TC_HD_ROW = 144;           // bytes per row of the HD transpose buffers (128 + 16: conflict-free)
constexpr uint32_t TC_MIN_SMEM = 116 * 1024;  // > half of the SM's shared memory: one CTA per SM (it owns all 512 TMEM columns)

// slots in flight and head accumulator regions per slot, fitted to the 512 TMEM columns
__host__ __device__ constexpr int tc_slots(int width, int nout) { return width > 64 ? 2 : (nout <= 16 ? 4 : 3); }
__host__ __device__ constexpr int tc_heads_per_slot(int width) { return width > 64 ? 2 : 1; }
// EN warp groups (4 warps each, group g encodes the blocks with run % groups == g) and A1 ring stages:
// a 64-wide MLP needs < 500 tensor cycles per block, less than one warp needs to encode its 32 rows
__host__ __device__ constexpr int tc_en_groups(int width) { return width > 64 ? 1 : 2; }
__host__ __device__ constexpr int tc_a1_stages(int width) { return width > 64 ? 4 : 8; }
// HE warp groups: 128 wide -- one group of 8 warps (64 columns each) serves both slots in turn;
// 64 wide -- groups of 4 warps (a whole row of 64 columns each), group g serving the slots s % groups == g
__host__ __device__ constexpr int tc_he_groups(int width, int nout) { return width > 64 ? 1 : (nout <= 16 ? 2 : 1); }
__host__ __device__ constexpr int tc_he_warps(int, int) { return 8; }
// a warp of its own for the head MMAs (and the weight loads): wide MLPs only.  For the 64- and 32-wide ones the
// slot warps issue their heads and slot warp 0 loads the weights: 24 warps instead of 25, i.e. 80 registers
// instead of 72 (ptxas budgets for the warp count rounded up to a multiple of four).
__host__ __device__ constexpr int tc_head_warp(int width) { return width > 64 ? 1 : 0; }
__host__ __device__ constexpr int tc_warps(int width, int nout) {
  return tc_slots(width, nout) + tc_head_warp(width) + 4 * tc_en_groups(width) + 4 + tc_he_warps(width, nout);
}
// warps: one MMA warp per slot, head MMA warp (also weight loader and TMEM owner), EN groups, 4 HD, HE groups

template <int NFREQ, int VIEWDIR, int WIDTH, int NOUT, int NH, int CONTACT = 0>
__global__ void __launch_bounds__(32 * tc_warps(WIDTH, NOUT), 1) mlp_tc_kernel(const TcParams p) {
  constexpr int IN = CONTACT ? 12 * NFREQ : 3 + 6 * NFREQ + 3 * VIEWDIR;   // CONTACT: gamma([d; delta]) of the paper's own mode
  constexpr int K1 = (IN + 2 + 15) / 16 * 16;
  constexpr int NSLOT = tc_slots(WIDTH, NOUT);
  constexpr int HPS = tc_heads_per_slot(WIDTH);   // head regions per slot (private to the slot's MMA warp)
  constexpr int NHS = NSLOT * HPS;
  constexpr int NEG = tc_en_groups(WIDTH), TC_NA1 = tc_a1_stages(WIDTH), NG = tc_he_groups(WIDTH, NOUT), HEW = tc_he_warps(WIDTH, NOUT) / NG;   // HE groups, warps per group
  static_assert(TC_NA1 % NEG == 0, "every ring stage belongs to one EN group");
  constexpr bool HEADW = tc_head_warp(WIDTH) != 0;
  constexpr int W_HM = HEADW ? NSLOT : 0;          // head warp, or slot warp 0 in its place as loader / TMEM owner
  constexpr int W_EN = NSLOT + (HEADW ? 1 : 0), W_HD = W_EN + 4 * NEG, W_HE = W_HD + 4;   // first warp of each group
  constexpr int SLOT_COLS = WIDTH + WIDTH / 2 + 8;
  constexpr int HEAD_COL0 = NSLOT * SLOT_COLS;
  static_assert(HEAD_COL0 + NHS * NOUT <= 512, "TMEM columns");
  constexpr uint32_t A1_BYTES = MS_ROWS * K1 * 2;
  constexpr uint32_t IMG_BYTES = tc_image_bytes(K1, WIDTH, NH, NOUT);
  extern __shared__ __align__(1024) uint8_t smem[];
  // [ weight image | A1 ring | HD transpose buffers (wide head only) ]
  __shared__ uint64_t bars[2 + 2 * TC_NA1 + 3 * NSLOT + 2 * NHS];
  __shared__ uint32_t tmem_base_s;
  uint8_t *s_img = smem;
  uint8_t *s_a1 = smem + IMG_BYTES;
  uint8_t *s_hd = s_a1 + TC_NA1 * A1_BYTES;
  const uint32_t bar_w_full = smem_u32(&bars[0]), bar_w_free = smem_u32(&bars[1]);
  const uint32_t bar_a1_full = smem_u32(&bars[2]), bar_a1_free = bar_a1_full + 8 * TC_NA1;
  const uint32_t bar_d_full = bar_a1_free + 8 * TC_NA1, bar_a_ready = bar_d_full + 8 * NSLOT;
  const uint32_t bar_a3_ready = bar_a_ready + 8 * NSLOT;   // the block's last epilogue is done: input of the head
  const uint32_t bar_h_full = bar_a3_ready + 8 * NSLOT, bar_h_free = bar_h_full + 8 * NHS;

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  if (tid == 0) {
    mbar_init(bar_w_full, 1);
    mbar_init(bar_w_free, NSLOT + (HEADW ? 1 : 0));
    for (int i = 0; i < TC_NA1; ++i) { mbar_init(bar_a1_full + 8 * i, 4); mbar_init(bar_a1_free + 8 * i, 1); }
    for (int i = 0; i < NSLOT; ++i) { mbar_init(bar_d_full + 8 * i, 1); mbar_init(bar_a_ready + 8 * i, HEW); mbar_init(bar_a3_ready + 8 * i, HEW); }
    for (int i = 0; i < NHS; ++i) { mbar_init(bar_h_full + 8 * i, 1); mbar_init(bar_h_free + 8 * i, 4); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == W_HM) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&tmem_base_s)), "r"(512));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = tmem_base_s;
  if (warp >= W_HE && warp < W_HE + 4) {  // the two constant 1 columns (bf16 pair 1,1 then zeros) of every slot's A operand
    uint32_t ones[8] = {0x3f803f80u, 0u, 0u, 0u, 0u, 0u, 0u, 0u};
#pragma unroll
    for (int s = 0; s < NSLOT; ++s)
      tmem_st8(tmem + s * SLOT_COLS + WIDTH + WIDTH / 2 + ((uint32_t)((warp & 3) * 32) << 16), ones);
    tmem_st_wait();
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();

  const uint2 srange = *p.segs.range;
  const uint32_t n_blocks = p.segs.blk_off[srange.y] - p.segs.blk_off[srange.x];
  const uint32_t slot0 = p.segs.band->slot0;
  const uint32_t b0 = (uint32_t)(((uint64_t)n_blocks * blockIdx.x) / gridDim.x);
  const uint32_t b1 = (uint32_t)(((uint64_t)n_blocks * (blockIdx.x + 1)) / gridDim.x);

  if (warp < NSLOT) {
    // ===== MMA issuer of slot s = warp (all 32 lanes walk the schedule; mma_* elect one lane) =====
    const int s = warp;
    SegWalk w(p.segs, srange, b0, b1);
    int prim; uint32_t sg, first, count, seg = 0;
    uint32_t run0 = 0;                 // running index of the segment's first block (ring positions)
    uint32_t pa = 0;                   // parity of the next a_ready[s] completion
    constexpr uint32_t idesc_w = umma_idesc(WIDTH);
    const uint32_t img = smem_u32(s_img);
    const uint32_t a1_base = smem_u32(s_a1);
    const uint32_t d_tmem = tmem + s * SLOT_COLS, a_tmem = d_tmem + WIDTH;
    const uint32_t bar_a_ready_s = bar_a_ready + 8 * s, bar_d_full_s = bar_d_full + 8 * s;
    uint32_t cnt = 0;                  // !HEADW: heads this warp has issued (head region s*HPS + cnt%HPS, use cnt/HPS)
    SegWalk wl(p.segs, srange, b0, b1);   // !HEADW, slot warp 0: the weight loader's walk, one segment ahead
    if (!HEADW && s == 0) {
      int lp; uint32_t ls, lf, lc;
      if (wl.next(ls, lp, lf, lc) && lane == 0) {
        mbar_expect_tx(bar_w_full, IMG_BYTES);
        bulk_g2s(img, p.image + (size_t)lp * IMG_BYTES, IMG_BYTES, bar_w_full);
      }
      __syncwarp();
    }
    while (w.next(sg, prim, first, count)) {
      mbar_wait(bar_w_full, seg & 1);
      tc_fence_after();
      const uint32_t n_s = (count + NSLOT - 1 - s) / NSLOT;   // blocks of this segment that run in slot s
      for (uint32_t j = 0; j <= n_s; ++j) {
        if (j > 0) {  // the previous block's last epilogue has read D; its head: the head warp's business, or issued here
          mbar_wait(bar_a_ready_s, pa);
          pa ^= 1u;
          if constexpr (!HEADW) {
            constexpr uint32_t idesc_o = umma_idesc(NOUT);
            const uint32_t hs = s * HPS + cnt % HPS;
            mbar_wait(bar_h_free + 8 * hs, ((cnt / HPS) & 1u) ^ 1u);
            ++cnt;
            tc_fence_after();
            const uint32_t h_tmem = tmem + HEAD_COL0 + hs * NOUT;
#pragma unroll
            for (int q = 0; q <= WIDTH / 16; ++q) {
              const uint64_t db = umma_desc(img + tc_off_w(K1, WIDTH, NH) + q * 2 * (NOUT * 16), NOUT * 16, 128);
              mma_ts(h_tmem, a_tmem + q * 8, db, idesc_o, q > 0);
            }
            mma_commit(bar_h_full + 8 * hs);
          }
        }
        if (j == n_s) break;
        {  // layer 1 of the slot's next block: A from the A1 ring
          const uint32_t run = run0 + j * NSLOT + s, st = run % TC_NA1;
          mbar_wait(bar_a1_full + 8 * st, (run / TC_NA1) & 1u);
          tc_fence_after();
          const uint32_t a1 = a1_base + st * A1_BYTES;
#pragma unroll
          for (int q = 0; q < K1 / 16; ++q) {
            const uint64_t da = umma_desc(a1 + q * 2 * (MS_ROWS * 16), MS_ROWS * 16, 128);
            const uint64_t db = umma_desc(img + q * 2 * (WIDTH * 16), WIDTH * 16, 128);
            mma_ss(d_tmem, da, db, idesc_w, q > 0);
          }
          mma_commit(bar_a1_free + 8 * st);
          mma_commit(bar_d_full_s);
        }
#pragma unroll
        for (int l = 1; l < NH; ++l) {
          mbar_wait(bar_a_ready_s, pa);
          pa ^= 1u;
          tc_fence_after();
#pragma unroll
          for (int q = 0; q <= WIDTH / 16; ++q) {
            const uint64_t db = umma_desc(img + tc_off_w(K1, WIDTH, l) + q * 2 * (WIDTH * 16), WIDTH * 16, 128);
            mma_ts(d_tmem, a_tmem + q * 8, db, idesc_w, q > 0);
          }
          mma_commit(bar_d_full_s);
        }
      }
      mma_commit(bar_w_free);  // arrives once every MMA this warp issued in the segment has read its weights
      if (!HEADW && s == 0) {  // loader duty: the next primitive's image once every slot is done with this one
        mbar_wait(bar_w_free, seg & 1);
        int lp; uint32_t ls, lf, lc;
        if (wl.next(ls, lp, lf, lc) && lane == 0) {
          mbar_expect_tx(bar_w_full, IMG_BYTES);
          bulk_g2s(img, p.image + (size_t)lp * IMG_BYTES, IMG_BYTES, bar_w_full);
        }
        __syncwarp();
      }
      run0 += count;
      ++seg;
    }
    if (seg > 0) mbar_wait(bar_w_free, (seg - 1) & 1);  // no asynchronous arrive may outlive the CTA
  } else if (HEADW && warp == W_HM) {
    // ===== head MMA issuer: the N = NOUT head MMAs are issue-bound (~25 cycles each for a few cycles
    // of tensor work); from a warp of their own they slip into the pipe between the slots' wide MMAs
    // It is also the weight loader: one bulk async copy of the next primitive's image once every
    // MMA of the segment has read the current one (w_free), issued by lane 0.
    SegWalk w(p.segs, srange, b0, b1), wl(p.segs, srange, b0, b1);
    int prim; uint32_t sg, first, count, seg = 0;
    constexpr uint32_t idesc_o = umma_idesc(NOUT);
    const uint32_t img = smem_u32(s_img);
    uint32_t cum[NSLOT];                          // blocks each slot has taken in earlier segments
#pragma unroll
    for (int s = 0; s < NSLOT; ++s) cum[s] = 0;
    {
      int lp; uint32_t ls, lf, lc;
      if (wl.next(ls, lp, lf, lc) && lane == 0) {
        mbar_expect_tx(bar_w_full, IMG_BYTES);
        bulk_g2s(img, p.image + (size_t)lp * IMG_BYTES, IMG_BYTES, bar_w_full);
      }
      __syncwarp();
    }
    while (w.next(sg, prim, first, count)) {
      mbar_wait(bar_w_full, seg & 1);
      for (uint32_t i = 0; i < count; ++i) {
        const uint32_t slot = i % NSLOT;
        uint32_t cnt = i / NSLOT;                   // the slot's block counter (uses of its barriers)
#pragma unroll
        for (int s = 0; s < NSLOT; ++s) cnt += slot == (uint32_t)s ? cum[s] : 0u;
        const uint32_t hs = slot * HPS + cnt % HPS;
        mbar_wait(bar_a3_ready + 8 * slot, cnt & 1u);
        mbar_wait(bar_h_free + 8 * hs, ((cnt / HPS) & 1u) ^ 1u);
        tc_fence_after();
        const uint32_t a_tmem = tmem + slot * SLOT_COLS + WIDTH;
        const uint32_t h_tmem = tmem + HEAD_COL0 + hs * NOUT;
#pragma unroll
        for (int q = 0; q <= WIDTH / 16; ++q) {
          const uint64_t db = umma_desc(img + tc_off_w(K1, WIDTH, NH) + q * 2 * (NOUT * 16), NOUT * 16, 128);
          mma_ts(h_tmem, a_tmem + q * 8, db, idesc_o, q > 0);
        }
        mma_commit(bar_h_full + 8 * hs);
      }
      mma_commit(bar_w_free);
#pragma unroll
      for (int s = 0; s < NSLOT; ++s) cum[s] += (count + NSLOT - 1 - s) / NSLOT;
      mbar_wait(bar_w_free, seg & 1);             // every MMA of the segment is done with the image
      {
        int lp; uint32_t ls, lf, lc;
        if (wl.next(ls, lp, lf, lc) && lane == 0) {
          mbar_expect_tx(bar_w_full, IMG_BYTES);
          bulk_g2s(img, p.image + (size_t)lp * IMG_BYTES, IMG_BYTES, bar_w_full);
        }
        __syncwarp();
      }
      ++seg;
    }
  } else if (warp >= W_HE) {
    // ===== HE: hidden-layer epilogues =====
    const int quarter = warp & 3;                 // TMEM lanes this warp may touch: 32*quarter .. +31
    const int grp = (warp - W_HE) / HEW;            // this warp serves the slots with s % NG == grp
    const int ch = ((warp - W_HE) % HEW) >> 2;      // column group
    constexpr int HC = WIDTH / (HEW / 4);         // columns per warp (64)
    const uint32_t lane_addr = (uint32_t)(quarter * 32) << 16;
    uint32_t pd = 0;                              // bit s: parity of the next d_full[s] completion
    uint32_t cum[NSLOT];                          // blocks each slot has taken in earlier segments
#pragma unroll
    for (int s = 0; s < NSLOT; ++s) cum[s] = 0;
    SegWalk w(p.segs, srange, b0, b1);
    int prim; uint32_t sg, first, count;
    while (w.next(sg, prim, first, count)) {
      const uint32_t jmax = (count + NSLOT - 1) / NSLOT;
      for (uint32_t j = 0; j < jmax; ++j) {
#pragma unroll 1
        for (int l = 0; l < NH; ++l) {
#pragma unroll
          for (int s = 0; s < NSLOT; ++s) {
            const uint32_t n_s = (count + NSLOT - 1 - s) / NSLOT;
            if (j >= n_s || s % NG != grp) continue;
            const uint32_t d_tmem = tmem + s * SLOT_COLS + lane_addr + ch * HC;
            const uint32_t a_tmem = tmem + s * SLOT_COLS + WIDTH + lane_addr + ch * (HC / 2);
            mbar_wait(bar_d_full + 8 * s, (pd >> s) & 1u);
            pd ^= 1u << s;
            tc_fence_after();
            const uint32_t prev = cum[s] + j;       // blocks the slot has finished before this one
            if constexpr (WIDTH > 64 || !HEADW) {
              uint32_t r[HC];
#pragma unroll
              for (int c0 = 0; c0 < HC; c0 += 32) tmem_ld32(d_tmem + c0, r + c0);
              tmem_ld_wait();
              if (HEADW && l == 0 && prev > 0) {    // A still feeds the previous block's head MMAs
                mbar_wait(bar_h_full + 8 * (s * HPS + (prev - 1) % HPS), ((prev - 1) / HPS) & 1u);
                tc_fence_after();
              }
#pragma unroll
              for (int c0 = 0; c0 < HC; c0 += 32) {
                uint32_t o[16];
#pragma unroll
                for (int q = 0; q < 16; ++q)
                  o[q] = relu_pack_bf16(__uint_as_float(r[c0 + 2 * q]), __uint_as_float(r[c0 + 2 * q + 1]));
                tmem_st16(a_tmem + c0 / 2, o);
              }
            } else {                                // 72-register budget: 32 columns at a time
#pragma unroll
              for (int c0 = 0; c0 < HC; c0 += 32) {
                uint32_t r[32], o[16];
                tmem_ld32(d_tmem + c0, r);
                tmem_ld_wait();
#pragma unroll
                for (int q = 0; q < 16; ++q) o[q] = relu_pack_bf16(__uint_as_float(r[2 * q]), __uint_as_float(r[2 * q + 1]));
                if (HEADW && c0 == 0 && l == 0 && prev > 0) {
                  mbar_wait(bar_h_full + 8 * (s * HPS + (prev - 1) % HPS), ((prev - 1) / HPS) & 1u);
                  tc_fence_after();
                }
                tmem_st16(a_tmem + c0 / 2, o);
              }
            }
            tmem_st_wait();
            tc_fence_before();
            __syncwarp();
            if (lane == 0) {
              mbar_arrive(bar_a_ready + 8 * s);
              if (HEADW && l == NH - 1) mbar_arrive(bar_a3_ready + 8 * s);
            }
          }
        }
      }
#pragma unroll
      for (int s = 0; s < NSLOT; ++s) cum[s] += (count + NSLOT - 1 - s) / NSLOT;
    }
  } else if (warp >= W_HD) {
    // ===== HD: head epilogue: raw -> rgb = sigmoid, sigma = softplus, e = exp(-sigma delta) =====
    const int quarter = warp & 3;
    const int row = quarter * 32 + lane;          // sample row inside the block = TMEM lane
    const uint32_t lane_addr = (uint32_t)(quarter * 32) << 16;
    const uint32_t K = (uint32_t)p.K;
    const uint32_t dj = MS_ROWS / K, dk = MS_ROWS - dj * K;
    uint32_t cum[NSLOT];                          // blocks each slot has taken in earlier segments
#pragma unroll
    for (int s = 0; s < NSLOT; ++s) cum[s] = 0;
    SegWalk w(p.segs, srange, b0, b1);
    int prim; uint32_t sg, first, count;
    while (w.next(sg, prim, first, count)) {
      const uint32_t iv_first = p.segs.iv0[sg], iv_count = p.segs.cnt ? p.segs.cnt[sg] : p.segs.iv0[sg + 1] - iv_first;
      const uint64_t s0 = (uint64_t)first * MS_ROWS + (uint32_t)row;
      uint32_t j = (uint32_t)(s0 / K), k = (uint32_t)(s0 - (uint64_t)j * K);
      float4 q0 = make_float4(0.f, 0.f, 0.f, 0.f);   // (ray, t_in, delta, slot) of the row's interval
      float4 q1 = q0;                                // CONTACT: (d, -) of the row's interval, for the falloff
      if (j < iv_count) {
        q0 = __ldg(reinterpret_cast<const float4 *>(p.intervals + iv_first + j));
        if (CONTACT) q1 = __ldg(reinterpret_cast<const float4 *>(p.intervals + iv_first + j) + 1);
      }
      float Al[9], mu[3];
      if (CONTACT) {
#pragma unroll
        for (int q = 0; q < 9; ++q) Al[q] = __ldg(p.A + 9 * (size_t)prim + q);
#pragma unroll
        for (int q = 0; q < 3; ++q) mu[q] = __ldg(p.center + 3 * (size_t)prim + q);
      }
      for (uint32_t i = 0; i < count; ++i) {
        const uint32_t slot = i % NSLOT;
        uint32_t cnt = i / NSLOT;                   // the slot's head counter for this block (see the MMA warp)
#pragma unroll
        for (int s = 0; s < NSLOT; ++s) cnt += slot == (uint32_t)s ? cum[s] : 0u;
        const uint32_t hs = slot * HPS + cnt % HPS;
        const bool valid = j < iv_count;
        const float delta = q0.z;
        const size_t out_idx = (size_t)((uint32_t)__float_as_int(q0.w) - slot0) * K + k;
        float fall = 1.0f;                           // CONTACT: g = exp(-(9/2) |p* - mu|^2_Lambda)
        if (CONTACT && valid) {
          const float dd[3] = {q1.x, q1.y, q1.z};
          float uu[3];
          ms_sample_u(Al, mu, p.cam.o, dd, q0.y, uu);
          fall = __expf(-p.falloff * (uu[0] * uu[0] + uu[1] * uu[1] + uu[2] * uu[2]));
          if (p.staging_gate) p.staging_gate[out_idx] = ms_slot_gates(uu);   // Eq.7 gates for stage (e)
        }
        k += dk; j += dj;
        if (k >= K) { k -= K; ++j; }
        if (i + 1 < count && j < iv_count) {
          q0 = __ldg(reinterpret_cast<const float4 *>(p.intervals + iv_first + j));
          if (CONTACT) q1 = __ldg(reinterpret_cast<const float4 *>(p.intervals + iv_first + j) + 1);
        }
        mbar_wait(bar_h_full + 8 * hs, (cnt / HPS) & 1u);
        tc_fence_after();
        const uint32_t h_tmem = tmem + HEAD_COL0 + hs * NOUT + lane_addr;
        uint32_t r[NOUT > 16 ? 36 : 4];
        const bool feat = NOUT > 16 && p.staging_feat != nullptr;
        if constexpr (NOUT > 16) {
          if (feat) {
            tmem_ld16(h_tmem, r);
            tmem_ld16(h_tmem + 16, r + 16);
            tmem_ld4(h_tmem + 32, r + 32);
          } else {
            tmem_ld4(h_tmem, r);
          }
        } else {
          tmem_ld4(h_tmem, r);
        }
        tmem_ld_wait();
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(bar_h_free + 8 * hs);
        if (valid) {
          const float r0 = __uint_as_float(r[0]), r1 = __uint_as_float(r[1]);
          const float r2 = __uint_as_float(r[2]), r3 = __uint_as_float(r[3]);
          float4 v;
          v.x = __fdividef(1.0f, 1.0f + __expf(-r0));
          v.y = __fdividef(1.0f, 1.0f + __expf(-r1));
          v.z = __fdividef(1.0f, 1.0f + __expf(-r2));
          const float sigma = fmaxf(r3, 0.0f) + __logf(1.0f + __expf(-fabsf(r3)));
          v.w = __expf(-sigma * delta);
          if (CONTACT) v.w = 1.0f - (1.0f - v.w) * fall;   // alpha = (1 - exp(-sigma l)) g
          p.staging[out_idx] = v;
          if constexpr (NOUT > 16) if (feat && p.n_feat != 32) {
            float *f = reinterpret_cast<float *>(p.staging_feat) + out_idx * (size_t)p.n_feat;
#pragma unroll
            for (int c = 0; c < 32; ++c)
              if (c < p.n_feat) f[c] = __uint_as_float(r[4 + c]);
          }
        }
        if constexpr (NOUT > 16) if (feat && p.n_feat == 32) {
          // 32 feature channels, staged as fp16 (the contraction's operands are bf16; fp16 keeps three more bits):
          // one 64 B row per sample.  A lane storing its own row would touch 32 lines per instruction (one LSU
          // wavefront each -- measured in round 1: HD was the slowest role of CFG5, and at 128 B per sample the
          // kernel wrote 2.7 TB/s); transposed through shared memory, four lanes store one row and an instruction
          // touches 8 rows.  Row stride 80 B: conflict-free for the 16-byte accesses on both sides.
          constexpr uint32_t HROW = 80;
          uint8_t *buf = s_hd + (warp - W_HD) * (32 * TC_HD_ROW);
#pragma unroll
          for (int c = 0; c < 4; ++c) {
            uint4 v;
            v.x = pack_f16(__uint_as_float(r[4 + 8 * c + 0]), __uint_as_float(r[4 + 8 * c + 1]));
            v.y = pack_f16(__uint_as_float(r[4 + 8 * c + 2]), __uint_as_float(r[4 + 8 * c + 3]));
            v.z = pack_f16(__uint_as_float(r[4 + 8 * c + 4]), __uint_as_float(r[4 + 8 * c + 5]));
            v.w = pack_f16(__uint_as_float(r[4 + 8 * c + 6]), __uint_as_float(r[4 + 8 * c + 7]));
            *reinterpret_cast<uint4 *>(buf + lane * HROW + c * 16) = v;
          }
          __syncwarp();
          const unsigned long long my = valid ? (unsigned long long)out_idx : ~0ull;
          uint8_t *fbase = reinterpret_cast<uint8_t *>(p.staging_feat);
#pragma unroll
          for (int it = 0; it < 4; ++it) {
            const int rr = it * 8 + (lane >> 2);
            const unsigned long long idx = __shfl_sync(0xffffffffu, my, rr);
            const uint4 v = *reinterpret_cast<const uint4 *>(buf + rr * HROW + (lane & 3) * 16);
            if (idx != ~0ull) *reinterpret_cast<uint4 *>(fbase + (size_t)idx * 64 + (lane & 3) * 16) = v;
          }
          __syncwarp();
        }
      }
#pragma unroll
      for (int s = 0; s < NSLOT; ++s) cum[s] += (count + NSLOT - 1 - s) / NSLOT;
    }
  } else {
    // ===== EN: sample -> u -> encoding -> A1 ring =====
    const int row = ((warp - W_EN) & 3) * 32 + lane;
    const uint32_t grp = (uint32_t)(warp - W_EN) >> 2;   // this group encodes the blocks with run % NEG == grp
    const uint32_t K = (uint32_t)p.K;
    const uint32_t dj = (NEG * MS_ROWS) / K, dk = NEG * MS_ROWS - dj * K;   // NEG blocks ahead
    uint32_t run0 = 0;
    SegWalk w(p.segs, srange, b0, b1);
    int prim; uint32_t sg, first, count;
    while (w.next(sg, prim, first, count)) {
      const uint32_t iv_first = p.segs.iv0[sg], iv_count = p.segs.cnt ? p.segs.cnt[sg] : p.segs.iv0[sg + 1] - iv_first;
      float Al[9], mu[3];
#pragma unroll
      for (int q = 0; q < 9; ++q) Al[q] = __ldg(p.A + 9 * (size_t)prim + q);
#pragma unroll
      for (int q = 0; q < 3; ++q) mu[q] = __ldg(p.center + 3 * (size_t)prim + q);
      // interval index j and sample index k of this thread's row in block i; advanced by 128 samples per block
      const uint32_t i0 = (grp + NEG - run0 % NEG) % NEG;   // first block of the segment that is this group's
      const uint64_t s0 = (uint64_t)(first + i0) * MS_ROWS + (uint32_t)row;
      uint32_t j = (uint32_t)(s0 / K), k = (uint32_t)(s0 - (uint64_t)j * K);
      float4 q0 = make_float4(0.f, 0.f, 0.f, 0.f), q1 = q0;   // interval record of the block about to be encoded
      if (j < iv_count) {
        const float4 *ivp = reinterpret_cast<const float4 *>(p.intervals + iv_first + j);
        q0 = __ldg(ivp); q1 = __ldg(ivp + 1);
      }
      for (uint32_t i = i0; i < count; i += NEG) {
        const uint32_t run = run0 + i, st = run % TC_NA1;
        const bool valid = j < iv_count;
        const float4 c0 = q0, c1 = q1;
        const uint32_t kk = k;
        // prefetch the next block's interval record
        k += dk; j += dj;
        if (k >= K) { k -= K; ++j; }
        if (i + NEG < count && j < iv_count) {
          const float4 *ivp = reinterpret_cast<const float4 *>(p.intervals + iv_first + j);
          q0 = __ldg(ivp); q1 = __ldg(ivp + 1);
        }
        float u[3] = {0.f, 0.f, 0.f}, d[3] = {0.f, 0.f, 0.f};
        float z[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};   // CONTACT: [d; mu - p*]
        if (valid) {
          const float t = ms_sample_tm(c0.y, c0.z, (int)kk, CONTACT);
          d[0] = c1.x; d[1] = c1.y; d[2] = c1.z;
          if (CONTACT) {
#pragma unroll
            for (int c = 0; c < 3; ++c) {
              z[c] = d[c];
              z[3 + c] = __fsub_rn(mu[c], __fadd_rn(p.cam.o[c], __fmul_rn(t, d[c])));
            }
          } else {
            ms_sample_u(Al, mu, p.cam.o, d, t, u);
          }
        }
        mbar_wait(bar_a1_free + 8 * st, ((run / TC_NA1) & 1u) ^ 1u);
        if constexpr (CONTACT) encode_contact_row<NFREQ, K1>(z, s_a1 + st * A1_BYTES + row * 16);
        else encode_row<NFREQ, VIEWDIR, K1>(u, d, s_a1 + st * A1_BYTES + row * 16);
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        __syncwarp();
        if (lane == 0) mbar_arrive(bar_a1_full + 8 * st);
      }
      run0 += count;
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == W_HM) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"(512));
}

// ---------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------
float bf16_round(float f) {  // RNE to a bf16-representable value
  uint32_t u;
  memcpy(&u, &f, 4);
  if ((u & 0x7f800000u) == 0x7f800000u) return f;
  uint32_t lsb = (u >> 16) & 1u;
  u = (u + 0x7fffu + lsb) & 0xffff0000u;
  memcpy(&f, &u, 4);
  return f;
}
uint16_t bf16_bits(float f) {  // of a bf16-representable value
  uint32_t u;
  memcpy(&u, &f, 4);
  return (uint16_t)(u >> 16);
}

// W [in][out] row-major and b [out] -> [W; b_hi; b_lo; 0]^T as B operand: element (n = out, k) at
// chunk (k/8) slab [n_pad rows x 16 B], row n, position k%8.  Rows k = in, in+1 carry the bias.
void pack_wT(const float *W, const float *b, int in, int out, int k_pad, int n_pad, uint8_t *dst) {
  uint16_t *d = reinterpret_cast<uint16_t *>(dst);
  for (int k = 0; k < k_pad; ++k)
    for (int n = 0; n < n_pad; ++n) {
      float v = 0.0f;
      if (n < out) {
        if (k < in) v = bf16_round(W[(size_t)k * out + n]);
        else if (k == in) v = bf16_round(b[n]);
        else if (k == in + 1) v = bf16_round(b[n] - bf16_round(b[n]));
      }
      d[(size_t)(k / 8) * (n_pad * 8) + (size_t)n * 8 + (k % 8)] = bf16_bits(v);
    }
}

using KernelFn = void (*)(const TcParams);

KernelFn select_kernel(int n_freq, int viewdir, int width, int nout, int nh, int contact) {
  if (contact) {   // the paper's own shape: gamma([d; delta]) 72-d, 32 wide, two hidden layers
    if (n_freq == 6 && viewdir == 0 && width == 32 && nout == 16 && nh == 2) return mlp_tc_kernel<6, 0, 32, 16, 2, 1>;
    return nullptr;
  }
#define MS_TC_CASE(F, V, W, O, H) \
  if (n_freq == F && viewdir == V && width == W && nout == O && nh == H) return mlp_tc_kernel<F, V, W, O, H>;
  MS_TC_CASE(4, 0, 64, 16, 3)
  MS_TC_CASE(4, 1, 64, 16, 3)
  MS_TC_CASE(4, 1, 64, 48, 3)
  MS_TC_CASE(4, 0, 64, 48, 3)
  MS_TC_CASE(6, 0, 128, 16, 3)
  MS_TC_CASE(6, 1, 128, 16, 3)
  MS_TC_CASE(4, 0, 128, 16, 3)
  MS_TC_CASE(4, 1, 128, 16, 3)
  MS_TC_CASE(6, 0, 64, 16, 3)
  MS_TC_CASE(4, 0, 64, 16, 2)
  MS_TC_CASE(6, 0, 128, 16, 2)
#undef MS_TC_CASE
  return nullptr;
}

int nout_pad(int out_dim) { return out_dim <= 16 ? 16 : (out_dim <= 36 ? 48 : 0); }

}  // namespace

int ms_tc_pack(const MsMlpShape &sh, int n_prims, const float *weights, MsTcWeights *out) {
  out->valid = false;
  const int nout = nout_pad(sh.out_dim);
  if (nout == 0 || !select_kernel(sh.n_freq, sh.use_viewdir, sh.width, nout, sh.n_hidden, sh.mode == MS_MODE_CONTACT)) return MS_OK;  // shape not covered
  const int k1 = (sh.in_dim + 2 + 15) / 16 * 16;
  const TcLayout L = tc_layout(k1, sh.width, sh.n_hidden, nout);
  std::vector<uint8_t> img;
  try {
    img.assign((size_t)n_prims * L.bytes, 0);
  } catch (...) {
    return MS_ERR_OUT_OF_MEMORY;
  }
  auto pack_range = [&](int i0, int i1) {
    for (int i = i0; i < i1; ++i) {
      const float *w = weights + (size_t)i * sh.params;
      uint8_t *dst = img.data() + (size_t)i * L.bytes;
      int in = sh.in_dim;
      for (int l = 0; l <= sh.n_hidden; ++l) {
        const bool last = l == sh.n_hidden;
        const int o = last ? sh.out_dim : sh.width;
        const float *b = w + (size_t)in * o;
        pack_wT(w, b, in, o, l == 0 ? k1 : sh.width + 16, last ? nout : sh.width, dst + L.off_w[l]);
        w = b + o;
        in = o;
      }
    }
  };
  {  // primitives are independent: the host's cores share them (4096 x 88.5 KB took 0.6 s on one)
    unsigned nt = std::thread::hardware_concurrency();
    if (nt < 1) nt = 1;
    if (nt > 16) nt = 16;
    if ((unsigned)n_prims < 4 * nt) nt = 1;
    std::vector<std::thread> th;
    try {
      for (unsigned t = 1; t < nt; ++t)
        th.emplace_back(pack_range, (int)((long long)n_prims * t / nt), (int)((long long)n_prims * (t + 1) / nt));
    } catch (...) {
      for (auto &x : th) x.join();
      th.clear();
      pack_range((int)((long long)n_prims / nt), n_prims);
      nt = 1;   // the rest was done inline
    }
    pack_range(0, (int)((long long)n_prims / nt));
    for (auto &x : th) x.join();
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
  if (!w.valid) return cudaErrorNotSupported;
  KernelFn fn = select_kernel(a.shape.n_freq, a.shape.use_viewdir, a.shape.width, w.n_out_pad, a.shape.n_hidden,
                              a.shape.mode == MS_MODE_CONTACT);
  if (!fn) return cudaErrorNotSupported;
  TcParams p;
  p.cam = a.cam; p.K = a.K; p.n_feat = a.shape.n_feat; p.falloff = a.falloff;
  p.center = a.center; p.A = a.A; p.segs = a.segs; p.intervals = a.intervals;
  p.image = (const uint8_t *)w.image;
  p.staging = a.staging; p.staging_feat = a.staging_feat; p.staging_gate = a.staging_gate;
  size_t smem = w.bytes_per_prim + tc_a1_stages(a.shape.width) * ((size_t)MS_ROWS * w.k1_pad * 2);
  if (w.n_out_pad > 16) smem += 4 * 32 * TC_HD_ROW;
  if (smem < TC_MIN_SMEM) smem = TC_MIN_SMEM;
  static int n_sm = 0;
  if (n_sm == 0) {
    int dev = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
  }
  cudaError_t e = cudaFuncSetAttribute((const void *)fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  // one persistent CTA per SM; the launch's block count lives on the device (a CTA with an empty range leaves at once)
  unsigned grid = (unsigned)n_sm;
  if (a.n_blocks_hint > 0 && a.n_blocks_hint < grid) grid = a.n_blocks_hint;
  const int threads = 32 * tc_warps(a.shape.width, w.n_out_pad);
  fn<<<grid, threads, smem, s>>>(p);
  MS_LAUNCHED();
  return cudaGetLastError();
}
