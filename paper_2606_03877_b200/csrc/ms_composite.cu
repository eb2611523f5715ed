// ms_composite.cu -- stage (e): per-ray merge of the hit intervals' sample streams in
// (t, primitive id, k) order and front-to-back compositing (Eq.6, Eq.14):
//   w = T (1 - e); C += w rgb; F += w feat; T <- T e; stop once T < t_stop (NS (e), Q9).
//
// One warp per ray.  Each stream t_k = t_in + (k + 1/2) delta is non-decreasing in k (fp32 rounding
// is monotone), so the position of a sample in the merged order has a closed form: its own k plus,
// for every other hit of the ray, the number of that hit's samples that precede (t, prim) -- 0 or K
// when the two t-ranges do not overlap (two compares), else a binary search over k.  No cursors, no
// sort.  The ray's staged samples (16 B each, one contiguous run) are gathered in merged order
// straight from global memory -- only the order (4 B per sample) lives in shared memory, so 40+
// warps fit per SM; each lane composites a run of consecutive merged samples, one warp product
// scan per window links the runs.  Features
// (32 channels): four 128 B rows per warp load.  Eq.7 slot features: composite_kernel<2> leaves per-hit coefficients,
// slot_feature_tile_kernel sums the embeddings tile by tile.
// HBM-bound by design: reads 16 B (+ 4 n_feat B) per sample and 16 B per hit, once.
#include <cuda_fp16.h>

#include "ms_internal.cuh"

namespace {

constexpr int CW = 4;        // warps (rays) per CTA
constexpr int CAP = 448;     // samples per window (a ray with more is processed in rank windows)
constexpr int HCAP = 32;     // hits cached in shared memory per ray (one per lane)
constexpr unsigned FULL = 0xffffffffu;

struct WarpSmem {
  uint32_t ord[CAP];    // ord[rank - r0] = sample index s = h*K + k inside the ray
  float4 key[HCAP];     // (t of sample 0, t of sample K-1, prim bits, unused)
  float2 geo[HCAP];     // (t_in, delta)
  uint2 pre[HCAP];      // (samples of streams entirely before this one, mask of streams that overlap it)
};

__device__ __forceinline__ bool precedes(float t2, float t, bool tie_lt) { return t2 < t || (t2 == t && tie_lt); }

// number of samples of stream (ti2, dl2, first tf, last tl, prim p2) that precede (t, prim)
__device__ __forceinline__ uint32_t count_before(float tf, float tl, float ti2, float dl2, int p2, float t, int prim, int K) {
  const bool tie_lt = p2 < prim;
  if (!precedes(tf, t, tie_lt)) return 0u;
  if (precedes(tl, t, tie_lt)) return (uint32_t)K;
  // precedes(sample 0) holds, precedes(sample K-1) does not: the count c is in [1, K-1].  The stream
  // is an arithmetic progression, so c ~ (t - t_in2)/delta2 + 1/2; the estimate is then corrected
  // against the canonical fp32 sample positions (usually one test on each side), so the result is
  // exactly the count the definition gives.
  int c = __float2int_rn(__fdividef(t - ti2, dl2));
  c = c < 1 ? 1 : (c > K - 1 ? K - 1 : c);
  while (c > 1 && !precedes(ms_sample_t(ti2, dl2, c - 1), t, tie_lt)) --c;
  while (c < K - 1 && precedes(ms_sample_t(ti2, dl2, c), t, tie_lt)) ++c;
  return (uint32_t)c;
}

// rank of sample (h, k) in the order (t, prim, k).  n <= HCAP: stream-level classification in
// sm.pre (streams entirely before / after need no per-sample work); else every stream is tested.
__device__ __forceinline__ uint32_t sample_rank(const WarpSmem &sm, const MsHit *__restrict__ hits, int n, int K, int h,
                                                int k, float *t_out, int contact) {
  if (n <= HCAP) {
    const float t = ms_sample_tm(sm.geo[h].x, sm.geo[h].y, k, contact);
    const int prim = __float_as_int(sm.key[h].z);
    *t_out = t;
    const uint2 pr = sm.pre[h];
    uint32_t rank = (uint32_t)k + pr.x;
    uint32_t m = pr.y;
    while (m) {
      const int h2 = __ffs(m) - 1;
      m &= m - 1;
      const float4 q = sm.key[h2];
      const float2 g = sm.geo[h2];
      rank += count_before(q.x, q.y, g.x, g.y, __float_as_int(q.z), t, prim, K);
    }
    return rank;
  }
  const MsHit me = hits[h];
  const float t = ms_sample_tm(me.t_in, me.delta, k, contact);
  *t_out = t;
  uint32_t rank = (uint32_t)k;
  for (int h2 = 0; h2 < n; ++h2) {
    if (h2 == h) continue;
    const MsHit g = hits[h2];
    rank += count_before(ms_sample_tm(g.t_in, g.delta, 0, contact), ms_sample_tm(g.t_in, g.delta, K - 1, contact), g.t_in, g.delta, g.prim, t,
                         me.prim, K);
  }
  return rank;
}

// n <= HCAP: lane h caches hit h and classifies every other stream against it
__device__ __forceinline__ void load_hits(WarpSmem &sm, const MsHit *__restrict__ hits, int n, int K, int lane, int contact) {
  if (n > HCAP) return;
  float tf = 0.f, tl = 0.f;
  int prim = 0;
  if (lane < n) {
    const MsHit g = hits[lane];
    tf = ms_sample_tm(g.t_in, g.delta, 0, contact); tl = ms_sample_tm(g.t_in, g.delta, K - 1, contact); prim = g.prim;
    sm.key[lane] = make_float4(tf, tl, __int_as_float(prim), 0.f);
    sm.geo[lane] = make_float2(g.t_in, g.delta);
  }
  __syncwarp();
  if (lane < n) {
    uint32_t before = 0, mask = 0;
    for (int h2 = 0; h2 < n; ++h2) {
      const float4 q = sm.key[h2];
      const bool tie_lt = __float_as_int(q.z) < prim;
      const bool all_before = precedes(q.y, tf, tie_lt);    // its last sample precedes my first
      const bool some_before = precedes(q.x, tl, tie_lt);   // its first sample precedes my last
      before += all_before ? (uint32_t)K : 0u;
      mask |= (some_before && !all_before && h2 != lane) ? (1u << h2) : 0u;
    }
    sm.pre[lane] = make_uint2(before, mask);
  }
}

template <int FEAT, bool DBG>  // FEAT 0: rgb/alpha only; 1: + linear head features; 2: + Eq.7 slot features (contact mode, K = 1); DBG: record the order (MS_FLAG_KEEP_ORDER)
__global__ void __launch_bounds__(CW * 32, FEAT == 0 ? 12 : 8) composite_kernel(MsCompositeArgs a) {
  __shared__ WarpSmem s_all[CW];
  __shared__ float s_w[FEAT ? CW : 1][FEAT ? CAP : 1];   // weight of the window's r-th merged sample (features only)
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  if (a.counters && a.counters[MS_CNT_OVERFLOW]) return;   // a no-sync render that overflowed its scratch: view invalid
  const MsBand band = a.band;
  WarpSmem &sm = s_all[warp];
  const int K = a.K, nf = a.n_feat;
  uint32_t n_stopped = 0;                                   // rays of this warp that stopped before their last sample
  // one warp per ray slot of the band (tile-major ray order: consecutive slots are neighbouring pixels of one
  // tile, and their staged samples are consecutive runs of the band's staging buffer)
  // one CTA per CW consecutive slots: the hardware's CTA scheduler balances the rays, which differ widely in cost
  // (0 .. 40+ hits); a persistent split, static or through a cursor, measured 0.6 - 1.5 ms slower on CFG4
  for (uint32_t q = band.q_lo + blockIdx.x * CW + warp; q < band.q_hi; q = band.q_hi) {
  int px, py;
  if (!ms_slot_pixel_dev(a.grid, q, &px, &py)) continue;     // padding slot of a tile that overhangs the image
  const size_t ray = (size_t)py * a.grid.W + px;
  __syncwarp();                                           // the previous ray is done with the warp's shared memory
  const uint32_t off = a.ray_off[q];
  const int n = (int)(a.ray_off[q + 1] - off);
  float T = 1.0f, C0 = 0.f, C1 = 0.f, C2 = 0.f;
  float F[MS_MAX_OUT / 32] = {0.f, 0.f};
  float4 F4 = make_float4(0.f, 0.f, 0.f, 0.f);   // n_feat == 32: channels 4*(lane%8)..+3 of the samples of lane group lane/8
  float4 G4 = make_float4(0.f, 0.f, 0.f, 0.f);   // fp16 staging: F4, G4 = channels 8*(lane%4)..+7 of lane group lane/4
  if (n > 0) {
    const MsHit *hits = a.hits + off;
    const size_t loc = (size_t)(off - band.slot0);        // the ray's first hit inside the band's staging buffers
    const float4 *stg = a.staging + loc * (size_t)K;
    const uint32_t S = (uint32_t)n * (uint32_t)K;
    const bool one_hit = FEAT == 0 && n == 1 && K > 1 && K <= 32;   // a single interval: its samples are in order
    if ((FEAT != 1 && K == 1 && n <= 32) || one_hit) {
      // At most one sample per lane.  K = 1 (the contact-point mode's usual ray): lane j holds hit j, its rank is the
      // number of hits that precede it in (t, prim) order.  One hit with K <= 32 samples (the usual ray of a sparse
      // scene): lane k holds sample k, already in order.  One product scan composites the ray.
      const int m = one_hit ? K : n;
      float t = 0.f;
      int prim = 0x7fffffff;
      if (!one_hit && lane < n) {
        const MsHit g = hits[lane];
        t = ms_sample_tm(g.t_in, g.delta, 0, a.contact);
        prim = g.prim;
      }
      uint32_t rank = 0;
      if (!one_hit) {
        for (int j = 0; j < n; ++j) {
          const float t2 = __shfl_sync(FULL, t, j);
          const int p2 = __shfl_sync(FULL, prim, j);
          rank += (j != lane && precedes(t2, t, p2 < prim)) ? 1u : 0u;
        }
      }
      if (a.tile_order || one_hit) rank = (uint32_t)lane;      // the shared per-tile order: the hits as stage (c) wrote them
      if (lane < m) {
        sm.ord[rank] = (uint32_t)lane;
        if (DBG) a.dbg_ord[(size_t)off * (size_t)K + rank] = (uint32_t)lane;
      }
      __syncwarp();
      const bool valid = lane < m;
      uint32_t slot = 0;
      float4 v = make_float4(0.f, 0.f, 0.f, 1.f);
      if (valid) {
        slot = sm.ord[lane];
        v = __ldg(stg + slot);
      }
      float p = v.w;  // inclusive product scan of e over the lanes
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const float q = __shfl_up_sync(FULL, p, o);
        if (lane >= o) p *= q;
      }
      float excl = __shfl_up_sync(FULL, p, 1);
      if (lane == 0) excl = 1.0f;
      const unsigned stop = __ballot_sync(FULL, valid && p < a.t_stop);
      const int last = stop ? __ffs(stop) - 1 : 31;          // Q9: the stopping sample still contributes
      const float w = (valid && lane <= last) ? excl * (1.0f - v.w) : 0.f;
      C0 = w * v.x; C1 = w * v.y; C2 = w * v.z;
      T = __shfl_sync(FULL, p, stop ? last : 31);
      n_stopped += (stop && last + 1 < m) ? 1u : 0u;
      if (FEAT == 2 && valid) {
        const float4 g = __ldg(a.gates + loc + slot);
        a.coef[loc + slot] = make_float4(w * g.x, w * g.y, w * g.z, w * g.w);
      }
    } else {
    load_hits(sm, hits, n, K, lane, a.contact);
    if (FEAT == 2 && S > (uint32_t)CAP)   // a ray that stops early leaves its later windows unvisited: their coefficients are 0
      for (uint32_t s = lane; s < S; s += 32) a.coef[loc + s] = make_float4(0.f, 0.f, 0.f, 0.f);
    __syncwarp();
    bool stopped = false;
    for (uint32_t r0 = 0; r0 < S && (!stopped || DBG); r0 += CAP) {
      const uint32_t cnt = S - r0 < (uint32_t)CAP ? S - r0 : (uint32_t)CAP;
      // ---- rank pass: ord[] (and, for a multi-window ray, val[] by rank) ----
      int h = lane / K, k = lane - h * K;
      const int dh = 32 / K, dk = 32 - dh * K;
      for (uint32_t s = lane; s < S; s += 32) {
        float t;
        const uint32_t rk = (a.tile_order ? s : sample_rank(sm, hits, n, K, h, k, &t, a.contact)) - r0;
        if (rk < cnt) {
          sm.ord[rk] = s;
          if (DBG) a.dbg_ord[(size_t)off * (size_t)K + r0 + rk] = s;
        }
        h += dh; k += dk;
        if (k >= K) { k -= K; ++h; }
      }
      __syncwarp();
      if (DBG && stopped) continue;                // MS_FLAG_KEEP_ORDER: the windows behind the stop are ranked only
      // ---- composite the window: lane l takes the l-th run of CH consecutive merged samples ----
      // One product scan over the lanes' run products gives every lane its entry transmittance; the
      // run itself is sequential (T <- T e).  The first sample, in merged order, whose T drops
      // below t_stop still contributes (Q9); every later one contributes nothing.
      const uint32_t CH = (cnt + 31u) >> 5;
      const uint32_t rb = lane * CH < cnt ? lane * CH : cnt, re = rb + CH < cnt ? rb + CH : cnt;
      float pl = 1.0f;
      for (uint32_t r = rb; r < re; ++r) pl *= __ldg(&stg[sm.ord[r]].w);
      float p = pl;  // inclusive product scan of the run products over the lanes
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const float q = __shfl_up_sync(FULL, p, o);
        if (lane >= o) p *= q;
      }
      float Tl = __shfl_up_sync(FULL, p, 1);
      Tl = lane == 0 ? T : T * Tl;                 // transmittance in front of the lane's first sample
      float c0 = 0.f, c1 = 0.f, c2 = 0.f;
      uint32_t lstop = 0xffffffffu;                // the lane's first sample that crosses the threshold
      for (uint32_t r = rb; r < re && lstop == 0xffffffffu; ++r) {
        const float4 v = __ldg(stg + sm.ord[r]);   // 16 B gather inside the ray's contiguous staging run (second touch: L1)
        const float w = Tl * (1.0f - v.w);
        c0 = fmaf(w, v.x, c0); c1 = fmaf(w, v.y, c1); c2 = fmaf(w, v.z, c2);
        if (FEAT) s_w[FEAT ? warp : 0][FEAT ? r : 0] = w;
        Tl *= v.w;
        if (Tl < a.t_stop) lstop = r;
      }
      const unsigned stop = __ballot_sync(FULL, lstop != 0xffffffffu);
      uint32_t done = cnt;                         // samples of this window that carry a weight
      if (stop) {
        const int ls = __ffs(stop) - 1;            // runs are in merged order: the lowest lane stops first
        if (lane > ls) { c0 = 0.f; c1 = 0.f; c2 = 0.f; }
        done = __shfl_sync(FULL, lstop, ls) + 1u;
        T = __shfl_sync(FULL, Tl, ls);
        stopped = true;
        n_stopped += (r0 + done < S) ? 1u : 0u;
      } else {
        T = __shfl_sync(FULL, Tl, 31);             // lane 31 leaves with T times the product of the whole window
      }
      C0 += c0; C1 += c1; C2 += c2;
      if (FEAT == 2) {
        // Eq.7: F = sum_i (T_i alpha_i) sum_k g_ik e_ik.  This kernel only turns every hit's gates into
        // its coefficients (T alpha) g_k; slot_feature_tile_kernel sums the embeddings.
        __syncwarp();
        const float4 *gates = a.gates + loc;
        float4 *coef = a.coef + loc;
        for (uint32_t r = lane; r < cnt; r += 32) {
          const uint32_t s = sm.ord[r];
          const float w = r < done ? s_w[FEAT ? warp : 0][FEAT ? r : 0] : 0.0f;
          const float4 g = __ldg(gates + s);
          coef[s] = make_float4(w * g.x, w * g.y, w * g.z, w * g.w);
        }
      }
      if (FEAT == 1) {
        __syncwarp();
        const float *fbase = reinterpret_cast<const float *>(a.staging_feat) + loc * (size_t)K * (size_t)nf;
        if (nf == 32 && a.feat_half) {
          // fp16 rows of 64 B (tensor path): lane group g = lane/4 takes sample r+g, lane%4 the channels
          // 8*(lane%4)..+7: one warp load covers eight rows; four loads in flight per lane before the FMAs.
          const uint4 *hbase = reinterpret_cast<const uint4 *>(a.staging_feat) + loc * (size_t)K * 4;
          const int g = lane >> 2, c8 = lane & 3;
          for (uint32_t r = 0; r < done; r += 32) {
            uint4 f[4];
            float wv[4];
#pragma unroll
            for (int q = 0; q < 4; ++q) {
              const uint32_t rr = r + 8 * q + g;
              f[q] = make_uint4(0u, 0u, 0u, 0u);
              wv[q] = 0.f;
              if (rr < done) {
                const uint32_t s = sm.ord[rr];
                wv[q] = s_w[FEAT ? warp : 0][FEAT ? rr : 0];
                f[q] = __ldg(hbase + (size_t)s * 4 + c8);
              }
            }
#pragma unroll
            for (int q = 0; q < 4; ++q) {
              const float2 a0 = __half22float2(*reinterpret_cast<const __half2 *>(&f[q].x));
              const float2 a1 = __half22float2(*reinterpret_cast<const __half2 *>(&f[q].y));
              const float2 a2 = __half22float2(*reinterpret_cast<const __half2 *>(&f[q].z));
              const float2 a3 = __half22float2(*reinterpret_cast<const __half2 *>(&f[q].w));
              F4.x = fmaf(wv[q], a0.x, F4.x); F4.y = fmaf(wv[q], a0.y, F4.y);
              F4.z = fmaf(wv[q], a1.x, F4.z); F4.w = fmaf(wv[q], a1.y, F4.w);
              G4.x = fmaf(wv[q], a2.x, G4.x); G4.y = fmaf(wv[q], a2.y, G4.y);
              G4.z = fmaf(wv[q], a3.x, G4.z); G4.w = fmaf(wv[q], a3.y, G4.w);
            }
          }
        } else if (nf == 32) {
          // lane group g = lane/8 takes sample r+g, lane%8 takes channels 4*(lane%8)..+3: one warp
          // load covers four 128 B rows; four loads in flight per lane before the FMAs.
          const int g = lane >> 3, c4 = lane & 7;
          for (uint32_t r = 0; r < done; r += 16) {
            float4 f[4];
            float wv[4];
#pragma unroll
            for (int q = 0; q < 4; ++q) {
              const uint32_t rr = r + 4 * q + g;
              f[q] = make_float4(0.f, 0.f, 0.f, 0.f);
              wv[q] = 0.f;
              if (rr < done) {
                const uint32_t s = sm.ord[rr];
                wv[q] = s_w[FEAT ? warp : 0][FEAT ? rr : 0];
                f[q] = __ldg(reinterpret_cast<const float4 *>(fbase + (size_t)s * 32) + c4);
              }
            }
#pragma unroll
            for (int q = 0; q < 4; ++q) {
              F4.x = fmaf(wv[q], f[q].x, F4.x); F4.y = fmaf(wv[q], f[q].y, F4.y);
              F4.z = fmaf(wv[q], f[q].z, F4.z); F4.w = fmaf(wv[q], f[q].w, F4.w);
            }
          }
        } else {
          for (uint32_t r = 0; r < done; ++r) {
            const uint32_t s = sm.ord[r];
            const float w = s_w[FEAT ? warp : 0][FEAT ? r : 0];
#pragma unroll
            for (int q = 0; q < MS_MAX_OUT / 32; ++q) {
              const int c = lane + 32 * q;
              if (c < nf) F[q] = fmaf(w, __ldg(fbase + (size_t)s * (size_t)nf + c), F[q]);
            }
          }
        }
      }
      __syncwarp();
    }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      C0 += __shfl_xor_sync(FULL, C0, o);
      C1 += __shfl_xor_sync(FULL, C1, o);
      C2 += __shfl_xor_sync(FULL, C2, o);
    }
  }
  if (lane < 3) a.out_rgb[3 * ray + lane] = lane == 0 ? C0 : (lane == 1 ? C1 : C2);
  if (lane == 3) a.out_alpha[ray] = 1.0f - T;
  if (FEAT == 1) {
    if (nf == 32 && a.feat_half) {
#pragma unroll
      for (int o = 4; o < 32; o <<= 1) {
        F4.x += __shfl_xor_sync(FULL, F4.x, o); F4.y += __shfl_xor_sync(FULL, F4.y, o);
        F4.z += __shfl_xor_sync(FULL, F4.z, o); F4.w += __shfl_xor_sync(FULL, F4.w, o);
        G4.x += __shfl_xor_sync(FULL, G4.x, o); G4.y += __shfl_xor_sync(FULL, G4.y, o);
        G4.z += __shfl_xor_sync(FULL, G4.z, o); G4.w += __shfl_xor_sync(FULL, G4.w, o);
      }
      if (lane < 4) {
        reinterpret_cast<float4 *>(a.out_feat + ray * 32)[2 * lane] = F4;
        reinterpret_cast<float4 *>(a.out_feat + ray * 32)[2 * lane + 1] = G4;
      }
    } else if (nf == 32) {
#pragma unroll
      for (int o = 8; o < 32; o <<= 1) {
        F4.x += __shfl_xor_sync(FULL, F4.x, o); F4.y += __shfl_xor_sync(FULL, F4.y, o);
        F4.z += __shfl_xor_sync(FULL, F4.z, o); F4.w += __shfl_xor_sync(FULL, F4.w, o);
      }
      if (lane < 8) reinterpret_cast<float4 *>(a.out_feat + ray * 32)[lane] = F4;
    } else {
#pragma unroll
      for (int q2 = 0; q2 < MS_MAX_OUT / 32; ++q2) {
        const int c = lane + 32 * q2;
        if (c < nf) a.out_feat[ray * nf + c] = F[q2];
      }
    }
  }
  }
  if (lane == 0 && n_stopped && a.counters) atomicAdd(&a.counters[MS_CNT_STOPPED_RAYS], n_stopped);
}

// Eq.7 features, tile-owned accumulation.  A ray's hits are a subsequence of its tile's sorted list (stage (c) writes
// them in list order), so the CTA of a tile walks that list ONCE: the four embedding rows of a primitive are loaded
// once per (tile, 128-channel chunk) instead of once per group of four rays, and a primitive that no pixel of the warp
// hits costs one ballot.  CTA = (tile, block of up to 256 ray slots, chunk of 128 channels); a warp owns 32 consecutive
// ray slots (two rows of a 16 x 16 tile): lane l keeps the hit-list cursor of slot l AND the accumulators of the channels
// 4 l .. 4 l + 3 of all 32 slots (128 registers).  Per primitive of the list: ballot of the slots whose next hit it
// is, their coefficients through shared memory (one broadcast LDS.128 per hit), 16 FMAs per hit and lane.  The sum of
// a ray runs over its hits in list order whatever the band layout: deterministic.
constexpr int SF_CHUNK = 32;          // list entries staged per step (one per lane)

// V = the channels a lane owns: float4 (chunks of 128 channels, 128 accumulator registers, one CTA per SM)
__device__ __forceinline__ float4 sf_zero(float4) { return make_float4(0.f, 0.f, 0.f, 0.f); }
__device__ __forceinline__ void sf_fma(float4 &F, const float4 c, const float4 e0, const float4 e1, const float4 e2, const float4 e3) {
  F.x = fmaf(c.w, e3.x, fmaf(c.z, e2.x, fmaf(c.y, e1.x, fmaf(c.x, e0.x, F.x))));
  F.y = fmaf(c.w, e3.y, fmaf(c.z, e2.y, fmaf(c.y, e1.y, fmaf(c.x, e0.y, F.y))));
  F.z = fmaf(c.w, e3.z, fmaf(c.z, e2.z, fmaf(c.y, e1.z, fmaf(c.x, e0.z, F.z))));
  F.w = fmaf(c.w, e3.w, fmaf(c.z, e2.w, fmaf(c.y, e1.w, fmaf(c.x, e0.w, F.w))));
}

template <typename V>
__global__ void __launch_bounds__(256, sizeof(V) == 8 ? 2 : 1) slot_feature_tile_kernel(MsCompositeArgs a, int blocks_per_tile, int n_chunks) {
  constexpr int VW = (int)(sizeof(V) / 4);
  __shared__ float4 sC[8][32];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  if (a.counters && a.counters[MS_CNT_OVERFLOW]) return;
  const MsBand band = a.band;
  const uint32_t T2 = (uint32_t)(a.grid.tile * a.grid.tile);
  const int chunk = blockIdx.x % n_chunks;
  const int blk = (blockIdx.x / n_chunks) % blocks_per_tile;
  const uint32_t pos = band.q_lo / T2 + blockIdx.x / (uint32_t)(n_chunks * blocks_per_tile);
  const ushort2 txy = a.grid.pos_xy[pos];
  const int tile_id = (int)txy.y * a.grid.tiles_x + (int)txy.x;
  const uint32_t q = pos * T2 + (uint32_t)blk * 256u + threadIdx.x;      // this lane's ray slot
  int px, py;
  const bool live = q < band.q_hi && ms_slot_pixel_dev(a.grid, q, &px, &py);
  const uint32_t off = live ? a.ray_off[q] : 0u;
  const uint32_t nh = live ? a.ray_off[q + 1] - off : 0u;
  // the cursor of this lane's hit list, with the next coefficient and the two next primitives already loaded: the
  // loads a hit triggers are consumed one hit later
  uint32_t cur = 0;
  int nxt = nh ? __ldg(&a.hits[off].prim) : -1;
  int nxt2 = nh > 1 ? __ldg(&a.hits[off + 1].prim) : -1;
  const float4 *coef = a.coef + (off - band.slot0);
  float4 cnext = nh ? __ldg(coef) : make_float4(0.f, 0.f, 0.f, 0.f);
  V F[32];
#pragma unroll
  for (int j = 0; j < 32; ++j) F[j] = sf_zero(V());
  const uint64_t pmask = (1ull << a.prim_bits) - 1ull;
  const uint32_t beg = a.tile_start[tile_id], end = a.tile_start[tile_id + 1];
  const size_t cf = (size_t)a.c_f, cf4 = cf / VW, prow = 4 * cf4;     // in units of V: a row, a primitive's four rows
  const V *slots4 = reinterpret_cast<const V *>(a.slots) + 32 * chunk + lane;
  const unsigned any_hits = __ballot_sync(FULL, nh > 0);
  // list entry i: its primitive, or -1 past the end / for a pair without hits
  auto entry = [&](uint32_t i) -> int {
    if (i < end && (!a.pair_hits || __ldg(a.pair_hits + i) > 0u)) return (int)(__ldg(a.keys + i) & pmask);
    return -1;
  };
  if (any_hits && beg < end) {
    int my_p = entry(beg + lane);                          // lane c stages entry base + c of the current chunk ...
    V e0, e1, e2, e3;                                 // the embedding rows of the current entry (this lane's channels)
    {
      const int p0 = __shfl_sync(FULL, my_p, 0);
      const V *e = slots4 + (size_t)(p0 < 0 ? 0 : p0) * prow;
      e0 = __ldg(e); e1 = __ldg(e + cf4); e2 = __ldg(e + 2 * cf4); e3 = __ldg(e + 3 * cf4);
    }
    for (uint32_t base = beg; base < end; base += SF_CHUNK) {
      const int my_p2 = entry(base + SF_CHUNK + lane);     // ... and of the one after it
      const int nc = (int)(end - base < (uint32_t)SF_CHUNK ? end - base : (uint32_t)SF_CHUNK);
      for (int c = 0; c < nc; ++c) {
        const int p = __shfl_sync(FULL, my_p, c);
        // the rows of the entry after this one are on their way while this one is summed
        const int pn = c + 1 < SF_CHUNK ? __shfl_sync(FULL, my_p, (c + 1) & 31) : __shfl_sync(FULL, my_p2, 0);
        const V *en = slots4 + (size_t)(pn < 0 ? 0 : pn) * prow;
        const V n0 = __ldg(en), n1 = __ldg(en + cf4), n2 = __ldg(en + 2 * cf4), n3 = __ldg(en + 3 * cf4);
        const bool has = p >= 0 && nxt == p;
        const unsigned m = __ballot_sync(FULL, has);
        if (m) {
          sC[warp][lane] = has ? cnext : make_float4(0.f, 0.f, 0.f, 0.f);
          if (has) {
            ++cur;
            nxt = nxt2;
            if (cur < nh) cnext = __ldg(coef + cur);
            nxt2 = cur + 1 < nh ? __ldg(&a.hits[off + cur + 1].prim) : -1;
          }
          __syncwarp();
          // groups of four neighbouring slots: a group with a hit is summed whole (zero coefficients where there is
          // none) -- straight-line code with four independent broadcast loads and sixteen FMA chains in flight
#pragma unroll
          for (int g = 0; g < 8; ++g) {
            if ((m >> (4 * g)) & 15u) {
              float4 cj[4];
#pragma unroll
              for (int u = 0; u < 4; ++u) cj[u] = sC[warp][4 * g + u];
#pragma unroll
              for (int u = 0; u < 4; ++u) {
                sf_fma(F[4 * g + u], cj[u], e0, e1, e2, e3);
              }
            }
          }
          __syncwarp();
        }
        e0 = n0; e1 = n1; e2 = n2; e3 = n3;
      }
      my_p = my_p2;
    }
  }
  // pixel j of the warp: 32 lanes x sizeof(V) contiguous bytes of its feature row
  const unsigned lv = __ballot_sync(FULL, live);
  const long long my_pix = live ? (long long)py * a.grid.W + px : 0;
#pragma unroll
  for (int j = 0; j < 32; ++j) {
    const long long pix = __shfl_sync(FULL, my_pix, j);
    if ((lv >> j) & 1u) reinterpret_cast<V *>(a.out_feat + (size_t)pix * cf)[32 * chunk + lane] = F[j];
  }
}

// Backward of the compositing (S:Sec.8(f) NEXT-4; Eq.6, Eq.14): for one ray with dL/dC = g,
//   dL/dc_j = T_j (1 - e_j) g,     dL/de_j = -T_j (c_j . g) + (sum_{m > j} T_m (1 - e_m) (c_m . g)) / e_j,
// in the merged (t, primitive, k) order of the forward pass (the same closed-form ranks), samples behind the early
// stop (Q9) carrying nothing.  One warp per ray: ranks into a global order buffer, a forward product scan that leaves
// T_j in the output slot, a reverse sum scan that turns it into the two gradients.  Output per sample, at its
// staging index: (dL/dc_r, dL/dc_g, dL/dc_b, dL/de).
__global__ void __launch_bounds__(CW * 32) composite_bwd_kernel(MsCompositeBwdArgs a) {
  __shared__ WarpSmem s_all[CW];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const uint32_t q = blockIdx.x * CW + warp;
  if (q >= (uint32_t)a.grid.n_tiles << (2 * a.grid.tshift)) return;
  int px, py;
  if (!ms_slot_pixel_dev(a.grid, q, &px, &py)) return;
  WarpSmem &sm = s_all[warp];
  const uint32_t off = a.ray_off[q];
  const int n = (int)(a.ray_off[q + 1] - off);
  if (n == 0) return;
  const int K = a.K;
  const size_t ray = (size_t)py * a.grid.W + px;
  const float g0 = a.d_rgb[3 * ray], g1 = a.d_rgb[3 * ray + 1], g2 = a.d_rgb[3 * ray + 2];
  const MsHit *hits = a.hits + off;
  const float4 *stg = a.staging + (size_t)off * (size_t)K;
  float4 *gst = a.gstage + (size_t)off * (size_t)K;
  uint32_t *ord = a.ord + (size_t)off * (size_t)K;
  const uint32_t S = (uint32_t)n * (uint32_t)K;
  load_hits(sm, hits, n, K, lane, 0);
  __syncwarp();
  for (uint32_t s = lane; s < S; s += 32) {
    const int h = (int)(s / (uint32_t)K), k = (int)(s - (uint32_t)h * (uint32_t)K);
    float t;
    ord[sample_rank(sm, hits, n, K, h, k, &t, 0)] = s;
  }
  __syncwarp();
  // forward: transmittance in front of every sample, the stop
  float T = 1.0f;
  uint32_t n_used = S;
  for (uint32_t base = 0; base < S; base += 32) {
    const uint32_t r = base + lane;
    const bool valid = r < S;
    uint32_t s = 0;
    float e = 1.0f;
    if (valid) { s = ord[r]; e = stg[s].w; }
    float p = e;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const float v = __shfl_up_sync(FULL, p, o);
      if (lane >= o) p *= v;
    }
    float excl = __shfl_up_sync(FULL, p, 1);
    if (lane == 0) excl = 1.0f;
    if (valid) gst[s].w = T * excl;                           // T_j, replaced by dL/de_j below
    const unsigned stop = __ballot_sync(FULL, valid && T * p < a.t_stop);
    if (stop) { n_used = base + (uint32_t)__ffs(stop); break; }   // the stopping sample still counts (Q9)
    T *= __shfl_sync(FULL, p, 31);
  }
  __syncwarp();
  // backward: suffix sums of T_m (1 - e_m) (c_m . g), from the last used sample to the first
  float carry = 0.0f;
  for (int base = (int)((S - 1) / 32) * 32; base >= 0; base -= 32) {
    const uint32_t r = (uint32_t)base + lane;
    const bool valid = r < S;
    const bool used = r < n_used;
    uint32_t s = 0;
    float4 v = make_float4(0.f, 0.f, 0.f, 1.f);
    float Tj = 0.0f;
    if (valid) { s = ord[r]; v = stg[s]; Tj = gst[s].w; }
    const float cg = v.x * g0 + v.y * g1 + v.z * g2;
    const float term = used ? Tj * (1.0f - v.w) * cg : 0.0f;
    float sum = term;                                          // inclusive sum over the lanes at and above this one
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const float t = __shfl_down_sync(FULL, sum, o);
      if (lane + o < 32) sum += t;
    }
    const float suffix = carry + sum - term;
    if (valid) {
      float4 out = make_float4(0.f, 0.f, 0.f, 0.f);
      if (used) {
        const float w = Tj * (1.0f - v.w);
        out.x = w * g0; out.y = w * g1; out.z = w * g2;
        out.w = -Tj * cg + (v.w > 0.0f ? suffix / v.w : 0.0f);
      }
      gst[s] = out;
    }
    carry += __shfl_sync(FULL, sum, 0);
  }
}

}  // namespace

cudaError_t ms_composite(const MsCompositeArgs &a, cudaStream_t s) {
  const size_t slots = (size_t)a.band.q_hi - a.band.q_lo;
  if (slots == 0) return cudaSuccess;
  const unsigned grid = (unsigned)((slots + CW - 1) / CW);
  const bool feat = a.n_feat > 0 && a.out_feat && a.staging_feat;
  const bool slot_feat = a.c_f > 0 && a.out_feat && a.gates && a.coef && a.slots && a.K == 1;
  const bool dbg = a.dbg_ord != nullptr;
  if (slot_feat) { if (dbg) composite_kernel<2, true><<<grid, CW * 32, 0, s>>>(a); else composite_kernel<2, false><<<grid, CW * 32, 0, s>>>(a); }
  else if (!feat) { if (dbg) composite_kernel<0, true><<<grid, CW * 32, 0, s>>>(a); else composite_kernel<0, false><<<grid, CW * 32, 0, s>>>(a); }
  else { if (dbg) composite_kernel<1, true><<<grid, CW * 32, 0, s>>>(a); else composite_kernel<1, false><<<grid, CW * 32, 0, s>>>(a); }
  MS_LAUNCHED();
  if (slot_feat) {
    const size_t T2 = (size_t)a.grid.tile * a.grid.tile;
    // bands are runs of whole tiles; the tile lists are those of stage (b)
    if (!(a.keys && a.tile_start && a.grid.pos_xy && a.band.q_lo % T2 == 0 && slots % T2 == 0 && a.c_f % 128 == 0))
      return cudaErrorInvalidValue;
    const int threads = (int)(T2 < 256 ? T2 : 256), bpt = (int)((T2 + 255) / 256);
    const size_t n_tiles = slots / T2;
    // float2 per lane (64-channel chunks, two CTAs per SM) measured slower: 2.75 against 2.64 ms on next2
    slot_feature_tile_kernel<float4><<<(unsigned)(n_tiles * bpt * (a.c_f / 128)), threads, 0, s>>>(a, bpt, a.c_f / 128);
    MS_LAUNCHED();
  }
  return cudaGetLastError();
}

cudaError_t ms_composite_bwd(const MsCompositeBwdArgs &a, cudaStream_t s) {
  const size_t slots = (size_t)a.grid.n_tiles * a.grid.tile * a.grid.tile;
  if (slots == 0) return cudaSuccess;
  composite_bwd_kernel<<<(unsigned)((slots + CW - 1) / CW), CW * 32, 0, s>>>(a);
  MS_LAUNCHED();
  return cudaGetLastError();
}
