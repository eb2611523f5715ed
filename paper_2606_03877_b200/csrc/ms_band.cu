// ms_band.cu -- bands and depth waves (S:Sec.8(f) NEXT-3; P:437 Sec.B.2 "The sorted primitives are processed
// sequentially ... We further adopt early t[ermination]").
//
// Stage (d) wants all samples of one primitive together, stage (e) all samples of one ray together; the staging
// buffer between them is what stage (d) writes and stage (e) reads.  To keep it small (and L2-resident) the frame
// is cut into BANDS: runs of consecutive tiles, in macro-tile order, whose hits fill a byte budget.  (c)-count and
// the ray_off scan run once per frame; this file then orders the (tile, primitive) pairs by
// (band, wave, primitive) -- one radix sort of P keys -- so that every (band, wave) owns a contiguous range of
// SEGMENTS (= the intervals of one primitive inside one band and wave), of intervals and of 128-row blocks.
// Stages (d) and (e) are then launched per band on a staging buffer of one band's size.
//
// Depth WAVES give the early termination of P:437 real effect: a tile's list is sorted by entry depth, so wave w of
// a band -- the list ranks [first(w), first(w+1)) of every tile -- holds the primitives behind those of the earlier
// waves.  Before wave w >= 1 every ray knows B = the smallest t_in among its own hits still to come; the samples
// already evaluated with t < B precede everything not yet evaluated, and the transmittance over them is a product,
// independent of their order.  A ray whose product is already below t_stop/2 stops inside that prefix whatever
// the later hits hold (the factor 2 covers fp32 rounding in the final compositing order), so its later intervals
// are dropped before they are encoded.  The image is bitwise the one without waves.
#include "ms_internal.cuh"
#include "ms_cta_scan.cuh"

namespace {

constexpr int WB = 3;   // bits of the wave field (MS_MAX_WAVES <= 8)
static_assert(MS_MAX_WAVES <= (1 << WB), "wave field");

__device__ __forceinline__ void tile_stats_body(const MsGrid &g, int pos, const uint32_t *ray_off, const uint32_t *tile_start,
                                                uint32_t *counters, uint32_t hit_cap) {
  const uint32_t T2 = (uint32_t)(g.tile * g.tile);
  if (pos < g.n_tiles) {
    const uint32_t h = ray_off[(size_t)(pos + 1) * T2] - ray_off[(size_t)pos * T2];   // exact even if the scan wrapped
    if (h) {
      atomicMax(&counters[MS_CNT_MAX_TILE_HITS], h);
      atomicAdd(reinterpret_cast<unsigned long long *>(counters + MS_CNT_HITS), (unsigned long long)h);
    }
    const uint32_t len = tile_start[pos + 1] - tile_start[pos];
    if (len) atomicMax(&counters[MS_CNT_MAX_LIST], len);
  }
  // no-sync renders: the hits must fit the scratch sized from the previous view (hit_cap = 0: no check)
  if (pos == 0 && hit_cap && ray_off[(size_t)g.n_tiles * T2] > hit_cap) {
    counters[MS_CNT_OVERFLOW] = 1u;
    counters[MS_CNT_STICKY_OVERFLOW] = 1u;       // survives the per-view reset: any view of a batch
  }
}

__global__ void tile_stats_kernel(MsGrid g, const uint32_t *__restrict__ ray_off, const uint32_t *__restrict__ tile_start,
                                  uint32_t *__restrict__ counters, uint32_t hit_cap) {
  tile_stats_body(g, blockIdx.x * blockDim.x + threadIdx.x, ray_off, tile_start, counters, hit_cap);
}

// ---- single band, single wave: segments = primitives, pairs in stage (a)'s emission order ----------------------
__device__ __forceinline__ void pair_single_body(const MsBandArgs &a, size_t i) {
  const uint64_t key = a.keys[i];
  const int prim = (int)(key & ((1ull << a.prim_bits) - 1ull));
  const int tile = (int)(key >> (32 + a.prim_bits));
  const int tx = tile % a.grid.tiles_x, ty = tile / a.grid.tiles_x;
  const int4 rc = a.rect[prim];
  const uint32_t emit = a.emit_off[prim] + (uint32_t)((ty - rc.y) * (rc.z - rc.x + 1) + (tx - rc.x));
  a.slot_of[i] = emit;
  a.pair_hits_j[emit] = a.pair_hits_i[i];
}

__global__ void pair_single_kernel(MsBandArgs a) {
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  const size_t P = a.P_dev ? (*a.P_dev < a.P ? (size_t)*a.P_dev : a.P) : a.P;
  if (i < P) pair_single_body(a, i);
}

__device__ __forceinline__ void seg_single_body(const MsBandArgs &a, int p) {
  const uint32_t cap = (uint32_t)a.P;       // no-sync renders: emit offsets beyond the capacity (an overflowed view)
  const uint32_t s = a.pair_off[a.emit_off[p] < cap ? a.emit_off[p] : cap];
  a.grp_iv0[p] = s;
  if (p < a.n_prims) {
    const uint32_t e = a.pair_off[a.emit_off[p + 1] < cap ? a.emit_off[p + 1] : cap];
    a.grp_blocks[p] = (uint32_t)(((uint64_t)(e - s) * (uint64_t)a.K + MS_ROWS - 1) / MS_ROWS);
  }
}

__global__ void seg_single_kernel(MsBandArgs a) {
  const int p = blockIdx.x * blockDim.x + threadIdx.x;
  if (p <= a.n_prims) seg_single_body(a, p);
}

__device__ __forceinline__ void tables_single_body(const MsBandArgs &a) {
  const uint32_t T2 = (uint32_t)(a.grid.tile * a.grid.tile);
  // a no-sync render whose pairs or hits overflowed the scratch evaluates nothing (the view is reported invalid)
  a.bw[0] = make_uint2(0u, a.counters[MS_CNT_OVERFLOW] ? 0u : (uint32_t)a.n_prims);
  for (int w = 1; w < MS_MAX_WAVES; ++w) a.bw[w] = make_uint2((uint32_t)a.n_prims, (uint32_t)a.n_prims);
  MsBand b;
  b.q_lo = 0u; b.q_hi = (uint32_t)a.grid.n_tiles * T2; b.slot0 = 0u; b.pad = 0u;
  a.bands[0] = b;
  a.counters[MS_CNT_SEGS] = (uint32_t)a.n_prims;
  a.counters[MS_CNT_BLOCKS] = a.blk_off[a.n_prims];
}

__global__ void tables_single_kernel(MsBandArgs a) { tables_single_body(a); }

// small frames: the five steps of ms_order_single by one CTA, one launch
constexpr int OS_THREADS = 1024;
constexpr size_t OS_MAX = 32768;
__global__ void __launch_bounds__(OS_THREADS) order_single_small_kernel(MsBandArgs a) {
  __shared__ uint32_t wt[OS_THREADS / 32 + 1];
  if (a.fuse_ray_scan) {
    cta_exclusive_scan_u32<OS_THREADS>(a.ray_hits, a.ray_off_w, a.R, wt);
    __syncthreads();
  }
  if (a.fuse_stats) {
    const int n = a.grid.n_tiles > 0 ? a.grid.n_tiles : 1;
    for (int pos = threadIdx.x; pos < n; pos += OS_THREADS)
      tile_stats_body(a.grid, pos, a.ray_off, a.tile_start, a.counters, a.hit_cap);
    __syncthreads();
  }
  const size_t P = a.P_dev ? (*a.P_dev < a.P ? (size_t)*a.P_dev : a.P) : a.P;
  for (size_t i = threadIdx.x; i < P; i += OS_THREADS) pair_single_body(a, i);
  __syncthreads();
  cta_exclusive_scan_u32<OS_THREADS>(a.pair_hits_j, a.pair_off, a.P, wt);
  __syncthreads();
  for (int p = threadIdx.x; p <= a.n_prims; p += OS_THREADS) seg_single_body(a, p);
  __syncthreads();
  cta_exclusive_scan_u32<OS_THREADS>(a.grp_blocks, a.blk_off, (size_t)a.n_prims, wt);
  __syncthreads();
  if (threadIdx.x == 0) tables_single_body(a);
}

// ---- bands x waves --------------------------------------------------------------------------------------------
// first tile position whose hit prefix reaches v
__device__ __forceinline__ int first_pos_at(const MsGrid &g, const uint32_t *__restrict__ ray_off, uint64_t v) {
  const uint32_t T2 = (uint32_t)(g.tile * g.tile);
  int lo = 0, hi = g.n_tiles;       // answer in [0, n_tiles]
  while (lo < hi) {
    const int mid = (lo + hi) >> 1;
    if ((uint64_t)ray_off[(size_t)mid * T2] >= v) hi = mid; else lo = mid + 1;
  }
  return lo;
}

__global__ void band_table_kernel(MsBandArgs a) {
  const int b = blockIdx.x * blockDim.x + threadIdx.x;
  if (b >= a.n_bands) return;
  const uint32_t T2 = (uint32_t)(a.grid.tile * a.grid.tile);
  const int lo = b == 0 ? 0 : first_pos_at(a.grid, a.ray_off, (uint64_t)b * a.cap_hits);
  const int hi = b == a.n_bands - 1 ? a.grid.n_tiles : first_pos_at(a.grid, a.ray_off, (uint64_t)(b + 1) * a.cap_hits);
  MsBand t;
  t.q_lo = (uint32_t)lo * T2; t.q_hi = (uint32_t)hi * T2; t.slot0 = a.ray_off[(size_t)lo * T2]; t.pad = 0u;
  a.bands[b] = t;
}

// band of a tile position: the band whose [b cap, (b+1) cap) holds the tile's hit prefix -- but a tile with the
// same prefix as its predecessor (no hits in between) must land where band_table_kernel's lower bound puts it
__device__ __forceinline__ int band_of_pos(const MsBandArgs &a, int pos) {
  const uint32_t T2 = (uint32_t)(a.grid.tile * a.grid.tile);
  int b = (int)(a.ray_off[(size_t)pos * T2] / a.cap_hits);
  if (b > a.n_bands - 1) b = a.n_bands - 1;
  return b;
}

__global__ void key2_kernel(MsBandArgs a, int ib) {
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= a.P) return;
  const uint64_t key = a.keys[i];
  const uint64_t prim = key & ((1ull << a.prim_bits) - 1ull);
  const int tile = (int)(key >> (32 + a.prim_bits));
  const int tx = tile % a.grid.tiles_x, ty = tile / a.grid.tiles_x;
  const int pos = ms_tile_pos(a.grid, tx, ty);
  const uint64_t band = (uint64_t)band_of_pos(a, pos);
  const uint64_t wave = (uint64_t)ms_wave_of_rank((uint32_t)(i - a.tile_start[tile]), a.wave_c);
  a.key2_a[i] = ((((band << WB) | wave) << a.prim_bits | prim) << ib) | (uint64_t)i;
}

__global__ void pair_banded_kernel(MsBandArgs a, const uint64_t *__restrict__ key2, int ib) {
  const size_t j = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= a.P) return;
  const uint64_t key = key2[j];
  const size_t i = (size_t)(key & ((1ull << ib) - 1ull));
  a.slot_of[i] = (uint32_t)j;
  a.pair_hits_j[j] = a.pair_hits_i[i];
  a.flags[j] = (j == 0 || (key >> ib) != (key2[j - 1] >> ib)) ? 1u : 0u;
}

__global__ void seg_banded_kernel(MsBandArgs a, const uint64_t *__restrict__ key2, int ib) {
  const size_t j = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= a.P) return;
  if (a.flags[j]) {
    const uint32_t g = a.gid[j];
    const uint32_t gk = (uint32_t)(key2[j] >> ib);
    a.grp_key[g] = gk;
    a.grp_prim[g] = gk & ((1u << a.prim_bits) - 1u);
    a.grp_iv0[g] = a.pair_off[j];
  }
  if (j == 0) a.grp_iv0[a.gid[a.P]] = a.pair_off[a.P];
}

__global__ void blocks_banded_kernel(MsBandArgs a) {
  const size_t g = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (g >= a.P) return;
  const uint32_t n_seg = a.gid[a.P];
  uint32_t b = 0;
  if (g < n_seg) b = (uint32_t)(((uint64_t)(a.grp_iv0[g + 1] - a.grp_iv0[g]) * (uint64_t)a.K + MS_ROWS - 1) / MS_ROWS);
  a.grp_blocks[g] = b;
}

__global__ void bw_table_kernel(MsBandArgs a) {
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  const uint32_t n_seg = a.gid[a.P];
  if (t == 0) {
    a.counters[MS_CNT_SEGS] = n_seg;
    a.counters[MS_CNT_BLOCKS] = a.blk_off[n_seg];
  }
  if (t >= a.n_bands * MS_MAX_WAVES) return;
  const uint32_t b = (uint32_t)(t / MS_MAX_WAVES), w = (uint32_t)(t % MS_MAX_WAVES);
  const uint32_t want = (b << WB) | w;
  uint32_t r[2];
#pragma unroll
  for (int e = 0; e < 2; ++e) {     // first segment whose (band, wave) >= want + e
    uint32_t lo = 0, hi = n_seg;
    while (lo < hi) {
      const uint32_t mid = (lo + hi) >> 1;
      if ((a.grp_key[mid] >> a.prim_bits) >= want + (uint32_t)e) hi = mid; else lo = mid + 1;
    }
    r[e] = lo;
  }
  a.bw[t] = make_uint2(r[0], r[1]);
}

// ---- depth waves ----------------------------------------------------------------------------------------------
constexpr unsigned FULL = 0xffffffffu;

__global__ void __launch_bounds__(256) wave_alive_kernel(MsWaveArgs a) {
  const int lane = threadIdx.x & 31;
  const uint32_t warp_g = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, n_warps = (gridDim.x * blockDim.x) >> 5;
  const MsBand band = a.bands[a.band];
  const uint32_t K = (uint32_t)a.K;
  uint32_t n_dead = 0;
  for (uint32_t q = band.q_lo + warp_g; q < band.q_hi; q += n_warps) {
    if (!a.alive[q]) continue;
    const uint32_t off = a.ray_off[q];
    const uint32_t n = a.ray_off[q + 1] - off;
    if (n == 0) continue;
    const MsHit *hits = a.hits + off;
    // The ray's hits are in list order, so those of earlier waves (all evaluated: the ray is alive) are a prefix
    // [0, m).  B = the smallest t_in among the hits still to come: every sample not yet evaluated lies at t >= B
    // (t_k = t_in + (k + 1/2) delta >= t_in in canonical fp32), so the evaluated samples with t < B precede all of
    // them in the (t, primitive, k) order whatever their values turn out to be.
    uint32_t m = 0;
    float B = 3.0e38f;
    for (uint32_t h = lane; h < n; h += 32) {
      const MsHit g = hits[h];
      if (g.wave < a.wave) ++m;
      else B = fminf(B, g.t_in);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      m += __shfl_xor_sync(FULL, m, o);
      B = fminf(B, __shfl_xor_sync(FULL, B, o));
    }
    if (m == n || m == 0) continue;                      // nothing left to drop / nothing evaluated yet
    const float4 *stg = a.staging + (size_t)(off - band.slot0) * K;
    float *hitE = a.hit_e + off;
    // Lane h takes hit h.  A hit whose last sample lies in front of B contributes the product of all its K samples,
    // which is cached per hit the first time it is needed (B only grows from wave to wave, so it stays valid): every
    // staged e is then read about once per frame instead of once per later wave.  A hit that straddles B contributes
    // its samples with t < B and is not cached.
    float p = 1.0f;
    for (uint32_t h0 = 0; h0 < m; h0 += 32) {
      const uint32_t h = h0 + lane;
      const bool have = h < m;
      MsHit g;
      g.prim = 0; g.t_in = 0.f; g.delta = 0.f; g.wave = 0;
      if (have) g = hits[h];
      const float tf = ms_sample_tm(g.t_in, g.delta, 0, a.contact), tl = ms_sample_tm(g.t_in, g.delta, (int)K - 1, a.contact);
      const bool full = have && tl < B, part = have && !full && tf < B;
      float val = 1.0f;
      bool need = part;
      if (full) {
        val = hitE[h];
        need = !(val == val);                             // not cached yet (the buffer starts as NaN)
      }
      unsigned todo = __ballot_sync(FULL, need);
      while (todo) {
        const int hh = __ffs(todo) - 1;
        todo &= todo - 1;
        const float t_in2 = __shfl_sync(FULL, g.t_in, hh), dl2 = __shfl_sync(FULL, g.delta, hh);
        const bool full2 = __shfl_sync(FULL, full ? 1 : 0, hh) != 0;
        float pr = 1.0f;
        for (uint32_t k = lane; k < K; k += 32)
          if (full2 || ms_sample_tm(t_in2, dl2, (int)k, a.contact) < B) pr *= __ldg(&stg[(size_t)(h0 + hh) * K + k].w);
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) pr *= __shfl_xor_sync(FULL, pr, o);
        if (lane == hh) {
          val = pr;
          if (full2) hitE[h] = pr;
        }
      }
      p *= val;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) p *= __shfl_xor_sync(FULL, p, o);
    // the transmittance over that prefix is a product, independent of the order: below t_stop / 2 the ray stops
    // inside the prefix (the factor 2 covers fp32 rounding in the order the final compositing multiplies in)
    if (lane == 0 && p < 0.5f * a.t_stop) {
      a.alive[q] = 0;
      ++n_dead;
    }
  }
  if (lane == 0 && n_dead) atomicAdd(&a.counters[MS_CNT_DEAD_RAYS], n_dead);
}

// The intervals of a (band, wave) are one contiguous run (its segments are consecutive), so the compaction is flat:
// a thread per interval, the survivors appended to their segment's run in a SECOND interval buffer at
// iv0[g] + (a per-segment atomic counter), warp-aggregated.  The order inside a segment is then whatever the
// atomics make it -- it only decides which row of which 128-row block evaluates a sample, never its value or where
// its result is staged (the hit slot), so the image stays bitwise the same.  (A CTA per segment, in place, took
// 145 us per launch on cfg4_opaque: one primitive covering half a band is one CTA walking 1 000 chunks.)
__global__ void __launch_bounds__(256) wave_compact_kernel(MsWaveArgs a) {
  const int lane = threadIdx.x & 31;
  const uint2 r = a.bw[a.band * MS_MAX_WAVES + a.wave];
  if (r.x >= r.y) return;
  const uint32_t lo = a.grp_iv0[r.x], hi = a.grp_iv0[r.y];
  for (uint32_t i0 = lo + (blockIdx.x * blockDim.x + threadIdx.x - lane); i0 < hi; i0 += gridDim.x * blockDim.x) {
    const uint32_t i = i0 + lane;
    const bool valid = i < hi;
    MsInterval iv;
    iv.ray = 0; iv.prim = 0;
    if (valid) iv = a.intervals[i];
    const bool keep = valid && a.alive[(uint32_t)iv.ray] != 0;
    // the interval's segment: the one of this (band, wave) with its primitive (segments are sorted by primitive)
    uint32_t g = r.x;
    if (keep) {
      uint32_t l2 = r.x, h2 = r.y;            // last g with iv0[g] <= i
      while (h2 - l2 > 1) {
        const uint32_t mid = (l2 + h2) >> 1;
        if (a.grp_iv0[mid] <= i) l2 = mid; else h2 = mid;
      }
      g = l2;
    }
    const unsigned act = __ballot_sync(FULL, keep);
    if (keep) {
      const unsigned peers = __match_any_sync(act, g);
      const int leader = __ffs(peers) - 1;
      uint32_t base = 0;
      if (lane == leader) base = atomicAdd(&a.grp_cnt_c[g], (uint32_t)__popc(peers));
      base = __shfl_sync(peers, base, leader);
      a.intervals_c[a.grp_iv0[g] + base + __popc(peers & ((1u << lane) - 1u))] = iv;
    }
  }
}

// single CTA: block counts of the compacted segments, blk_off_c[r.x .. r.y] = their exclusive scan starting at 0
__global__ void __launch_bounds__(1024) wave_scan_kernel(MsWaveArgs a) {
  __shared__ uint32_t wsum[32];
  __shared__ uint32_t carry_s, skip_s;
  const uint2 r = a.bw[a.band * MS_MAX_WAVES + a.wave];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  if (threadIdx.x == 0) { carry_s = 0u; skip_s = 0u; }
  __syncthreads();
  uint32_t skipped = 0;
  for (uint32_t c = r.x; c < r.y; c += 1024) {
    const uint32_t g = c + threadIdx.x;
    uint32_t v = 0;
    if (g < r.y) {
      const uint32_t kept = a.grp_cnt_c[g];
      v = (uint32_t)(((uint64_t)kept * (uint64_t)a.K + MS_ROWS - 1) / MS_ROWS);
      skipped += (a.grp_iv0[g + 1] - a.grp_iv0[g]) - kept;
    }
    uint32_t inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const uint32_t t = __shfl_up_sync(FULL, inc, o);
      if (lane >= o) inc += t;
    }
    if (lane == 31) wsum[warp] = inc;
    __syncthreads();
    if (warp == 0) {
      uint32_t w = wsum[lane];
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const uint32_t t = __shfl_up_sync(FULL, w, o);
        if (lane >= o) w += t;
      }
      wsum[lane] = w;
    }
    __syncthreads();
    const uint32_t carry = carry_s;
    const uint32_t excl = carry + inc - v + (warp > 0 ? wsum[warp - 1] : 0u);
    if (g < r.y) a.blk_off_c[g] = excl;
    __syncthreads();
    if (threadIdx.x == 1023) carry_s = carry + wsum[31];
    __syncthreads();
  }
  if (skipped) atomicAdd(&skip_s, skipped);
  __syncthreads();
  if (threadIdx.x == 0) {
    a.blk_off_c[r.y] = carry_s;
    if (skip_s) atomicAdd(&a.counters[MS_CNT_SKIPPED], skip_s);
  }
}

inline unsigned grid_for(size_t n, int threads) { return (unsigned)((n + threads - 1) / threads); }

}  // namespace

#define MS_CHECK_LAUNCH()                 \
  do {                                    \
    MS_LAUNCHED();                        \
    cudaError_t _e = cudaGetLastError();  \
    if (_e != cudaSuccess) return _e;     \
  } while (0)

cudaError_t ms_tile_stats(const MsGrid &g, const uint32_t *ray_off, const uint32_t *tile_start, uint32_t *counters,
                          cudaStream_t s, uint32_t hit_cap) {
  tile_stats_kernel<<<grid_for((size_t)(g.n_tiles > 0 ? g.n_tiles : 1), 256), 256, 0, s>>>(g, ray_off, tile_start, counters,
                                                                                           hit_cap);
  MS_CHECK_LAUNCH();
  return cudaSuccess;
}

bool ms_order_single_is_small(size_t P, int n_prims) { return P <= OS_MAX && (size_t)n_prims <= OS_MAX; }

cudaError_t ms_order_single(const MsBandArgs &a, cudaStream_t s) {
  cudaError_t e;
  if (ms_order_single_is_small(a.P, a.n_prims)) {
    order_single_small_kernel<<<1, OS_THREADS, 0, s>>>(a);
    MS_CHECK_LAUNCH();
    return cudaSuccess;
  }
  if (a.P > 0) {
    pair_single_kernel<<<grid_for(a.P, 256), 256, 0, s>>>(a);
    MS_CHECK_LAUNCH();
  }
  e = ms_exclusive_scan_u32(a.pair_hits_j, a.pair_off, a.P, a.scan_scratch, s);
  if (e != cudaSuccess) return e;
  seg_single_kernel<<<grid_for((size_t)a.n_prims + 1, 128), 128, 0, s>>>(a);
  MS_CHECK_LAUNCH();
  e = ms_exclusive_scan_u32(a.grp_blocks, a.blk_off, (size_t)a.n_prims, a.scan_scratch, s);
  if (e != cudaSuccess) return e;
  tables_single_kernel<<<1, 1, 0, s>>>(a);
  MS_CHECK_LAUNCH();
  return cudaSuccess;
}

cudaError_t ms_order_banded(const MsBandArgs &a, cudaStream_t s) {
  cudaError_t e;
  int ib = 1;
  while ((1ull << ib) < a.P) ++ib;
  int bb = 1;
  while ((1 << bb) < a.n_bands) ++bb;
  band_table_kernel<<<grid_for((size_t)a.n_bands, 128), 128, 0, s>>>(a);
  MS_CHECK_LAUNCH();
  const uint64_t *key2 = a.key2_a;
  if (a.P > 0) {
    key2_kernel<<<grid_for(a.P, 256), 256, 0, s>>>(a, ib);
    MS_CHECK_LAUNCH();
    uint64_t *sorted = nullptr;
    e = ms_radix_sort_u64(a.key2_a, a.key2_b, a.P, ib, ib + a.prim_bits + WB + bb, a.sort_scratch, &sorted, s);
    if (e != cudaSuccess) return e;
    key2 = sorted;
    pair_banded_kernel<<<grid_for(a.P, 256), 256, 0, s>>>(a, key2, ib);
    MS_CHECK_LAUNCH();
  }
  e = ms_exclusive_scan_u32(a.pair_hits_j, a.pair_off, a.P, a.scan_scratch, s);
  if (e != cudaSuccess) return e;
  e = ms_exclusive_scan_u32(a.flags, a.gid, a.P, a.scan_scratch, s);
  if (e != cudaSuccess) return e;
  if (a.P > 0) {
    seg_banded_kernel<<<grid_for(a.P, 256), 256, 0, s>>>(a, key2, ib);
    MS_CHECK_LAUNCH();
    blocks_banded_kernel<<<grid_for(a.P, 256), 256, 0, s>>>(a);
    MS_CHECK_LAUNCH();
  }
  e = ms_exclusive_scan_u32(a.grp_blocks, a.blk_off, a.P, a.scan_scratch, s);
  if (e != cudaSuccess) return e;
  bw_table_kernel<<<grid_for((size_t)a.n_bands * MS_MAX_WAVES, 128), 128, 0, s>>>(a);
  MS_CHECK_LAUNCH();
  return cudaSuccess;
}

int ms_banded_key_bits(size_t P, int prim_bits, int n_bands, int *group_bits) {
  int ib = 1;
  while ((1ull << ib) < P) ++ib;
  int bb = 1;
  while ((1 << bb) < n_bands) ++bb;
  if (group_bits) *group_bits = prim_bits + WB + bb;
  return ib + prim_bits + WB + bb;
}

cudaError_t ms_wave_prepare(const MsWaveArgs &a, cudaStream_t s) {
  wave_alive_kernel<<<a.n_sm * 8, 256, 0, s>>>(a);
  MS_CHECK_LAUNCH();
  wave_compact_kernel<<<a.n_sm * 8, 256, 0, s>>>(a);
  MS_CHECK_LAUNCH();
  wave_scan_kernel<<<1, 1024, 0, s>>>(a);
  MS_CHECK_LAUNCH();
  return cudaSuccess;
}
