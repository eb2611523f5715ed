// ms_isect.cu -- stage (c): per-tile ray/ellipsoid intersection (NS (c)).  One CTA per tile,
// one thread per pixel; the CTA walks the tile's sorted list and every thread tests its ray
// against the primitive (canonical fp32 chord).  Two passes:
//   count: hits per ray slot and hits per (tile, primitive) pair (by tile-list index)
//   fill : after the scans and the pair ordering of ms_band.cu, each hit is written twice --
//          ray-major      hits[ray_off[q] + h]                       (stage (e) merges these per ray)
//          segment-major  intervals[pair_off[slot_of[i]] + rank]     (stage (d) batches samples by primitive)
// Rays are numbered tile by tile (ms_ray_slot order), so a band of tiles owns a contiguous run of hit slots.
// Deterministic (the only atomics are integer hit counters in shared memory).  Bytes: ~48 B written per
// hit; reads are L1/L2-resident lists.
#include "ms_internal.cuh"

namespace {

constexpr int IS_CHUNK = 32;   // primitives of the tile list staged in shared memory at a time

template <bool FILL>
__global__ void isect_kernel(MsIsectArgs a) {
  // The tile's list is walked in chunks of 32 primitives whose frames (A, o') and pair slots are staged
  // in shared memory by the first 32 threads: no dependent global load and no block barrier per primitive.
  __shared__ float sA[IS_CHUNK][12];        // A (9), o' = A (o - mu) (3)
  __shared__ int sPrim[IS_CHUNK];
  __shared__ uint32_t sBase[IS_CHUNK];      // FILL: pair_off[slot_of[i]]
  __shared__ uint32_t sCnt[IS_CHUNK][33];   // hits of the pair per warp (count pass: [c][32] = total)
  if (FILL && a.guard && a.guard[MS_CNT_OVERFLOW]) return;
  const int T = a.grid.tile;
  const int tile_id = blockIdx.x;
  const int tile_x = tile_id % a.grid.tiles_x, tile_y = tile_id / a.grid.tiles_x;
  const int lx = threadIdx.x % T, ly = threadIdx.x / T;
  const int x = tile_x * T + lx, y = tile_y * T + ly;
  const bool valid = x < a.cam.W && y < a.cam.H;
  const int pos = ms_tile_pos(a.grid, tile_x, tile_y);
  const uint32_t q = (uint32_t)pos * (uint32_t)(T * T) + threadIdx.x;   // ray slot
  if (!FILL && threadIdx.x == 0) a.pos_xy[pos] = make_ushort2((unsigned short)tile_x, (unsigned short)tile_y);
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const uint32_t lt = (1u << lane) - 1u;
  float d[3] = {0.f, 0.f, 1.f};
  if (valid) ms_camera_ray(a.cam, x, y, d);
  const float Kf = (float)a.K;
  const uint64_t pmask = (1ull << a.prim_bits) - 1ull;
  const uint32_t beg = a.tile_start[tile_id], end = a.tile_start[tile_id + 1];
  uint32_t my_hits = 0;
  uint32_t ray_base = 0;
  if (FILL) ray_base = a.ray_off[q];
  for (uint32_t base = beg; base < end; base += IS_CHUNK) {
    const int nc = (int)(end - base < (uint32_t)IS_CHUNK ? end - base : (uint32_t)IS_CHUNK);
    __syncthreads();                        // the previous chunk is done with the staging arrays
    if ((int)threadIdx.x < nc) {
      const int c = threadIdx.x;
      const int prim = (int)(a.keys[base + c] & pmask);
      const float *A = a.A + 9 * (size_t)prim;
      const float *op = a.oprime + 3 * (size_t)prim;
#pragma unroll
      for (int qq = 0; qq < 9; ++qq) sA[c][qq] = __ldg(A + qq);
#pragma unroll
      for (int qq = 0; qq < 3; ++qq) sA[c][9 + qq] = __ldg(op + qq);
      sPrim[c] = prim;
      if (FILL) sBase[c] = a.pair_off[a.slot_of[base + c]];
      if (!FILL) sCnt[c][32] = 0u;
    }
    __syncthreads();
    // pass 1 over the chunk: which primitives does this ray hit; hits per (primitive, warp)
    uint32_t hitmask = 0;
    for (int c = 0; c < nc; ++c) {
      float t_in, delta;
      const bool hit = valid && ms_intersect(sA[c], sA[c] + 9, d, a.cam.t_near, Kf, &t_in, &delta, a.contact);
      const uint32_t ballot = __ballot_sync(0xffffffffu, hit);
      hitmask |= hit ? (1u << c) : 0u;
      if (lane == 0 && ballot) {
        if (FILL) sCnt[c][warp] = __popc(ballot);
        else atomicAdd(&sCnt[c][32], (uint32_t)__popc(ballot));
      } else if (FILL && lane == 0) {
        sCnt[c][warp] = 0u;
      }
    }
    __syncthreads();
    if (!FILL) {
      if ((int)threadIdx.x < nc) a.pair_hits[base + threadIdx.x] = sCnt[threadIdx.x][32];
      my_hits += __popc(hitmask);
    } else {
      // pass 2: the hits are written in list order; rank inside the pair = hits of lower warps + lower lanes
      for (int c = 0; c < nc; ++c) {
        const bool hit = (hitmask >> c) & 1u;
        const uint32_t ballot = __ballot_sync(0xffffffffu, hit);
        if (hit) {
          float t_in = 0.f, delta = 0.f;
          ms_intersect(sA[c], sA[c] + 9, d, a.cam.t_near, Kf, &t_in, &delta, a.contact);
          uint32_t rank = __popc(ballot & lt);
          for (int w = 0; w < warp; ++w) rank += sCnt[c][w];
          const uint32_t slot = ray_base + my_hits;
          MsInterval iv;
          iv.ray = (int)q; iv.t_in = t_in; iv.delta = delta; iv.slot = (int)slot;
          iv.dx = d[0]; iv.dy = d[1]; iv.dz = d[2]; iv.prim = sPrim[c];
          a.intervals[sBase[c] + rank] = iv;
          MsHit h;
          h.prim = sPrim[c]; h.t_in = t_in; h.delta = delta;
          h.wave = ms_wave_of_rank(base + (uint32_t)c - beg, a.wave_c);
          a.hits[slot] = h;
          ++my_hits;
        }
      }
    }
  }
  if (!FILL) a.ray_hits[q] = my_hits;    // 0 for the padding slots of an overhanging tile
}

}  // namespace

cudaError_t ms_isect_count(const MsIsectArgs &a, cudaStream_t s) {
  if (a.grid.n_tiles == 0) return cudaSuccess;
  isect_kernel<false><<<a.grid.n_tiles, a.grid.tile * a.grid.tile, 0, s>>>(a);
  MS_LAUNCHED();
  return cudaGetLastError();
}

cudaError_t ms_isect_fill(const MsIsectArgs &a, cudaStream_t s) {
  if (a.grid.n_tiles == 0) return cudaSuccess;
  isect_kernel<true><<<a.grid.n_tiles, a.grid.tile * a.grid.tile, 0, s>>>(a);
  MS_LAUNCHED();
  return cudaGetLastError();
}
