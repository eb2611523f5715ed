// ms_internal.cuh -- shared declarations of the CUDA path (never included by oracle/).
// Canonical fp32 geometry: every operation below is an explicit
// round-to-nearest intrinsic, so nvcc can never contract a multiply and an add into an FMA.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "../../include/mlpsplat.h"

#define MS_MAX_WIDTH 128
#define MS_MAX_IN 80
#define MS_MAX_OUT 64
#define MS_MAX_K 64
#define MS_ROWS 128  // samples per MLP row block (one TMEM lane / one thread per sample)

struct MsCam {
  float fx, fy, cx, cy;
  float r[9];  // c2w rotation, row-major
  float o[3];  // eye
  float t_near;
  int W, H;
};

// interval of one (ray, primitive) hit in the primitive-major list consumed by stage (d)
struct __align__(16) MsInterval {
  int ray;      // ray slot q (tile-major ray order, ms_ray_slot)
  float t_in;
  float delta;  // (t_out - t_in)/K
  int slot;     // global hit index = ray_off[ray] + h ; sample k lives at staging[slot*K + k]
  float dx, dy, dz;  // unit world-frame ray direction (canonical)
  int prim;          // the primitive (the backward pass walks intervals without their segment)
};

// hit of one ray (ray-major list consumed by stage (e))
struct __align__(16) MsHit {
  int prim;
  float t_in;
  float delta;
  int wave;     // depth wave of the (tile, primitive) pair the hit comes from (0 when waves are off)
};

struct MsMlpShape {
  int n_freq, use_viewdir, n_hidden, width, n_feat;
  int in_dim, out_dim, n_layers, params;
  int mode;  // MS_MODE_LOCAL | MS_MODE_CONTACT
};

// ---------------------------------------------------------------------------------------------
// tile-major ray order, bands and depth waves (DESIGN.md Sec.6 "Bands and waves"; S:Sec.8(f) NEXT-3)
// ---------------------------------------------------------------------------------------------
// Tiles are enumerated macro-tile by macro-tile (G x G tiles, row-major inside), so that a run of
// consecutive tiles is a compact screen region whose primitives overlap; ray slot q = pos*T*T + ly*T + lx.
struct MsGrid {
  int tile, tiles_x, tiles_y, n_tiles, G;   // tile edge, tile grid, macro-tile edge in tiles
  int W, H;
  int tshift;                               // log2(tile)
  const ushort2 *pos_xy;                    // device [n_tiles]: tile (tx, ty) at position pos (written by stage (c))
};
__host__ __device__ __forceinline__ int ms_tile_pos(const MsGrid &g, int tx, int ty) {
  const int mx = tx / g.G, my = ty / g.G;
  const int h = g.tiles_y - my * g.G < g.G ? g.tiles_y - my * g.G : g.G;
  const int w = g.tiles_x - mx * g.G < g.G ? g.tiles_x - mx * g.G : g.G;
  return my * g.G * g.tiles_x + mx * g.G * h + (ty - my * g.G) * w + (tx - mx * g.G);
}
__host__ __device__ __forceinline__ void ms_pos_tile(const MsGrid &g, int pos, int *tx, int *ty) {
  const int my = pos / (g.G * g.tiles_x);
  const int rem = pos - my * g.G * g.tiles_x;
  const int h = g.tiles_y - my * g.G < g.G ? g.tiles_y - my * g.G : g.G;
  const int mcols = (g.tiles_x + g.G - 1) / g.G;
  int mx = rem / (g.G * h);
  if (mx > mcols - 1) mx = mcols - 1;
  const int rem2 = rem - mx * g.G * h;
  const int w = g.tiles_x - mx * g.G < g.G ? g.tiles_x - mx * g.G : g.G;
  *ty = my * g.G + rem2 / w;
  *tx = mx * g.G + rem2 % w;
}
// device: the same through the position table (no divisions)
__device__ __forceinline__ bool ms_slot_pixel_dev(const MsGrid &g, uint32_t q, int *x, int *y) {
  const uint32_t pos = q >> (2 * g.tshift), l = q & ((1u << (2 * g.tshift)) - 1u);
  const ushort2 t = __ldg(g.pos_xy + pos);
  *x = ((int)t.x << g.tshift) + (int)(l & ((1u << g.tshift) - 1u));
  *y = ((int)t.y << g.tshift) + (int)(l >> g.tshift);
  return *x < g.W && *y < g.H;
}
// pixel (x, y) of ray slot q; false for the padding slots of tiles that overhang the image
__host__ __device__ __forceinline__ bool ms_slot_pixel(const MsGrid &g, uint32_t q, int *x, int *y) {
  const int T2 = g.tile * g.tile;
  const int pos = (int)(q / (uint32_t)T2), l = (int)(q - (uint32_t)pos * (uint32_t)T2);
  int tx, ty;
  ms_pos_tile(g, pos, &tx, &ty);
  *x = tx * g.tile + l % g.tile;
  *y = ty * g.tile + l / g.tile;
  return *x < g.W && *y < g.H;
}

// Depth waves: wave w covers the ranks [w C, (w + 1) C) of a tile's sorted list; the last wave takes the rest.
// C == 0: a single wave.
#define MS_MAX_WAVES 6
__host__ __device__ __forceinline__ uint32_t ms_wave_first(int w, int C) {
  return w <= 0 ? 0u : (uint32_t)C * (uint32_t)w;
}
__host__ __device__ __forceinline__ int ms_wave_of_rank(uint32_t r, int C) {
  if (C <= 0) return 0;
  const uint32_t w = r / (uint32_t)C;
  return w < MS_MAX_WAVES - 1 ? (int)w : MS_MAX_WAVES - 1;
}

// One band = a run of consecutive tiles (in ms_tile_pos order) whose hits fill the staging budget.
struct MsBand {
  uint32_t q_lo, q_hi;   // ray slots of the band
  uint32_t slot0;        // first hit slot of the band: sample k of hit slot lives at staging[(slot - slot0) * K + k]
  uint32_t pad;
};
// Segment tables of stage (d): segment g = the intervals of one primitive inside one (band, wave).
struct MsSegs {
  const uint32_t *iv0;      // [n_seg + 1] first interval of the segment
  const uint32_t *cnt;      // [n_seg] intervals of the segment, or NULL: iv0[g + 1] - iv0[g]
  const uint32_t *blk_off;  // [n_seg + 1] exclusive scan of the segments' 128-row block counts (any base)
  const uint32_t *prim;     // [n_seg] primitive of the segment, or NULL: the segment index itself
  const uint2 *range;       // device: segments [x, y) of this launch
  const MsBand *band;       // device: the launch's band
};

// ---------------------------------------------------------------------------------------------
// canonical fp32 primitives
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ float ms_dot3(float a0, float a1, float a2, float b0, float b1, float b2) {
  return __fadd_rn(__fadd_rn(__fmul_rn(a0, b0), __fmul_rn(a1, b1)), __fmul_rn(a2, b2));
}

// ray through the image point (px, py) in pixel units; pixel (x, y) has its centre at (x + 0.5, y + 0.5)
__device__ __forceinline__ void ms_point_ray(const MsCam &c, float px, float py, float *d) {
  float dcx = __fdiv_rn(__fsub_rn(px, c.cx), c.fx);
  float dcy = __fdiv_rn(__fsub_rn(py, c.cy), c.fy);
  float wx = __fadd_rn(__fadd_rn(__fmul_rn(c.r[0], dcx), __fmul_rn(c.r[1], dcy)), c.r[2]);
  float wy = __fadd_rn(__fadd_rn(__fmul_rn(c.r[3], dcx), __fmul_rn(c.r[4], dcy)), c.r[5]);
  float wz = __fadd_rn(__fadd_rn(__fmul_rn(c.r[6], dcx), __fmul_rn(c.r[7], dcy)), c.r[8]);
  float n2 = __fadd_rn(__fadd_rn(__fmul_rn(wx, wx), __fmul_rn(wy, wy)), __fmul_rn(wz, wz));
  float nrm = __fsqrt_rn(n2);
  d[0] = __fdiv_rn(wx, nrm);
  d[1] = __fdiv_rn(wy, nrm);
  d[2] = __fdiv_rn(wz, nrm);
}

__device__ __forceinline__ void ms_camera_ray(const MsCam &c, int x, int y, float *d) {
  ms_point_ray(c, __fadd_rn((float)x, 0.5f), __fadd_rn((float)y, 0.5f), d);
}

// Eq.2's t* = max(-b/a, 0) of primitive (A, op = A (o - mu)) for the ray direction d (the tile-centre order)
__device__ __forceinline__ float ms_contact_t(const float *A, const float *op, const float *d) {
  float d0 = ms_dot3(A[0], A[1], A[2], d[0], d[1], d[2]);
  float d1 = ms_dot3(A[3], A[4], A[5], d[0], d[1], d[2]);
  float d2 = ms_dot3(A[6], A[7], A[8], d[0], d[1], d[2]);
  float a = ms_dot3(d0, d1, d2, d0, d1, d2);
  float b = ms_dot3(op[0], op[1], op[2], d0, d1, d2);
  float ts = __fdiv_rn(-b, a);
  return ts > 0.0f ? ts : 0.0f;
}

// ray / ellipsoid chord in the unit-sphere frame; op = A (o - mu) is per primitive per view.
// contact != 0 (MS_MODE_CONTACT, K = 1): *t_in is the contact point t* = max(-b/a, t_near) of Eq.2
// and *delta the chord length inside the support.
__device__ __forceinline__ bool ms_intersect(const float *A, const float *op, const float *d, float t_near,
                                             float Kf, float *t_in, float *delta, int contact = 0) {
  float d0 = ms_dot3(A[0], A[1], A[2], d[0], d[1], d[2]);
  float d1 = ms_dot3(A[3], A[4], A[5], d[0], d[1], d[2]);
  float d2 = ms_dot3(A[6], A[7], A[8], d[0], d[1], d[2]);
  float a = ms_dot3(d0, d1, d2, d0, d1, d2);
  float b = ms_dot3(op[0], op[1], op[2], d0, d1, d2);
  float c = __fsub_rn(ms_dot3(op[0], op[1], op[2], op[0], op[1], op[2]), 1.0f);
  float disc = __fsub_rn(__fmul_rn(b, b), __fmul_rn(a, c));
  if (!(disc > 0.0f)) return false;
  float sq = __fsqrt_rn(disc);
  float nb = -b;
  float t0 = __fdiv_rn(__fsub_rn(nb, sq), a);
  float t1 = __fdiv_rn(__fadd_rn(nb, sq), a);
  if (!(t1 > t_near)) return false;
  float ti = t0 > t_near ? t0 : t_near;
  float dl = __fdiv_rn(__fsub_rn(t1, ti), Kf);
  if (!(dl > 0.0f)) return false;
  if (contact) {
    const float ts = __fdiv_rn(nb, a);
    ti = ts > t_near ? ts : t_near;
  }
  *t_in = ti;
  *delta = dl;
  return true;
}

__device__ __forceinline__ float ms_sample_t(float t_in, float delta, int k) {
  float kf = __fadd_rn((float)k, 0.5f);
  return __fadd_rn(t_in, __fmul_rn(kf, delta));
}
// sample position of either mode: the contact point itself in MS_MODE_CONTACT
__device__ __forceinline__ float ms_sample_tm(float t_in, float delta, int k, int contact) {
  return contact ? t_in : ms_sample_t(t_in, delta, k);
}

// u = A ((o + t d) - mu)
__device__ __forceinline__ void ms_sample_u(const float *A, const float *mu, const float *o, const float *d,
                                            float t, float *u) {
  float w0 = __fsub_rn(__fadd_rn(o[0], __fmul_rn(t, d[0])), mu[0]);
  float w1 = __fsub_rn(__fadd_rn(o[1], __fmul_rn(t, d[1])), mu[1]);
  float w2 = __fsub_rn(__fadd_rn(o[2], __fmul_rn(t, d[2])), mu[2]);
  u[0] = ms_dot3(A[0], A[1], A[2], w0, w1, w2);
  u[1] = ms_dot3(A[3], A[4], A[5], w0, w1, w2);
  u[2] = ms_dot3(A[6], A[7], A[8], w0, w1, w2);
}

// Eq.7: slot gates g = softmax_k(a_k^T u_s), u_s = clip(R^T delta / s) = clip(-u) with
// u = A (p* - mu) the local coordinate of the contact point; a_k the canonical tetrahedral frame.
__device__ __forceinline__ float4 ms_slot_gates(const float *u) {
  const float c = 0.57735026918962576f;  // 1/sqrt(3)
  const float x = fminf(fmaxf(-u[0], -1.0f), 1.0f), y = fminf(fmaxf(-u[1], -1.0f), 1.0f), z = fminf(fmaxf(-u[2], -1.0f), 1.0f);
  const float z0 = (x + y + z) * c, z1 = (x - y - z) * c, z2 = (-x + y - z) * c, z3 = (-x - y + z) * c;
  const float m = fmaxf(fmaxf(z0, z1), fmaxf(z2, z3));
  const float e0 = expf(z0 - m), e1 = expf(z1 - m), e2 = expf(z2 - m), e3 = expf(z3 - m);
  const float inv = 1.0f / (e0 + e1 + e2 + e3);
  return make_float4(e0 * inv, e1 * inv, e2 * inv, e3 * inv);
}

// kernels launched so far by this host thread (bench.py reports the per-step count)
extern thread_local long long ms_launch_count;
#define MS_LAUNCHED() (++ms_launch_count)

// ---------------------------------------------------------------------------------------------
// host-side launchers (one per stage file)
// ---------------------------------------------------------------------------------------------
// ms_scan.cu: out[i] = sum_{j<i} in[j] for i in [0, n]; out has n+1 entries. scratch >= ms_scan_scratch_elems(n).
size_t ms_scan_scratch_elems(size_t n);
cudaError_t ms_exclusive_scan_u32(const uint32_t *in, uint32_t *out, size_t n, uint32_t *scratch, cudaStream_t s);

// ms_sort.cu: stable LSD radix sort of 64-bit keys on bits [first_bit, n_bits). Result ends in *result (a or b).
size_t ms_sort_scratch_elems(size_t n);
// n_dev != NULL: the number of keys is read from the device (<= n, the capacity the launches are sized for)
cudaError_t ms_radix_sort_u64(uint64_t *a, uint64_t *b, size_t n, int first_bit, int n_bits, uint32_t *scratch,
                              uint64_t **result, cudaStream_t s, const uint32_t *n_dev = nullptr);

// ms_bin.cu
cudaError_t ms_prep_prims(int n, const float *center, const float *quat, const float *scale, float *A, float *M,
                          int *bad, cudaStream_t s);
cudaError_t ms_project(int n, const float *center, const float *A, const float *M, MsCam cam, int tile,
                       float eye_guard, uint32_t *tile_count, int4 *rect, float *z_entry, float *oprime,
                       uint32_t *counters, cudaStream_t s);
// tile_order != 0: the depth field of the key is t*_{i,c} of the tile-centre ray (needs cam, tile, A, oprime)
cudaError_t ms_emit_keys(int n, const uint32_t *emit_off, const int4 *rect, const float *z_entry, int tiles_x,
                         int prim_bits, uint64_t *keys, int tile_order, MsCam cam, int tile, const float *A,
                         const float *oprime, cudaStream_t s, uint32_t cap = 0xffffffffu,
                         uint32_t *counters = nullptr);   // counters: no-sync views (pair count + overflow guard)
// small frames without host synchronisation: stages (a) + (b) in one launch of one CTA (ms_bin.cu)
constexpr int MS_SMALL_PRIMS = 4096;
constexpr size_t MS_BLOCK_SORT_MAX = 16384;   // keys one CTA sorts in one launch (ms_block_sort.cuh: SB_MAX)
bool ms_bin_sort_small_fits(int n_prims, size_t pair_cap);
cudaError_t ms_bin_sort_small(int n, const float *center, const float *A, const float *M, MsCam cam, int tile, float eye_guard,
                              int tiles_x, int n_tiles, int prim_bits, int tile_order, int n_bits, uint32_t cap,
                              uint32_t *tile_count, uint32_t *emit_off, int4 *rect, float *z_entry, float *oprime,
                              uint32_t *counters, uint64_t *keys_a, uint64_t *keys_b, uint32_t *tile_start,
                              uint32_t *pair_hits_j, cudaStream_t s);
cudaError_t ms_tile_ranges(const uint64_t *keys, size_t n_pairs, int n_tiles, int prim_bits, uint32_t *tile_start,
                           cudaStream_t s, const uint32_t *n_dev = nullptr);
// no-sync renders: counters[MS_CNT_P_EFF] = min(*total, cap); MS_CNT_OVERFLOW if the pairs do not fit

// ms_isect.cu
struct MsIsectArgs {
  MsCam cam;
  MsGrid grid;
  int K, prim_bits, contact, wave_c;
  const uint64_t *keys;        // sorted
  const uint32_t *tile_start;  // [n_tiles+1]
  const float *A;              // [N][9]
  const float *oprime;         // [N][3]
  ushort2 *pos_xy;             // [n_tiles] (count pass: out) tile coordinates by position
  uint32_t *pair_hits;         // [P]    (count pass: out)   indexed by tile-list index
  uint32_t *ray_hits;          // [R']   (count pass: out)   indexed by ray slot
  const uint32_t *slot_of;     // [P]    (fill pass: in)     tile-list index -> pair slot of the prim-major order
  const uint32_t *pair_off;    // [P+1]  (fill pass: in)     by pair slot
  const uint32_t *ray_off;     // [R'+1] (fill pass: in)
  const uint32_t *guard;       // counters (MS_CNT_OVERFLOW): a no-sync render that overflowed writes nothing; or NULL
  MsInterval *intervals;       // [n_hits] segment-major (fill pass: out)
  MsHit *hits;                 // [n_hits] ray-major      (fill pass: out)
};
cudaError_t ms_isect_count(const MsIsectArgs &a, cudaStream_t s);
cudaError_t ms_isect_fill(const MsIsectArgs &a, cudaStream_t s);

// ms_band.cu: orders the (tile, primitive) pairs for stage (d) and cuts the frame into bands and waves
struct MsBandArgs {
  MsGrid grid;
  int K, prim_bits, n_prims, wave_c, n_bands;
  uint32_t cap_hits;           // band budget in hits
  size_t P;                    // pairs, or their capacity when P_dev != NULL
  const uint32_t *P_dev;       // no-sync renders: the pair count on the device
  const uint64_t *keys;        // sorted tile lists
  const uint32_t *tile_start;
  const uint32_t *ray_off;     // [R'+1]
  // small frames without host synchronisation (ms_order_single): the CTA that orders the pairs also scans the ray hit
  // counts (fuse_ray_scan: ray_hits [R] -> ray_off_w [R + 1]) and takes the tile statistics (fuse_stats; hit_cap as in
  // ms_tile_stats)
  const uint32_t *ray_hits;
  uint32_t *ray_off_w;
  size_t R;
  uint32_t hit_cap;
  int fuse_ray_scan, fuse_stats;
  const uint32_t *emit_off;    // [N+1]  (single-band path)
  const int4 *rect;            // [N]    (single-band path)
  const uint32_t *pair_hits_i; // [P] by tile-list index
  uint64_t *key2_a, *key2_b;   // [P]
  uint32_t *sort_scratch;
  uint32_t *scan_scratch;
  uint32_t *slot_of;           // [P]
  uint32_t *pair_hits_j;       // [P+1] by pair slot
  uint32_t *pair_off;          // [P+2]
  uint32_t *flags, *gid;       // [P+2] group boundary flags and their exclusive scan
  uint32_t *grp_key;           // [n_seg_cap] (band, wave, prim) of segment g
  uint32_t *grp_prim;          // [n_seg_cap]
  uint32_t *grp_iv0;           // [n_seg_cap + 1]
  uint32_t *grp_blocks;        // [n_seg_cap + 1]
  uint32_t *blk_off;           // [n_seg_cap + 2]
  uint2 *bw;                   // [n_bands * MS_MAX_WAVES] segment range of (band, wave)
  MsBand *bands;               // [n_bands]
  uint32_t *counters;          // device counters (MsCounter)
};
// device counters of a view (uint32 each; HITS and PAIRS are 64-bit little-endian pairs, so a total that wrapped the
// 32-bit scans is seen)
enum MsCounter { MS_CNT_SEGS = 0, MS_CNT_BLOCKS, MS_CNT_HITS, MS_CNT_HITS_HI, MS_CNT_PAIRS, MS_CNT_PAIRS_HI,
                 MS_CNT_MAX_TILE_HITS, MS_CNT_MAX_LIST, MS_CNT_SKIPPED, MS_CNT_DEAD_RAYS, MS_CNT_VISIBLE,
                 MS_CNT_STOPPED_RAYS, MS_CNT_P_EFF, MS_CNT_OVERFLOW, MS_CNT_N,
                 MS_CNT_STICKY_OVERFLOW = MS_CNT_N + 1 /* not cleared per view: read and cleared by the host */ };
// after the ray_off scan: the hit total (64-bit), the largest tile's hit count and the longest tile list into counters
cudaError_t ms_tile_stats(const MsGrid &g, const uint32_t *ray_off, const uint32_t *tile_start, uint32_t *counters,
                          cudaStream_t s, uint32_t hit_cap = 0);
// one band, one wave: segments = primitives in emission order (the layout of small frames)
// one CTA orders the pairs of such a frame; it can take the ray scan and the tile statistics along (MsBandArgs)
bool ms_order_single_is_small(size_t P, int n_prims);
constexpr size_t MS_SMALL_RAYS = 65536;   // ray slots one CTA scans along the way
cudaError_t ms_order_single(const MsBandArgs &a, cudaStream_t s);
// bands x waves: pairs sorted by (band, wave, primitive), segments = runs of equal (band, wave, primitive)
cudaError_t ms_order_banded(const MsBandArgs &a, cudaStream_t s);
// bits of the (band, wave, primitive, pair index) sort key; the (band, wave, primitive) part must fit 32 bits
int ms_banded_key_bits(size_t P, int prim_bits, int n_bands, int *group_bits);

// depth waves (real early termination): before wave w >= 1 of a band, rays whose transmittance over the samples
// in front of the wave's nearest possible sample is already below t_stop/2 are dropped, the wave's interval lists
// are compacted and its block offsets rebuilt
struct MsWaveArgs {
  MsGrid grid;
  int K, prim_bits, wave_c, band, wave, contact;
  float t_stop, margin;
  const uint64_t *keys;
  const uint32_t *tile_start;
  const uint32_t *ray_off;
  const MsHit *hits;
  const float4 *staging;
  const MsBand *bands;
  const uint2 *bw;
  uint8_t *alive;              // [R'] 1 = the ray still needs its later hits
  float *hit_e;                // [n_hits] product of a hit's K staged e, cached by the wave check (NaN = not yet)
  const MsInterval *intervals; // the frame's interval lists (stage (c))
  MsInterval *intervals_c;     // second buffer: the compacted lists of the waves >= 1
  const uint32_t *grp_iv0;
  uint32_t *grp_cnt_c;         // [n_seg_cap] compacted interval count (zeroed once per frame)
  uint32_t *grp_blocks_c;      // [n_seg_cap] compacted 128-row block count
  uint32_t *blk_off_c;         // [n_seg_cap + 2] block offsets of the compacted wave (relative to its first segment)
  uint32_t *counters;
  int n_sm;
};
cudaError_t ms_wave_prepare(const MsWaveArgs &a, cudaStream_t s);

// ms_mlp_f32.cu
struct MsMlpArgs {
  MsMlpShape shape;
  MsCam cam;
  int K;
  float falloff;                  // contact mode: g = exp(-falloff |p* - mu|^2_Lambda)
  const float *center, *A;
  const float *weights_f32;       // [N][params]
  MsSegs segs;
  uint32_t n_blocks_hint;         // blocks of the launch if the host knows them, else 0
  const MsInterval *intervals;
  float4 *staging;                // band-local: [(slot - slot0)*K + k] (r,g,b,e)
  void *staging_feat;             // same indexing x n_feat, or NULL: fp32, or fp16 when feat_half
  int feat_half;                  // tensor path, n_feat == 32: features staged as fp16 rows of 64 B
  float4 *staging_gate;           // slot gates g_k of Eq.7 (contact mode) or NULL
};
cudaError_t ms_mlp_f32(const MsMlpArgs &a, cudaStream_t s);

// ms_composite.cu
struct MsCompositeArgs {
  MsGrid grid;
  int K, n_feat, contact;
  int tile_order;        // contact mode: the hits are already in the tile's shared order -- no per-ray merge
  float t_stop;
  MsBand band;           // ray slots and staging origin of this launch
  const uint32_t *ray_off;  // [R'+1]
  const MsHit *hits;
  const float4 *staging;
  const void *staging_feat;
  int feat_half;         // staging_feat holds fp16 rows (tensor path, n_feat == 32)
  const float4 *gates;   // slot gates (Eq.7) or NULL
  float4 *coef;          // (T alpha) g_k per hit: composite_kernel<2> -> slot_feature_tile_kernel
  const float *slots;    // [N][4][c_f] slot embeddings
  int c_f;
  // Eq.7 features, tile-owned accumulation (slot_feature_tile_kernel): the sorted tile lists and the hits per pair
  const uint64_t *keys;
  const uint32_t *tile_start;
  const uint32_t *pair_hits;   // by tile-list index, or NULL
  int prim_bits;
  uint32_t *counters;    // MS_CNT_STOPPED_RAYS
  uint32_t *dbg_ord;     // MS_FLAG_KEEP_ORDER: [n_hits*K] sample index (h*K + k) by (hit slot of the ray)*K + rank
  float *out_rgb, *out_alpha, *out_feat;
};
cudaError_t ms_composite(const MsCompositeArgs &a, cudaStream_t s);

// ---- backward pass (S:Sec.8(f) NEXT-4; ms_backward.cu, ms_composite.cu) -----------------------------------------
struct MsCompositeBwdArgs {
  MsGrid grid;
  int K;
  float t_stop;
  const uint32_t *ray_off;
  const MsHit *hits;
  const float4 *staging;   // whole frame (one band): (r, g, b, e) at slot * K + k
  const float *d_rgb;      // [H][W][3] dL/dC
  uint32_t *ord;           // [n_samples] scratch: sample index by (ray's first sample + rank)
  float4 *gstage;          // [n_samples] out: (dL/dc_r, dL/dc_g, dL/dc_b, dL/de) at slot * K + k
};
cudaError_t ms_composite_bwd(const MsCompositeBwdArgs &a, cudaStream_t s);

struct MsMlpBwdArgs {
  MsMlpShape shape;
  MsCam cam;
  int K, n_prims;
  size_t n_hits;
  const float *center, *A, *quat, *scale;
  const float *weights_f32;
  MsSegs segs;
  const MsInterval *intervals;
  const float4 *staging;
  const float4 *gstage;
  float *ivgrad;           // [n_hits][8] scratch, zeroed: dL/d(o'[3], d'[3], t_in, delta) of every interval
  float *gA;               // [N][9] scratch, zeroed: dL/dA
  float *g_weights;        // [N][params]  += dL/dtheta
  float *g_center;         // [N][3]       += dL/dmu
  float *g_quat;           // [N][4]       += dL/dq
  float *g_scale;          // [N][3]       += dL/ds
};
// smem bytes the MLP backward kernel needs for this shape (0: shape not covered)
size_t ms_mlp_bwd_smem(const MsMlpShape &sh);
cudaError_t ms_mlp_bwd(const MsMlpBwdArgs &a, cudaStream_t s);
