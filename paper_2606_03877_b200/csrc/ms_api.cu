// ms_api.cu -- the C ABI of include/mlpsplat.h: scene handle, scratch management and the
// per-view stage sequence (a) project/emit -> (b) sort/ranges -> (c) intersect count/scan/fill
// -> (d) grouped MLP -> (e) merge + composite.  Host code only orchestrates; every step of the
// path runs in the kernels of this directory.
#include <math.h>
#include <new>
#include <stdlib.h>
#include <string.h>
#include <vector>

#include "ms_internal.cuh"
#include "ms_mlp_tc.cuh"

thread_local long long ms_launch_count = 0;

namespace {

struct Buf {
  void *p = nullptr;
  size_t cap = 0;
};

}  // namespace

struct ms_scene {
  int device = 0;
  int n = 0;
  int dtype = MS_F32;
  MsMlpShape shape{};
  int last_cuda = 0;
  // scene-lifetime device data
  float *center = nullptr, *quat = nullptr, *scale = nullptr, *A = nullptr, *M = nullptr;
  float *weights_f32 = nullptr;
  MsTcWeights tc{};  // packed bf16 image for the tensor path (may be empty)
  int slot_cf = 0;           // Eq.7 slot embeddings: width C_f (0 = none)
  float *slots = nullptr;    // device [N][4][slot_cf]
  // per-view scratch
  Buf tile_count, emit_off, rect, z_entry, oprime, keys_a, keys_b, sort_scratch, tile_start, pair_hits, pair_off,
      ray_hits, ray_off, scan_scratch, prim_start, prim_blocks, blk_off, intervals, hits, staging, staging_feat, staging_gate, staging_coef,
      host_rgb, host_alpha, host_feat, dbg;
  uint32_t *pinned = nullptr;  // [4] host-pinned readback
  cudaEvent_t ev[MS_N_STAGES + 1] = {};
  bool ev_valid = false;
  bool ev_pending = false;         // events of the last view not yet added to stage_sum
  double stage_sum[MS_N_STAGES] = {};
  int64_t stage_views = 0;
  // last view
  ms_stats stats{};
  bool debug_valid = false;
  int dbg_H = 0, dbg_W = 0, dbg_tile = 0, dbg_K = 0, dbg_prim_bits = 0, dbg_n_tiles = 0;
  uint64_t *dbg_keys = nullptr;
  float dbg_t_stop = 0.f;
  int dbg_tile_order = 0;
};

namespace {

#define CK(call)                                    \
  do {                                              \
    cudaError_t _e = (call);                        \
    if (_e != cudaSuccess) {                        \
      sc->last_cuda = (int)_e;                      \
      return _e == cudaErrorMemoryAllocation ? MS_ERR_OUT_OF_MEMORY : MS_ERR_CUDA; \
    }                                               \
  } while (0)

int ensure(ms_scene *sc, Buf &b, size_t bytes) {
  if (bytes <= b.cap && b.p) return MS_OK;
  if (b.p) {
    cudaFree(b.p);
    b.p = nullptr;
    b.cap = 0;
  }
  size_t want = bytes + bytes / 4 + 256;
  cudaError_t e = cudaMalloc(&b.p, want);
  if (e != cudaSuccess) {
    (void)cudaGetLastError();
    e = cudaMalloc(&b.p, bytes + 256);  // retry without slack
    want = bytes + 256;
  }
  if (e != cudaSuccess) {
    sc->last_cuda = (int)e;
    b.p = nullptr;
    (void)cudaGetLastError();
    return MS_ERR_OUT_OF_MEMORY;
  }
  b.cap = want;
  return MS_OK;
}

#define ENS(buf, bytes)                         \
  do {                                          \
    int _r = ensure(sc, buf, (size_t)(bytes));  \
    if (_r != MS_OK) return _r;                 \
  } while (0)

size_t scratch_total(const ms_scene *sc) {
  const Buf *all[] = {&sc->tile_count, &sc->emit_off, &sc->rect, &sc->z_entry, &sc->oprime, &sc->keys_a, &sc->keys_b,
                      &sc->sort_scratch, &sc->tile_start, &sc->pair_hits, &sc->pair_off, &sc->ray_hits, &sc->ray_off,
                      &sc->scan_scratch, &sc->prim_start, &sc->prim_blocks, &sc->blk_off, &sc->intervals, &sc->hits,
                      &sc->staging, &sc->staging_feat, &sc->staging_gate, &sc->staging_coef};
  size_t t = 0;
  for (const Buf *b : all) t += b->cap;
  return t;
}

int ceil_log2(uint64_t v) {
  int b = 0;
  while ((1ull << b) < v) ++b;
  return b;
}

float round_bf16(float f) {
  uint32_t u;
  memcpy(&u, &f, 4);
  if ((u & 0x7f800000u) == 0x7f800000u) return f;  // inf / nan unchanged
  uint32_t lsb = (u >> 16) & 1u;
  u = (u + 0x7fffu + lsb) & 0xffff0000u;
  memcpy(&f, &u, 4);
  return f;
}

// Adds the stage times of the previous view to the running sums.  Called right after a stream
// synchronisation (so the events have completed) -- never adds a synchronisation of its own.
void harvest_stage_times(ms_scene *sc) {
  if (!sc->ev_pending) return;
  sc->ev_pending = false;
  for (int i = 0; i < MS_N_STAGES; ++i) {
    float ms = 0.f;
    if (cudaEventElapsedTime(&ms, sc->ev[i], sc->ev[i + 1]) != cudaSuccess) {
      (void)cudaGetLastError();
      return;
    }
    sc->stage_sum[i] += ms;
  }
  sc->stage_views += 1;
}

MsCam make_cam(const ms_camera *c, int H, int W) {
  MsCam m;
  m.fx = c->fx; m.fy = c->fy; m.cx = c->cx; m.cy = c->cy;
  for (int r = 0; r < 3; ++r) {
    for (int k = 0; k < 3; ++k) m.r[3 * r + k] = c->c2w[4 * r + k];
    m.o[r] = c->c2w[4 * r + 3];
  }
  m.t_near = c->t_near;
  m.W = W; m.H = H;
  return m;
}

int render_view(ms_scene *sc, const ms_camera *camera, int H, int W, const ms_opts *opts, float *out_rgb,
                float *out_alpha, float *out_feat) {
  cudaStream_t st = (cudaStream_t)opts->stream;
  const int tile = opts->tile == 0 ? 16 : opts->tile;
  const int K = opts->K;
  const int N = sc->n;
  const int tiles_x = (W + tile - 1) / tile, tiles_y = (H + tile - 1) / tile;
  const int64_t n_tiles64 = (int64_t)tiles_x * tiles_y;
  const int64_t R64 = (int64_t)H * W;
  if (R64 >= (1ll << 31) - 1) return MS_ERR_UNSUPPORTED_SHAPE;
  const int n_tiles = (int)n_tiles64;
  const int R = (int)R64;
  const int prim_bits = ceil_log2((uint64_t)N) < 1 ? 1 : ceil_log2((uint64_t)N);
  const int tile_bits = ceil_log2((uint64_t)n_tiles) < 1 ? 1 : ceil_log2((uint64_t)n_tiles);
  if (prim_bits + tile_bits > 32) return MS_ERR_UNSUPPORTED_SHAPE;

  int path = opts->path;
  if (path == MS_PATH_AUTO)
    path = (sc->dtype == MS_BF16 && sc->tc.valid) ? MS_PATH_BF16_TC : MS_PATH_FP32;
  if (path == MS_PATH_BF16_TC && !sc->tc.valid) return MS_ERR_UNSUPPORTED_SHAPE;
  if (path != MS_PATH_BF16_TC && path != MS_PATH_FP32) return MS_ERR_INVALID_ARG;

  const bool timing = (opts->flags & MS_FLAG_STAGE_TIMES) != 0;
  sc->debug_valid = false;
  const MsCam cam = make_cam(camera, H, W);
  const long long launches0 = ms_launch_count;
  if (sc->ev_pending) {  // the previous view's events must be read before they are re-recorded
    CK(cudaEventSynchronize(sc->ev[MS_N_STAGES]));
    harvest_stage_times(sc);
  }
  sc->ev_valid = false;

  // ---- (a) projection + key emit ----------------------------------------------------------
  if (timing) CK(cudaEventRecord(sc->ev[0], st));
  ENS(sc->tile_count, (size_t)N * 4);
  ENS(sc->emit_off, (size_t)(N + 1) * 4);
  ENS(sc->rect, (size_t)N * sizeof(int4));
  ENS(sc->z_entry, (size_t)N * 4);
  ENS(sc->oprime, (size_t)N * 12);
  ENS(sc->scan_scratch, (ms_scan_scratch_elems((size_t)R > (size_t)N ? (size_t)R : (size_t)N) + 16) * 4);
  CK(ms_project(N, sc->center, sc->A, sc->M, cam, tile, tiles_x, tiles_y, (uint32_t *)sc->tile_count.p,
                (int4 *)sc->rect.p, (float *)sc->z_entry.p, (float *)sc->oprime.p, st));
  CK(ms_exclusive_scan_u32((uint32_t *)sc->tile_count.p, (uint32_t *)sc->emit_off.p, (size_t)N,
                           (uint32_t *)sc->scan_scratch.p, st));
  CK(cudaMemcpyAsync(sc->pinned, (uint32_t *)sc->emit_off.p + N, 4, cudaMemcpyDeviceToHost, st));
  CK(cudaStreamSynchronize(st));
  const size_t P = sc->pinned[0];
  if (P >= (1ull << 31)) return MS_ERR_UNSUPPORTED_SHAPE;
  ENS(sc->keys_a, (P + 1) * 8);
  ENS(sc->keys_b, (P + 1) * 8);
  ENS(sc->sort_scratch, ms_sort_scratch_elems(P) * 4);
  ENS(sc->tile_start, (size_t)(n_tiles + 1) * 4);
  ENS(sc->pair_hits, (P + 1) * 4);
  ENS(sc->pair_off, (P + 2) * 4);
  if (ms_scan_scratch_elems(P) + 16 > sc->scan_scratch.cap / 4) ENS(sc->scan_scratch, (ms_scan_scratch_elems(P) + 16) * 4);
  const int tile_order = (opts->flags & MS_FLAG_TILE_ORDER) != 0;
  CK(ms_emit_keys(N, (uint32_t *)sc->emit_off.p, (int4 *)sc->rect.p, (float *)sc->z_entry.p, tiles_x, prim_bits,
                  (uint64_t *)sc->keys_a.p, tile_order, cam, tile, sc->A, (float *)sc->oprime.p, st));

  // ---- (b) radix sort + tile ranges -------------------------------------------------------
  if (timing) CK(cudaEventRecord(sc->ev[1], st));
  uint64_t *sorted = nullptr;
  // stage (a) emits the keys primitive by primitive, i.e. already ordered by the id in their low prim_bits bits;
  // the sort is stable, so only the (tile | depth) bits above them need passes
  CK(ms_radix_sort_u64((uint64_t *)sc->keys_a.p, (uint64_t *)sc->keys_b.p, P, prim_bits, prim_bits + 32 + tile_bits,
                       (uint32_t *)sc->sort_scratch.p, &sorted, st));
  CK(ms_tile_ranges(sorted, P, n_tiles, prim_bits, (uint32_t *)sc->tile_start.p, st));

  // ---- (c) intersection: count, scans, fill -----------------------------------------------
  if (timing) CK(cudaEventRecord(sc->ev[2], st));
  ENS(sc->ray_hits, (size_t)R * 4);
  ENS(sc->ray_off, (size_t)(R + 1) * 4);
  ENS(sc->prim_start, (size_t)(N + 1) * 4);
  ENS(sc->prim_blocks, (size_t)(N + 1) * 4);
  ENS(sc->blk_off, (size_t)(N + 2) * 4);
  MsIsectArgs ia;
  ia.cam = cam; ia.tile = tile; ia.tiles_x = tiles_x; ia.n_tiles = n_tiles; ia.K = K; ia.prim_bits = prim_bits;
  ia.contact = sc->shape.mode == MS_MODE_CONTACT;
  ia.keys = sorted; ia.tile_start = (uint32_t *)sc->tile_start.p; ia.A = sc->A; ia.oprime = (float *)sc->oprime.p;
  ia.rect = (int4 *)sc->rect.p; ia.emit_off = (uint32_t *)sc->emit_off.p;
  ia.pair_hits = (uint32_t *)sc->pair_hits.p; ia.ray_hits = (uint32_t *)sc->ray_hits.p;
  ia.pair_off = (uint32_t *)sc->pair_off.p; ia.ray_off = (uint32_t *)sc->ray_off.p;
  ia.intervals = nullptr; ia.hits = nullptr;
  CK(ms_isect_count(ia, st));
  CK(ms_exclusive_scan_u32((uint32_t *)sc->pair_hits.p, (uint32_t *)sc->pair_off.p, P, (uint32_t *)sc->scan_scratch.p, st));
  CK(ms_exclusive_scan_u32((uint32_t *)sc->ray_hits.p, (uint32_t *)sc->ray_off.p, (size_t)R,
                           (uint32_t *)sc->scan_scratch.p, st));
  CK(ms_prim_blocks(N, (uint32_t *)sc->emit_off.p, (uint32_t *)sc->pair_off.p, K, (uint32_t *)sc->prim_start.p,
                    (uint32_t *)sc->prim_blocks.p, st));
  CK(ms_exclusive_scan_u32((uint32_t *)sc->prim_blocks.p, (uint32_t *)sc->blk_off.p, (size_t)N,
                           (uint32_t *)sc->scan_scratch.p, st));
  CK(cudaMemcpyAsync(sc->pinned + 1, (uint32_t *)sc->ray_off.p + R, 4, cudaMemcpyDeviceToHost, st));
  CK(cudaMemcpyAsync(sc->pinned + 2, (uint32_t *)sc->blk_off.p + N, 4, cudaMemcpyDeviceToHost, st));
  CK(cudaMemcpyAsync(sc->pinned + 3, (uint32_t *)sc->pair_off.p + P, 4, cudaMemcpyDeviceToHost, st));
  CK(cudaStreamSynchronize(st));
  const size_t n_hits = sc->pinned[1];
  const uint32_t n_blocks = sc->pinned[2];
  if (sc->pinned[3] != sc->pinned[1]) return MS_ERR_CUDA;  // the two scans must agree
  if (n_hits >= (1ull << 31)) return MS_ERR_UNSUPPORTED_SHAPE;
  const size_t n_samples = n_hits * (size_t)K;
  const bool want_feat = sc->shape.n_feat > 0 && out_feat != nullptr;
  ENS(sc->intervals, (n_hits + 1) * sizeof(MsInterval));
  ENS(sc->hits, (n_hits + 1) * sizeof(MsHit));
  ENS(sc->staging, (n_samples + 1) * sizeof(float4));
  if (want_feat) ENS(sc->staging_feat, (n_samples + 1) * (size_t)sc->shape.n_feat * 4);
  const bool want_slots = sc->slot_cf > 0 && out_feat != nullptr;   // Eq.7 features (contact mode, K = 1)
  if (want_slots) ENS(sc->staging_gate, (n_samples + 1) * sizeof(float4));
  if (want_slots) ENS(sc->staging_coef, (n_samples + 1) * sizeof(float4));
  ia.intervals = (MsInterval *)sc->intervals.p;
  ia.hits = (MsHit *)sc->hits.p;
  CK(ms_isect_fill(ia, st));

  // ---- (d) grouped per-primitive MLP ------------------------------------------------------
  if (timing) CK(cudaEventRecord(sc->ev[3], st));
  MsMlpArgs ma;
  ma.shape = sc->shape; ma.cam = cam; ma.K = K; ma.n_prims = N;
  ma.center = sc->center; ma.A = sc->A; ma.weights_f32 = sc->weights_f32;
  ma.prim_start = (uint32_t *)sc->prim_start.p; ma.blk_off = (uint32_t *)sc->blk_off.p; ma.n_blocks = n_blocks;
  ma.intervals = (MsInterval *)sc->intervals.p;
  ma.staging = (float4 *)sc->staging.p;
  ma.staging_feat = want_feat ? (float *)sc->staging_feat.p : nullptr;
  ma.staging_gate = want_slots ? (float4 *)sc->staging_gate.p : nullptr;
  if (path == MS_PATH_BF16_TC) CK(ms_mlp_tc(sc->tc, ma, st));
  else CK(ms_mlp_f32(ma, st));

  // ---- (e) merge + composite ---------------------------------------------------------------
  if (timing) CK(cudaEventRecord(sc->ev[4], st));
  MsCompositeArgs ca;
  ca.n_rays = R; ca.K = K; ca.n_feat = sc->shape.n_feat; ca.t_stop = opts->t_stop;
  ca.contact = sc->shape.mode == MS_MODE_CONTACT;
  ca.tile_order = tile_order;
  ca.ray_off = (uint32_t *)sc->ray_off.p; ca.hits = (MsHit *)sc->hits.p; ca.staging = (float4 *)sc->staging.p;
  ca.staging_feat = want_feat ? (float *)sc->staging_feat.p : nullptr;
  ca.gates = want_slots ? (const float4 *)sc->staging_gate.p : nullptr;
  ca.coef = want_slots ? (float4 *)sc->staging_coef.p : nullptr;
  ca.slots = sc->slots; ca.c_f = sc->slot_cf;
  ca.out_rgb = out_rgb; ca.out_alpha = out_alpha; ca.out_feat = (want_feat || want_slots) ? out_feat : nullptr;
  CK(ms_composite(ca, st));
  if (timing) {
    CK(cudaEventRecord(sc->ev[5], st));
    sc->ev_valid = true;
    sc->ev_pending = true;
  }
  sc->stats.n_launches = (int64_t)(ms_launch_count - launches0);

  sc->stats.n_pairs = (int64_t)P;
  sc->stats.n_intervals = (int64_t)n_hits;
  sc->stats.n_samples = (int64_t)n_samples;
  sc->stats.n_blocks = (int64_t)n_blocks;
  sc->stats.n_visible = -1;
  sc->stats.scratch_bytes = (int64_t)scratch_total(sc);
  if (opts->flags & MS_FLAG_KEEP_DEBUG) {
    sc->debug_valid = true;
    sc->dbg_H = H; sc->dbg_W = W; sc->dbg_tile = tile; sc->dbg_K = K; sc->dbg_prim_bits = prim_bits;
    sc->dbg_n_tiles = n_tiles; sc->dbg_keys = sorted; sc->dbg_t_stop = opts->t_stop;
    sc->dbg_tile_order = tile_order;
  }
  return MS_OK;
}

int check_render_args(ms_scene *sc, const ms_camera *cams, int n_views, int H, int W, const ms_opts *o, const void *rgb,
                      const void *alpha) {
  if (!sc || !cams || !o || !rgb || !alpha || n_views < 1 || H < 1 || W < 1) return MS_ERR_INVALID_ARG;
  if (o->K < 1 || o->K > MS_MAX_K || !(o->t_stop >= 0.0f)) return MS_ERR_INVALID_ARG;
  if (sc->shape.mode == MS_MODE_CONTACT && o->K != 1) return MS_ERR_INVALID_ARG;   // one evaluation per hit
  if ((o->flags & MS_FLAG_TILE_ORDER) && sc->shape.mode != MS_MODE_CONTACT) return MS_ERR_INVALID_ARG;
  if (o->tile != 0 && o->tile != 8 && o->tile != 16 && o->tile != 32) return MS_ERR_INVALID_ARG;
  for (int v = 0; v < n_views; ++v)
    if (!(cams[v].fx > 0.f) || !(cams[v].fy > 0.f) || !(cams[v].t_near >= 0.f)) return MS_ERR_INVALID_ARG;
  return MS_OK;
}

void free_buf(Buf &b) {
  if (b.p) cudaFree(b.p);
  b.p = nullptr;
  b.cap = 0;
}

}  // namespace

extern "C" {

int ms_scene_create(const ms_prims *prims, const ms_mlp *mlp, ms_scene **out) {
  if (!prims || !mlp || !out) return MS_ERR_INVALID_ARG;
  *out = nullptr;
  if (prims->n < 1 || !prims->center || !prims->quat || !prims->scale || !mlp->weights) return MS_ERR_INVALID_ARG;
  if (mlp->n_freq < 0 || mlp->n_hidden < 1 || mlp->n_hidden > 4 || mlp->width < 1 || mlp->n_feat < 0)
    return MS_ERR_INVALID_ARG;
  if (mlp->dtype != MS_F32 && mlp->dtype != MS_BF16) return MS_ERR_INVALID_ARG;
  MsMlpShape sh;
  sh.n_freq = mlp->n_freq; sh.use_viewdir = mlp->use_viewdir ? 1 : 0; sh.n_hidden = mlp->n_hidden;
  sh.width = mlp->width; sh.n_feat = mlp->n_feat;
  if (mlp->mode != MS_MODE_LOCAL && mlp->mode != MS_MODE_CONTACT) return MS_ERR_INVALID_ARG;
  if (mlp->mode == MS_MODE_CONTACT && (mlp->n_freq < 1 || mlp->use_viewdir)) return MS_ERR_INVALID_ARG;
  sh.mode = mlp->mode;
  sh.in_dim = sh.mode == MS_MODE_CONTACT ? 12 * sh.n_freq : 3 + 6 * sh.n_freq + (sh.use_viewdir ? 3 : 0);
  sh.out_dim = 4 + sh.n_feat;
  sh.n_layers = sh.n_hidden + 1;
  if (sh.width > MS_MAX_WIDTH || sh.in_dim > MS_MAX_IN || sh.out_dim > MS_MAX_OUT) return MS_ERR_UNSUPPORTED_SHAPE;
  int params = 0, in = sh.in_dim;
  for (int l = 0; l < sh.n_layers; ++l) {
    int o = l == sh.n_layers - 1 ? sh.out_dim : sh.width;
    params += in * o + o;
    in = o;
  }
  sh.params = params;
  if ((size_t)params * sizeof(float) > 200 * 1024) return MS_ERR_UNSUPPORTED_SHAPE;
  const size_t n = (size_t)prims->n;
  if (mlp->n_weights != n * (size_t)params) return MS_ERR_INVALID_ARG;

  ms_scene *sc = new (std::nothrow) ms_scene();
  if (!sc) return MS_ERR_OUT_OF_MEMORY;
  sc->n = prims->n;
  sc->dtype = mlp->dtype;
  sc->shape = sh;
  int rc = MS_OK;
  int *d_bad = nullptr;
  std::vector<float> w;
  auto fail = [&](int code) {
    if (d_bad) cudaFree(d_bad);
    ms_scene_destroy(sc);
    return code;
  };
#define CKC(call)                                                                        \
  do {                                                                                   \
    cudaError_t _e = (call);                                                             \
    if (_e != cudaSuccess) {                                                             \
      (void)cudaGetLastError();                                                          \
      return fail(_e == cudaErrorMemoryAllocation ? MS_ERR_OUT_OF_MEMORY : MS_ERR_CUDA); \
    }                                                                                    \
  } while (0)
  CKC(cudaGetDevice(&sc->device));
  CKC(cudaMalloc(&sc->center, n * 12));
  CKC(cudaMalloc(&sc->quat, n * 16));
  CKC(cudaMalloc(&sc->scale, n * 12));
  CKC(cudaMalloc(&sc->A, n * 36));
  CKC(cudaMalloc(&sc->M, n * 36));
  CKC(cudaMalloc(&sc->weights_f32, n * (size_t)params * 4));
  CKC(cudaMalloc(&d_bad, 4));
  CKC(cudaMemset(d_bad, 0, 4));
  CKC(cudaMemcpy(sc->center, prims->center, n * 12, cudaMemcpyHostToDevice));
  CKC(cudaMemcpy(sc->quat, prims->quat, n * 16, cudaMemcpyHostToDevice));
  CKC(cudaMemcpy(sc->scale, prims->scale, n * 12, cudaMemcpyHostToDevice));
  try {
    w.assign(mlp->weights, mlp->weights + n * (size_t)params);
  } catch (...) {
    return fail(MS_ERR_OUT_OF_MEMORY);
  }
  if (mlp->dtype == MS_BF16) {  // Q18: weight matrices to bf16 (RNE); biases stay fp32
    for (size_t i = 0; i < n; ++i) {
      float *p = w.data() + i * (size_t)params;
      int li = sh.in_dim;
      for (int l = 0; l < sh.n_layers; ++l) {
        int o = l == sh.n_layers - 1 ? sh.out_dim : sh.width;
        for (int q = 0; q < li * o; ++q) p[q] = round_bf16(p[q]);
        p += li * o + o;
        li = o;
      }
    }
  }
  CKC(cudaMemcpy(sc->weights_f32, w.data(), n * (size_t)params * 4, cudaMemcpyHostToDevice));
  CKC(ms_prep_prims(sc->n, sc->center, sc->quat, sc->scale, sc->A, sc->M, d_bad, 0));
  int bad = 0;
  CKC(cudaMemcpy(&bad, d_bad, 4, cudaMemcpyDeviceToHost));
  if (bad) return fail(MS_ERR_INVALID_ARG);
  for (size_t i = 0; i < n * 3; ++i)
    if (!isfinite(prims->center[i])) return fail(MS_ERR_INVALID_ARG);
  CKC(cudaMallocHost(&sc->pinned, 16));
  for (int i = 0; i <= MS_N_STAGES; ++i) CKC(cudaEventCreate(&sc->ev[i]));
  if (mlp->dtype == MS_BF16) {
    rc = ms_tc_pack(sh, sc->n, w.data(), &sc->tc);  // leaves tc.valid = false if the shape is not covered
    if (rc != MS_OK) return fail(rc);
  }
  CKC(cudaDeviceSynchronize());
  cudaFree(d_bad);
  *out = sc;
  return MS_OK;
#undef CKC
}

int ms_scene_set_slots(ms_scene *sc, int32_t c_f, const float *emb) {
  if (!sc || !emb || c_f < 1) return MS_ERR_INVALID_ARG;
  if (sc->shape.mode != MS_MODE_CONTACT || sc->shape.n_feat != 0) return MS_ERR_INVALID_ARG;
  if (c_f % 128 != 0 || c_f > 512) return MS_ERR_UNSUPPORTED_SHAPE;   // one float4 per lane per 128 channels
  const size_t bytes = (size_t)sc->n * 4 * (size_t)c_f * sizeof(float);
  float *d = nullptr;
  cudaError_t e = cudaMalloc(&d, bytes);
  if (e != cudaSuccess) { (void)cudaGetLastError(); sc->last_cuda = (int)e; return MS_ERR_OUT_OF_MEMORY; }
  e = cudaMemcpy(d, emb, bytes, cudaMemcpyHostToDevice);
  if (e != cudaSuccess) { cudaFree(d); sc->last_cuda = (int)e; return MS_ERR_CUDA; }
  cudaFree(sc->slots);
  sc->slots = d;
  sc->slot_cf = c_f;
  return MS_OK;
}

int ms_scene_destroy(ms_scene *sc) {
  if (!sc) return MS_OK;
  cudaFree(sc->center); cudaFree(sc->quat); cudaFree(sc->scale); cudaFree(sc->A); cudaFree(sc->M);
  cudaFree(sc->weights_f32);
  cudaFree(sc->slots);
  ms_tc_free(&sc->tc);
  Buf *all[] = {&sc->tile_count, &sc->emit_off, &sc->rect, &sc->z_entry, &sc->oprime, &sc->keys_a, &sc->keys_b,
                &sc->sort_scratch, &sc->tile_start, &sc->pair_hits, &sc->pair_off, &sc->ray_hits, &sc->ray_off,
                &sc->scan_scratch, &sc->prim_start, &sc->prim_blocks, &sc->blk_off, &sc->intervals, &sc->hits,
                &sc->staging, &sc->staging_feat, &sc->staging_gate, &sc->staging_coef, &sc->host_rgb, &sc->host_alpha, &sc->host_feat, &sc->dbg};
  for (Buf *b : all) free_buf(*b);
  if (sc->pinned) cudaFreeHost(sc->pinned);
  for (int i = 0; i <= MS_N_STAGES; ++i)
    if (sc->ev[i]) cudaEventDestroy(sc->ev[i]);
  (void)cudaGetLastError();
  delete sc;
  return MS_OK;
}

int ms_render(ms_scene *sc, const ms_camera *camera, int32_t H, int32_t W, const ms_opts *opts, float *out_rgb,
              float *out_alpha, float *out_feat) {
  int rc = check_render_args(sc, camera, 1, H, W, opts, out_rgb, out_alpha);
  if (rc != MS_OK) return rc;
  return render_view(sc, camera, H, W, opts, out_rgb, out_alpha, out_feat);
}

int ms_render_batch(ms_scene *sc, const ms_camera *cams, int32_t n_views, int32_t H, int32_t W, const ms_opts *opts,
                    float *out_rgb, float *out_alpha, float *out_feat) {
  int rc = check_render_args(sc, cams, n_views, H, W, opts, out_rgb, out_alpha);
  if (rc != MS_OK) return rc;
  const size_t px = (size_t)H * W;
  for (int v = 0; v < n_views; ++v) {
    rc = render_view(sc, cams + v, H, W, opts, out_rgb + v * px * 3, out_alpha + v * px,
                     out_feat ? out_feat + v * px * (size_t)(sc->slot_cf ? sc->slot_cf : sc->shape.n_feat) : nullptr);
    if (rc != MS_OK) return rc;
  }
  return MS_OK;
}

int ms_render_host(ms_scene *sc, const ms_camera *cams, int32_t n_views, int32_t H, int32_t W, const ms_opts *opts,
                   float *host_rgb, float *host_alpha, float *host_feat) {
  int rc = check_render_args(sc, cams, n_views, H, W, opts, host_rgb, host_alpha);
  if (rc != MS_OK) return rc;
  cudaStream_t st = (cudaStream_t)opts->stream;
  const size_t px = (size_t)H * W;
  const int nf = sc->slot_cf ? sc->slot_cf : sc->shape.n_feat;
  const bool feat = nf > 0 && host_feat;
  ENS(sc->host_rgb, px * 12);
  ENS(sc->host_alpha, px * 4);
  if (feat) ENS(sc->host_feat, px * (size_t)nf * 4);
  for (int v = 0; v < n_views; ++v) {
    rc = render_view(sc, cams + v, H, W, opts, (float *)sc->host_rgb.p, (float *)sc->host_alpha.p,
                     feat ? (float *)sc->host_feat.p : nullptr);
    if (rc != MS_OK) return rc;
    CK(cudaMemcpyAsync(host_rgb + v * px * 3, sc->host_rgb.p, px * 12, cudaMemcpyDeviceToHost, st));
    CK(cudaMemcpyAsync(host_alpha + v * px, sc->host_alpha.p, px * 4, cudaMemcpyDeviceToHost, st));
    if (feat) CK(cudaMemcpyAsync(host_feat + v * px * nf, sc->host_feat.p, px * (size_t)nf * 4, cudaMemcpyDeviceToHost, st));
  }
  CK(cudaStreamSynchronize(st));
  return MS_OK;
}

int ms_last_stats(ms_scene *sc, ms_stats *out) {
  if (!sc || !out) return MS_ERR_INVALID_ARG;
  *out = sc->stats;
  return MS_OK;
}

int ms_last_stage_ms(ms_scene *sc, float *ms) {
  if (!sc || !ms || !sc->ev_valid) return MS_ERR_INVALID_ARG;
  CK(cudaEventSynchronize(sc->ev[MS_N_STAGES]));
  for (int i = 0; i < MS_N_STAGES; ++i) CK(cudaEventElapsedTime(&ms[i], sc->ev[i], sc->ev[i + 1]));
  return MS_OK;
}

int ms_stage_accum(ms_scene *sc, double *ms_sum, int64_t *n_views, int32_t reset) {
  if (!sc) return MS_ERR_INVALID_ARG;
  if (sc->ev_pending) {
    CK(cudaEventSynchronize(sc->ev[MS_N_STAGES]));
    harvest_stage_times(sc);
  }
  if (ms_sum)
    for (int i = 0; i < MS_N_STAGES; ++i) ms_sum[i] = sc->stage_sum[i];
  if (n_views) *n_views = sc->stage_views;
  if (reset) {
    for (int i = 0; i < MS_N_STAGES; ++i) sc->stage_sum[i] = 0.0;
    sc->stage_views = 0;
  }
  return MS_OK;
}

int ms_debug_tile_lists(ms_scene *sc, int64_t *tile_offsets, int32_t *prim_ids, uint32_t *zbits, size_t cap, size_t *n) {
  if (!sc || !sc->debug_valid) return MS_ERR_INVALID_ARG;
  CK(cudaDeviceSynchronize());
  const size_t P = (size_t)sc->stats.n_pairs;
  if (n) *n = P;
  if (cap < P) return MS_ERR_CAPACITY;
  std::vector<uint64_t> keys(P);
  std::vector<uint32_t> ts((size_t)sc->dbg_n_tiles + 1);
  if (P) CK(cudaMemcpy(keys.data(), sc->dbg_keys, P * 8, cudaMemcpyDeviceToHost));
  CK(cudaMemcpy(ts.data(), sc->tile_start.p, ts.size() * 4, cudaMemcpyDeviceToHost));
  if (tile_offsets)
    for (size_t i = 0; i < ts.size(); ++i) tile_offsets[i] = ts[i];
  const uint64_t pmask = (1ull << sc->dbg_prim_bits) - 1;
  for (size_t i = 0; i < P; ++i) {
    if (prim_ids) prim_ids[i] = (int32_t)(keys[i] & pmask);
    if (zbits) zbits[i] = (uint32_t)((keys[i] >> sc->dbg_prim_bits) & 0xffffffffull);
  }
  return MS_OK;
}

int ms_debug_intervals(ms_scene *sc, int64_t *hit_offsets, int32_t *prim, float *t_in, float *delta, size_t cap,
                       size_t *n) {
  if (!sc || !sc->debug_valid) return MS_ERR_INVALID_ARG;
  CK(cudaDeviceSynchronize());
  const size_t nh = (size_t)sc->stats.n_intervals;
  const size_t R = (size_t)sc->dbg_H * sc->dbg_W;
  if (n) *n = nh;
  if (cap < nh) return MS_ERR_CAPACITY;
  std::vector<uint32_t> ro(R + 1);
  std::vector<MsHit> h(nh);
  CK(cudaMemcpy(ro.data(), sc->ray_off.p, (R + 1) * 4, cudaMemcpyDeviceToHost));
  if (nh) CK(cudaMemcpy(h.data(), sc->hits.p, nh * sizeof(MsHit), cudaMemcpyDeviceToHost));
  if (hit_offsets)
    for (size_t i = 0; i <= R; ++i) hit_offsets[i] = ro[i];
  for (size_t i = 0; i < nh; ++i) {
    if (prim) prim[i] = h[i].prim;
    if (t_in) t_in[i] = h[i].t_in;
    if (delta) delta[i] = h[i].delta;
  }
  return MS_OK;
}

int ms_debug_sample_order(ms_scene *sc, int32_t ray, int32_t *prim, int32_t *k, float *t, size_t cap, size_t *n) {
  if (!sc || !sc->debug_valid || ray < 0 || ray >= sc->dbg_H * sc->dbg_W) return MS_ERR_INVALID_ARG;
  CK(cudaDeviceSynchronize());
  uint32_t ro[2];
  CK(cudaMemcpy(ro, (uint32_t *)sc->ray_off.p + ray, 8, cudaMemcpyDeviceToHost));
  const size_t ns = (size_t)(ro[1] - ro[0]) * (size_t)sc->dbg_K;
  if (n) *n = ns;
  if (cap < ns) return MS_ERR_CAPACITY;
  if (ns == 0) return MS_OK;
  ENS(sc->dbg, ns * 12);
  int *dp = (int *)sc->dbg.p, *dk = dp + ns;
  float *dt = (float *)(dk + ns);
  MsCompositeArgs ca;
  memset(&ca, 0, sizeof(ca));
  ca.n_rays = sc->dbg_H * sc->dbg_W; ca.K = sc->dbg_K; ca.n_feat = 0; ca.t_stop = 0.f;
  ca.contact = sc->shape.mode == MS_MODE_CONTACT;
  ca.tile_order = sc->dbg_tile_order;
  ca.ray_off = (uint32_t *)sc->ray_off.p; ca.hits = (MsHit *)sc->hits.p; ca.staging = (float4 *)sc->staging.p;
  CK(ms_sample_order(ca, ray, dp, dk, dt, 0));
  CK(cudaDeviceSynchronize());
  if (prim) CK(cudaMemcpy(prim, dp, ns * 4, cudaMemcpyDeviceToHost));
  if (k) CK(cudaMemcpy(k, dk, ns * 4, cudaMemcpyDeviceToHost));
  if (t) CK(cudaMemcpy(t, dt, ns * 4, cudaMemcpyDeviceToHost));
  return MS_OK;
}

int ms_debug_prim_frames(ms_scene *sc, float *A, float *M) {
  if (!sc) return MS_ERR_INVALID_ARG;
  if (A) CK(cudaMemcpy(A, sc->A, (size_t)sc->n * 36, cudaMemcpyDeviceToHost));
  if (M) CK(cudaMemcpy(M, sc->M, (size_t)sc->n * 36, cudaMemcpyDeviceToHost));
  return MS_OK;
}

const char *ms_error_string(int code) {
  switch (code) {
    case MS_OK: return "ok";
    case MS_ERR_INVALID_ARG: return "invalid argument";
    case MS_ERR_OUT_OF_MEMORY: return "out of memory";
    case MS_ERR_CUDA: return "CUDA error";
    case MS_ERR_UNSUPPORTED_SHAPE: return "unsupported shape";
    case MS_ERR_CAPACITY: return "buffer too small";
    default: return "unknown error";
  }
}

int ms_last_cuda_error(ms_scene *sc) { return sc ? sc->last_cuda : 0; }

}  // extern "C"
