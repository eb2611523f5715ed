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
  int n_sm = 0;
  int dtype = MS_F32;
  MsMlpShape shape{};
  float falloff = MS_FALLOFF_DEFAULT;
  int last_cuda = 0;
  // scene-lifetime device data
  float *center = nullptr, *quat = nullptr, *scale = nullptr, *A = nullptr, *M = nullptr;
  float *weights_f32 = nullptr;      // fp32 path / backward; for a bf16 scene on the tensor path uploaded on first use
  std::vector<float> w_host;         // the (bf16-rounded) weight values until then
  MsTcWeights tc{};  // packed bf16 image for the tensor path (may be empty)
  int slot_cf = 0;           // Eq.7 slot embeddings: width C_f (0 = none)
  float *slots = nullptr;    // device [N][4][slot_cf]
  // per-view scratch
  Buf tile_count, emit_off, rect, z_entry, oprime, keys_a, keys_b, sort_scratch, tile_start, pair_hits_i, pair_hits_j,
      pair_off, slot_of, key2_a, key2_b, flags, gid, grp_key, grp_prim, grp_iv0, grp_blocks, blk_off, grp_cnt_c,
      grp_blocks_c, blk_off_c, bw, bands, counters, alive, ray_hits, ray_off, scan_scratch, intervals, intervals_c, hit_e, hits, staging,
      staging_feat, staging_gate, staging_coef, dbg_ord, pos_xy, host_rgb, host_alpha, host_feat;
  uint32_t *pinned = nullptr;  // host-pinned readback: [0] P, [1..] device counters
  MsBand *pinned_bands = nullptr;  // host-pinned readback of the band table
  size_t pinned_bands_cap = 0;
  // MS_FLAG_STAGE_TIMES: 4 + 2 per band events per view, in two alternating sets -- a view's events are read when the
  // view after the next begins (they have long completed then: no wait that would drain the stream)
  struct EvSet {
    std::vector<cudaEvent_t> ev;
    std::vector<cudaEvent_t> evc;  // overlapped bands: start / end of stage (e) of band b on the second stream (2b, 2b + 1)
    bool overlap = false;
    int bands = 0;
    bool pending = false;          // recorded, not yet added to stage_sum
  } evs[2];
  int ev_cur = 0;
  bool ev_valid = false;
  float last_stage_ms[MS_N_STAGES] = {};
  double stage_sum[MS_N_STAGES] = {};
  int64_t stage_views = 0;
  cudaEvent_t frame_done = nullptr;  // recorded after the counters' readback copy of the last view
  // banded views: stage (e) of band b runs on st2 while stage (d) of band b + 1 runs on the caller's stream
  cudaStream_t st2 = nullptr;
  // ms_render_host, several views: the copy of view v to the host runs on copy_st beside the render of view v + 1
  // (the outputs alternate between two device buffers: host_* and host2_*)
  cudaStream_t copy_st = nullptr;
  cudaEvent_t ev_rendered[2] = {nullptr, nullptr}, ev_copied[2] = {nullptr, nullptr};
  Buf host2_rgb, host2_alpha, host2_feat;
  cudaEvent_t ev_mlp[2] = {nullptr, nullptr}, ev_comp[2] = {nullptr, nullptr};
  bool frame_pending = false;
  bool prev_terminated = false;      // MS_WAVES_AUTO: the previous view had rays stopping early
  // last view
  struct LastView {
    bool valid = false;
    MsGrid grid{};
    MsCam cam{};
    int K = 0, n_bands = 0, n_waves = 0, banded = 0, path = 0;
    size_t n_hits = 0;
    float t_stop = 0.f;
  } last;
  struct History {            // MS_FLAG_NO_SYNC: the last synchronising view, whose scratch sizes the next ones
    bool valid = false;
    int H = 0, W = 0, tile = 0, K = 0, path = 0, feat = 0, slots = 0, tile_order = 0;
    size_t pairs = 0;         // its pair count
  } hist;
  bool frame_nosync = false;  // the pending view was rendered without host synchronisation
  bool clear_sticky = false;  // the sticky overflow flag has been seen: clear it before the next view
  Buf bwd_rgb, bwd_alpha, bwd_ord, bwd_gstage, bwd_ivgrad, bwd_gA;   // backward pass scratch
  ms_stats stats{};
  bool debug_valid = false, order_valid = false;
  int dbg_H = 0, dbg_W = 0, dbg_K = 0, dbg_prim_bits = 0;
  MsGrid dbg_grid{};
  uint64_t *dbg_keys = nullptr;
  int dbg_contact = 0;
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

#define ENS_HOST(sc, bytes)                                                     \
  do {                                                                          \
    if ((bytes) > (sc)->pinned_bands_cap) {                                     \
      if ((sc)->pinned_bands) cudaFreeHost((sc)->pinned_bands);                 \
      (sc)->pinned_bands = nullptr; (sc)->pinned_bands_cap = 0;                 \
      if (cudaMallocHost(&(sc)->pinned_bands, 2 * (bytes)) != cudaSuccess) {    \
        (void)cudaGetLastError();                                               \
        return MS_ERR_OUT_OF_MEMORY;                                            \
      }                                                                         \
      (sc)->pinned_bands_cap = 2 * (bytes);                                     \
    }                                                                           \
  } while (0)

#define ENS(buf, bytes)                         \
  do {                                          \
    int _r = ensure(sc, buf, (size_t)(bytes));  \
    if (_r != MS_OK) return _r;                 \
  } while (0)

std::vector<Buf *> scratch_bufs(ms_scene *sc) {
  return {&sc->tile_count, &sc->emit_off, &sc->rect, &sc->z_entry, &sc->oprime, &sc->keys_a, &sc->keys_b,
          &sc->sort_scratch, &sc->tile_start, &sc->pair_hits_i, &sc->pair_hits_j, &sc->pair_off, &sc->slot_of,
          &sc->key2_a, &sc->key2_b, &sc->flags, &sc->gid, &sc->grp_key, &sc->grp_prim, &sc->grp_iv0, &sc->grp_blocks,
          &sc->blk_off, &sc->grp_cnt_c, &sc->grp_blocks_c, &sc->blk_off_c, &sc->bw, &sc->bands, &sc->counters,
          &sc->alive, &sc->ray_hits, &sc->ray_off, &sc->scan_scratch, &sc->intervals, &sc->intervals_c, &sc->hit_e, &sc->hits, &sc->staging,
          &sc->staging_feat, &sc->staging_gate, &sc->staging_coef, &sc->dbg_ord, &sc->pos_xy};
}

size_t scratch_total(ms_scene *sc) {
  size_t t = 0;
  for (const Buf *b : scratch_bufs(sc)) t += b->cap;
  return t;
}

int ceil_log2(uint64_t v) {
  int b = 0;
  while ((1ull << b) < v) ++b;
  return b;
}

// Mid-frame read-backs (pair count, hit counters, band table) are written to pinned host memory by a kernel, not by
// a device-to-host copy: a copy would queue on the copy engine behind the image copies of the previous view, which
// ms_render_host runs on a stream of its own beside this view (a 300 MB copy ahead costs 5 ms of waiting).
__global__ void readback_kernel(uint32_t *dst_host, const uint32_t *src, int n) {
  for (int i = threadIdx.x; i < n; i += blockDim.x) dst_host[i] = src[i];
  __threadfence_system();
}
cudaError_t readback_words(void *dst_host, const void *src, size_t n_words, cudaStream_t st) {
  readback_kernel<<<1, 128, 0, st>>>((uint32_t *)dst_host, (const uint32_t *)src, (int)n_words);
  MS_LAUNCHED();
  return cudaGetLastError();
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

// Event layout of a view rendered with MS_FLAG_STAGE_TIMES: 0 start (a), 1 start (b), 2 start (c), 3 start of the band
// loop; per band b: 4 + 2b before stage (d), 5 + 2b between (d) and (e); 4 + 2 n_bands the end.
// Adds the stage times of the previous view to the running sums.  Called right after the last event has completed.
int harvest_stage_times(ms_scene *sc, int set) {
  ms_scene::EvSet &E = sc->evs[set];
  if (!E.pending) return MS_OK;
  if (cudaEventSynchronize(E.ev[3 + 2 * E.bands]) != cudaSuccess) { (void)cudaGetLastError(); return MS_ERR_CUDA; }
  E.pending = false;
  float ms[MS_N_STAGES] = {0.f, 0.f, 0.f, 0.f, 0.f};
  auto el = [&](int a, int b, float *out) {
    float v = 0.f;
    if (cudaEventElapsedTime(&v, E.ev[a], E.ev[b]) != cudaSuccess) { (void)cudaGetLastError(); return false; }
    *out += v;
    return true;
  };
  bool ok = el(0, 1, &ms[MS_STAGE_BIN]) && el(1, 2, &ms[MS_STAGE_SORT]) && el(2, 3, &ms[MS_STAGE_ISECT]);
  for (int b = 0; ok && b < E.bands; ++b) {
    ok = el(3 + 2 * b, 4 + 2 * b, &ms[MS_STAGE_MLP]);
    if (!ok) break;
    if (E.overlap) {            // stage (e) ran beside the next band's stage (d): its own duration on the second stream
      float v = 0.f;
      if (cudaEventElapsedTime(&v, E.evc[2 * b], E.evc[2 * b + 1]) != cudaSuccess) { (void)cudaGetLastError(); ok = false; }
      ms[MS_STAGE_COMPOSITE] += v;
    } else {
      ok = el(4 + 2 * b, 5 + 2 * b, &ms[MS_STAGE_COMPOSITE]);
    }
  }
  if (!ok) return MS_OK;
  for (int i = 0; i < MS_N_STAGES; ++i) { sc->stage_sum[i] += ms[i]; sc->last_stage_ms[i] = ms[i]; }
  sc->stage_views += 1;
  return MS_OK;
}

// Reads the device counters of the last view (waits for it) into sc->stats.
int finish_frame(ms_scene *sc) {
  if (!sc->frame_pending) return MS_OK;
  CK(cudaEventSynchronize(sc->frame_done));
  sc->frame_pending = false;
  const uint32_t *c = sc->pinned + 1;
  sc->stats.n_blocks = (int64_t)c[MS_CNT_BLOCKS];
  sc->stats.n_visible = (int64_t)c[MS_CNT_VISIBLE];
  sc->stats.n_dead_rays = (int64_t)c[MS_CNT_DEAD_RAYS];
  sc->stats.n_samples_evaluated = sc->stats.n_samples - (int64_t)c[MS_CNT_SKIPPED] * (int64_t)sc->dbg_K;
  sc->prev_terminated = c[MS_CNT_STOPPED_RAYS] > 0;
  if (sc->frame_nosync) {     // the counts the host never saw
    sc->frame_nosync = false;
    sc->stats.n_pairs = (int64_t)c[MS_CNT_PAIRS] | ((int64_t)c[MS_CNT_PAIRS_HI] << 32);
    sc->stats.n_intervals = (int64_t)c[MS_CNT_HITS] | ((int64_t)c[MS_CNT_HITS_HI] << 32);
    sc->stats.n_samples = sc->stats.n_intervals * (int64_t)sc->dbg_K;
    sc->stats.n_samples_evaluated = sc->stats.n_samples;
    sc->stats.overflow = (c[MS_CNT_OVERFLOW] || c[MS_CNT_STICKY_OVERFLOW]) ? 1 : 0;   // this view, or an earlier one of its batch
    if (c[MS_CNT_STICKY_OVERFLOW]) sc->clear_sticky = true;
    if (sc->stats.overflow) {
      sc->hist.valid = false;  // the next render takes the synchronising path and regrows the scratch
      sc->stats.n_samples_evaluated = 0;
    }
  }
  return MS_OK;
}

// MS_FLAG_NO_SYNC renders never wait for the previous view: its counters are read only if it has finished
int finish_frame_if_done(ms_scene *sc, bool no_block) {
  if (!sc->frame_pending) return MS_OK;
  if (no_block && cudaEventQuery(sc->frame_done) != cudaSuccess) {
    (void)cudaGetLastError();
    return MS_OK;
  }
  return finish_frame(sc);
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
  MsGrid grid;
  grid.tile = tile; grid.tiles_x = (W + tile - 1) / tile; grid.tiles_y = (H + tile - 1) / tile;
  grid.G = 64 / tile < 1 ? 1 : 64 / tile;          // macro-tiles of 64 x 64 pixels
  grid.W = W; grid.H = H;
  grid.tshift = tile == 8 ? 3 : (tile == 16 ? 4 : 5);
  grid.pos_xy = nullptr;
  const int64_t n_tiles64 = (int64_t)grid.tiles_x * grid.tiles_y;
  const int64_t R64 = n_tiles64 * tile * tile;      // ray slots: every tile padded to tile x tile
  if (R64 >= (1ll << 31) - 1) return MS_ERR_UNSUPPORTED_SHAPE;
  grid.n_tiles = (int)n_tiles64;
  const int n_tiles = grid.n_tiles;
  const size_t R = (size_t)R64;
  const int prim_bits = ceil_log2((uint64_t)N) < 1 ? 1 : ceil_log2((uint64_t)N);
  const int tile_bits = ceil_log2((uint64_t)n_tiles) < 1 ? 1 : ceil_log2((uint64_t)n_tiles);
  if (prim_bits + tile_bits > 32) return MS_ERR_UNSUPPORTED_SHAPE;

  int path = opts->path;
  if (path == MS_PATH_AUTO)
    path = (sc->dtype == MS_BF16 && sc->tc.valid) ? MS_PATH_BF16_TC : MS_PATH_FP32;
  if (path == MS_PATH_BF16_TC && !sc->tc.valid) return MS_ERR_UNSUPPORTED_SHAPE;
  if (path != MS_PATH_BF16_TC && path != MS_PATH_FP32) return MS_ERR_INVALID_ARG;

  const int tile_order = (opts->flags & MS_FLAG_TILE_ORDER) != 0;
  const bool want_feat = sc->shape.n_feat > 0 && out_feat != nullptr;
  const bool want_slots = sc->slot_cf > 0 && out_feat != nullptr;   // Eq.7 features (contact mode, K = 1)
  // the tensor path stages its 32 feature channels as fp16 (its operands are bf16); the fp32 path keeps fp32
  const bool feat_half = want_feat && path == MS_PATH_BF16_TC && sc->shape.n_feat == 32;
  const size_t feat_bytes = want_feat ? (size_t)sc->shape.n_feat * (feat_half ? 2 : 4) : 0;
  const size_t sample_bytes = sizeof(float4) + feat_bytes + (want_slots ? 2 * sizeof(float4) : 0);
  // MS_FLAG_NO_SYNC: no read-back at all if the previous synchronising view had the same shape, was one band without
  // waves, and left scratch to size this one from (its buffers carry 25 % of slack); the kernels clamp against those
  // capacities and raise MS_CNT_OVERFLOW, reported by ms_last_stats
  size_t P_cap = 0, hit_cap = 0;
  bool nosync = (opts->flags & MS_FLAG_NO_SYNC) != 0 && !(opts->flags & (MS_FLAG_KEEP_DEBUG | MS_FLAG_KEEP_ORDER)) &&
                sc->hist.valid && sc->hist.H == H && sc->hist.W == W && sc->hist.tile == tile && sc->hist.K == K &&
                sc->hist.path == path && sc->hist.feat == (want_feat ? 1 : 0) && sc->hist.slots == (want_slots ? 1 : 0) &&
                sc->hist.tile_order == tile_order && opts->waves <= 0;
  {  // the previous view's counters (its stats, whether its rays stopped early, whether it overflowed): a view that
     // may go without synchronisation does not wait for them
    int rc = finish_frame_if_done(sc, nosync);
    if (rc != MS_OK) return rc;
  }
  if (!sc->hist.valid || (opts->waves == 0 && sc->prev_terminated)) nosync = false;   // overflowed meanwhile / waves due
  if (nosync) {
    auto mn = [](size_t a, size_t b) { return a < b ? a : b; };
    P_cap = mn(mn(sc->keys_a.cap / 8, sc->keys_b.cap / 8), mn(sc->pair_hits_i.cap / 4, sc->slot_of.cap / 4));
    P_cap = mn(P_cap, mn(sc->pair_hits_j.cap / 4, sc->pair_off.cap / 4));
    P_cap = P_cap > 4 ? P_cap - 4 : 0;
    while (P_cap > 0 && (ms_sort_scratch_elems(P_cap) * 4 > sc->sort_scratch.cap ||
                         (ms_scan_scratch_elems(P_cap) + 16) * 4 > sc->scan_scratch.cap))
      P_cap = P_cap * 3 / 4;
    // a key set that fits one CTA's sort with a quarter of slack keeps to that capacity: one launch sorts it
    if (P_cap > MS_BLOCK_SORT_MAX && sc->hist.pairs + sc->hist.pairs / 4 + 64 <= MS_BLOCK_SORT_MAX) P_cap = MS_BLOCK_SORT_MAX;
    hit_cap = mn(mn(sc->intervals.cap / sizeof(MsInterval), sc->hits.cap / sizeof(MsHit)),
                 sc->staging.cap / (sizeof(float4) * (size_t)K));
    if (want_feat) hit_cap = mn(hit_cap, sc->staging_feat.cap / (feat_bytes * (size_t)K));
    if (want_slots) hit_cap = mn(hit_cap, mn(sc->staging_gate.cap, sc->staging_coef.cap) / (sizeof(float4) * (size_t)K));
    hit_cap = hit_cap > 2 ? hit_cap - 2 : 0;
    if (P_cap == 0 || hit_cap == 0 || P_cap >= (1ull << 31) || hit_cap >= (1ull << 31)) nosync = false;
  }
  if (path == MS_PATH_FP32 && !sc->weights_f32) {
    const size_t bytes = (size_t)N * (size_t)sc->shape.params * 4;
    if (sc->w_host.size() * 4 != bytes) return MS_ERR_CUDA;
    CK(cudaMalloc(&sc->weights_f32, bytes));
    CK(cudaMemcpy(sc->weights_f32, sc->w_host.data(), bytes, cudaMemcpyHostToDevice));
    std::vector<float>().swap(sc->w_host);
  }
  const bool timing = (opts->flags & MS_FLAG_STAGE_TIMES) != 0;
  const MsCam cam = make_cam(camera, H, W);
  const long long launches0 = ms_launch_count;
  if (timing) {   // this view records into the older set: its events (two views back) are read first
    sc->ev_cur ^= 1;
    int rc = harvest_stage_times(sc, sc->ev_cur);
    if (rc != MS_OK) return rc;
  }
  sc->ev_valid = false;
  auto rec = [&](int i) -> cudaError_t {
    if (!timing) return cudaSuccess;
    std::vector<cudaEvent_t> &ev = sc->evs[sc->ev_cur].ev;
    while ((int)ev.size() <= i) {
      cudaEvent_t e;
      cudaError_t r = cudaEventCreate(&e);
      if (r != cudaSuccess) return r;
      ev.push_back(e);
    }
    return cudaEventRecord(ev[i], st);
  };

  // ---- (a) projection + key emit ----------------------------------------------------------
  CK(rec(0));
  if (!sc->counters.p) {
    ENS(sc->counters, (MS_CNT_N + 4) * 4);
    CK(cudaMemsetAsync(sc->counters.p, 0, (MS_CNT_N + 4) * 4, st));
  }
  // small frames without host synchronisation: stages (a) + (b) are one launch of one CTA, which also resets the counters
  const bool small_ab = nosync && ms_bin_sort_small_fits(N, P_cap);
  if (!small_ab) CK(cudaMemsetAsync(sc->counters.p, 0, MS_CNT_N * 4, st));         // the sticky overflow flag behind them stays
  if (sc->clear_sticky) {
    CK(cudaMemsetAsync((uint32_t *)sc->counters.p + MS_CNT_STICKY_OVERFLOW, 0, 4, st));
    sc->clear_sticky = false;
  }
  uint32_t *counters = (uint32_t *)sc->counters.p;
  ENS(sc->tile_count, (size_t)N * 4);
  ENS(sc->emit_off, (size_t)(N + 1) * 4);
  ENS(sc->rect, (size_t)N * sizeof(int4));
  ENS(sc->z_entry, (size_t)N * 4);
  ENS(sc->oprime, (size_t)N * 12);
  ENS(sc->scan_scratch, (ms_scan_scratch_elems(R > (size_t)N ? R : (size_t)N) + 16) * 4);
  const float eye_guard = opts->eye_guard > 0.0f ? opts->eye_guard : MS_EYE_GUARD_DEFAULT;
  if (!small_ab) {
    CK(ms_project(N, sc->center, sc->A, sc->M, cam, tile, eye_guard, (uint32_t *)sc->tile_count.p,
                  (int4 *)sc->rect.p, (float *)sc->z_entry.p, (float *)sc->oprime.p, counters, st));
    CK(ms_exclusive_scan_u32((uint32_t *)sc->tile_count.p, (uint32_t *)sc->emit_off.p, (size_t)N,
                             (uint32_t *)sc->scan_scratch.p, st));
  }
  size_t P = 0;                       // the pair count, or (no-sync) the capacity the launches are sized for
  const uint32_t *P_dev = nullptr;    // no-sync: where the kernels read the count
  if (nosync) {
    P = P_cap;
    P_dev = counters + MS_CNT_P_EFF;
  } else {
    CK(readback_words(sc->pinned, (uint32_t *)sc->emit_off.p + N, 1, st));
    CK(readback_words(sc->pinned + 1 + MS_CNT_PAIRS_HI, counters + MS_CNT_PAIRS_HI, 1, st));
    CK(cudaStreamSynchronize(st));
    // the 32-bit scan total must agree with the 64-bit count of the projection kernel (a wrapped sum would size
    // every buffer below too small)
    if (sc->pinned[1 + MS_CNT_PAIRS_HI] != 0) return MS_ERR_UNSUPPORTED_SHAPE;
    P = sc->pinned[0];
    if (P >= (1ull << 31)) return MS_ERR_UNSUPPORTED_SHAPE;
  }
  ENS(sc->keys_a, (P + 1) * 8);
  ENS(sc->keys_b, (P + 1) * 8);
  // sized for the pairs the other buffers' 25 % of slack can hold: a no-sync view may use all of it
  const size_t P_slack = nosync ? P : P + P / 4 + 4096;
  ENS(sc->sort_scratch, ms_sort_scratch_elems(P_slack) * 4);
  ENS(sc->tile_start, (size_t)(n_tiles + 1) * 4);
  ENS(sc->pair_hits_i, (P + 1) * 4);
  ENS(sc->pair_hits_j, (P + 2) * 4);
  ENS(sc->pair_off, (P + 2) * 4);
  ENS(sc->slot_of, (P + 1) * 4);
  if (ms_scan_scratch_elems(P_slack) + 16 > sc->scan_scratch.cap / 4) ENS(sc->scan_scratch, (ms_scan_scratch_elems(P_slack) + 16) * 4);
  uint64_t *sorted = nullptr;
  if (small_ab) {
    CK(ms_bin_sort_small(N, sc->center, sc->A, sc->M, cam, tile, eye_guard, grid.tiles_x, n_tiles, prim_bits, tile_order,
                         prim_bits + 32 + tile_bits, (uint32_t)P_cap, (uint32_t *)sc->tile_count.p,
                         (uint32_t *)sc->emit_off.p, (int4 *)sc->rect.p, (float *)sc->z_entry.p, (float *)sc->oprime.p,
                         counters, (uint64_t *)sc->keys_a.p, (uint64_t *)sc->keys_b.p, (uint32_t *)sc->tile_start.p,
                         (uint32_t *)sc->pair_hits_j.p, st));
    sorted = (uint64_t *)sc->keys_b.p;
    CK(rec(1));                      // stage times: the fused launch counts as stage (a); stage (b) reads 0
  } else {
    CK(ms_emit_keys(N, (uint32_t *)sc->emit_off.p, (int4 *)sc->rect.p, (float *)sc->z_entry.p, grid.tiles_x, prim_bits,
                    (uint64_t *)sc->keys_a.p, tile_order, cam, tile, sc->A, (float *)sc->oprime.p, st,
                    nosync ? (uint32_t)P_cap : 0xffffffffu, nosync ? counters : nullptr));

    // ---- (b) radix sort + tile ranges -------------------------------------------------------
    CK(rec(1));
    // stage (a) emits the keys primitive by primitive, i.e. already ordered by the id in their low prim_bits bits;
    // the sort is stable, so only the (tile | depth) bits above them need passes
    CK(ms_radix_sort_u64((uint64_t *)sc->keys_a.p, (uint64_t *)sc->keys_b.p, P, prim_bits, prim_bits + 32 + tile_bits,
                         (uint32_t *)sc->sort_scratch.p, &sorted, st, P_dev));
    CK(ms_tile_ranges(sorted, P, n_tiles, prim_bits, (uint32_t *)sc->tile_start.p, st, P_dev));
  }

  // ---- (c) intersection: count, scan, pair order, fill ---------------------------------------
  CK(rec(2));
  ENS(sc->ray_hits, R * 4);
  ENS(sc->ray_off, (R + 1) * 4);
  ENS(sc->pos_xy, (size_t)(n_tiles + 1) * sizeof(ushort2));
  grid.pos_xy = (const ushort2 *)sc->pos_xy.p;
  MsIsectArgs ia;
  ia.cam = cam; ia.grid = grid; ia.K = K; ia.prim_bits = prim_bits;
  ia.contact = sc->shape.mode == MS_MODE_CONTACT;
  ia.wave_c = 0;
  ia.keys = sorted; ia.tile_start = (uint32_t *)sc->tile_start.p; ia.A = sc->A; ia.oprime = (float *)sc->oprime.p;
  ia.pos_xy = (ushort2 *)sc->pos_xy.p;
  ia.pair_hits = (uint32_t *)sc->pair_hits_i.p; ia.ray_hits = (uint32_t *)sc->ray_hits.p;
  ia.slot_of = (uint32_t *)sc->slot_of.p; ia.pair_off = (uint32_t *)sc->pair_off.p; ia.ray_off = (uint32_t *)sc->ray_off.p;
  ia.intervals = nullptr; ia.hits = nullptr; ia.guard = nullptr;
  CK(ms_isect_count(ia, st));
  // small frames without host synchronisation: the CTA that orders the pairs (below) takes the tile statistics along,
  // and the ray scan too when the frame has few enough rays
  const bool small_c = nosync && ms_order_single_is_small(P, N);
  const bool small_c_scan = small_c && R <= MS_SMALL_RAYS;
  if (!small_c_scan)
    CK(ms_exclusive_scan_u32((uint32_t *)sc->ray_hits.p, (uint32_t *)sc->ray_off.p, R, (uint32_t *)sc->scan_scratch.p, st));
  if (!small_c)
    CK(ms_tile_stats(grid, (uint32_t *)sc->ray_off.p, (uint32_t *)sc->tile_start.p, counters, st,
                     nosync ? (uint32_t)hit_cap : 0u));
  size_t n_hits = hit_cap, max_tile_hits = 0;     // no-sync: the capacity stands in for the count
  uint32_t max_list = 0;
  if (!nosync) {
    CK(readback_words(sc->pinned + 1, counters, MS_CNT_N, st));
    CK(cudaStreamSynchronize(st));
    if (sc->pinned[1 + MS_CNT_HITS_HI] != 0) return MS_ERR_UNSUPPORTED_SHAPE;   // 64-bit hit total beyond 32 bits
    n_hits = sc->pinned[1 + MS_CNT_HITS];
    max_tile_hits = sc->pinned[1 + MS_CNT_MAX_TILE_HITS];
    max_list = sc->pinned[1 + MS_CNT_MAX_LIST];
    if (n_hits >= (1ull << 31)) return MS_ERR_UNSUPPORTED_SHAPE;
  }
  const size_t n_samples = n_hits * (size_t)K;
  if (n_samples >= (1ull << 40)) return MS_ERR_UNSUPPORTED_SHAPE;

  // bands: the staging bytes of one sample decide how many hits fit the budget
  const int64_t budget = opts->band_bytes == 0 ? MS_BAND_BYTES_DEFAULT : opts->band_bytes;
  size_t cap_hits = n_hits + 1;
  if (budget > 0) {
    cap_hits = (size_t)budget / (sample_bytes * (size_t)K);
    if (cap_hits < 1) cap_hits = 1;
  }
  if (nosync) cap_hits = n_hits + 1;                 // the history says: one band
  int n_bands = n_hits <= cap_hits ? 1 : (int)(n_hits / cap_hits) + 1;
  while (n_bands > 1 && prim_bits + 3 + ceil_log2((uint64_t)n_bands) > 32) {   // (band, wave, prim) must fit 32 bits
    cap_hits *= 2;
    n_bands = n_hits <= cap_hits ? 1 : (int)(n_hits / cap_hits) + 1;
  }
  // MS_FLAG_OVERLAP, two or more bands: the budget becomes two halves, stage (e) of one beside stage (d) of the next
  const bool overlap = n_bands > 1 && (opts->flags & MS_FLAG_OVERLAP) != 0;
  if (overlap) {
    cap_hits = cap_hits > 1 ? cap_hits / 2 : 1;
    n_bands = (int)(n_hits / cap_hits) + 1;
    while (prim_bits + 3 + ceil_log2((uint64_t)n_bands) > 32) {
      cap_hits *= 2;
      n_bands = (int)(n_hits / cap_hits) + 1;
    }
  }
  // depth waves: asked for, or (auto) the previous view had rays stopping early
  int wave_c = 0;
  if (opts->t_stop > 0.0f && !tile_order && !nosync) {
    if (opts->waves > 0) wave_c = opts->waves;
    else if (opts->waves == MS_WAVES_AUTO && sc->prev_terminated) wave_c = 4;   // measured on cfg4_opaque: C = 4 and 6 within noise, 4 skips more
  }
  int n_waves = 1;
  if (wave_c > 0 && max_list > 0) n_waves = ms_wave_of_rank(max_list - 1, wave_c) + 1;
  if (n_waves == 1) wave_c = 0;
  const bool banded = n_bands > 1 || wave_c > 0;
  const size_t seg_cap = (banded ? P : (size_t)N) + 2;
  const size_t band_hits_cap = n_bands == 1 ? n_hits : cap_hits + max_tile_hits;

  ENS(sc->grp_iv0, (seg_cap + 1) * 4);
  ENS(sc->grp_blocks, (seg_cap + 1) * 4);
  ENS(sc->blk_off, (seg_cap + 2) * 4);
  ENS(sc->bw, (size_t)n_bands * MS_MAX_WAVES * sizeof(uint2));
  ENS(sc->bands, (size_t)n_bands * sizeof(MsBand));
  if (banded) {
    ENS(sc->key2_a, (P + 1) * 8);
    ENS(sc->key2_b, (P + 1) * 8);
    ENS(sc->flags, (P + 2) * 4);
    ENS(sc->gid, (P + 2) * 4);
    ENS(sc->grp_key, seg_cap * 4);
    ENS(sc->grp_prim, seg_cap * 4);
  }
  if (wave_c > 0) {
    ENS(sc->grp_cnt_c, seg_cap * 4);
    ENS(sc->grp_blocks_c, seg_cap * 4);
    ENS(sc->blk_off_c, (seg_cap + 2) * 4);
    ENS(sc->alive, R);
    CK(cudaMemsetAsync(sc->alive.p, 1, R, st));
    CK(cudaMemsetAsync(sc->grp_cnt_c.p, 0, seg_cap * 4, st));
    ENS(sc->intervals_c, (n_hits + 1) * sizeof(MsInterval));
    ENS(sc->hit_e, (n_hits + 1) * 4);
    CK(cudaMemsetAsync(sc->hit_e.p, 0xff, (n_hits + 1) * 4, st));   // NaN: no product cached yet
  }
  ENS(sc->intervals, (n_hits + 1) * sizeof(MsInterval));
  ENS(sc->hits, (n_hits + 1) * sizeof(MsHit));
  const size_t band_samples = band_hits_cap * (size_t)K + 1;     // per staging half
  const size_t n_half = overlap ? 2 : 1;
  ENS(sc->staging, n_half * band_samples * sizeof(float4));
  if (want_feat) ENS(sc->staging_feat, n_half * band_samples * feat_bytes);
  if (want_slots) ENS(sc->staging_gate, n_half * band_samples * sizeof(float4));
  if (want_slots) ENS(sc->staging_coef, (band_hits_cap * (size_t)K + 1) * sizeof(float4));
  const bool keep_order = (opts->flags & MS_FLAG_KEEP_ORDER) != 0;
  if (keep_order) {
    ENS(sc->dbg_ord, (n_samples + 1) * 4);
    CK(cudaMemsetAsync(sc->dbg_ord.p, 0xff, (n_samples + 1) * 4, st));   // a rank stage (e) never writes is seen
  }

  MsBandArgs ba;
  ba.grid = grid; ba.K = K; ba.prim_bits = prim_bits; ba.n_prims = N; ba.wave_c = wave_c; ba.n_bands = n_bands;
  ba.cap_hits = (uint32_t)(cap_hits > 0xffffffffull ? 0xffffffffull : cap_hits); ba.P = P; ba.P_dev = P_dev;
  ba.keys = sorted; ba.tile_start = (uint32_t *)sc->tile_start.p; ba.ray_off = (uint32_t *)sc->ray_off.p;
  ba.emit_off = (uint32_t *)sc->emit_off.p; ba.rect = (int4 *)sc->rect.p; ba.pair_hits_i = (uint32_t *)sc->pair_hits_i.p;
  ba.key2_a = (uint64_t *)sc->key2_a.p; ba.key2_b = (uint64_t *)sc->key2_b.p;
  ba.sort_scratch = (uint32_t *)sc->sort_scratch.p; ba.scan_scratch = (uint32_t *)sc->scan_scratch.p;
  ba.slot_of = (uint32_t *)sc->slot_of.p; ba.pair_hits_j = (uint32_t *)sc->pair_hits_j.p; ba.pair_off = (uint32_t *)sc->pair_off.p;
  ba.flags = (uint32_t *)sc->flags.p; ba.gid = (uint32_t *)sc->gid.p;
  ba.grp_key = (uint32_t *)sc->grp_key.p; ba.grp_prim = (uint32_t *)sc->grp_prim.p; ba.grp_iv0 = (uint32_t *)sc->grp_iv0.p;
  ba.grp_blocks = (uint32_t *)sc->grp_blocks.p; ba.blk_off = (uint32_t *)sc->blk_off.p;
  ba.bw = (uint2 *)sc->bw.p; ba.bands = (MsBand *)sc->bands.p; ba.counters = counters;
  ba.ray_hits = (uint32_t *)sc->ray_hits.p; ba.ray_off_w = (uint32_t *)sc->ray_off.p; ba.R = R;
  ba.hit_cap = nosync ? (uint32_t)hit_cap : 0u;
  ba.fuse_ray_scan = small_c_scan && !banded ? 1 : 0; ba.fuse_stats = small_c && !banded ? 1 : 0;
  if (nosync && !small_ab) CK(cudaMemsetAsync(sc->pair_hits_j.p, 0, (P + 2) * 4, st));   // slots beyond the device's pair count
  if (banded) CK(ms_order_banded(ba, st));
  else CK(ms_order_single(ba, st));
  // the band table comes back to the host: stage (e) is launched with one CTA per four rays of the band (the
  // hardware's CTA scheduler balances them; see ms_composite.cu).  A single band is the whole frame: no readback.
  std::vector<MsBand> band_tab((size_t)n_bands);
  if (n_bands == 1) {
    band_tab[0].q_lo = 0u; band_tab[0].q_hi = (uint32_t)R; band_tab[0].slot0 = 0u; band_tab[0].pad = 0u;
  } else {
    ENS_HOST(sc, (size_t)n_bands * sizeof(MsBand));
    CK(readback_words(sc->pinned_bands, sc->bands.p, (size_t)n_bands * sizeof(MsBand) / 4, st));
    CK(cudaStreamSynchronize(st));
    memcpy(band_tab.data(), sc->pinned_bands, (size_t)n_bands * sizeof(MsBand));
  }

  ia.wave_c = wave_c;
  ia.guard = nosync ? counters : nullptr;
  ia.intervals = (MsInterval *)sc->intervals.p;
  ia.hits = (MsHit *)sc->hits.p;
  CK(ms_isect_fill(ia, st));

  // ---- per band: (d) grouped per-primitive MLP, wave by wave, then (e) merge + composite ----------------
  MsMlpArgs ma;
  ma.shape = sc->shape; ma.cam = cam; ma.K = K; ma.falloff = sc->falloff;
  ma.center = sc->center; ma.A = sc->A; ma.weights_f32 = sc->weights_f32;
  ma.segs.iv0 = (uint32_t *)sc->grp_iv0.p; ma.segs.cnt = nullptr; ma.segs.blk_off = (uint32_t *)sc->blk_off.p;
  ma.segs.prim = banded ? (uint32_t *)sc->grp_prim.p : nullptr;
  ma.n_blocks_hint = 0;
  ma.intervals = (MsInterval *)sc->intervals.p;
  ma.staging = (float4 *)sc->staging.p;
  ma.staging_feat = want_feat ? sc->staging_feat.p : nullptr;
  ma.feat_half = feat_half ? 1 : 0;
  ma.staging_gate = want_slots ? (float4 *)sc->staging_gate.p : nullptr;
  MsCompositeArgs ca;
  ca.grid = grid; ca.K = K; ca.n_feat = sc->shape.n_feat; ca.t_stop = opts->t_stop;
  ca.contact = sc->shape.mode == MS_MODE_CONTACT;
  ca.tile_order = tile_order;
  ca.ray_off = (uint32_t *)sc->ray_off.p; ca.hits = (MsHit *)sc->hits.p; ca.staging = (float4 *)sc->staging.p;
  ca.staging_feat = want_feat ? sc->staging_feat.p : nullptr;
  ca.feat_half = feat_half ? 1 : 0;
  ca.gates = want_slots ? (const float4 *)sc->staging_gate.p : nullptr;
  ca.coef = want_slots ? (float4 *)sc->staging_coef.p : nullptr;
  ca.slots = sc->slots; ca.c_f = sc->slot_cf;
  ca.keys = sorted; ca.tile_start = (uint32_t *)sc->tile_start.p; ca.pair_hits = (uint32_t *)sc->pair_hits_i.p;
  ca.prim_bits = prim_bits;
  ca.dbg_ord = keep_order ? (uint32_t *)sc->dbg_ord.p : nullptr;
  ca.counters = counters;
  ca.out_rgb = out_rgb; ca.out_alpha = out_alpha; ca.out_feat = (want_feat || want_slots) ? out_feat : nullptr;
  MsWaveArgs wa;
  wa.grid = grid; wa.K = K; wa.prim_bits = prim_bits; wa.wave_c = wave_c; wa.contact = ca.contact;
  wa.t_stop = opts->t_stop;
  wa.margin = 1e-4f * (1.0f + fabsf(cam.o[0]) + fabsf(cam.o[1]) + fabsf(cam.o[2]));
  wa.keys = sorted; wa.tile_start = (uint32_t *)sc->tile_start.p; wa.ray_off = (uint32_t *)sc->ray_off.p;
  wa.hits = (MsHit *)sc->hits.p; wa.staging = (float4 *)sc->staging.p; wa.bands = (MsBand *)sc->bands.p;
  wa.bw = (uint2 *)sc->bw.p; wa.alive = (uint8_t *)sc->alive.p; wa.intervals = (MsInterval *)sc->intervals.p;
  wa.intervals_c = (MsInterval *)sc->intervals_c.p; wa.hit_e = (float *)sc->hit_e.p;
  wa.grp_iv0 = (uint32_t *)sc->grp_iv0.p; wa.grp_cnt_c = (uint32_t *)sc->grp_cnt_c.p;
  wa.grp_blocks_c = (uint32_t *)sc->grp_blocks_c.p; wa.blk_off_c = (uint32_t *)sc->blk_off_c.p;
  wa.counters = counters; wa.n_sm = sc->n_sm;
  if (overlap && !sc->st2) {
    CK(cudaStreamCreateWithFlags(&sc->st2, cudaStreamNonBlocking));
    for (int i = 0; i < 2; ++i) {
      CK(cudaEventCreateWithFlags(&sc->ev_mlp[i], cudaEventDisableTiming));
      CK(cudaEventCreateWithFlags(&sc->ev_comp[i], cudaEventDisableTiming));
    }
  }
  auto recc = [&](int i) -> cudaError_t {           // stage (e) events of an overlapped view, on the second stream
    if (!timing) return cudaSuccess;
    std::vector<cudaEvent_t> &ev = sc->evs[sc->ev_cur].evc;
    while ((int)ev.size() <= i) {
      cudaEvent_t e;
      cudaError_t r = cudaEventCreate(&e);
      if (r != cudaSuccess) return r;
      ev.push_back(e);
    }
    return cudaEventRecord(ev[i], sc->st2);
  };
  for (int b = 0; b < n_bands; ++b) {
    const int half = overlap ? (b & 1) : 0;
    ma.staging = (float4 *)sc->staging.p + (size_t)half * band_samples;
    ma.staging_feat = want_feat ? (void *)((char *)sc->staging_feat.p + (size_t)half * band_samples * feat_bytes) : nullptr;
    ma.staging_gate = want_slots ? (float4 *)sc->staging_gate.p + (size_t)half * band_samples : nullptr;
    ca.staging = ma.staging; ca.staging_feat = ma.staging_feat; ca.gates = ma.staging_gate;
    wa.staging = ma.staging;
    if (overlap && b >= 2) CK(cudaStreamWaitEvent(st, sc->ev_comp[half], 0));   // stage (e) of band b - 2 has left this half
    CK(rec(3 + 2 * b));
    ma.segs.band = (MsBand *)sc->bands.p + b;
    for (int w = 0; w < n_waves; ++w) {
      ma.segs.range = (uint2 *)sc->bw.p + (size_t)b * MS_MAX_WAVES + w;
      if (w > 0) {    // rays that have stopped drop out of this wave before their samples are encoded
        wa.band = b; wa.wave = w;
        CK(ms_wave_prepare(wa, st));
        ma.segs.cnt = (uint32_t *)sc->grp_cnt_c.p; ma.segs.blk_off = (uint32_t *)sc->blk_off_c.p;
        ma.intervals = (MsInterval *)sc->intervals_c.p;
      } else {
        ma.segs.cnt = nullptr; ma.segs.blk_off = (uint32_t *)sc->blk_off.p;
        ma.intervals = (MsInterval *)sc->intervals.p;
      }
      if (path == MS_PATH_BF16_TC) CK(ms_mlp_tc(sc->tc, ma, st));
      else CK(ms_mlp_f32(ma, st));
    }
    CK(rec(4 + 2 * b));
    ca.band = band_tab[b];
    if (overlap) {
      CK(cudaEventRecord(sc->ev_mlp[half], st));
      CK(cudaStreamWaitEvent(sc->st2, sc->ev_mlp[half], 0));
      CK(recc(2 * b));
      CK(ms_composite(ca, sc->st2));
      CK(recc(2 * b + 1));
      CK(cudaEventRecord(sc->ev_comp[half], sc->st2));
    } else {
      CK(ms_composite(ca, st));
    }
  }
  if (overlap) CK(cudaStreamWaitEvent(st, sc->ev_comp[(n_bands - 1) & 1], 0));   // st2 is in order: this covers every band
  CK(rec(3 + 2 * n_bands));
  if (timing) {
    sc->evs[sc->ev_cur].bands = n_bands;
    sc->evs[sc->ev_cur].overlap = overlap;
    sc->evs[sc->ev_cur].pending = true;
    sc->ev_valid = true;
  }
  CK(cudaMemcpyAsync(sc->pinned + 1, counters, (MS_CNT_N + 2) * 4, cudaMemcpyDeviceToHost, st));
  CK(cudaEventRecord(sc->frame_done, st));
  sc->frame_pending = true;
  sc->stats = ms_stats{};
  sc->stats.n_launches = (int64_t)(ms_launch_count - launches0);
  sc->stats.n_pairs = (int64_t)P;                    // no-sync: capacities, replaced by the counts in finish_frame
  sc->stats.n_intervals = (int64_t)n_hits;
  sc->stats.n_samples = (int64_t)n_samples;
  sc->stats.n_samples_evaluated = (int64_t)n_samples;
  sc->frame_nosync = nosync;
  sc->stats.no_sync = nosync ? 1 : 0;
  if (!nosync) {
    sc->hist.valid = n_bands == 1 && !banded;
    sc->hist.H = H; sc->hist.W = W; sc->hist.tile = tile; sc->hist.K = K; sc->hist.path = path;
    sc->hist.feat = want_feat ? 1 : 0; sc->hist.slots = want_slots ? 1 : 0; sc->hist.tile_order = tile_order;
    sc->hist.pairs = P;
  }
  sc->stats.n_bands = n_bands;
  sc->stats.n_waves = n_waves;
  sc->stats.staging_bytes = (int64_t)(n_half * band_hits_cap * (size_t)K * sample_bytes);   // what this view needed
  sc->stats.scratch_bytes = (int64_t)scratch_total(sc);
  sc->dbg_K = K;
  sc->last.valid = true; sc->last.grid = grid; sc->last.cam = cam; sc->last.K = K; sc->last.n_bands = n_bands;
  sc->last.n_waves = n_waves; sc->last.banded = banded ? 1 : 0; sc->last.path = path; sc->last.n_hits = n_hits;
  sc->last.t_stop = opts->t_stop;
  if (opts->flags & MS_FLAG_KEEP_DEBUG) {
    sc->debug_valid = true;
    sc->order_valid = keep_order;
    sc->dbg_H = H; sc->dbg_W = W; sc->dbg_prim_bits = prim_bits;
    sc->dbg_grid = grid; sc->dbg_keys = sorted;
    sc->dbg_contact = ca.contact;
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
  if (mlp->mode == MS_MODE_CONTACT && !(mlp->falloff >= 0.0f)) return MS_ERR_INVALID_ARG;
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
  sc->falloff = mlp->falloff;
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
  CKC(cudaDeviceGetAttribute(&sc->n_sm, cudaDevAttrMultiProcessorCount, sc->device));
  CKC(cudaMalloc(&sc->center, n * 12));
  CKC(cudaMalloc(&sc->quat, n * 16));
  CKC(cudaMalloc(&sc->scale, n * 12));
  CKC(cudaMalloc(&sc->A, n * 36));
  CKC(cudaMalloc(&sc->M, n * 36));
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
  CKC(ms_prep_prims(sc->n, sc->center, sc->quat, sc->scale, sc->A, sc->M, d_bad, 0));
  int bad = 0;
  CKC(cudaMemcpy(&bad, d_bad, 4, cudaMemcpyDeviceToHost));
  if (bad) return fail(MS_ERR_INVALID_ARG);
  for (size_t i = 0; i < n * 3; ++i)
    if (!isfinite(prims->center[i])) return fail(MS_ERR_INVALID_ARG);
  CKC(cudaMallocHost(&sc->pinned, (MS_CNT_N + 4) * 4));
  memset(sc->pinned, 0, (MS_CNT_N + 4) * 4);
  CKC(cudaEventCreateWithFlags(&sc->frame_done, cudaEventDisableTiming));
  if (mlp->dtype == MS_BF16) {
    rc = ms_tc_pack(sh, sc->n, w.data(), &sc->tc);  // leaves tc.valid = false if the shape is not covered
    if (rc != MS_OK) return fail(rc);
  }
  if (sc->tc.valid) {
    sc->w_host.swap(w);       // the tensor path needs only the packed image: the fp32 copy (633 MB at CFG4) goes
                              // to the device when the fp32 path or the backward pass is first asked for
  } else {
    CKC(cudaMalloc(&sc->weights_f32, n * (size_t)params * 4));
    CKC(cudaMemcpy(sc->weights_f32, w.data(), n * (size_t)params * 4, cudaMemcpyHostToDevice));
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
  for (Buf *b : scratch_bufs(sc)) free_buf(*b);
  free_buf(sc->bwd_rgb); free_buf(sc->bwd_alpha); free_buf(sc->bwd_ord); free_buf(sc->bwd_gstage);
  free_buf(sc->bwd_ivgrad); free_buf(sc->bwd_gA);
  free_buf(sc->host_rgb); free_buf(sc->host_alpha); free_buf(sc->host_feat);
  free_buf(sc->host2_rgb); free_buf(sc->host2_alpha); free_buf(sc->host2_feat);
  for (int i = 0; i < 2; ++i) {
    if (sc->ev_rendered[i]) cudaEventDestroy(sc->ev_rendered[i]);
    if (sc->ev_copied[i]) cudaEventDestroy(sc->ev_copied[i]);
  }
  if (sc->copy_st) cudaStreamDestroy(sc->copy_st);
  if (sc->pinned) cudaFreeHost(sc->pinned);
  if (sc->pinned_bands) cudaFreeHost(sc->pinned_bands);
  for (auto &E : sc->evs) {
    for (cudaEvent_t e : E.ev) cudaEventDestroy(e);
    for (cudaEvent_t e : E.evc) cudaEventDestroy(e);
  }
  if (sc->frame_done) cudaEventDestroy(sc->frame_done);
  for (int i = 0; i < 2; ++i) {
    if (sc->ev_mlp[i]) cudaEventDestroy(sc->ev_mlp[i]);
    if (sc->ev_comp[i]) cudaEventDestroy(sc->ev_comp[i]);
  }
  if (sc->st2) cudaStreamDestroy(sc->st2);
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
  const bool two = n_views > 1;            // several views: copy view v beside the render of view v + 1
  if (two) {
    ENS(sc->host2_rgb, px * 12);
    ENS(sc->host2_alpha, px * 4);
    if (feat) ENS(sc->host2_feat, px * (size_t)nf * 4);
    if (!sc->copy_st) {
      CK(cudaStreamCreateWithFlags(&sc->copy_st, cudaStreamNonBlocking));
      for (int i = 0; i < 2; ++i) {
        CK(cudaEventCreateWithFlags(&sc->ev_rendered[i], cudaEventDisableTiming));
        CK(cudaEventCreateWithFlags(&sc->ev_copied[i], cudaEventDisableTiming));
      }
    }
  }
  for (int v = 0; v < n_views; ++v) {
    const int b = two ? (v & 1) : 0;
    float *d_rgb = (float *)(b ? sc->host2_rgb.p : sc->host_rgb.p), *d_alpha = (float *)(b ? sc->host2_alpha.p : sc->host_alpha.p);
    float *d_feat = feat ? (float *)(b ? sc->host2_feat.p : sc->host_feat.p) : nullptr;
    if (two && v >= 2) CK(cudaStreamWaitEvent(st, sc->ev_copied[b], 0));      // view v - 2 has left this buffer
    rc = render_view(sc, cams + v, H, W, opts, d_rgb, d_alpha, d_feat);
    if (rc != MS_OK) {
      if (two) cudaStreamSynchronize(sc->copy_st);
      return rc;
    }
    cudaStream_t cs = st;
    if (two) {
      CK(cudaEventRecord(sc->ev_rendered[b], st));
      CK(cudaStreamWaitEvent(sc->copy_st, sc->ev_rendered[b], 0));
      cs = sc->copy_st;
    }
    CK(cudaMemcpyAsync(host_rgb + v * px * 3, d_rgb, px * 12, cudaMemcpyDeviceToHost, cs));
    CK(cudaMemcpyAsync(host_alpha + v * px, d_alpha, px * 4, cudaMemcpyDeviceToHost, cs));
    if (feat) CK(cudaMemcpyAsync(host_feat + v * px * nf, d_feat, px * (size_t)nf * 4, cudaMemcpyDeviceToHost, cs));
    if (two) CK(cudaEventRecord(sc->ev_copied[b], sc->copy_st));
  }
  if (two) CK(cudaStreamSynchronize(sc->copy_st));
  CK(cudaStreamSynchronize(st));
  if (opts->flags & MS_FLAG_NO_SYNC) {   // a view that outgrew the scratch sized from its predecessor: once more, sizing
    rc = finish_frame(sc);
    if (rc != MS_OK) return rc;
    if (sc->stats.overflow) {
      ms_opts o2 = *opts;
      o2.flags &= ~MS_FLAG_NO_SYNC;
      return ms_render_host(sc, cams, n_views, H, W, &o2, host_rgb, host_alpha, host_feat);
    }
  }
  return MS_OK;
}

int ms_backward(ms_scene *sc, const ms_camera *camera, int32_t H, int32_t W, const ms_opts *opts, const float *d_rgb,
                float *g_weights, float *g_center, float *g_quat, float *g_scale) {
  if (!d_rgb || !g_weights || !g_center) return MS_ERR_INVALID_ARG;
  int rc = check_render_args(sc, camera, 1, H, W, opts, d_rgb, d_rgb);
  if (rc != MS_OK) return rc;
  if (sc->shape.mode != MS_MODE_LOCAL || ms_mlp_bwd_smem(sc->shape) == 0) return MS_ERR_UNSUPPORTED_SHAPE;
  cudaStream_t st = (cudaStream_t)opts->stream;
  // forward stages (a)-(e) on the fp32 path with the whole frame staged (one band, no waves): the backward kernels
  // read the staged (rgb, e) of every sample
  ms_opts o2 = *opts;
  o2.band_bytes = -1; o2.waves = -1; o2.path = MS_PATH_FP32;
  o2.flags &= ~(MS_FLAG_KEEP_ORDER | MS_FLAG_TILE_ORDER | MS_FLAG_STAGE_TIMES);
  const size_t px = (size_t)H * W;
  ENS(sc->bwd_rgb, px * 12);
  ENS(sc->bwd_alpha, px * 4);
  rc = render_view(sc, camera, H, W, &o2, (float *)sc->bwd_rgb.p, (float *)sc->bwd_alpha.p, nullptr);
  if (rc != MS_OK) return rc;
  if (!sc->last.valid || sc->last.n_bands != 1 || sc->last.banded) return MS_ERR_CUDA;
  const size_t n_hits = sc->last.n_hits, n_samples = n_hits * (size_t)sc->last.K;
  if (n_hits == 0) return MS_OK;
  const long long launches0 = ms_launch_count;
  ENS(sc->bwd_ord, (n_samples + 1) * 4);
  ENS(sc->bwd_gstage, (n_samples + 1) * sizeof(float4));
  ENS(sc->bwd_ivgrad, (n_hits + 1) * 32);
  ENS(sc->bwd_gA, (size_t)sc->n * 36);
  CK(cudaMemsetAsync(sc->bwd_ivgrad.p, 0, (n_hits + 1) * 32, st));
  CK(cudaMemsetAsync(sc->bwd_gA.p, 0, (size_t)sc->n * 36, st));
  MsCompositeBwdArgs cb;
  cb.grid = sc->last.grid; cb.K = sc->last.K; cb.t_stop = sc->last.t_stop;
  cb.ray_off = (uint32_t *)sc->ray_off.p; cb.hits = (MsHit *)sc->hits.p; cb.staging = (float4 *)sc->staging.p;
  cb.d_rgb = d_rgb; cb.ord = (uint32_t *)sc->bwd_ord.p; cb.gstage = (float4 *)sc->bwd_gstage.p;
  CK(ms_composite_bwd(cb, st));
  MsMlpBwdArgs mb;
  mb.shape = sc->shape; mb.cam = sc->last.cam; mb.K = sc->last.K; mb.n_prims = sc->n; mb.n_hits = n_hits;
  mb.center = sc->center; mb.A = sc->A; mb.quat = sc->quat; mb.scale = sc->scale; mb.weights_f32 = sc->weights_f32;
  mb.segs.iv0 = (uint32_t *)sc->grp_iv0.p; mb.segs.cnt = nullptr; mb.segs.blk_off = (uint32_t *)sc->blk_off.p;
  mb.segs.prim = nullptr; mb.segs.range = (uint2 *)sc->bw.p; mb.segs.band = (MsBand *)sc->bands.p;
  mb.intervals = (MsInterval *)sc->intervals.p; mb.staging = (float4 *)sc->staging.p;
  mb.gstage = (float4 *)sc->bwd_gstage.p; mb.ivgrad = (float *)sc->bwd_ivgrad.p; mb.gA = (float *)sc->bwd_gA.p;
  mb.g_weights = g_weights; mb.g_center = g_center; mb.g_quat = g_quat; mb.g_scale = g_scale;
  CK(ms_mlp_bwd(mb, st));
  sc->stats.n_launches += (int64_t)(ms_launch_count - launches0);
  return MS_OK;
}

int ms_last_stats(ms_scene *sc, ms_stats *out) {
  if (!sc || !out) return MS_ERR_INVALID_ARG;
  int rc = finish_frame(sc);
  if (rc != MS_OK) return rc;
  *out = sc->stats;
  return sc->stats.overflow ? MS_ERR_CAPACITY : MS_OK;
}

int ms_last_stage_ms(ms_scene *sc, float *ms) {
  if (!sc || !ms || !sc->ev_valid) return MS_ERR_INVALID_ARG;
  int rc = harvest_stage_times(sc, sc->ev_cur ^ 1);      // older view first: last_stage_ms ends as the newest
  if (rc == MS_OK) rc = harvest_stage_times(sc, sc->ev_cur);
  if (rc != MS_OK) return rc;
  for (int i = 0; i < MS_N_STAGES; ++i) ms[i] = sc->last_stage_ms[i];
  return MS_OK;
}

int ms_stage_accum(ms_scene *sc, double *ms_sum, int64_t *n_views, int32_t reset) {
  if (!sc) return MS_ERR_INVALID_ARG;
  int rc = harvest_stage_times(sc, sc->ev_cur ^ 1);
  if (rc == MS_OK) rc = harvest_stage_times(sc, sc->ev_cur);
  if (rc != MS_OK) return rc;
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
  std::vector<uint32_t> ts((size_t)sc->dbg_grid.n_tiles + 1);
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

// ray slot of pixel index y*W + x
static uint32_t slot_of_pixel(const MsGrid &g, size_t pix) {
  const int x = (int)(pix % (size_t)g.W), y = (int)(pix / (size_t)g.W);
  const int tx = x / g.tile, ty = y / g.tile;
  return (uint32_t)ms_tile_pos(g, tx, ty) * (uint32_t)(g.tile * g.tile) + (uint32_t)((y - ty * g.tile) * g.tile + (x - tx * g.tile));
}

int ms_debug_intervals(ms_scene *sc, int64_t *hit_offsets, int32_t *prim, float *t_in, float *delta, size_t cap,
                       size_t *n) {
  if (!sc || !sc->debug_valid) return MS_ERR_INVALID_ARG;
  CK(cudaDeviceSynchronize());
  const size_t nh = (size_t)sc->stats.n_intervals;
  const MsGrid &g = sc->dbg_grid;
  const size_t R = (size_t)sc->dbg_H * sc->dbg_W, Rs = (size_t)g.n_tiles * g.tile * g.tile;
  if (n) *n = nh;
  if (cap < nh) return MS_ERR_CAPACITY;
  std::vector<uint32_t> ro(Rs + 1);
  std::vector<MsHit> h(nh);
  CK(cudaMemcpy(ro.data(), sc->ray_off.p, (Rs + 1) * 4, cudaMemcpyDeviceToHost));
  if (nh) CK(cudaMemcpy(h.data(), sc->hits.p, nh * sizeof(MsHit), cudaMemcpyDeviceToHost));
  // the device numbers its rays tile by tile; the export is in pixel order y*W + x
  size_t tot = 0;
  for (size_t pix = 0; pix < R; ++pix) {
    const uint32_t q = slot_of_pixel(g, pix);
    if (hit_offsets) hit_offsets[pix] = (int64_t)tot;
    for (uint32_t i = ro[q]; i < ro[q + 1]; ++i, ++tot) {
      if (prim) prim[tot] = h[i].prim;
      if (t_in) t_in[tot] = h[i].t_in;
      if (delta) delta[tot] = h[i].delta;
    }
  }
  if (hit_offsets) hit_offsets[R] = (int64_t)tot;
  return MS_OK;
}

// canonical sample position, host side: this file is compiled without FMA contraction
static float host_sample_t(float t_in, float delta, int k, int contact) {
  if (contact) return t_in;
  volatile float kf = (float)k + 0.5f;
  volatile float m = kf * delta;
  return t_in + m;
}

int ms_debug_sample_order(ms_scene *sc, int32_t ray, int32_t *prim, int32_t *k, float *t, size_t cap, size_t *n) {
  if (!sc || !sc->debug_valid || !sc->order_valid || ray < 0 || ray >= sc->dbg_H * sc->dbg_W) return MS_ERR_INVALID_ARG;
  CK(cudaDeviceSynchronize());
  const uint32_t q = slot_of_pixel(sc->dbg_grid, (size_t)ray);
  uint32_t ro[2];
  CK(cudaMemcpy(ro, (uint32_t *)sc->ray_off.p + q, 8, cudaMemcpyDeviceToHost));
  const size_t K = (size_t)sc->dbg_K, nh = ro[1] - ro[0], ns = nh * K;
  if (n) *n = ns;
  if (cap < ns) return MS_ERR_CAPACITY;
  if (ns == 0) return MS_OK;
  std::vector<uint32_t> ord(ns);
  std::vector<MsHit> h(nh);
  CK(cudaMemcpy(ord.data(), (uint32_t *)sc->dbg_ord.p + (size_t)ro[0] * K, ns * 4, cudaMemcpyDeviceToHost));
  CK(cudaMemcpy(h.data(), (MsHit *)sc->hits.p + ro[0], nh * sizeof(MsHit), cudaMemcpyDeviceToHost));
  for (size_t r = 0; r < ns; ++r) {
    const uint32_t s = ord[r];
    if (s >= ns) return MS_ERR_CUDA;       // stage (e) never wrote this rank
    const size_t hh = s / K;
    const int kk = (int)(s % K);
    if (prim) prim[r] = h[hh].prim;
    if (k) k[r] = kk;
    if (t) t[r] = host_sample_t(h[hh].t_in, h[hh].delta, kk, sc->dbg_contact);
  }
  return MS_OK;
}

int ms_debug_sample_order_all(ms_scene *sc, int32_t *prim, int32_t *k, size_t cap, size_t *n) {
  if (!sc || !sc->debug_valid || !sc->order_valid) return MS_ERR_INVALID_ARG;
  CK(cudaDeviceSynchronize());
  const MsGrid &g = sc->dbg_grid;
  const size_t K = (size_t)sc->dbg_K, nh = (size_t)sc->stats.n_intervals, ns = nh * K;
  const size_t R = (size_t)sc->dbg_H * sc->dbg_W, Rs = (size_t)g.n_tiles * g.tile * g.tile;
  if (n) *n = ns;
  if (cap < ns) return MS_ERR_CAPACITY;
  std::vector<uint32_t> ro(Rs + 1), ord(ns);
  std::vector<MsHit> h(nh);
  CK(cudaMemcpy(ro.data(), sc->ray_off.p, (Rs + 1) * 4, cudaMemcpyDeviceToHost));
  if (ns) CK(cudaMemcpy(ord.data(), sc->dbg_ord.p, ns * 4, cudaMemcpyDeviceToHost));
  if (nh) CK(cudaMemcpy(h.data(), sc->hits.p, nh * sizeof(MsHit), cudaMemcpyDeviceToHost));
  size_t tot = 0;
  for (size_t pix = 0; pix < R; ++pix) {
    const uint32_t q = slot_of_pixel(g, pix);
    const size_t base = (size_t)ro[q] * K, cnt = (size_t)(ro[q + 1] - ro[q]) * K;
    for (size_t r = 0; r < cnt; ++r, ++tot) {
      const uint32_t s = ord[base + r];
      if (s >= cnt) return MS_ERR_CUDA;    // stage (e) never wrote this rank
      if (prim) prim[tot] = h[ro[q] + s / K].prim;
      if (k) k[tot] = (int32_t)(s % K);
    }
  }
  return MS_OK;
}

int ms_debug_prim_frames(ms_scene *sc, float *A, float *M) {
  if (!sc) return MS_ERR_INVALID_ARG;
  if (A) CK(cudaMemcpy(A, sc->A, (size_t)sc->n * 36, cudaMemcpyDeviceToHost));
  if (M) CK(cudaMemcpy(M, sc->M, (size_t)sc->n * 36, cudaMemcpyDeviceToHost));
  return MS_OK;
}

int64_t ms_launch_count_total(void) { return (int64_t)ms_launch_count; }

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
