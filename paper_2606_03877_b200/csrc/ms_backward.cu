// ms_backward.cu -- backward pass of the render, fp32 SIMT (S:Sec.8(f) NEXT-4; the losses of P:132-134 Eq.8 need
// dL/dtheta_i and dL/d(mu_i, s_i, q_i)).  North-star (K-sample) mode.  After the forward stages (a)-(d) and the
// compositing backward of ms_composite.cu (which leaves (dL/dc, dL/de) per sample):
//   mlp_bwd_kernel       one CTA per 128-sample row block of one primitive, one thread per sample: recomputes the
//                        sample's activations into shared memory, backpropagates through sigmoid / softplus,
//                        the Linear+ReLU layers and Eq.5; the weight gradients of the block are the
//                        contractions X_l^T G_l over its 128 samples (threads over (in, out) pairs), added to
//                        g_weights with one atomic per weight and block; dL/du goes on to the interval:
//                        u = o' + t d'  ->  dL/do' += du, dL/dd' += t du, dL/dt_in += du.d', dL/ddelta += (k+1/2) du.d'
//   mlp_bwd_t_kernel     the same chain for widths that are multiples of 4, as register-tiled GEMMs (see its header):
//                        the kernel that runs for every configuration of the bench; mlp_bwd_kernel serves the rest
//   interval_bwd_kernel  one thread per (ray, primitive) interval: through delta = (t1 - t_in)/K, t_in = max(t0, t_near),
//                        t0,1 = (-b -+ s)/a, s = sqrt(b^2 - a c), a = d'.d', b = o'.d', c = o'.o' - 1 to (o', d'), then
//                        o' = A (o - mu), d' = A d: dL/dA += ..., dL/dmu -= A^T dL/do'
//   prim_bwd_kernel      one thread per primitive: A = diag(1/s) R(q/|q|)^T  ->  dL/ds, dL/dq
// Written from the chain rule itself; it shares no code with the test oracle, which states the same chain in fp64.
#include "ms_internal.cuh"
#include "ms_tile_gemm.cuh"

namespace {

constexpr int BT = MS_ROWS;   // threads per CTA = samples per row block

// odd leading dimension: a thread walking its own row and a warp walking one column are both conflict-free
__host__ __device__ inline int ld_of(int n) { return n | 1; }

struct BwdLayout {
  int ld0, ldw, ldg;          // leading dimensions of X0 (encoded input), H_l (hidden), G (gradients)
  size_t off_h[5];            // float offsets of X0 (index 0) and H_1..H_nh
  size_t off_g0, off_g1;      // the two gradient buffers
  size_t floats;
};
__host__ __device__ inline BwdLayout bwd_layout(const MsMlpShape &sh) {
  BwdLayout L;
  const int gmax = sh.width > sh.in_dim ? sh.width : sh.in_dim;
  L.ld0 = ld_of(sh.in_dim); L.ldw = ld_of(sh.width); L.ldg = ld_of(gmax);
  size_t o = 0;
  L.off_h[0] = o; o += (size_t)BT * L.ld0;
  for (int l = 1; l <= sh.n_hidden; ++l) { L.off_h[l] = o; o += (size_t)BT * L.ldw; }
  L.off_g0 = o; o += (size_t)BT * L.ldg;
  L.off_g1 = o; o += (size_t)BT * L.ldg;
  L.floats = o;
  return L;
}

__device__ __forceinline__ int find_seg(const uint32_t *__restrict__ bo, int n, uint32_t base, uint32_t b) {
  int lo = 0, hi = n;
  while (hi - lo > 1) {
    int mid = (lo + hi) >> 1;
    if (bo[mid] - base <= b) lo = mid; else hi = mid;
  }
  return lo;
}

__global__ void __launch_bounds__(BT) mlp_bwd_kernel(MsMlpBwdArgs a) {
  extern __shared__ __align__(16) float sm[];
  __shared__ int s_seg;
  const MsMlpShape &sh = a.shape;
  const BwdLayout L = bwd_layout(sh);
  const int tid = threadIdx.x;
  const uint2 r = *a.segs.range;
  const uint32_t *bo = a.segs.blk_off + r.x;
  const uint32_t base = bo[0], n_blocks = bo[r.y - r.x] - base;
  const int nh = sh.n_hidden, NL = nh + 1;
  for (uint32_t blk = blockIdx.x; blk < n_blocks; blk += gridDim.x) {
    __syncthreads();
    if (tid == 0) s_seg = find_seg(bo, (int)(r.y - r.x), base, blk);
    __syncthreads();
    const uint32_t g = r.x + (uint32_t)s_seg;
    const int prim = a.segs.prim ? (int)a.segs.prim[g] : (int)g;
    const uint32_t first = a.segs.iv0[g], count = a.segs.cnt ? a.segs.cnt[g] : a.segs.iv0[g + 1] - first;
    const uint64_t srow = (uint64_t)(blk - (bo[s_seg] - base)) * BT + tid;
    const uint32_t j = (uint32_t)(srow / (uint32_t)a.K);
    const int k = (int)(srow % (uint32_t)a.K);
    const bool live = j < count;
    const float *wp = a.weights_f32 + (size_t)prim * sh.params;
    const float *Ap = a.A + 9 * (size_t)prim, *mu = a.center + 3 * (size_t)prim;
    MsInterval iv;
    iv.t_in = 0.f; iv.delta = 0.f; iv.slot = 0; iv.dx = 0.f; iv.dy = 0.f; iv.dz = 1.f; iv.ray = 0; iv.prim = prim;
    if (live) iv = a.intervals[first + j];
    const float d[3] = {iv.dx, iv.dy, iv.dz};
    const float t = ms_sample_t(iv.t_in, iv.delta, k);
    float u[3];
    ms_sample_u(Ap, mu, a.cam.o, d, t, u);
    // ---- forward, activations into shared memory (a dead row carries zeros) ----
    float *X0 = sm + L.off_h[0] + (size_t)tid * L.ld0;
    {
      int ni = 0;
      X0[ni++] = u[0]; X0[ni++] = u[1]; X0[ni++] = u[2];
      float scale = 1.0f;
      for (int l = 0; l < sh.n_freq; ++l) {
        float sv[3], cv[3];
#pragma unroll
        for (int c = 0; c < 3; ++c) sincospif(scale * u[c], &sv[c], &cv[c]);
        X0[ni++] = sv[0]; X0[ni++] = sv[1]; X0[ni++] = sv[2];
        X0[ni++] = cv[0]; X0[ni++] = cv[1]; X0[ni++] = cv[2];
        scale *= 2.0f;
      }
      if (sh.use_viewdir) { X0[ni++] = d[0]; X0[ni++] = d[1]; X0[ni++] = d[2]; }
    }
    int off_w[5], n_in_l[5];
    {
      int off = 0, nin = sh.in_dim;
      for (int l = 0; l < NL; ++l) {
        const int no = l == nh ? sh.out_dim : sh.width;
        off_w[l] = off; n_in_l[l] = nin;
        off += nin * no + no; nin = no;
      }
    }
    for (int l = 0; l < nh; ++l) {
      const float *src = sm + L.off_h[l] + (size_t)tid * (l == 0 ? L.ld0 : L.ldw);
      float *dst = sm + L.off_h[l + 1] + (size_t)tid * L.ldw;
      const float *w = wp + off_w[l];
      const int nin = n_in_l[l], no = sh.width;
      const float *bias = w + nin * no;
      for (int o = 0; o < no; ++o) {
        float acc = __ldg(bias + o);
        for (int i = 0; i < nin; ++i) acc = fmaf(src[i], __ldg(w + i * no + o), acc);
        dst[o] = acc > 0.0f ? acc : 0.0f;
      }
    }
    float raw[4];
    {
      const float *src = sm + L.off_h[nh] + (size_t)tid * L.ldw;
      const float *w = wp + off_w[nh];
      const int nin = sh.width, no = sh.out_dim;
#pragma unroll
      for (int o = 0; o < 4; ++o) {
        float acc = __ldg(w + nin * no + o);
        for (int i = 0; i < nin; ++i) acc = fmaf(src[i], __ldg(w + i * no + o), acc);
        raw[o] = acc;
      }
    }
    // ---- gradient of the head's four outputs ----
    float *G = sm + L.off_g0, *Gn = sm + L.off_g1;
    float g_delta = 0.0f;
    {
      float gr[4] = {0.f, 0.f, 0.f, 0.f};
      if (live) {
        const size_t idx = (size_t)(uint32_t)iv.slot * (size_t)a.K + (size_t)k;
        const float4 gs = a.gstage[idx];
        const float e = a.staging[idx].w;
        const float c0 = 1.0f / (1.0f + expf(-raw[0])), c1 = 1.0f / (1.0f + expf(-raw[1])), c2 = 1.0f / (1.0f + expf(-raw[2]));
        gr[0] = gs.x * c0 * (1.0f - c0); gr[1] = gs.y * c1 * (1.0f - c1); gr[2] = gs.z * c2 * (1.0f - c2);
        const float sigma = fmaxf(raw[3], 0.0f) + log1pf(expf(-fabsf(raw[3])));
        gr[3] = -iv.delta * e * gs.w / (1.0f + expf(-raw[3]));     // softplus' = sigmoid
        g_delta = -sigma * e * gs.w;
      }
      float *gp = G + (size_t)tid * L.ldg;
#pragma unroll
      for (int o = 0; o < 4; ++o) gp[o] = gr[o];
    }
    // ---- layers, last to first: weight gradients of the block, then the gradient of the layer's input ----
    for (int l = nh; l >= 0; --l) {
      __syncthreads();                                   // G of every sample is written
      const int nin = n_in_l[l];
      const int no_ld = l == nh ? sh.out_dim : sh.width;   // stride of W's rows
      const int no = l == nh ? 4 : sh.width;               // outputs that carry a gradient
      const float *Xl = sm + L.off_h[l];
      const int ldx = l == 0 ? L.ld0 : L.ldw;
      float *gw = a.g_weights + (size_t)prim * sh.params + off_w[l];
      for (int idx = tid; idx < nin * no; idx += BT) {
        const int i = idx / no, o = idx - i * no;
        float acc = 0.0f;
        for (int s = 0; s < BT; ++s) acc = fmaf(Xl[(size_t)s * ldx + i], G[(size_t)s * L.ldg + o], acc);
        if (acc != 0.0f) atomicAdd(gw + i * no_ld + o, acc);
      }
      for (int o = tid; o < no; o += BT) {
        float acc = 0.0f;
        for (int s = 0; s < BT; ++s) acc += G[(size_t)s * L.ldg + o];
        if (acc != 0.0f) atomicAdd(gw + nin * no_ld + o, acc);
      }
      // gradient of this thread's layer input (ReLU of the previous layer folded in)
      const float *w = wp + off_w[l];
      const float *gp = G + (size_t)tid * L.ldg;
      const float *xin = Xl + (size_t)tid * ldx;
      float *gn = Gn + (size_t)tid * L.ldg;
      for (int i = 0; i < nin; ++i) {
        float acc = 0.0f;
        for (int o = 0; o < no; ++o) acc = fmaf(__ldg(w + i * no_ld + o), gp[o], acc);
        gn[i] = (l > 0 && !(xin[i] > 0.0f)) ? 0.0f : acc;
      }
      float *tmp = G; G = Gn; Gn = tmp;
    }
    // ---- Eq.5: dL/du, then the interval ----
    if (live) {
      const float *gx = G + (size_t)tid * L.ldg;
      float gu[3] = {gx[0], gx[1], gx[2]};
      float scale = 3.14159265358979323846f;
      for (int l = 0; l < sh.n_freq; ++l) {
#pragma unroll
        for (int c = 0; c < 3; ++c) {
          const float sn = X0[3 + 6 * l + c], cs = X0[3 + 6 * l + 3 + c];
          gu[c] += scale * (cs * gx[3 + 6 * l + c] - sn * gx[3 + 6 * l + 3 + c]);
        }
        scale *= 2.0f;
      }
      float dp[3];
#pragma unroll
      for (int rr = 0; rr < 3; ++rr) dp[rr] = Ap[3 * rr] * d[0] + Ap[3 * rr + 1] * d[1] + Ap[3 * rr + 2] * d[2];
      const float gt = gu[0] * dp[0] + gu[1] * dp[1] + gu[2] * dp[2];
      float *ig = a.ivgrad + (size_t)(first + j) * 8;
      atomicAdd(ig + 0, gu[0]); atomicAdd(ig + 1, gu[1]); atomicAdd(ig + 2, gu[2]);
      atomicAdd(ig + 3, t * gu[0]); atomicAdd(ig + 4, t * gu[1]); atomicAdd(ig + 5, t * gu[2]);
      atomicAdd(ig + 6, gt);
      atomicAdd(ig + 7, ((float)k + 0.5f) * gt + g_delta);
    }
  }
}

// The same computation as three register-tiled fp32 GEMMs per layer (any hidden width that is a multiple of 4).
// Activations and gradients live in shared memory FEATURE-major, X^T[feature][sample] with leading dimension BS + 4
// (= 4 mod 32 words): a thread owns a 4 x 4 tile and a warp is 8 tile columns x 4 tile rows, so every operand fetch is
// one float4 per lane with 8 (or 4) distinct 16-byte chunks per warp -- one shared-memory wavefront per 16 FMA
// instructions, where a thread per sample needs one wavefront per FMA instruction or four per float4 of weights.
//   forward   Z^T[o][s]  = b[o] + sum_i W[i][o] X^T[i][s]      tile = 4 outputs x 4 samples, weights staged as W[i][o]
//   dX        gX^T[i][s] = sum_o W[i][o] gZ^T[o][s]            tile = 4 inputs x 4 samples, weights staged as W^T[o][i]
//   dW        gW[i][o]   = sum_s X^T[i][s] gZ^T[o][s]          tile = 4 inputs x 4 outputs, a warp = 32 inputs x 16 outputs
// 512 threads per CTA, one CTA per SM (the activations of BS samples fill shared memory; BS = 128 = one row block, or
// 64 = half of one when 128 do not fit -- width 128, or four hidden layers of 64).  The forward sums run in the order of
// the generic kernel (bias first, inputs ascending); the backward sums differ from it only in the order of the fp32
// additions.
constexpr int TNT = TG_NT;            // threads per CTA
constexpr int TNW = TG_NW;            // warps per CTA
constexpr int TKP = TG_KP;            // contraction steps of one staged weight panel

__device__ __forceinline__ float4 lds4(const float *p) { return tg_lds4(p); }
__device__ __forceinline__ void sts4(float *p, float x, float y, float z, float w) { tg_sts4(p, x, y, z, w); }

struct TLayout {
  int R0, LS, LW;             // rows of X0^T (in_dim rounded up to 4), leading dimensions of the activations / the panel
  size_t off_x[5];            // float offsets of X0^T (index 0) and H_1^T..H_nh^T; the gradient of a layer's input
                              // overwrites that input in place (the owner of a tile reads its mask, then writes)
  size_t off_g0;              // ... except X0^T, which Eq.5's backward still needs: dL/dX0 has rows of its own
  size_t off_hd;              // 8 rows: the head's raw outputs (0..3) and their gradients (4..7)
  size_t off_ws;              // weight panel
  size_t off_acc;             // weight-gradient accumulators of the primitive being walked (0 floats if they do not fit)
  int acc_w[5], acc_b[5];     // per layer: float offset of its tile slots / bias slots inside the accumulators
  int acc_floats;
  size_t floats;
};
// weight-gradient slots of layer l: one per (warp tile, tile element, lane) -- lane-contiguous, so a warp adds its
// 16 tile elements without a bank conflict
__host__ __device__ inline int t_warp_tiles(int n_in, int n_out, bool head) {
  return ((n_in + 31) >> 5) * (head ? 1 : (n_out + 15) >> 4);
}
__host__ __device__ inline TLayout t_layout(const MsMlpShape &sh, int bs, bool with_acc) {
  TLayout L;
  L.R0 = (sh.in_dim + 3) & ~3;
  L.LS = bs + 4;
  L.LW = (sh.width > L.R0 ? sh.width : L.R0) + 4;
  size_t o = 0;
  L.off_x[0] = o; o += (size_t)L.R0 * L.LS;
  for (int l = 1; l <= sh.n_hidden; ++l) { L.off_x[l] = o; o += (size_t)sh.width * L.LS; }
  L.off_g0 = o; o += (size_t)L.R0 * L.LS;
  L.off_hd = o; o += (size_t)8 * L.LS;
  L.off_ws = o; o += (size_t)TKP * L.LW;
  L.off_acc = o;
  int ac = 0, nin = sh.in_dim;
  for (int l = 0; l <= sh.n_hidden; ++l) {
    const bool head = l == sh.n_hidden;
    const int no = head ? 4 : sh.width;
    L.acc_w[l] = ac; ac += t_warp_tiles(nin, no, head) * 512;
    L.acc_b[l] = ac; ac += (no + 15) & ~15;
    nin = sh.width;
  }
  L.acc_floats = with_acc ? ac : 0;
  o += (size_t)L.acc_floats;
  L.floats = o;
  return L;
}

template <int BS, bool ACC>
__global__ void __launch_bounds__(TNT, 1) mlp_bwd_t_kernel(MsMlpBwdArgs a) {
  constexpr int PASSES = BT / BS;     // passes per 128-row block
  constexpr int NCG = TNT / BS;       // threads per sample in the per-sample steps
  constexpr int NSW = BS / 32;        // warps side by side over the samples (8 sample tiles = 32 samples each)
  constexpr int NFW = (TNW / NSW) * 4;   // feature tiles (of 4) the CTA covers in one pass of a GEMM
  extern __shared__ __align__(16) float sm[];
  __shared__ int s_seg;
  const MsMlpShape &sh = a.shape;
  const TLayout L = t_layout(sh, BS, ACC);
  const int LS = L.LS, LW = L.LW, WD = sh.width;
  float *const DWS = sm + L.off_acc;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int srow_in = tid & (BS - 1), cg = tid / BS;      // per-sample steps: sample, helper index
  const int sg = (warp % NSW) * 8 + (lane & 7);           // GEMMs: sample tile (samples 4 sg .. 4 sg + 3)
  const int ft = (warp / NSW) * 4 + (lane >> 3);          //        feature tile inside a pass
  float *const WS = sm + L.off_ws;
  const uint2 r = *a.segs.range;
  const uint32_t *bo = a.segs.blk_off + r.x;
  const uint32_t base = bo[0], n_blocks = bo[r.y - r.x] - base;
  const int nh = sh.n_hidden, NL = nh + 1;
  int off_w[5], n_in_l[5];
  {
    int off = 0, nin = sh.in_dim;
    for (int l = 0; l < NL; ++l) {
      const int no = l == nh ? sh.out_dim : WD;
      off_w[l] = off; n_in_l[l] = nin;
      off += nin * no + no; nin = no;
    }
  }

  auto gemm_fwd = [&](const float *XT, int n_in, const float *Wg, int ldw, int n_out, bool relu, float *OUT) {
    tg_fwd<BS>(XT, n_in, Wg, ldw, n_out, relu, OUT, WS, LS, LW);
  };

  // gX^T = W gZ^T over the n_out leading outputs, masked by the ReLU of the layer below (XT = its output, or null)
  auto gemm_dx = [&](const float *G, int n_out, const float *Wg, int ldw, int n_in, const float *XT, float *GIN) {
    const int n_pad = (n_in + 3) & ~3, n_it = n_pad >> 2;
    for (int f0 = 0; f0 < n_it; f0 += NFW) {
      const int f = f0 + ft;
      const bool on = f < n_it;
      float acc[4][4];
#pragma unroll
      for (int q = 0; q < 4; ++q)
#pragma unroll
        for (int p = 0; p < 4; ++p) acc[q][p] = 0.0f;
      for (int o0 = 0; o0 < n_out; o0 += TKP) {
        const int kp = min(TKP, n_out - o0);
        __syncthreads();
        for (int e = tid; e < n_pad * kp; e += TNT) {      // W^T[o][i], inputs past n_in read as 0
          const int i = e / kp, c = e - i * kp;
          WS[c * LW + i] = i < n_in ? __ldg(Wg + (size_t)i * ldw + o0 + c) : 0.0f;
        }
        __syncthreads();
        if (on) {
          const float *gp = G + (size_t)o0 * LS + 4 * sg, *wq = WS + 4 * f;
#pragma unroll 4
          for (int c = 0; c < kp; ++c) {
            const float4 g4 = lds4(gp + (size_t)c * LS), w4 = lds4(wq + c * LW);
            const float gs[4] = {g4.x, g4.y, g4.z, g4.w}, ws[4] = {w4.x, w4.y, w4.z, w4.w};
#pragma unroll
            for (int q = 0; q < 4; ++q)
#pragma unroll
              for (int p = 0; p < 4; ++p) acc[q][p] = fmaf(ws[q], gs[p], acc[q][p]);
          }
        }
      }
      if (on) {
#pragma unroll
        for (int q = 0; q < 4; ++q) {
          const size_t at = (size_t)(4 * f + q) * LS + 4 * sg;
          if (XT) {
            const float4 x4 = lds4(XT + at);
            sts4(GIN + at, x4.x > 0.0f ? acc[q][0] : 0.0f, x4.y > 0.0f ? acc[q][1] : 0.0f,
                 x4.z > 0.0f ? acc[q][2] : 0.0f, x4.w > 0.0f ? acc[q][3] : 0.0f);
          } else {
            sts4(GIN + at, acc[q][0], acc[q][1], acc[q][2], acc[q][3]);
          }
        }
      }
    }
  };

  // gW += X G^T over the samples of the pass (and the bias row: sum_s gZ^T[o][s]).  A warp = 32 inputs x 16 outputs:
  // lane (it, ot) holds the inputs 32 iw + 8 q + it and the outputs 16 ow + 4 q' + ot, rows that sit 4 banks apart.
  // The head (4 outputs) gives its 4 lane rows to a further split of the samples instead.
  auto gemm_dw = [&](const float *XT, int n_in, const float *G, int n_out, bool head, float *gw, int ldw, int l) {
    const int n_iw = (n_in + 31) >> 5, n_ow = head ? 1 : (n_out + 15) >> 4;
    const int n_wt = n_iw * n_ow;
    const int it = lane & 7, ot = lane >> 3;
    // one (warp tile, sample part) item: acc[q][p] = sum_s X^T[i_q][s] gZ^T[o_p][s], bsum[p] = sum_s gZ^T[o_p][s]
    auto item_sums = [&](int wt, int part, int SS, float (&acc)[4][4], float (&bsum)[4]) {
      const int iw = wt / n_ow, ow = wt - iw * n_ow;
      int s_n = BS / SS, s_lo = part * s_n;
      if (head) { s_n >>= 2; s_lo += ot * s_n; }
      const float *xr = XT + (size_t)(32 * iw + it) * LS + s_lo;
      const float *gr = G + (size_t)(head ? 0 : 16 * ow + ot) * LS + s_lo;
      const int gstep = head ? LS : 4 * LS;
      const bool do_bias = iw == 0;                        // warp-uniform
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        bsum[q] = 0.0f;
#pragma unroll
        for (int p = 0; p < 4; ++p) acc[q][p] = 0.0f;
      }
      for (int s0 = 0; s0 < s_n; s0 += 4) {
        float4 x[4], g4[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) {
          x[q] = lds4(xr + (size_t)(8 * q) * LS + s0);
          g4[q] = lds4(gr + (size_t)q * gstep + s0);
        }
#pragma unroll
        for (int q = 0; q < 4; ++q)
#pragma unroll
          for (int p = 0; p < 4; ++p) {
            float v = acc[q][p];
            v = fmaf(x[q].x, g4[p].x, v); v = fmaf(x[q].y, g4[p].y, v);
            v = fmaf(x[q].z, g4[p].z, v); v = fmaf(x[q].w, g4[p].w, v);
            acc[q][p] = v;
          }
        if (do_bias) {
#pragma unroll
          for (int p = 0; p < 4; ++p) bsum[p] += (g4[p].x + g4[p].y) + (g4[p].z + g4[p].w);
        }
      }
    };
    // bias slot of output o_p of this lane (the head's four lane rows are sample parts: a slot each)
    auto bias_slot = [&](int ow, int p) { return head ? 4 * p + ot : 16 * ow + 4 * p + ot; };
    float acc[4][4], bsum[4];
    if (ACC) {
      // into the primitive's accumulators, slot (warp tile, element, lane): every slot has ONE owner -- with two
      // sample parts per tile the odd part hands its sums over through the idle weight panel
      float *const BSC = sm + L.off_hd;                    // rows 0..3 (the head's raw outputs, consumed): bias hand-over
      const bool two = 2 * n_wt <= TNW && BS / 2 >= (head ? 16 : 4) && n_wt * 512 <= TKP * LW;
      if (!two) {
        for (int wt = warp; wt < n_wt; wt += TNW) {
          item_sums(wt, 0, 1, acc, bsum);
          float *slot = DWS + L.acc_w[l] + wt * 512 + lane;
#pragma unroll
          for (int q = 0; q < 4; ++q)
#pragma unroll
            for (int p = 0; p < 4; ++p) slot[(q * 4 + p) * 32] += acc[q][p];
          if (wt < n_ow && it == 0) {
#pragma unroll
            for (int p = 0; p < 4; ++p) DWS[L.acc_b[l] + bias_slot(wt, p)] += bsum[p];
          }
        }
      } else {
        const int wt = warp >> 1, part = warp & 1;
        const bool active = wt < n_wt;
        if (active) item_sums(wt, part, 2, acc, bsum);
        if (active && part == 1) {
#pragma unroll
          for (int q = 0; q < 4; ++q)
#pragma unroll
            for (int p = 0; p < 4; ++p) WS[wt * 512 + (q * 4 + p) * 32 + lane] = acc[q][p];
          if (wt < n_ow && it == 0) {
#pragma unroll
            for (int p = 0; p < 4; ++p) BSC[bias_slot(wt, p)] = bsum[p];
          }
        }
        __syncthreads();
        if (active && part == 0) {
          float *slot = DWS + L.acc_w[l] + wt * 512 + lane;
#pragma unroll
          for (int q = 0; q < 4; ++q)
#pragma unroll
            for (int p = 0; p < 4; ++p) slot[(q * 4 + p) * 32] += acc[q][p] + WS[wt * 512 + (q * 4 + p) * 32 + lane];
          if (wt < n_ow && it == 0) {
#pragma unroll
            for (int p = 0; p < 4; ++p) DWS[L.acc_b[l] + bias_slot(wt, p)] += bsum[p] + BSC[bias_slot(wt, p)];
          }
        }
      }
      return;
    }
    int SS = 1;
    while (2 * SS * n_wt <= TNW && BS / (2 * SS) >= (head ? 16 : 4)) SS *= 2;
    for (int item = warp; item < n_wt * SS; item += TNW) {
      const int wt = item / SS, part = item - wt * SS;
      const int iw = wt / n_ow, ow = wt - iw * n_ow;
      item_sums(wt, part, SS, acc, bsum);
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        const int i = 32 * iw + 8 * q + it;
        if (i >= n_in) continue;
#pragma unroll
        for (int p = 0; p < 4; ++p) {
          const int o = head ? p : 16 * ow + 4 * p + ot;
          if (o < n_out && acc[q][p] != 0.0f) atomicAdd(gw + (size_t)i * ldw + o, acc[q][p]);
        }
      }
      if (iw == 0 && it == 0) {
#pragma unroll
        for (int p = 0; p < 4; ++p) {
          const int o = head ? p : 16 * ow + 4 * p + ot;
          if (o < n_out && bsum[p] != 0.0f) atomicAdd(gw + (size_t)n_in * ldw + o, bsum[p]);
        }
      }
    }
  };

  // the accumulators of one primitive go to g_weights (one atomic per non-zero slot) and are cleared
  auto flush_acc = [&](int prim) {
    __syncthreads();
    float *gwp = a.g_weights + (size_t)prim * sh.params;
    for (int l = 0; l < NL; ++l) {
      const bool head = l == nh;
      const int n_in = n_in_l[l], n_out = head ? 4 : WD, ldw = head ? sh.out_dim : WD;
      const int n_ow = head ? 1 : (n_out + 15) >> 4;
      const int n_slots = t_warp_tiles(n_in, n_out, head) * 512;
      float *gw = gwp + off_w[l];
      for (int e = tid; e < n_slots; e += TNT) {
        const float v = DWS[L.acc_w[l] + e];
        if (v == 0.0f) continue;
        DWS[L.acc_w[l] + e] = 0.0f;
        const int wt = e >> 9, qp = (e >> 5) & 15, ln = e & 31;
        const int iw = wt / n_ow, ow = wt - iw * n_ow;
        const int i = 32 * iw + 8 * (qp >> 2) + (ln & 7), o = head ? (qp & 3) : 16 * ow + 4 * (qp & 3) + (ln >> 3);
        if (i < n_in && o < n_out) atomicAdd(gw + (size_t)i * ldw + o, v);
      }
      for (int o = tid; o < n_out; o += TNT) {
        float v;
        if (head) {                   // a slot per sample part
          float *b = DWS + L.acc_b[l] + 4 * o;
          v = (b[0] + b[1]) + (b[2] + b[3]);
          b[0] = b[1] = b[2] = b[3] = 0.0f;
        } else {
          v = DWS[L.acc_b[l] + o];
          DWS[L.acc_b[l] + o] = 0.0f;
        }
        if (v != 0.0f) atomicAdd(gw + (size_t)n_in * ldw + o, v);
      }
    }
    __syncthreads();
  };

  if (ACC) {
    for (int e = tid; e < L.acc_floats; e += TNT) DWS[e] = 0.0f;
  }
  int acc_prim = -1;
  // with accumulators a CTA walks a contiguous run of (row block, pass) units -- consecutive units mostly belong to
  // one primitive; without, the CTAs interleave (neighbouring CTAs then share a primitive's weights in L2)
  const uint32_t n_units = n_blocks * PASSES;
  const uint32_t unit_lo = ACC ? (uint32_t)(((uint64_t)n_units * blockIdx.x) / gridDim.x) : blockIdx.x;
  const uint32_t unit_hi = ACC ? (uint32_t)(((uint64_t)n_units * (blockIdx.x + 1)) / gridDim.x) : n_units;
  const uint32_t unit_step = ACC ? 1u : gridDim.x;
  for (uint32_t unit = unit_lo; unit < unit_hi; unit += unit_step) {
    const uint32_t blk = unit / PASSES, pass = unit % PASSES;
    __syncthreads();
    if (tid == 0) s_seg = find_seg(bo, (int)(r.y - r.x), base, blk);
    __syncthreads();
    const uint32_t g = r.x + (uint32_t)s_seg;
    const int prim = a.segs.prim ? (int)a.segs.prim[g] : (int)g;
    if (ACC && prim != acc_prim) {                         // block-uniform
      if (acc_prim >= 0) flush_acc(acc_prim);
      acc_prim = prim;
    }
    const uint32_t first = a.segs.iv0[g], count = a.segs.cnt ? a.segs.cnt[g] : a.segs.iv0[g + 1] - first;
    const uint64_t srow = (uint64_t)(blk - (bo[s_seg] - base)) * BT + pass * BS + srow_in;
    const uint32_t j = (uint32_t)(srow / (uint32_t)a.K);
    const int k = (int)(srow % (uint32_t)a.K);
    const bool live = j < count;
    const float *wp = a.weights_f32 + (size_t)prim * sh.params;
    const float *Ap = a.A + 9 * (size_t)prim, *mu = a.center + 3 * (size_t)prim;
    MsInterval iv;
    iv.t_in = 0.f; iv.delta = 0.f; iv.slot = 0; iv.dx = 0.f; iv.dy = 0.f; iv.dz = 1.f; iv.ray = 0; iv.prim = prim;
    if (live) iv = a.intervals[first + j];
    const float d[3] = {iv.dx, iv.dy, iv.dz};
    const float t = ms_sample_t(iv.t_in, iv.delta, k);
    float *X0 = sm + L.off_x[0] + srow_in;                 // this sample's column of X0^T: feature i at X0[i LS]
    {                                 // the encoded input of the sample: frequency l by helper l mod NCG
      float u[3];
      ms_sample_u(Ap, mu, a.cam.o, d, t, u);
      if (cg == 0) {
        X0[0] = u[0]; X0[LS] = u[1]; X0[2 * LS] = u[2];
        if (sh.use_viewdir) { float *v = X0 + (size_t)(3 + 6 * sh.n_freq) * LS; v[0] = d[0]; v[LS] = d[1]; v[2 * LS] = d[2]; }
        for (int i = sh.in_dim; i < L.R0; ++i) X0[(size_t)i * LS] = 0.0f;
      }
      for (int l = cg; l < sh.n_freq; l += NCG) {
        const float scale = (float)(1 << l);
        float sv[3], cv[3];
#pragma unroll
        for (int c = 0; c < 3; ++c) sincospif(scale * u[c], &sv[c], &cv[c]);
        float *x = X0 + (size_t)(3 + 6 * l) * LS;
        x[0] = sv[0]; x[LS] = sv[1]; x[2 * LS] = sv[2];
        x[3 * LS] = cv[0]; x[4 * LS] = cv[1]; x[5 * LS] = cv[2];
      }
    }
    // ---- forward ----
    for (int l = 0; l < nh; ++l)
      gemm_fwd(sm + L.off_x[l], n_in_l[l], wp + off_w[l], WD, WD, true, sm + L.off_x[l + 1]);
    float *const RAW = sm + L.off_hd, *const GH = RAW + 4 * (size_t)LS;
    const int no_h = sh.out_dim;
    gemm_fwd(sm + L.off_x[nh], WD, wp + off_w[nh], no_h, 4, false, RAW);    // raw colour and density
    float g_delta = 0.0f;
    if (cg == 0) {                    // gradient of the head's four outputs (sigmoid colour, softplus density)
      const float *pp = RAW + srow_in;
      const float raw[4] = {pp[0], pp[LS], pp[2 * LS], pp[3 * LS]};
      float gr[4] = {0.f, 0.f, 0.f, 0.f};
      if (live) {
        const size_t idx = (size_t)(uint32_t)iv.slot * (size_t)a.K + (size_t)k;
        const float4 gs = a.gstage[idx];
        const float e = a.staging[idx].w;
        const float c0 = 1.0f / (1.0f + expf(-raw[0])), c1 = 1.0f / (1.0f + expf(-raw[1])), c2 = 1.0f / (1.0f + expf(-raw[2]));
        gr[0] = gs.x * c0 * (1.0f - c0); gr[1] = gs.y * c1 * (1.0f - c1); gr[2] = gs.z * c2 * (1.0f - c2);
        const float sigma = fmaxf(raw[3], 0.0f) + log1pf(expf(-fabsf(raw[3])));
        gr[3] = -iv.delta * e * gs.w / (1.0f + expf(-raw[3]));
        g_delta = -sigma * e * gs.w;
      }
      float *gq = GH + srow_in;
      gq[0] = gr[0]; gq[LS] = gr[1]; gq[2 * LS] = gr[2]; gq[3 * LS] = gr[3];
    }
    // ---- backward: the gradient of a layer's input replaces that input (X0^T keeps its values: Eq.5 needs them) ----
    for (int l = nh; l >= 0; --l) {
      __syncthreads();
      const bool head = l == nh;
      const int ldw = head ? no_h : WD, n_out = head ? 4 : WD;
      float *XT = sm + L.off_x[l];
      const float *G = head ? GH : sm + L.off_x[l + 1];
      gemm_dw(XT, n_in_l[l], G, n_out, head, a.g_weights + (size_t)prim * sh.params + off_w[l], ldw, l);
      gemm_dx(G, n_out, wp + off_w[l], ldw, n_in_l[l], l > 0 ? XT : nullptr, l > 0 ? XT : sm + L.off_g0);
    }
    __syncthreads();
    if (cg == 0) {                    // warps 0 .. BS / 32 - 1, whole
      float o8[8] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
      if (live) {
        const float *gx = sm + L.off_g0 + srow_in;
        float gu[3] = {gx[0], gx[LS], gx[2 * LS]};
        float scale = 3.14159265358979323846f;
        for (int l = 0; l < sh.n_freq; ++l) {
#pragma unroll
          for (int c = 0; c < 3; ++c) {
            const size_t is = (size_t)(3 + 6 * l + c) * LS, ic = (size_t)(3 + 6 * l + 3 + c) * LS;
            gu[c] += scale * (X0[ic] * gx[is] - X0[is] * gx[ic]);
          }
          scale *= 2.0f;
        }
        float dp[3];
#pragma unroll
        for (int rr = 0; rr < 3; ++rr) dp[rr] = Ap[3 * rr] * d[0] + Ap[3 * rr + 1] * d[1] + Ap[3 * rr + 2] * d[2];
        const float gt = gu[0] * dp[0] + gu[1] * dp[1] + gu[2] * dp[2];
        o8[0] = gu[0]; o8[1] = gu[1]; o8[2] = gu[2];
        o8[3] = t * gu[0]; o8[4] = t * gu[1]; o8[5] = t * gu[2];
        o8[6] = gt; o8[7] = ((float)k + 0.5f) * gt + g_delta;
      }
      // the K samples of an interval sit in K neighbouring lanes when K is a power of two up to 32 (row blocks start
      // at multiples of 128): summed by shuffles, one lane adds
      const int K = a.K;
      const bool grouped = K <= 32 && (K & (K - 1)) == 0;
      if (grouped) {
#pragma unroll
        for (int e = 0; e < 8; ++e)
          for (int o = K >> 1; o > 0; o >>= 1) o8[e] += __shfl_xor_sync(0xffffffffu, o8[e], o);
      }
      if (live && (!grouped || k == 0)) {
        float *ig = a.ivgrad + (size_t)(first + j) * 8;
#pragma unroll
        for (int e = 0; e < 8; ++e) atomicAdd(ig + e, o8[e]);
      }
    }
  }
  if (ACC && acc_prim >= 0) flush_acc(acc_prim);
}

__global__ void interval_bwd_kernel(MsMlpBwdArgs a) {
  const size_t i0 = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  const bool valid = i0 < a.n_hits;
  const size_t i = valid ? i0 : a.n_hits - 1;             // a lane past the end repeats the last interval and adds zeros
  const MsInterval iv = a.intervals[i];
  const int prim = iv.prim;
  const float *A = a.A + 9 * (size_t)prim, *mu = a.center + 3 * (size_t)prim;
  const float *ig = a.ivgrad + i * 8;
  const float v[3] = {a.cam.o[0] - mu[0], a.cam.o[1] - mu[1], a.cam.o[2] - mu[2]};
  const float d[3] = {iv.dx, iv.dy, iv.dz};
  float op[3], dp[3];
#pragma unroll
  for (int r = 0; r < 3; ++r) {
    op[r] = A[3 * r] * v[0] + A[3 * r + 1] * v[1] + A[3 * r + 2] * v[2];
    dp[r] = A[3 * r] * d[0] + A[3 * r + 1] * d[1] + A[3 * r + 2] * d[2];
  }
  const float qa = dp[0] * dp[0] + dp[1] * dp[1] + dp[2] * dp[2];
  const float qb = op[0] * dp[0] + op[1] * dp[1] + op[2] * dp[2];
  const float qc = op[0] * op[0] + op[1] * op[1] + op[2] * op[2] - 1.0f;
  const float disc = qb * qb - qa * qc;
  const float s = sqrtf(disc > 1e-30f ? disc : 1e-30f);
  const float t0 = (-qb - s) / qa, t1 = (-qb + s) / qa;
  const float Kf = (float)a.K;
  const float G1 = ig[7] / Kf;
  const float G0 = t0 > a.cam.t_near ? ig[6] - ig[7] / Kf : 0.0f;     // t_in clamped at t_near does not move
  const float ia = 1.0f / qa;
  const float gb = -(G0 + G1) * ia + (G1 - G0) * ia * qb / s;
  const float ga = -(G0 * t0 + G1 * t1) * ia - (G1 - G0) * ia * qc / (2.0f * s);
  const float gc = -(G1 - G0) / (2.0f * s);
  float gop[3], gdp[3];
#pragma unroll
  for (int r = 0; r < 3; ++r) {
    gop[r] = ig[r] + dp[r] * gb + 2.0f * op[r] * gc;
    gdp[r] = ig[3 + r] + 2.0f * dp[r] * ga + op[r] * gb;
  }
  // 12 sums per primitive: the intervals of a primitive are contiguous, so a warp mostly holds ONE primitive -- its
  // lanes are summed by shuffles and one lane adds; a warp that straddles primitives adds lane by lane
  float out[12];
#pragma unroll
  for (int r = 0; r < 3; ++r)
#pragma unroll
    for (int c = 0; c < 3; ++c) out[3 * r + c] = valid ? gop[r] * v[c] + gdp[r] * d[c] : 0.0f;
#pragma unroll
  for (int c = 0; c < 3; ++c) out[9 + c] = valid ? -(A[c] * gop[0] + A[3 + c] * gop[1] + A[6 + c] * gop[2]) : 0.0f;
  float *gA = a.gA + 9 * (size_t)prim, *gc3 = a.g_center + 3 * (size_t)prim;
  const bool uniform = __all_sync(0xffffffffu, prim == __shfl_sync(0xffffffffu, prim, 0));
  if (uniform) {
#pragma unroll
    for (int e = 0; e < 12; ++e) {
      float x = out[e];
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
      out[e] = x;
    }
    if ((threadIdx.x & 31) == 0) {
#pragma unroll
      for (int e = 0; e < 9; ++e) atomicAdd(gA + e, out[e]);
#pragma unroll
      for (int c = 0; c < 3; ++c) atomicAdd(gc3 + c, out[9 + c]);
    }
  } else if (valid) {
#pragma unroll
    for (int e = 0; e < 9; ++e) atomicAdd(gA + e, out[e]);
#pragma unroll
    for (int c = 0; c < 3; ++c) atomicAdd(gc3 + c, out[9 + c]);
  }
}

__global__ void prim_bwd_kernel(MsMlpBwdArgs a) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= a.n_prims) return;
  const float *A = a.A + 9 * (size_t)i, *gA = a.gA + 9 * (size_t)i, *sc = a.scale + 3 * (size_t)i;
  float G[9];     // dL/dR
#pragma unroll
  for (int r = 0; r < 3; ++r) {
    float gs = 0.0f;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      gs -= gA[3 * r + c] * A[3 * r + c] / sc[r];
      G[3 * c + r] = gA[3 * r + c] / sc[r];            // A[r][c] = R[c][r] / s[r]
    }
    if (a.g_scale) a.g_scale[3 * (size_t)i + r] += gs;
  }
  if (!a.g_quat) return;
  const float *qq = a.quat + 4 * (size_t)i;
  const float nr = sqrtf(qq[0] * qq[0] + qq[1] * qq[1] + qq[2] * qq[2] + qq[3] * qq[3]);
  const float w = qq[0] / nr, x = qq[1] / nr, y = qq[2] / nr, z = qq[3] / nr;
  float gq[4];
  gq[0] = 2 * (-z * G[1] + y * G[2] + z * G[3] - x * G[5] - y * G[6] + x * G[7]);
  gq[1] = 2 * (y * G[1] + z * G[2] + y * G[3] - 2 * x * G[4] - w * G[5] + z * G[6] + w * G[7] - 2 * x * G[8]);
  gq[2] = 2 * (-2 * y * G[0] + x * G[1] + w * G[2] + x * G[3] + z * G[5] - w * G[6] + z * G[7] - 2 * y * G[8]);
  gq[3] = 2 * (-2 * z * G[0] - w * G[1] + x * G[2] + w * G[3] - 2 * z * G[4] + y * G[5] + x * G[6] + y * G[7]);
  const float dot = gq[0] * w + gq[1] * x + gq[2] * y + gq[3] * z;
  const float qn[4] = {w, x, y, z};
#pragma unroll
  for (int c = 0; c < 4; ++c) a.g_quat[4 * (size_t)i + c] += (gq[c] - dot * qn[c]) / nr;   // through q / |q|
}

}  // namespace

// which kernel serves the shape: 2..5 = register-tiled GEMMs (widths that are multiples of 4) over 128 or 64 samples,
// with or without the primitive's weight-gradient accumulators in shared memory; 1 = generic
static int bwd_kind(const MsMlpShape &sh, size_t *smem) {
  *smem = 0;
  if (sh.mode != MS_MODE_LOCAL || sh.n_hidden > 4 || sh.n_hidden < 1) return 0;
  const size_t cap = 226 * 1024;
  if (sh.width % 4 == 0 && sh.width >= 8 && sh.out_dim >= 4) {
    for (int kind = 2; kind <= 5; ++kind) {              // 128 + acc, 128, 64 + acc, 64
      const size_t b = t_layout(sh, kind <= 3 ? 128 : 64, (kind & 1) == 0).floats * sizeof(float);
      if (b <= cap) { *smem = b; return kind; }
    }
  }
  const size_t b = bwd_layout(sh).floats * sizeof(float);
  if (b > 220 * 1024) return 0;
  *smem = b;
  return 1;
}

size_t ms_mlp_bwd_smem(const MsMlpShape &sh) {
  size_t b = 0;
  bwd_kind(sh, &b);
  return b;
}

cudaError_t ms_mlp_bwd(const MsMlpBwdArgs &a, cudaStream_t s) {
  size_t smem = 0;
  const int kind = bwd_kind(a.shape, &smem);
  if (kind == 0) return cudaErrorNotSupported;
  void (*fn)(MsMlpBwdArgs) = mlp_bwd_kernel;
  int threads = BT;
  if (kind >= 2) {
    threads = TNT;
    fn = kind == 2 ? mlp_bwd_t_kernel<128, true> : kind == 3 ? mlp_bwd_t_kernel<128, false>
       : kind == 4 ? mlp_bwd_t_kernel<64, true> : mlp_bwd_t_kernel<64, false>;
  }
  cudaError_t e = cudaFuncSetAttribute((const void *)fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  static int n_sm = 0;
  if (n_sm == 0) {
    int dev = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
  }
  int occ = 1;
  if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, (const void *)fn, threads, smem) != cudaSuccess || occ < 1) {
    (void)cudaGetLastError();
    occ = 1;
  }
  fn<<<(unsigned)(n_sm * occ * (kind >= 2 ? 1 : 4)), threads, smem, s>>>(a);
  MS_LAUNCHED();
  e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  if (a.n_hits > 0) {
    interval_bwd_kernel<<<(unsigned)((a.n_hits + 255) / 256), 256, 0, s>>>(a);
    MS_LAUNCHED();
    e = cudaGetLastError();
    if (e != cudaSuccess) return e;
  }
  prim_bwd_kernel<<<(unsigned)((a.n_prims + 127) / 128), 128, 0, s>>>(a);
  MS_LAUNCHED();
  return cudaGetLastError();
}
