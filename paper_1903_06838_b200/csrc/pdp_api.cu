// pdp_api.cu — host side of the C ABI declared in include/pdp.h: validation, derived maps, launch
// configuration, the launches of one batch, and the double-buffered host feed.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "../../include/pdp.h"
#include "pdp_chain.cuh"
#include "pdp_dense.cuh"
#include "pdp_fused.cuh"
#include "pdp_post.cuh"
#include "pdp_staged.cuh"

using pdp::CParams;
using pdp::KParams;
using pdp::PostParams;

namespace pdp {
using ChainFn = void (*)(const CParams);
ChainFn chain_lookup_v8(int nv, int lps, int mode);   // pdp_chain_v8.cu
ChainFn chain_lookup_v4(int nv, int lps, int mode);   // pdp_chain_v4.cu
ChainFn chain_lookup_v2(int nv, int lps, int mode);   // pdp_chain_v2.cu
using DenseFn = void (*)(const DParams);
DenseFn dense_lookup_v8(int nv, int mode);
DenseFn dense_lookup_v4(int nv, int mode);
DenseFn dense_lookup_v2(int nv, int mode);
}  // namespace pdp

namespace {

thread_local std::string g_last_error;  // errors raised before a context exists


// small-batch kernel (pdp_fused.cuh): band x chunk items with decoupled look-back
struct LaunchPlan {
  bool ok = false;
  int V = 0, G = 0;      // kernel variant
  int R = 0, TR = 0, WPR = 0, bands_per_panel = 0, n_bands = 0;
  int threads = 0;
  uint32_t stage_bytes = 0, off_v1 = 0, off_ctab = 0, off_cand = 0, off_accum = 0, off_misc = 0, smem = 0;
};

// throughput kernel (pdp_chain.cuh)
struct ChainVariant {
  int V, NV, LPS;
};
struct ChainPlan {
  bool ok = false;
  ChainVariant v{0, 0, 0};
  int R = 0, NWD = 0, NWS = 0, NB = 0, bands_per_panel = 0, n_bands = 0;
  uint32_t off_cm = 0, off_flag = 0, off_done = 0, off_pref = 0, off_phot = 0, off_sparse = 0,
           sparse_stride = 0, off_ring = 0, off_maps = 0, ring_warp_bytes = 0, maps_warp_bytes = 0, smem = 0;
};

// Preference order per vector width: the first entry that covers S with at most 25 % padding wins, otherwise
// the one with the least padding.  Entries with LPS < 32 put several frames side by side in a warp.
const ChainVariant kVariants[] = {   // measured order of preference
    {8, 3, 16}, {8, 1, 32}, {8, 2, 32}, {8, 4, 16}, {8, 2, 16}, {8, 3, 32}, {8, 4, 32}, {8, 6, 8}, {8, 4, 8},
    {4, 1, 32}, {4, 2, 32}, {4, 4, 32}, {4, 8, 32},
    {2, 13, 8}, {2, 7, 16}, {2, 1, 32}, {2, 2, 32}, {2, 4, 32}, {2, 8, 32}, {2, 16, 32},
};
// The guarded-mean and no-common-mode variants prefer fewer pixels per lane (maps in registers, two frames per warp):
// measured on configs 0 and 2 (S = 194): <2,7,16> 2.10 / 1.63 ms against <2,13,8> 2.61 / 2.16 ms; the median is
// the other way round (5.20 against 4.68 ms).
const ChainVariant kVariantsLight[] = {{2, 7, 16}, {8, 2, 16}};   // S = 256: <8,2,16> 17.6 / 15.6 ms against <8,1,32> 22.0 / 17.9 (config 4)

pdp::ChainFn chain_kernel(const ChainVariant &v, int mode) {
  switch (v.V) {
    case 8: return pdp::chain_lookup_v8(v.NV, v.LPS, mode);
    case 4: return pdp::chain_lookup_v4(v.NV, v.LPS, mode);
    case 2: return pdp::chain_lookup_v2(v.NV, v.LPS, mode);
  }
  return nullptr;
}

}  // namespace

struct pdp_ctx {
  pdp_geometry geo{};
  pdp_params prm{};
  int device = 0, num_sms = 0;
  size_t smem_limit = 0;
  size_t npix = 0;
  float *d_ped = nullptr, *d_gain = nullptr, *d_rg = nullptr;
  float *d_K = nullptr, *d_npf = nullptr;   // dense passes: 2^23 + rint(ped), -(ped - rint(ped))/gain
  double *d_rg64 = nullptr;
  unsigned long long *d_lookback = nullptr;
  unsigned *d_ticket = nullptr;
  uint32_t *d_seed_scratch = nullptr;       // throughput kernel: seed buffers [SMs][12 warps][6][seed_cap] (build_chain_plans)
  int seed_cap = 0;
  int n_stages = 0;                         // pdp_set_cm_stages: 0 = the hot path's single row-segment stage
  pdp_cm_stage stages[3] = {};
  float *d_st_v = nullptr;                  // staged path: working image [st_chunk][npix] and the stage estimates
  float *d_st_est = nullptr;
  int st_chunk = 0;
  size_t st_est_floats = 0;
  uint32_t *d_dense_ws = nullptr;           // per-CTA partial frame totals (pdp_process_dense), grown on demand
  size_t dense_ws_words = 0;
  uint32_t *d_hist_ws = nullptr;            // per-CTA partial histograms (pdp_histograms), grown on demand
  size_t hist_ws_words = 0;
  float *d_cm = nullptr;                    // optional kept common-mode estimates
  int keep_cm = 0;
  int64_t cm_frames = 0;                    // frames of the last call whose estimates are in d_cm
  LaunchPlan plan;
  uint32_t *h_stat = nullptr, *d_stat = nullptr;   // mapped host words {hits, frames} of the last batch (pdp_accum_kernel)
  ChainPlan cplan[3];                       // 4, 8, 12 sparse warps (16, 12, 8 dense ones): sparse ... dense data
  int sparse_override = 0;                  // pdp_debug_set("sparse_warps"): 0 default (4), 4, 8
  ChainVariant forced{0, 0, 0};             // pdp_debug_set("variant")
  int kernel_override = 0;                  // pdp_debug_set("kernel"): 0 auto, 1 look-back kernel, 2 throughput kernel
  int chunk_frames_override = 0;            // pdp_debug_set("chunk_frames")
  // host-feed state
  uint16_t *d_feed[2] = {nullptr, nullptr};
  int64_t feed_frames = 0;
  cudaStream_t copy_stream = nullptr;
  cudaEvent_t ev_ready[2] = {nullptr, nullptr}, ev_free[2] = {nullptr, nullptr};
  int launches = 0;
  const char *last_kernel = "";             // name of the dense-pass kernel of the last call
  char last_kernel_buf[64] = {0};
  std::string last_error;
};

namespace {

int fail(pdp_ctx *ctx, int code, const std::string &msg) {
  if (ctx) ctx->last_error = msg;
  g_last_error = msg;
  return code;
}

int cuda_fail(pdp_ctx *ctx, cudaError_t e, const char *what) {
  return fail(ctx, PDP_E_CUDA, std::string(what) + ": " + cudaGetErrorString(e));
}

#define PDP_CUDA(ctx, call)                                   \
  do {                                                        \
    cudaError_t e_ = (call);                                  \
    if (e_ != cudaSuccess) return cuda_fail(ctx, e_, #call);  \
  } while (0)

int validate_params(const pdp_params *p) {
  if (!std::isfinite(p->seed_adu) || !std::isfinite(p->cm_adu) || !std::isfinite(p->photon_adu)) return PDP_E_VALUE;
  if (!(p->photon_adu > 0.f) || !(p->cm_adu >= 0.f)) return PDP_E_VALUE;
  if (p->cm_mode < 0 || p->cm_mode > 2 || p->cm_min_count < 0) return PDP_E_VALUE;
  return PDP_OK;
}

// Small-batch kernel: the variant (V pixels per vector, G vectors per lane) with the fewest register slots
// per lane, and the tallest band that fits the warp and shared-memory budgets.
bool make_plan(const pdp_geometry &g, size_t smem_limit, LaunchPlan &pl) {
  const int S = g.seg_cols, W = g.cols, nseg = W / S;
  int bestN = 1 << 30;
  for (int V : {8, 4, 2}) {
    if (S % V || W % V) continue;
    const int vecs = S / V, G = (vecs + 31) / 32;
    if (G > 4) continue;
    if (V * G < bestN) {
      bestN = V * G;
      pl.V = V;
      pl.G = G;
    }
  }
  if (pl.V == 0) return false;
  pl.WPR = (W + 31) / 32;
  for (int R = pdp::kMaxWarps / nseg - 2; R >= 1; --R) {
    if (R > g.rows) continue;
    const int TR = R + 2;
    if (R * pl.WPR > pdp::kThreads) continue;
    uint32_t off = 0;
    const uint32_t stage = ((uint32_t)TR * W * 2u + 32u + 127u) & ~127u;
    off += stage * pdp::kStages;
    const uint32_t off_v1 = off;
    off += (uint32_t)TR * W * 4u;
    const uint32_t off_ctab = off;
    off += ((uint32_t)TR * nseg * 4u + 15u) & ~15u;
    const uint32_t off_cand = off;
    off += ((uint32_t)R * pl.WPR * 4u + 15u) & ~15u;
    const uint32_t off_accum = off;
    off += (uint32_t)R * W * 4u;
    const uint32_t off_misc = (off + 15u) & ~15u;
    off = off_misc + 8u * pdp::kStages + 80u * 4u;
    if (off > smem_limit) continue;
    pl.R = R;
    pl.TR = TR;
    pl.bands_per_panel = (g.rows + R - 1) / R;
    pl.n_bands = pl.bands_per_panel * g.panels;
    const int warps = std::max(TR * nseg, (R * pl.WPR + 31) / 32);
    pl.threads = warps * 32;
    pl.stage_bytes = stage;
    pl.off_v1 = off_v1;
    pl.off_ctab = off_ctab;
    pl.off_cand = off_cand;
    pl.off_accum = off_accum;
    pl.off_misc = off_misc;
    pl.smem = off;
    pl.ok = true;
    return true;
  }
  return false;
}

bool pick_variant(const pdp_geometry &g, int cm_mode, ChainVariant &out) {
  const int S = g.seg_cols, W = g.cols;
  int V = 0;
  for (int v : {8, 4, 2})
    if (S % v == 0 && W % v == 0) {
      V = v;
      break;
    }
  if (!V) return false;
  if (cm_mode != PDP_CM_MEDIAN)
    for (const ChainVariant &c : kVariantsLight) {
      const int cap = c.V * c.NV * c.LPS, pad = cap - S;
      if (c.V == V && pad >= 0 && 4 * pad <= cap) {
        out = c;
        return true;
      }
    }
  const ChainVariant *best = nullptr;
  int best_pad = 1 << 30;
  for (const ChainVariant &c : kVariants) {
    if (c.V != V) continue;
    const int cap = c.V * c.NV * c.LPS, pad = cap - S;
    if (pad < 0) continue;
    if (4 * pad <= cap) {   // first preferred entry with at most 25 % padding
      out = c;
      return true;
    }
    if (pad < best_pad) best_pad = pad, best = &c;
  }
  if (!best) return false;
  out = *best;
  return true;
}

// The throughput kernel: one dense warp per (band row, segment), R = dense warps / segments rows per band.
bool make_plan_chain(const pdp_geometry &g, const ChainVariant &v, int dense_warps_max, int nws, size_t smem_limit,
                     ChainPlan &pl) {
  const int nseg = g.cols / g.seg_cols;
  const int N = v.V * v.NV;
  if (v.V * v.NV * v.LPS < g.seg_cols || nseg > dense_warps_max) return false;
  if (nseg > 255 || g.cols >= (1 << 20)) return false;   // packed item / candidate descriptors
  const int NB = nws + 3;       // band slots of the rings: every sparse warp can own a band in flight, plus slack
  auto al = [](uint32_t x) { return (x + 127u) & ~127u; };
  for (int R = std::min(std::min(dense_warps_max / nseg, (int)g.rows), 254); R >= 1; --R) {
    if (R < 2 && g.rows > 1) return false;   // the sparse stage needs the previous band's last two rows in the ring
    const uint32_t ring = (uint32_t)NB * (uint32_t)R;
    const int NWD = R * nseg;
    uint32_t off = 0;
    pl.off_cm = off;      off = al(off + pdp::kFCH * ring * (uint32_t)nseg * 4u);
    pl.off_flag = off;    off = al(off + pdp::kFCH * ring * (uint32_t)nseg * 8u);
    pl.off_done = off;    off = al(off + 2u * (uint32_t)NB * 4u);
    pl.off_pref = off;    off = al(off + (uint32_t)NB * pdp::kFCH * 4u);
    pl.off_phot = off;    off = al(off + (uint32_t)NB * pdp::kFCH * 4u);
    // per sparse warp: item list + masks, candidate list, per-frame working totals
    pl.sparse_stride = al((uint32_t)(2 * pdp::kItemCap + pdp::kListCap + 3 * pdp::kFCH) * 4u);
    pl.off_sparse = off;  off = al(off + (uint32_t)nws * pl.sparse_stride);
    pl.ring_warp_bytes = (uint32_t)pdp::kRingD * 32u * (uint32_t)N * 2u;
    pl.off_ring = off;    off = al(off + (uint32_t)NWD * pl.ring_warp_bytes);
    pl.maps_warp_bytes = 2u * (uint32_t)v.LPS * (uint32_t)N * 4u;   // pedestal and 1/gain
    pl.off_maps = off;    off = al(off + (uint32_t)NWD * pl.maps_warp_bytes);
    if (off > smem_limit) continue;
    pl.v = v;
    pl.R = R;
    pl.NWD = NWD;
    pl.NWS = nws;
    pl.NB = NB;
    pl.bands_per_panel = (g.rows + R - 1) / R;
    pl.n_bands = pl.bands_per_panel * g.panels;
    pl.smem = off;
    pl.ok = true;
    return true;
  }
  return false;
}

using KernelFn = void (*)(const KParams);

KernelFn kernel_for(int V, int G) {
  switch (V * 10 + G) {
    case 21: return pdp::pdp_fused_kernel<2, 1>;
    case 22: return pdp::pdp_fused_kernel<2, 2>;
    case 23: return pdp::pdp_fused_kernel<2, 3>;
    case 24: return pdp::pdp_fused_kernel<2, 4>;
    case 41: return pdp::pdp_fused_kernel<4, 1>;
    case 42: return pdp::pdp_fused_kernel<4, 2>;
    case 43: return pdp::pdp_fused_kernel<4, 3>;
    case 44: return pdp::pdp_fused_kernel<4, 4>;
    case 81: return pdp::pdp_fused_kernel<8, 1>;
    case 82: return pdp::pdp_fused_kernel<8, 2>;
    case 83: return pdp::pdp_fused_kernel<8, 3>;
    case 84: return pdp::pdp_fused_kernel<8, 4>;
  }
  return nullptr;
}

void free_ctx(pdp_ctx *c) {
  if (!c) return;
  if (c->h_stat) cudaFreeHost(c->h_stat);
  cudaFree(c->d_ped);
  cudaFree(c->d_gain);
  cudaFree(c->d_K);
  cudaFree(c->d_rg);
  cudaFree(c->d_npf);
  cudaFree(c->d_rg64);
  cudaFree(c->d_lookback);
  cudaFree(c->d_ticket);
  cudaFree(c->d_cm);
  cudaFree(c->d_hist_ws);
  cudaFree(c->d_seed_scratch);
  cudaFree(c->d_st_v);
  cudaFree(c->d_st_est);
  cudaFree(c->d_dense_ws);
  for (int i = 0; i < 2; ++i) {
    cudaFree(c->d_feed[i]);
    if (c->ev_ready[i]) cudaEventDestroy(c->ev_ready[i]);
    if (c->ev_free[i]) cudaEventDestroy(c->ev_free[i]);
  }
  if (c->copy_stream) cudaStreamDestroy(c->copy_stream);
  delete c;
}

int alloc_staged(pdp_ctx *c);   // defined with the general common-mode path below

// (Re)build the throughput-kernel plans for the current variant choice.
int build_chain_plans(pdp_ctx *c) {
  ChainVariant v{0, 0, 0};
  for (ChainPlan &pl : c->cplan) pl = ChainPlan{};
  if (c->forced.V) v = c->forced;
  else if (!pick_variant(c->geo, c->prm.cm_mode, v)) return PDP_OK;   // no variant: the small-batch kernel serves every batch
  make_plan_chain(c->geo, v, 16, 4, c->smem_limit, c->cplan[0]);
  make_plan_chain(c->geo, v, 12, 8, c->smem_limit, c->cplan[1]);
  make_plan_chain(c->geo, v, 8, 12, c->smem_limit, c->cplan[2]);
  for (int i = 0; i < 3; ++i) {
    if (!c->cplan[i].ok) continue;
    for (int mode = 0; mode < 3; ++mode) {
      pdp::ChainFn fn = chain_kernel(v, mode);
      if (!fn) {
        c->cplan[i].ok = false;
        break;
      }
      PDP_CUDA(c, cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                       (int)std::max(std::max(c->cplan[0].smem, c->cplan[1].smem), c->cplan[2].smem)));
    }
  }
  if (c->forced.V && !c->cplan[0].ok) return fail(c, PDP_E_GEOMETRY, "pdp_debug_set: variant does not fit this geometry");
  // Workspace of the throughput kernel, allocated here (pdp_create / replanning), never on the pdp_process path.
  int r_max = 0;
  for (const ChainPlan &pl : c->cplan)
    if (pl.ok) r_max = std::max(r_max, pl.R);
  if (r_max > 0 && !c->d_seed_scratch) {
    // a band of all 16 frame slots can hold at most 16 * R * W / 2 seeds per panel row block; 8192 buffered seeds
    // let several bands be evaluated at the same time even on dense data (a full buffer only chains earlier)
    const long long most = (long long)pdp::kFCH * (r_max + 1) * ((c->geo.cols + 1) / 2);
    c->seed_cap = (int)std::min<long long>(8192, std::max<long long>(256, (most + 31) / 32 * 32));
    PDP_CUDA(c, cudaMalloc(&c->d_seed_scratch, (size_t)c->num_sms * 12 * 6 * (size_t)c->seed_cap * sizeof(uint32_t)));
  }
  if (r_max > 0 && !c->h_stat) {   // density hint of the last batch, written by pdp_accum_kernel (failure to map: no hint)
    if (cudaHostAlloc(&c->h_stat, 2 * sizeof(uint32_t), cudaHostAllocMapped) == cudaSuccess) {
      c->h_stat[0] = c->h_stat[1] = 0u;
      if (cudaHostGetDevicePointer(&c->d_stat, c->h_stat, 0) != cudaSuccess) c->d_stat = nullptr;
    } else {
      c->h_stat = nullptr;
      (void)cudaGetLastError();
    }
  }
  return PDP_OK;
}

}  // namespace

extern "C" {

int pdp_version(void) { return PDP_VERSION; }

const char *pdp_strerror(int code) {
  switch (code) {
    case PDP_OK: return "ok";
    case PDP_E_NULL: return "null pointer argument";
    case PDP_E_GEOMETRY: return "invalid or unsupported geometry";
    case PDP_E_VALUE: return "invalid value (non-finite map/threshold, zero gain, non-positive photon_adu, bad mode)";
    case PDP_E_BATCH: return "n_frames out of range";
    case PDP_E_ALIGN: return "raw batch pointer must be 16-byte aligned";
    case PDP_E_CUDA: return "CUDA runtime error";
    case PDP_E_NO_SM100: return "current device is not sm_100 (no fallback path exists)";
    case PDP_E_NOMEM: return "out of memory";
  }
  return "unknown pdp status";
}

const char *pdp_last_error(const pdp_ctx *ctx) { return ctx ? ctx->last_error.c_str() : g_last_error.c_str(); }

int pdp_create(const pdp_geometry *geo, const float *ped, const float *gain, const pdp_params *prm,
               pdp_ctx **out_ctx) {
  if (out_ctx) *out_ctx = nullptr;
  if (!geo || !ped || !gain || !prm || !out_ctx) return fail(nullptr, PDP_E_NULL, "pdp_create: null argument");
  if (geo->panels < 1 || geo->rows < 1 || geo->cols < 2 || geo->seg_cols < 2 || geo->max_frames_per_batch < 1 ||
      geo->cols % geo->seg_cols || (geo->cols & 1) || (geo->seg_cols & 1) || geo->seg_cols > 1024 ||
      geo->cols / geo->seg_cols > 6)
    return fail(nullptr, PDP_E_GEOMETRY, "pdp_create: unsupported geometry");
  const size_t npix = (size_t)geo->panels * geo->rows * geo->cols;
  if (npix > 0xffffffffull) return fail(nullptr, PDP_E_GEOMETRY, "pdp_create: frame exceeds 2^32 pixels");
  if (int rc = validate_params(prm)) return fail(nullptr, rc, "pdp_create: invalid params");

  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return cuda_fail(nullptr, e, "cudaGetDevice");
  cudaDeviceProp prop;
  e = cudaGetDeviceProperties(&prop, dev);
  if (e != cudaSuccess) return cuda_fail(nullptr, e, "cudaGetDeviceProperties");
  if (prop.major != 10) return fail(nullptr, PDP_E_NO_SM100, "pdp_create: device is not compute capability 10.x");

  // derived maps, evaluated in double: rg = 1/gain (float and double); for the small-batch kernel
  // K = 2^23 + rint(ped), npf = -(ped - rint(ped))/gain, so that v1 = fma((2^23 + raw) - K, rg, npf)
  std::vector<float> K, rg, npf;
  std::vector<double> rg64;
  try {
    rg64.resize(npix);
    K.resize(npix);
    rg.resize(npix);
    npf.resize(npix);
  } catch (const std::bad_alloc &) {
    return fail(nullptr, PDP_E_NOMEM, "pdp_create: host allocation failed");
  }
  for (size_t i = 0; i < npix; ++i) {
    const double p = ped[i], g = gain[i];
    if (!std::isfinite(p) || !std::isfinite(g) || g == 0.0 || std::fabs(p) > 4.0e6)
      return fail(nullptr, PDP_E_VALUE, "pdp_create: non-finite or out-of-range pedestal/gain");
    const double pi = std::nearbyint(p), r = 1.0 / g;
    K[i] = (float)(8388608.0 + pi);
    rg[i] = (float)r;
    rg64[i] = r;
    npf[i] = (float)(-(p - pi) * r);
  }

  pdp_ctx *c = new (std::nothrow) pdp_ctx();
  if (!c) return fail(nullptr, PDP_E_NOMEM, "pdp_create: host allocation failed");
  c->geo = *geo;
  c->prm = *prm;
  c->device = dev;
  c->num_sms = prop.multiProcessorCount;
  c->smem_limit = prop.sharedMemPerBlockOptin;
  c->npix = npix;
  if (!make_plan(*geo, c->smem_limit, c->plan)) {
    free_ctx(c);
    return fail(nullptr, PDP_E_GEOMETRY, "pdp_create: no kernel variant fits this geometry");
  }
  KernelFn fn = kernel_for(c->plan.V, c->plan.G);
  e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->plan.smem);
  if (e == cudaSuccess)
    e = cudaFuncSetAttribute(pdp::pdp_accum_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->smem_limit);
  if (e == cudaSuccess)
    e = cudaFuncSetAttribute(pdp::pdp_hist_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 3 * 16384 * 4);
  if (e != cudaSuccess) {
    free_ctx(c);
    return cuda_fail(nullptr, e, "cudaFuncSetAttribute");
  }
  if (int rc = build_chain_plans(c)) {
    free_ctx(c);
    return rc;
  }
  const size_t mb = npix * sizeof(float);
  const size_t lb = (size_t)geo->max_frames_per_batch * c->plan.n_bands * sizeof(unsigned long long);
  cudaError_t errs[] = {cudaMalloc(&c->d_ped, mb),      cudaMalloc(&c->d_gain, mb),
                        cudaMalloc(&c->d_K, mb),        cudaMalloc(&c->d_rg, mb),
                        cudaMalloc(&c->d_npf, mb),      cudaMalloc(&c->d_lookback, lb),
                        cudaMalloc(&c->d_ticket, 256),  cudaMalloc(&c->d_rg64, npix * sizeof(double))};
  for (cudaError_t x : errs)
    if (x != cudaSuccess) {
      free_ctx(c);
      return cuda_fail(nullptr, x, "cudaMalloc");
    }
  e = cudaMemcpy(c->d_rg64, rg64.data(), npix * sizeof(double), cudaMemcpyHostToDevice);
  const void *srcs[] = {ped, gain, K.data(), rg.data(), npf.data()};
  float *dsts[] = {c->d_ped, c->d_gain, c->d_K, c->d_rg, c->d_npf};
  for (int i = 0; i < 5 && e == cudaSuccess; ++i) e = cudaMemcpy(dsts[i], srcs[i], mb, cudaMemcpyHostToDevice);
  if (e != cudaSuccess) {
    free_ctx(c);
    return cuda_fail(nullptr, e, "cudaMemcpy(maps)");
  }
  *out_ctx = c;
  return PDP_OK;
}

int pdp_set_params(pdp_ctx *ctx, const pdp_params *prm) {
  if (!ctx || !prm) return fail(ctx, PDP_E_NULL, "pdp_set_params: null argument");
  if (int rc = validate_params(prm)) return fail(ctx, rc, "pdp_set_params: invalid params");
  const bool replan = (prm->cm_mode == PDP_CM_MEDIAN) != (ctx->prm.cm_mode == PDP_CM_MEDIAN);
  ctx->prm = *prm;
  if (replan) return build_chain_plans(ctx);   // the layout preference depends on the estimator
  return PDP_OK;
}

int pdp_set_cm_stages(pdp_ctx *ctx, const pdp_cm_stage *stages, int32_t n_stages) {
  if (!ctx || (n_stages > 0 && !stages)) return fail(ctx, PDP_E_NULL, "pdp_set_cm_stages: null argument");
  if (n_stages < 0 || n_stages > 3) return fail(ctx, PDP_E_VALUE, "pdp_set_cm_stages: 0 to 3 stages");
  for (int s = 0; s < n_stages; ++s) {
    const pdp_cm_stage &g = stages[s];
    if (g.group_rows < 1 || g.group_cols < 1 || ctx->geo.rows % g.group_rows || ctx->geo.cols % g.group_cols)
      return fail(ctx, PDP_E_GEOMETRY, "pdp_set_cm_stages: a group shape must tile the panel");
    if (g.cm_mode < 0 || g.cm_mode > 2 || g.cm_min_count < 0) return fail(ctx, PDP_E_VALUE, "pdp_set_cm_stages: bad estimator");
  }
  ctx->n_stages = n_stages;
  for (int s = 0; s < n_stages; ++s) ctx->stages[s] = stages[s];
  if (n_stages > 0) return alloc_staged(ctx);
  return PDP_OK;
}

int pdp_destroy(pdp_ctx *ctx) {
  free_ctx(ctx);
  return PDP_OK;
}

int pdp_last_launch_count(const pdp_ctx *ctx) { return ctx ? ctx->launches : 0; }

const char *pdp_last_kernel_name(const pdp_ctx *ctx) { return ctx ? ctx->last_kernel : ""; }

int pdp_debug_set(pdp_ctx *ctx, const char *key, int64_t value) {
  if (!ctx || !key) return fail(ctx, PDP_E_NULL, "pdp_debug_set: null argument");
  if (!std::strcmp(key, "kernel")) {
    if (value < 0 || value > 2) return fail(ctx, PDP_E_VALUE, "pdp_debug_set: kernel must be 0, 1 or 2");
    ctx->kernel_override = (int)value;
    return PDP_OK;
  }
  if (!std::strcmp(key, "chunk_frames")) {
    if (value < 0) return fail(ctx, PDP_E_VALUE, "pdp_debug_set: chunk_frames must be >= 0");
    ctx->chunk_frames_override = (int)value;
    return PDP_OK;
  }
  if (!std::strcmp(key, "sparse_warps")) {
    if (value != 0 && value != 4 && value != 8 && value != 12)
      return fail(ctx, PDP_E_VALUE, "pdp_debug_set: sparse_warps must be 0, 4, 8 or 12");
    ctx->sparse_override = (int)value;
    return PDP_OK;
  }
  if (!std::strcmp(key, "variant")) {   // V * 10000 + NV * 100 + LPS, 0 = automatic
    ctx->forced = ChainVariant{(int)(value / 10000), (int)((value / 100) % 100), (int)(value % 100)};
    return build_chain_plans(ctx);
  }
  return fail(ctx, PDP_E_VALUE, "pdp_debug_set: unknown key");
}

int pdp_keep_common_mode(pdp_ctx *ctx, int32_t enable) {
  if (!ctx) return fail(nullptr, PDP_E_NULL, "pdp_keep_common_mode: null ctx");
  ctx->keep_cm = enable ? 1 : 0;
  if (ctx->keep_cm && !ctx->d_cm) {
    const size_t n = (size_t)ctx->geo.max_frames_per_batch * (ctx->npix / ctx->geo.seg_cols) * sizeof(float);
    PDP_CUDA(ctx, cudaMalloc(&ctx->d_cm, n));
  }
  return PDP_OK;
}

int pdp_get_common_mode(pdp_ctx *ctx, float *cm_device, int64_t n_floats, void *stream) {
  if (!ctx || !cm_device) return fail(ctx, PDP_E_NULL, "pdp_get_common_mode: null argument");
  if (!ctx->d_cm) return fail(ctx, PDP_E_VALUE, "pdp_get_common_mode: pdp_keep_common_mode was not enabled");
  const int64_t have = ctx->cm_frames * (int64_t)(ctx->npix / ctx->geo.seg_cols);
  if (n_floats > have) return fail(ctx, PDP_E_BATCH, "pdp_get_common_mode: more floats requested than kept");
  PDP_CUDA(ctx, cudaMemcpyAsync(cm_device, ctx->d_cm, (size_t)n_floats * sizeof(float), cudaMemcpyDeviceToDevice,
                                (cudaStream_t)stream));
  return PDP_OK;
}

}  // extern "C"

namespace {

int enqueue_accum(pdp_ctx *c, int n, cudaStream_t st, const pdp_output &o);

// The throughput path: pdp_chain_kernel (dense pass + sparse stage, one launch) followed by pdp_accum_kernel
// (the accumulated image from the finished lists, no global atomics).
int enqueue_chain(pdp_ctx *c, const ChainPlan &pl, const uint16_t *raw, int n, cudaStream_t st, const pdp_output &o,
                  bool keep_cm) {
  CParams k{};
  k.raw = raw;
  k.n_frames = n;
  k.ped = c->d_ped;
  k.rg = c->d_rg;
  k.mapK = c->d_K;
  k.mapNpf = c->d_npf;
  k.rg64 = c->d_rg64;
  k.P = c->geo.panels;
  k.H = c->geo.rows;
  k.W = c->geo.cols;
  k.S = c->geo.seg_cols;
  k.nseg = k.W / k.S;
  k.R = pl.R;
  k.bands_per_panel = pl.bands_per_panel;
  k.n_bands = pl.n_bands;
  k.NWD = pl.NWD;
  k.NWS = pl.NWS;
  k.NB = pl.NB;
  k.off_done = pl.off_done;
  k.T_seed = c->prm.seed_adu;
  k.T_cm = c->prm.cm_adu;
  k.E_ph = c->prm.photon_adu;
  k.sqrtS = (float)std::sqrt((double)k.S);
  // candidates: a superset of the seeds; the margin covers the fp32 rounding of v1 and of c
  k.cand_thr = (float)((double)c->prm.seed_adu - std::max(1e-3, 4e-6 * std::fabs((double)c->prm.seed_adu)));
  // BIG: the value of every pixel outside the mask; a power of two >= 4 * N * T_cm so that the sum of a lane's
  // values splits exactly into (count outside the mask) * BIG + (sum inside)
  {
    const double need = std::max(1024.0, 4.0 * (double)(pl.v.V * pl.v.NV) * (double)c->prm.cm_adu + 1.0);
    double big = 1024.0;
    while (big < need) big *= 2.0;
    k.big = (float)big;
  }
  k.dT_seed = (double)c->prm.seed_adu;
  k.dE_ph = (double)c->prm.photon_adu;
  k.dinv_E_ph = 1.0 / (double)c->prm.photon_adu;
  k.cm_mode = c->prm.cm_mode;
  k.cm_min_count = c->prm.cm_min_count > 0 ? c->prm.cm_min_count : (int)std::ceil(std::sqrt((double)k.S));
  k.cap = o.hit_capacity;
  k.hit_count = o.hit_count;
  k.hit_pixel = o.hit_pixel;
  k.hit_charge = o.hit_charge;
  k.hit_nphot = o.hit_nphot;
  k.hit_dx = o.hit_dx;
  k.hit_dy = o.hit_dy;
  k.frame_photons = o.frame_photons;
  k.accum = o.accum;
  k.status = o.status;
  k.cm_keep = keep_cm ? c->d_cm : nullptr;
  k.seed_scratch = c->d_seed_scratch;
  k.seed_cap = c->seed_cap;
  k.off_cm = pl.off_cm;
  k.off_flag = pl.off_flag;
  k.off_pref = pl.off_pref;
  k.off_phot = pl.off_phot;
  k.off_sparse = pl.off_sparse;
  k.sparse_stride = pl.sparse_stride;
  k.off_ring = pl.off_ring;
  k.off_maps = pl.off_maps;
  k.ring_warp_bytes = pl.ring_warp_bytes;
  k.maps_warp_bytes = pl.maps_warp_bytes;
  const int grid = std::min(c->num_sms, n);
  pdp::ChainFn fn = chain_kernel(pl.v, c->prm.cm_mode);
  fn<<<grid, (pl.NWD + pl.NWS) * 32, pl.smem, st>>>(k);
  PDP_CUDA(c, cudaGetLastError());
  c->launches += 1;
  if (int rc = enqueue_accum(c, n, st, o)) return rc;
  std::snprintf(c->last_kernel_buf, sizeof(c->last_kernel_buf), "pdp_chain_kernel<%d,%d,%d,%d>", pl.v.V, pl.v.NV, pl.v.LPS,
                c->prm.cm_mode);
  c->last_kernel = c->last_kernel_buf;
  return PDP_OK;
}

// The accumulated image from the finished lists: owner-computes scatter by pixel range (no global atomics).
int enqueue_accum(pdp_ctx *c, int n, cudaStream_t st, const pdp_output &o) {
  PostParams q{};
  q.n_frames = n;
  q.cap = o.hit_capacity;
  q.npix = (uint32_t)c->npix;
  const uint32_t span_max = (uint32_t)((c->smem_limit - 1024) / 4);
  q.span = std::min(span_max, (uint32_t)((c->npix + c->num_sms - 1) / c->num_sms));
  q.span = std::max(q.span, 1u);
  q.hit_count = o.hit_count;
  q.hit_pixel = o.hit_pixel;
  q.hit_nphot = o.hit_nphot;
  q.accum = o.accum;
  q.stat = c->d_stat;
  const int grid_a = (int)((c->npix + q.span - 1) / q.span);
  pdp::pdp_accum_kernel<<<grid_a, pdp::kPostThreads, (size_t)q.span * 4, st>>>(q);
  PDP_CUDA(c, cudaGetLastError());
  c->launches += 1;
  return PDP_OK;
}

// Working image and estimate buffers of the general common-mode path: allocated when the stages are set
// (pdp_set_cm_stages), never on the pdp_process path.
int alloc_staged(pdp_ctx *c) {
  const size_t npix = c->npix;
  if (!c->d_st_v) {
    const size_t budget = (size_t)1 << 30;   // ~1 GiB of working image
    c->st_chunk = (int)std::max<size_t>(1, std::min<size_t>((size_t)c->geo.max_frames_per_batch, budget / (npix * 4)));
    PDP_CUDA(c, cudaMalloc(&c->d_st_v, (size_t)c->st_chunk * npix * sizeof(float)));
  }
  size_t est_per_frame = 0;
  for (int s = 0; s < c->n_stages; ++s)
    est_per_frame += npix / ((size_t)c->stages[s].group_rows * c->stages[s].group_cols);
  if (c->st_est_floats < est_per_frame * c->st_chunk) {
    cudaFree(c->d_st_est);
    c->d_st_est = nullptr;
    c->st_est_floats = 0;
    PDP_CUDA(c, cudaMalloc(&c->d_st_est, est_per_frame * c->st_chunk * sizeof(float)));
    c->st_est_floats = est_per_frame * c->st_chunk;
  }
  return PDP_OK;
}

// The general common-mode path (pdp_staged.cuh): calibrate into a working image, one kernel per stage, the finder,
// the accumulated image; frames in chunks that bound the working image.
int enqueue_staged(pdp_ctx *c, const uint16_t *raw, int n, cudaStream_t st, const pdp_output &o) {
  const size_t npix = c->npix;
  for (int f0 = 0; f0 < n; f0 += c->st_chunk) {
    const int m = std::min(c->st_chunk, n - f0);
    pdp::StParams k{};
    k.raw = raw + (size_t)f0 * npix;
    k.n_frames = m;
    k.mapK = c->d_K;
    k.rg = c->d_rg;
    k.mapNpf = c->d_npf;
    k.ped = c->d_ped;
    k.rg64 = c->d_rg64;
    k.P = c->geo.panels;
    k.H = c->geo.rows;
    k.W = c->geo.cols;
    k.npix = (uint32_t)npix;
    k.v = c->d_st_v;
    k.T_cm = c->prm.cm_adu;
    k.cand_thr = (float)((double)c->prm.seed_adu - std::max(1e-3, 4e-6 * std::fabs((double)c->prm.seed_adu)));
    k.dT_seed = (double)c->prm.seed_adu;
    k.dE_ph = (double)c->prm.photon_adu;
    k.n_stages = c->n_stages;
    float *est = c->d_st_est;
    for (int s = 0; s < c->n_stages; ++s) {
      pdp::StageDesc &d = k.st[s];
      d.gh = c->stages[s].group_rows;
      d.gw = c->stages[s].group_cols;
      d.ngr = k.H / d.gh;
      d.ngc = k.W / d.gw;
      d.mode = c->stages[s].cm_mode;
      d.min_count = c->stages[s].cm_min_count > 0 ? c->stages[s].cm_min_count
                                                  : (int)std::ceil(std::sqrt((double)d.gh * d.gw));
      d.sqrtG = (float)std::sqrt((double)d.gh * d.gw);
      d.est = est;
      est += (size_t)m * k.P * d.ngr * d.ngc;
    }
    k.cap = o.hit_capacity;
    k.hit_count = o.hit_count + f0;
    k.frame_photons = o.frame_photons + f0;
    const size_t off = (size_t)f0 * o.hit_capacity;
    k.hit_pixel = o.hit_pixel + off;
    k.hit_charge = o.hit_charge + off;
    k.hit_nphot = o.hit_nphot + off;
    k.hit_dx = o.hit_dx + off;
    k.hit_dy = o.hit_dy + off;
    k.accum = o.accum;
    k.status = o.status;
    const int grid_e = (int)std::min<size_t>((size_t)c->num_sms * 8, ((size_t)m * npix / 2 + pdp::kStThreads - 1) / pdp::kStThreads);
    pdp::pdp_st_calib_kernel<<<std::max(grid_e, 1), pdp::kStThreads, 0, st>>>(k);
    PDP_CUDA(c, cudaGetLastError());
    c->launches += 1;
    for (int s = 0; s < c->n_stages; ++s) {
      const pdp::StageDesc &sd = k.st[s];
      const long long items = (long long)m * k.P * sd.ngr * sd.ngc;
      // guarded-mean stages whose rows can be read with 128-bit loads take the coalesced kernels (pdp_staged.cuh)
      const bool vec4 = sd.mode == PDP_CM_MEAN_GUARDED && k.W % 4 == 0 && npix % 4 == 0;
      const long long gpx = (long long)sd.gh * sd.gw;
      if (sd.mode == PDP_CM_MEDIAN && gpx <= 1024) {   // a warp per group, the values in registers
        const long long ctas = (items + pdp::kStThreads / 32 - 1) / (pdp::kStThreads / 32);
        const int grid_s = (int)std::min<long long>(ctas, (long long)c->num_sms * 8);
        if (gpx <= 256) pdp::pdp_st_median_small_kernel<8><<<grid_s, pdp::kStThreads, 0, st>>>(k, s);
        else if (gpx <= 512) pdp::pdp_st_median_small_kernel<16><<<grid_s, pdp::kStThreads, 0, st>>>(k, s);
        else if (gpx <= 768) pdp::pdp_st_median_small_kernel<24><<<grid_s, pdp::kStThreads, 0, st>>>(k, s);
        else pdp::pdp_st_median_small_kernel<32><<<grid_s, pdp::kStThreads, 0, st>>>(k, s);
      } else if (vec4 && sd.gw % 4 == 0 && sd.gw >= 8 && (long long)sd.gh * sd.gw <= 2048) {   // a warp per group
        const long long ctas = (items + pdp::kStThreads / 32 - 1) / (pdp::kStThreads / 32);
        pdp::pdp_st_mean_small_kernel<<<(int)std::min<long long>(ctas, (long long)c->num_sms * 8), pdp::kStThreads, 0, st>>>(k, s);
      } else if (vec4 && sd.gw % 4 == 0 && sd.gw >= 8) {
        const int threads = (long long)sd.gh * sd.gw >= 32768 ? 1024 : pdp::kStThreads;
        const int grid_s = (int)std::min<long long>(items, (long long)c->num_sms * (threads == 1024 ? 2 : 8));
        pdp::pdp_st_mean_wide_kernel<<<grid_s, threads, 0, st>>>(k, s);
      } else if (vec4 && (sd.gw == 1 || sd.gw == 2 || sd.gw == 4)) {
        const long long citems = (long long)m * k.P * sd.ngr * ((k.W + pdp::kStColChunk - 1) / pdp::kStColChunk);
        pdp::pdp_st_mean_cols_kernel<<<(int)std::min<long long>(citems, (long long)c->num_sms * 8), pdp::kStThreads, 0, st>>>(k, s);
      } else {
        const int grid_s = (int)std::min<long long>(items, (long long)c->num_sms * 8);
        pdp::pdp_st_stage_kernel<<<grid_s, pdp::kStThreads, 0, st>>>(k, s);
      }
      PDP_CUDA(c, cudaGetLastError());
      c->launches += 1;
    }
    pdp::pdp_st_find_kernel<<<std::min(m, c->num_sms * 4), pdp::kStThreads, 0, st>>>(k);
    PDP_CUDA(c, cudaGetLastError());
    c->launches += 1;
  }
  c->last_kernel = "pdp_st_stage_kernel";
  return enqueue_accum(c, n, st, o);
}

// Enqueue the chain for n frames at `raw` (device); outputs are already offset to this batch.
int enqueue(pdp_ctx *c, const uint16_t *raw, int n, cudaStream_t st, const pdp_output &o, bool keep_cm) {
  if (c->n_stages > 0) return enqueue_staged(c, raw, n, st, o);
  // ---- large batches: the throughput kernel (frame-owner CTAs) ----
  {
    // Sparse warps: 4 by default; 8 when the previous batch was dense in hits (measured: above 1 % of
    // the pixels in any mode, above 0.25 % in the guarded-mean and no-common-mode variants, whose dense pass is light);
    // 12 above 2 % in those two variants.
    // The density is a hint read from mapped host memory without synchronisation; results never depend on it.
    int which = 0;
    if (c->sparse_override) which = c->sparse_override == 12 ? 2 : (c->sparse_override == 8 ? 1 : 0);
    else if (c->h_stat) {
      const uint32_t hits = ((volatile uint32_t *)c->h_stat)[0], fr = ((volatile uint32_t *)c->h_stat)[1];
      if (fr) {
        const double dens = (double)hits / ((double)fr * (double)c->npix);
        if (dens > 0.01 || (dens > 0.0025 && c->prm.cm_mode != PDP_CM_MEDIAN)) which = 1;
        if (dens > 0.02 && c->prm.cm_mode != PDP_CM_MEDIAN) which = 2;   // config 3: 5.6 -> 4.9 ms (mean), 6.3 -> 5.0 ms (none)
      }
    }
    if (!c->cplan[which].ok) which = 0;
    const bool can = c->cplan[which].ok;
    // measured crossover (configs 0, 1, 4): the frame-owner kernel wins from about 24 frames on (6 n >= SMs); below
    // that a frame's bands have to be spread over several CTAs, which only the look-back kernel does
    const bool use_chain = can && (c->kernel_override == 2 || (c->kernel_override == 0 && 6 * n >= c->num_sms));
    if (c->kernel_override == 2 && !can)
      return fail(c, PDP_E_GEOMETRY, "pdp_debug_set(kernel=2): the throughput kernel does not support this geometry");
    if (use_chain) return enqueue_chain(c, c->cplan[which], raw, n, st, o, keep_cm);
  }
  // ---- small batches: band x chunk items with decoupled look-back ----
  const LaunchPlan &pl = c->plan;
  KParams k{};
  k.raw = raw;
  k.n_frames = n;
  k.ped = c->d_ped;
  k.gain = c->d_gain;
  k.mapK = c->d_K;
  k.mapRg = c->d_rg;
  k.mapNpf = c->d_npf;
  k.P = c->geo.panels;
  k.H = c->geo.rows;
  k.W = c->geo.cols;
  k.S = c->geo.seg_cols;
  k.nseg = k.W / k.S;
  k.R = pl.R;
  k.TR = pl.TR;
  k.WPR = pl.WPR;
  k.bands_per_panel = pl.bands_per_panel;
  k.n_bands = pl.n_bands;
  // frames per work item: enough items for ~16 waves of CTAs, at least 8 frames each so that the
  // per-item map reload (12 B/pixel from L2) stays small against 2 B/pixel/frame of raw data
  int fc = c->chunk_frames_override;
  if (fc <= 0) {
    const long long want_items = 16LL * c->num_sms;
    long long chunks = std::max(1LL, want_items / pl.n_bands);
    fc = (int)std::max(8LL, std::min(64LL, (long long)((n + chunks - 1) / chunks)));
  }
  k.FC = std::min(fc, n);
  k.n_chunks = (n + k.FC - 1) / k.FC;
  k.n_items = k.n_chunks * k.n_bands;
  k.T_seed = c->prm.seed_adu;
  k.T_cm = c->prm.cm_adu;
  k.E_ph = c->prm.photon_adu;
  k.sqrtS = (float)std::sqrt((double)k.S);
  k.cand_margin = std::max(1e-3f, 4e-6f * std::fabs(c->prm.seed_adu));
  k.dT_seed = (double)c->prm.seed_adu;
  k.dE_ph = (double)c->prm.photon_adu;
  k.cm_mode = c->prm.cm_mode;
  k.cm_min_count = c->prm.cm_min_count > 0 ? c->prm.cm_min_count : (int)std::ceil(std::sqrt((double)k.S));
  k.cap = o.hit_capacity;
  k.hit_count = o.hit_count;
  k.hit_pixel = o.hit_pixel;
  k.hit_charge = o.hit_charge;
  k.hit_nphot = o.hit_nphot;
  k.hit_dx = o.hit_dx;
  k.hit_dy = o.hit_dy;
  k.frame_photons = o.frame_photons;
  k.accum = o.accum;
  k.status = o.status;
  k.cm_keep = keep_cm ? c->d_cm : nullptr;
  k.lookback = c->d_lookback;
  k.ticket = c->d_ticket;
  k.stage_bytes = pl.stage_bytes;
  k.off_v1 = pl.off_v1;
  k.off_ctab = pl.off_ctab;
  k.off_cand = pl.off_cand;
  k.off_accum = pl.off_accum;
  k.off_misc = pl.off_misc;
  PDP_CUDA(c, cudaMemsetAsync(c->d_lookback, 0, (size_t)n * pl.n_bands * sizeof(unsigned long long), st));
  PDP_CUDA(c, cudaMemsetAsync(c->d_ticket, 0, sizeof(unsigned), st));
  const int grid = std::min(k.n_items, c->num_sms);
  KernelFn fn = kernel_for(pl.V, pl.G);
  fn<<<grid, pl.threads, pl.smem, st>>>(k);
  PDP_CUDA(c, cudaGetLastError());
  c->launches += 1;
  c->last_kernel = "pdp_fused_kernel";
  return PDP_OK;
}

int check_output(pdp_ctx *c, const pdp_output *o) {
  if (!o || !o->hit_count || !o->hit_pixel || !o->hit_charge || !o->hit_nphot || !o->hit_dx || !o->hit_dy ||
      !o->frame_photons || !o->accum || !o->status)
    return fail(c, PDP_E_NULL, "pdp_process: null output pointer");
  return PDP_OK;
}

}  // namespace

extern "C" {

int pdp_process(pdp_ctx *ctx, const pdp_batch *batch, void *stream, const pdp_output *out) {
  if (!ctx || !batch) return fail(ctx, PDP_E_NULL, "pdp_process: null argument");
  if (int rc = check_output(ctx, out)) return rc;
  if (batch->n_frames < 0 || batch->n_frames > ctx->geo.max_frames_per_batch)
    return fail(ctx, PDP_E_BATCH, "pdp_process: n_frames out of range");
  ctx->launches = 0;
  if (batch->n_frames == 0) return PDP_OK;
  if (!batch->data) return fail(ctx, PDP_E_NULL, "pdp_process: null batch data");
  if (reinterpret_cast<uintptr_t>(batch->data) & 15) return fail(ctx, PDP_E_ALIGN, "pdp_process: batch not 16-byte aligned");
  ctx->cm_frames = ctx->keep_cm ? batch->n_frames : 0;
  return enqueue(ctx, batch->data, batch->n_frames, (cudaStream_t)stream, *out, ctx->keep_cm != 0);
}

int pdp_process_pinned(pdp_ctx *ctx, const uint16_t *raw_host, int32_t n_frames, int32_t chunk_frames,
                       void *compute_stream, void *copy_stream, const pdp_output *out) {
  if (!ctx || (!raw_host && n_frames > 0)) return fail(ctx, PDP_E_NULL, "pdp_process_pinned: null argument");
  if (int rc = check_output(ctx, out)) return rc;
  if (n_frames < 0 || chunk_frames < 1 || chunk_frames > ctx->geo.max_frames_per_batch)
    return fail(ctx, PDP_E_BATCH, "pdp_process_pinned: n_frames / chunk_frames out of range");
  ctx->launches = 0;
  if (n_frames == 0) return PDP_OK;
  cudaStream_t st = (cudaStream_t)compute_stream;
  const size_t frame_bytes = ctx->npix * sizeof(uint16_t);
  if (ctx->feed_frames < chunk_frames) {
    for (int i = 0; i < 2; ++i) {
      cudaFree(ctx->d_feed[i]);
      ctx->d_feed[i] = nullptr;
      PDP_CUDA(ctx, cudaMalloc(&ctx->d_feed[i], (size_t)chunk_frames * frame_bytes));
    }
    ctx->feed_frames = chunk_frames;
  }
  if (!ctx->ev_ready[0]) {
    for (int i = 0; i < 2; ++i) {
      PDP_CUDA(ctx, cudaEventCreateWithFlags(&ctx->ev_ready[i], cudaEventDisableTiming));
      PDP_CUDA(ctx, cudaEventCreateWithFlags(&ctx->ev_free[i], cudaEventDisableTiming));
    }
  }
  cudaStream_t cs = (cudaStream_t)copy_stream;
  if (!cs) {   // no copy stream given: the context's own side stream
    if (!ctx->copy_stream) PDP_CUDA(ctx, cudaStreamCreateWithFlags(&ctx->copy_stream, cudaStreamNonBlocking));
    cs = ctx->copy_stream;
  }
  // The copy stream must not overwrite a feed buffer that an earlier call's kernels still read: ev_free[b] was recorded
  // after the last kernel that read buffer b (below), on whatever stream that call used, and a wait on an event that
  // was never recorded is a no-op.  Nothing is recorded here, so back-to-back calls keep the copy engine busy while the
  // previous call's last chunk is still being processed.
  int launches = 0;
  for (int f0 = 0, i = 0; f0 < n_frames; f0 += chunk_frames, ++i) {
    const int b = i & 1, n = std::min(chunk_frames, n_frames - f0);
    PDP_CUDA(ctx, cudaStreamWaitEvent(cs, ctx->ev_free[b], 0));
    PDP_CUDA(ctx, cudaMemcpyAsync(ctx->d_feed[b], raw_host + (size_t)f0 * ctx->npix, (size_t)n * frame_bytes,
                                  cudaMemcpyHostToDevice, cs));
    PDP_CUDA(ctx, cudaEventRecord(ctx->ev_ready[b], cs));
    PDP_CUDA(ctx, cudaStreamWaitEvent(st, ctx->ev_ready[b], 0));
    pdp_output o = *out;
    o.hit_count += f0;
    o.frame_photons += f0;
    const size_t off = (size_t)f0 * out->hit_capacity;
    o.hit_pixel += off;
    o.hit_charge += off;
    o.hit_nphot += off;
    o.hit_dx += off;
    o.hit_dy += off;
    ctx->launches = 0;
    if (int rc = enqueue(ctx, ctx->d_feed[b], n, st, o, false)) return rc;
    launches += ctx->launches;
    PDP_CUDA(ctx, cudaEventRecord(ctx->ev_free[b], st));
  }
  ctx->launches = launches;
  ctx->cm_frames = 0;
  return PDP_OK;
}

int pdp_process_host(pdp_ctx *ctx, const uint16_t *raw_host, int32_t n_frames, int32_t chunk_frames, void *stream,
                     const pdp_output *out) {
  return pdp_process_pinned(ctx, raw_host, n_frames, chunk_frames, stream, nullptr, out);
}

int pdp_process_dense(pdp_ctx *ctx, const pdp_batch *batch, void *stream, float zero_below_adu, uint32_t *image,
                      uint32_t *frame_totals) {
  if (!ctx || !batch || !image) return fail(ctx, PDP_E_NULL, "pdp_process_dense: null argument");
  if (batch->n_frames < 0 || batch->n_frames > ctx->geo.max_frames_per_batch)
    return fail(ctx, PDP_E_BATCH, "pdp_process_dense: n_frames out of range");
  if (std::isnan(zero_below_adu)) return fail(ctx, PDP_E_VALUE, "pdp_process_dense: zero_below_adu is NaN");
  ctx->launches = 0;
  if (batch->n_frames == 0) return PDP_OK;
  if (!batch->data) return fail(ctx, PDP_E_NULL, "pdp_process_dense: null batch data");
  if (reinterpret_cast<uintptr_t>(batch->data) & 15) return fail(ctx, PDP_E_ALIGN, "pdp_process_dense: batch not 16-byte aligned");
  const int S = ctx->geo.seg_cols, W = ctx->geo.cols, n = batch->n_frames;
  int V = 0;
  for (int v : {8, 4, 2})
    if (S % v == 0 && W % v == 0) {
      V = v;
      break;
    }
  int NV = (S + 32 * V - 1) / (32 * V);
  pdp::DenseFn fn = nullptr;
  for (; NV <= 16 && !fn; ++NV)   // the next instantiated vector count that covers S
    fn = V == 8 ? pdp::dense_lookup_v8(NV, ctx->prm.cm_mode) : (V == 4 ? pdp::dense_lookup_v4(NV, ctx->prm.cm_mode) : pdp::dense_lookup_v2(NV, ctx->prm.cm_mode));
  --NV;
  if (!fn) return fail(ctx, PDP_E_GEOMETRY, "pdp_process_dense: no kernel variant covers seg_cols");
  pdp::DParams k{};
  k.raw = batch->data;
  k.n_frames = n;
  k.ped = ctx->d_ped;
  k.rg = ctx->d_rg;
  k.rg64 = ctx->d_rg64;
  k.P = ctx->geo.panels;
  k.H = ctx->geo.rows;
  k.W = W;
  k.S = S;
  k.nseg = W / S;
  k.n_tasks = k.P * k.H * k.nseg;
  k.T_cm = ctx->prm.cm_adu;
  k.sqrtS = (float)std::sqrt((double)S);
  {
    const double need = std::max(1024.0, 4.0 * (double)(V * NV) * (double)ctx->prm.cm_adu + 1.0);
    double big = 1024.0;
    while (big < need) big *= 2.0;
    k.big = (float)big;
  }
  k.zero_below = zero_below_adu;
  k.dzero_below = (double)zero_below_adu;
  k.inv_Eph = (float)(1.0 / (double)ctx->prm.photon_adu);
  k.dE_ph = (double)ctx->prm.photon_adu;
  k.cm_mode = ctx->prm.cm_mode;
  k.cm_min_count = ctx->prm.cm_min_count > 0 ? ctx->prm.cm_min_count : (int)std::ceil(std::sqrt((double)S));
  k.image = image;
  k.dinv_E_ph = 1.0 / (double)ctx->prm.photon_adu;
  const int nwarps = pdp::kDenseThreads / 32;
  // A warp owns a row segment; with few segments (small detectors) the frames of a segment are split into slices so
  // that every warp slot of the GPU gets about three tasks (slices of at least 64 frames); the slices accumulate into
  // their own images, merged by pdp_dense_merge_kernel.
  {
    const long long slots = (long long)ctx->num_sms * nwarps;
    long long ns = (3 * slots + k.n_tasks - 1) / k.n_tasks;
    ns = std::max(1LL, std::min<long long>(std::min<long long>(ns, 16), n / 64));
    k.n_slices = (int)ns;
    k.slice_frames = (n + k.n_slices - 1) / k.n_slices;
  }
  const long long tasks_all = (long long)k.n_tasks * k.n_slices;
  const int grid = (int)std::max<long long>(1, std::min<long long>(ctx->num_sms, (tasks_all + nwarps - 1) / nwarps));
  const size_t tot_bytes = frame_totals ? (((size_t)n * 4 + 127) & ~(size_t)127) : 0;
  const size_t smem = tot_bytes + (size_t)nwarps * pdp::kDenseRing * 32 * (size_t)(V * NV) * 2;
  if (smem > ctx->smem_limit) return fail(ctx, PDP_E_BATCH, "pdp_process_dense: too many frames per call for the per-frame totals");
  const size_t img_words = k.n_slices > 1 ? (size_t)k.n_slices * ctx->npix : 0;
  {
    const size_t need = (frame_totals ? (size_t)grid * n : 0) + img_words;
    if (ctx->dense_ws_words < need) {
      cudaFree(ctx->d_dense_ws);
      ctx->d_dense_ws = nullptr;
      ctx->dense_ws_words = 0;
      PDP_CUDA(ctx, cudaMalloc(&ctx->d_dense_ws, need * sizeof(uint32_t)));
      ctx->dense_ws_words = need;
    }
  }
  if (img_words) k.partial_image = ctx->d_dense_ws;
  if (frame_totals) {
    k.partial_totals = ctx->d_dense_ws + img_words;
    k.frame_totals = frame_totals;
    k.n_partials = grid;
  }
  PDP_CUDA(ctx, cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ctx->smem_limit));
  cudaStream_t st = (cudaStream_t)stream;
  fn<<<grid, pdp::kDenseThreads, smem, st>>>(k);
  PDP_CUDA(ctx, cudaGetLastError());
  ctx->launches = 1;
  if (k.n_slices > 1) {
    pdp::pdp_dense_merge_kernel<<<(int)std::min<size_t>((ctx->npix + 255) / 256, (size_t)ctx->num_sms * 8), 256, 0, st>>>(k);
    PDP_CUDA(ctx, cudaGetLastError());
    ctx->launches += 1;
  }
  if (frame_totals) {
    pdp::pdp_dense_totals_kernel<<<(n + 255) / 256, 256, 0, st>>>(k);
    PDP_CUDA(ctx, cudaGetLastError());
    ctx->launches += 1;
  }
  std::snprintf(ctx->last_kernel_buf, sizeof(ctx->last_kernel_buf), "pdp_dense_kernel<%d,%d,%d>", V, NV, ctx->prm.cm_mode);
  ctx->last_kernel = ctx->last_kernel_buf;
  return PDP_OK;
}

int pdp_histograms(pdp_ctx *ctx, const pdp_output *lists, int32_t n_frames, const pdp_hist_spec *energy,
                   uint32_t *hist_energy, const pdp_hist_spec *dxy, uint32_t *hist_dx, uint32_t *hist_dy, void *stream) {
  if (!ctx || !lists || !lists->hit_count || !lists->hit_charge || !lists->hit_dx || !lists->hit_dy)
    return fail(ctx, PDP_E_NULL, "pdp_histograms: null argument");
  if ((energy && !hist_energy) || (dxy && (!hist_dx || !hist_dy))) return fail(ctx, PDP_E_NULL, "pdp_histograms: null histogram");
  if (n_frames < 0) return fail(ctx, PDP_E_BATCH, "pdp_histograms: n_frames < 0");
  for (const pdp_hist_spec *s : {energy, dxy})
    if (s && (!std::isfinite(s->lo) || !std::isfinite(s->width) || !(s->width > 0.f) || s->nbins < 1 || s->nbins > 16384))
      return fail(ctx, PDP_E_VALUE, "pdp_histograms: invalid histogram specification");
  ctx->launches = 0;
  if (n_frames == 0 || (!energy && !dxy)) return PDP_OK;
  pdp::HistParams q{};
  q.n_frames = n_frames;
  q.cap = lists->hit_capacity;
  q.hit_count = lists->hit_count;
  q.hit_charge = lists->hit_charge;
  q.hit_dx = lists->hit_dx;
  q.hit_dy = lists->hit_dy;
  if (energy) q.e_lo = energy->lo, q.e_w = energy->width, q.e_bins = energy->nbins;
  if (dxy) q.d_lo = dxy->lo, q.d_w = dxy->width, q.d_bins = dxy->nbins;
  const int total = q.e_bins + 2 * q.d_bins;
  const int grid = std::min(ctx->num_sms, n_frames);
  const size_t need = (size_t)grid * total;
  if (ctx->hist_ws_words < need) {
    cudaFree(ctx->d_hist_ws);
    ctx->d_hist_ws = nullptr;
    ctx->hist_ws_words = 0;
    PDP_CUDA(ctx, cudaMalloc(&ctx->d_hist_ws, need * sizeof(uint32_t)));
    ctx->hist_ws_words = need;
  }
  q.partial = ctx->d_hist_ws;
  q.n_partials = grid;
  q.hist_e = hist_energy;
  q.hist_dx = hist_dx;
  q.hist_dy = hist_dy;
  cudaStream_t st = (cudaStream_t)stream;
  pdp::pdp_hist_kernel<<<grid, pdp::kPostThreads, (size_t)total * 4, st>>>(q);
  PDP_CUDA(ctx, cudaGetLastError());
  pdp::pdp_hist_merge_kernel<<<(total + 255) / 256, 256, 0, st>>>(q);
  PDP_CUDA(ctx, cudaGetLastError());
  ctx->launches = 2;
  ctx->last_kernel = "pdp_hist_kernel";
  return PDP_OK;
}

}  // extern "C"
